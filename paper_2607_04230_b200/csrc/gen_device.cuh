// gen_device.cuh — the arithmetic of H3 strand generation as device functions (PAPER.md:50, 62-64,
// Code 1 PAPER.md:353-443), shared by k_generate (vertices to HBM) and k_raster_fused (vertices stay in registers,
// the paper's own arrangement PAPER.md:58-64). One source, so both produce the same bits for a vertex.
#pragma once
#include "hair_internal.cuh"

namespace gen {
struct F3 {
  float x, y, z;
};
__device__ __forceinline__ F3 f3(float x, float y, float z) { return {x, y, z}; }
__device__ __forceinline__ F3 operator+(F3 a, F3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ F3 operator-(F3 a, F3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ F3 operator*(float s, F3 a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ float dot(F3 a, F3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ F3 cross(F3 a, F3 b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
__device__ __forceinline__ F3 normalize(F3 a) {
  float d = dot(a, a);
  return d > 0.f ? rsqrtf(d) * a : f3(0.f, 0.f, 0.f);
}
__device__ __forceinline__ F3 shfl3(F3 v, int src) {
  return {__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src), __shfl_sync(0xffffffffu, v.z, src)};
}
__device__ __forceinline__ F3 shfl3_up(F3 v) {
  return {__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1), __shfl_up_sync(0xffffffffu, v.z, 1)};
}
__device__ __forceinline__ F3 shfl3_down(F3 v) {
  return {__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1),
          __shfl_down_sync(0xffffffffu, v.z, 1)};
}


// Row of the per-bundle table (HAIR_ROW = 44 floats):
//  [0..3]  E0.xyz, AO0     [4..7]  E1.xyz, AO1     [8..11] E2.xyz, AO2
//  [12..15] dE0.xyz, w     [16..19] dE1.xyz, curl amplitude     [20..23] dE2.xyz, frizz amplitude
//  [24..27] c.xyz, clump factor   [28..31] Tc.xyz, frizz smoothstep   [32..35] Ef.xyz, frizz cell (int bits)
//  [36..39] cos/sin twist angle, cos/sin of the curl turn angle 2*pi*turns*w

// stages 1 + 2 for one bundle (whole warp): lanes = cage layers (edge polylines, Catmull-Rom tangents by shuffles),
// then lanes = control points (the three edge splines, their derivatives, centre curve, frame edge, styling scalars)
// into tab[C][HAIR_ROW] (shared memory of this warp). Ends with __syncwarp().
__device__ __forceinline__ void build_table(const GroomDev& g, uint32_t t, uint32_t C, float* __restrict__ tab,
                                            uint32_t lane) {
  const uint32_t Lv = g.Lv, ops = g.op_mask;
  // ---- stage 1: lanes = layers. Edge polylines X^k_i, AO, Catmull-Rom tangents via shuffles.
  F3 X[3], m[3];
  float ao[3];
  {
    const uint32_t li = min(lane, Lv - 1);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      uint32_t v = __ldg(&g.idx[t * 3 + k]);
      const float* p = g.pos + ((size_t)li * g.V + v) * 3;
      X[k] = f3(__ldg(p), __ldg(p + 1), __ldg(p + 2));
      ao[k] = g.ao ? __ldg(&g.ao[(size_t)li * g.V + v]) : 1.0f;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      F3 prev = shfl3_up(X[k]), next = shfl3_down(X[k]);
      if (lane == 0) m[k] = next - X[k];  // R4: one-sided at the ends
      else if (lane >= Lv - 1) m[k] = X[k] - prev;
      else m[k] = 0.5f * (next - prev);
    }
  }
  __syncwarp();
  // ---- stage 2: lanes = control points. Build the per-bundle table.
  const uint32_t den = C - 1;
  const float inv_den = 1.0f / (float)den;
  for (uint32_t j0 = 0; j0 < C; j0 += 32) {
    const uint32_t j = min(j0 + lane, C - 1);
    const uint32_t num = j * (Lv - 1);
    const uint32_t i = min(num / den, Lv - 2);  // R5
    const float tt = (float)(num - i * den) * inv_den;
    const float w = (float)j * inv_den;
    const float t2 = tt * tt, t3 = t2 * tt;
    const float h00 = 2.f * t3 - 3.f * t2 + 1.f, h10 = t3 - 2.f * t2 + tt, h01 = -2.f * t3 + 3.f * t2, h11 = t3 - t2;
    const float d00 = 6.f * t2 - 6.f * tt, d10 = 3.f * t2 - 4.f * tt + 1.f, d01 = -d00, d11 = 3.f * t2 - 2.f * tt;
    F3 E[3], dE[3];
    float aoj[3];
    F3 e0a, e0b, e1a, e1b;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      F3 Pa = shfl3(X[k], i), Pb = shfl3(X[k], i + 1), ma = shfl3(m[k], i), mb = shfl3(m[k], i + 1);
      float aa = __shfl_sync(0xffffffffu, ao[k], i), ab = __shfl_sync(0xffffffffu, ao[k], i + 1);
      E[k] = h00 * Pa + h10 * ma + h01 * Pb + h11 * mb;  // cubic Hermite
      dE[k] = d00 * Pa + d10 * ma + d01 * Pb + d11 * mb;
      aoj[k] = (1.f - tt) * aa + tt * ab;  // R25
      if (k == 0) {
        e0a = Pa;
        e1a = Pb;
      }
      if (k == 1) {
        e0b = Pa;
        e1b = Pb;
      }
    }
    if (j0 + lane < C) {
      float* row = tab + (size_t)j * HAIR_ROW;
      const F3 c = (1.0f / 3.0f) * (E[0] + E[1] + E[2]);
      const F3 Tc = normalize(dE[0] + dE[1] + dE[2]);
      const F3 Ef = (1.f - tt) * (e0b - e0a) + tt * (e1b - e1a);
      float clump = 0.f, ct = 1.f, st = 0.f, cc = 1.f, sc_ = 0.f, camp = 0.f, famp = 0.f, fs = 0.f;
      uint32_t cell = 0;
      if (ops & HAIR_OP_CLUMP) {
        float we = 1.f;
        for (uint32_t k = 0; k < g.clump_exp; ++k) we *= w;
        clump = g.clump_strength * we;
      }
      if (ops & HAIR_OP_TWIST) sincospif(2.f * g.twist_turns * w, &st, &ct);
      if (ops & HAIR_OP_CURL) {
        sincospif(2.f * g.curl_turns * w, &sc_, &cc);
        camp = g.curl_radius * (g.curl_ramp_w0 > 0.f ? fminf(w / g.curl_ramp_w0, 1.f) : 1.f);
      }
      if (ops & HAIR_OP_FRIZZ) {
        const uint32_t cells = max(g.frizz_cells, 1u);
        // x = w*cells evaluated as (j*cells)/den in integers: the cell index is exact
        const uint32_t xn = j * cells;
        cell = min(xn / den, cells - 1);
        const float fr = (float)(xn - cell * den) * inv_den;
        fs = fr * fr * (3.f - 2.f * fr);
        famp = g.frizz_sigma * (g.frizz_ramp_w0 > 0.f ? fminf(w / g.frizz_ramp_w0, 1.f) : 1.f);
      }
      float4* r4 = reinterpret_cast<float4*>(row);
      r4[0] = make_float4(E[0].x, E[0].y, E[0].z, aoj[0]);
      r4[1] = make_float4(E[1].x, E[1].y, E[1].z, aoj[1]);
      r4[2] = make_float4(E[2].x, E[2].y, E[2].z, aoj[2]);
      r4[3] = make_float4(dE[0].x, dE[0].y, dE[0].z, w);
      r4[4] = make_float4(dE[1].x, dE[1].y, dE[1].z, camp);
      r4[5] = make_float4(dE[2].x, dE[2].y, dE[2].z, famp);
      r4[6] = make_float4(c.x, c.y, c.z, clump);
      r4[7] = make_float4(Tc.x, Tc.y, Tc.z, fs);
      r4[8] = make_float4(Ef.x, Ef.y, Ef.z, __uint_as_float(cell));
      r4[9] = make_float4(ct, st, cc, sc_);
    }
  }
  __syncwarp();
}

// per strand, once: root barycentrics (R6) as (b1, b2), cos / sin of the curl phase; `base` = the strand's hash base
struct Strand {
  float b1, b2, cphi, sphi;
  uint32_t base, a1, a2;  // a1, a2: the folded 24-bit root coordinates themselves (b = a 2^-24)
};
__device__ __forceinline__ Strand strand_setup(const GroomDev& g, uint32_t id_local) {
  Strand s;
  s.base = pcg(g.seed_h + id_local);
  uint32_t a1 = pcg(s.base + 1u) >> 8, a2 = pcg(s.base + 2u) >> 8;
  if (a1 + a2 > 16777216u) {  // R6: fold on the integers
    a1 = 16777216u - a1;
    a2 = 16777216u - a2;
  }
  s.sphi = 0.f, s.cphi = 1.f;
  if (g.op_mask & HAIR_OP_CURL) sincospif(2.f * ((float)(pcg(s.base + 3u) >> 8) * (1.0f / 16777216.0f)), &s.sphi, &s.cphi);
  s.a1 = a1, s.a2 = a2;
  s.b1 = (float)a1 * (1.0f / 16777216.0f);
  s.b2 = (float)a2 * (1.0f / 16777216.0f);
  return s;
}

// b0 r0 + b1 r1 + b2 r2 on two components at once
__device__ __forceinline__ float2 blend2(float b0, float b1, float b2, float2 r0, float2 r1, float2 r2) {
  return __ffma2_rn(make_float2(b2, b2), r2, __ffma2_rn(make_float2(b1, b1), r1, __fmul2_rn(make_float2(b0, b0), r0)));
}

// stage 3 for one vertex: control point j of a strand, from the bundle table row and the strand's record; M = the
// instance transform (R-inst, applied last) or nullptr. Returns (x, y, z, ao).
__device__ __forceinline__ float4 vertex(const float* __restrict__ tab, uint32_t j, float b1, float b2, float cphi,
                                         float sphi, uint32_t base, uint32_t ops, const float* M) {
  const float4 sr = make_float4(b1, b2, cphi, sphi);
  const float b0 = (1.0f - b1) - b2;
  const float4* r4 = reinterpret_cast<const float4*>(tab + (size_t)j * HAIR_ROW);
  const float4 E0 = r4[0], E1 = r4[1], E2 = r4[2];
  // barycentric blend of the three table rows in packed fp32 (sm_100 FFMA2: the (x, y) and (z, ao) halves of a row
  // are register pairs as loaded; one issue slot for two FMAs)
  const float2 pxy = blend2(b0, b1, b2, make_float2(E0.x, E0.y), make_float2(E1.x, E1.y), make_float2(E2.x, E2.y));
  const float2 pza = blend2(b0, b1, b2, make_float2(E0.z, E0.w), make_float2(E1.z, E1.w), make_float2(E2.z, E2.w));
  F3 p = f3(pxy.x, pxy.y, pza.x);
  float aov = fminf(fmaxf(pza.y, 0.f), 1.f);
  if (ops) {
    if (ops & (HAIR_OP_CLUMP | HAIR_OP_TWIST)) {
      const float4 cc4 = r4[6];
      const F3 c = f3(cc4.x, cc4.y, cc4.z);
      if (ops & HAIR_OP_CLUMP) p = p + cc4.w * (c - p);
      if (ops & HAIR_OP_TWIST) {
        const float4 tc4 = r4[7], cs4 = r4[9];
        const F3 Tc = f3(tc4.x, tc4.y, tc4.z);
        const F3 d = p - c;  // Rodrigues rotation about Tc
        const F3 dr = cs4.x * d + cs4.y * cross(Tc, d) + (dot(Tc, d) * (1.f - cs4.x)) * Tc;
        p = c + dr;
      }
    }
    if (ops & (HAIR_OP_CURL | HAIR_OP_FRIZZ)) {
      // frame from the UNSTYLED base spline: T = normalised derivative, N from the cage edge
      const float4 D0 = r4[3], D1 = r4[4], D2 = r4[5];
      const float2 dxy = blend2(b0, b1, b2, make_float2(D0.x, D0.y), make_float2(D1.x, D1.y), make_float2(D2.x, D2.y));
      const float2 dzw = blend2(b0, b1, b2, make_float2(D0.z, D0.w), make_float2(D1.z, D1.w), make_float2(D2.z, D2.w));
      const F3 T = normalize(f3(dxy.x, dxy.y, dzw.x));  // (dzw.y blends the rows' styling scalars: unused)
      const float4 ef4 = r4[8];
      const F3 Ef = f3(ef4.x, ef4.y, ef4.z);
      F3 Nn = Ef - dot(Ef, T) * T;
      float nn = dot(Nn, Nn);
      if (nn < 1e-20f) {
        const float ax = fabsf(T.x), ay = fabsf(T.y), az = fabsf(T.z);
        const F3 a = (ax <= ay && ax <= az) ? f3(1, 0, 0) : (ay <= az ? f3(0, 1, 0) : f3(0, 0, 1));
        Nn = a - dot(a, T) * T;
        nn = dot(Nn, Nn);
      }
      const F3 N = (nn > 0.f ? rsqrtf(nn) : 0.f) * Nn;
      const F3 B = cross(T, N);
      if (ops & HAIR_OP_CURL) {
        const float4 cs4 = r4[9];
        const float ct = sr.z * cs4.z - sr.w * cs4.w, st = sr.w * cs4.z + sr.z * cs4.w;  // angle addition
        p = p + D1.w * (ct * N + st * B);
      }
      if (ops & HAIR_OP_FRIZZ) {
        const uint32_t cell = __float_as_uint(ef4.w);
        const float s = r4[7].w;
        float n[2];
#pragma unroll
        for (uint32_t ch = 0; ch < 2; ++ch) {
          const uint32_t h0 = pcg(base + 16u + 2u * cell + ch), h1 = pcg(base + 16u + 2u * (cell + 1u) + ch);
          const int s0 = (int)(__vsadu4(h0, 0u)) - 510, s1 = (int)(__vsadu4(h1, 0u)) - 510;  // byte sums
          const float g0 = (float)s0 * 0.0067658652f, g1 = (float)s1 * 0.0067658652f;       // 1/sqrt(21845)
          n[ch] = (1.f - s) * g0 + s * g1;
        }
        p = p + D2.w * (n[0] * N + n[1] * B);
      }
    }
  }
  if (M)  // R-inst: instance transform applied last
    p = f3(M[0] * p.x + M[1] * p.y + M[2] * p.z + M[3], M[4] * p.x + M[5] * p.y + M[6] * p.z + M[7],
           M[8] * p.x + M[9] * p.y + M[10] * p.z + M[11]);
  return make_float4(p.x, p.y, p.z, aov);
}

}  // namespace gen
