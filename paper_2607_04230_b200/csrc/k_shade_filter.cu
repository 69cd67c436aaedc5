// k_shade_filter.cu — H6 deferred shading and H7 reconstruction filter.
//
// H6: one thread per pixel reads the 16-byte word pair with one 128-bit
// load; pixels with a centre hit locate the winning segment (strand id -> vertex run), interpolate
// position / AO / calcTangent at the stored parameter and evaluate the stand-in
// hair shading model (R23). Only visible hits are shaded — the point of deferring.
// H7 (Eq. 9-10, Code 2): single pass doing strand connection (promotion of
// conservative-only pixels), the elliptical bilateral filter, fly-away blending and the alpha
// estimate. Sample classification (integer depth compare) and the strip test (fixed-order fp32)
// match the oracle bit for bit; weights and sums are fast fp32.
#include "hair_internal.cuh"

struct F3 {
  float x, y, z;
};
__device__ __forceinline__ F3 f3(float x, float y, float z) { return {x, y, z}; }
__device__ __forceinline__ F3 f3(float4 v) { return {v.x, v.y, v.z}; }
__device__ __forceinline__ F3 operator+(F3 a, F3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ F3 operator-(F3 a, F3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ F3 operator*(float s, F3 a) { return {s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ float dot(F3 a, F3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ F3 normalize(F3 a) {
  float d = dot(a, a);
  return d > 0.f ? rsqrtf(d) * a : f3(0.f, 0.f, 0.f);
}
// PAPER.md:353-359 calcTangent
__device__ __forceinline__ F3 calc_tangent(int idx, int count, F3 prev, F3 curr, F3 next) {
  if (idx == 0) return normalize(next - curr);
  else if (idx == count - 1) return normalize(curr - prev);
  else return normalize(next - prev);
}

// the frame's colour output: fp32 RGBA, or (HAIR_FLAG_RGB16F) IEEE half RGBA in 8 bytes per pixel, rounded to nearest
__device__ __forceinline__ void store_rgba(float4* __restrict__ out, size_t p, float4 v, uint32_t rgb16) {
  if (rgb16) {
    uint2 h;
    asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(h.x) : "f"(v.y), "f"(v.x));
    asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(h.y) : "f"(v.w), "f"(v.z));
    reinterpret_cast<uint2*>(out)[p] = h;
  } else
    out[p] = v;
}

// fast non-decision arithmetic of the shading model (everything here is far inside the 2e-3 RGB tolerance)
__device__ __forceinline__ float fast_sqrt(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float fast_rcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// asin on [-1, 1]: pi/2 - sqrt(1 - |x|) P7(|x|), |error| <= 2e-8 (Abramowitz & Stegun 4.4.46)
__device__ __forceinline__ float fast_asin(float x) {
  const float a = fabsf(x);
  float p = -0.0012624911f;
  p = fmaf(p, a, 0.0066700901f);
  p = fmaf(p, a, -0.0170881256f);
  p = fmaf(p, a, 0.0308918810f);
  p = fmaf(p, a, -0.0501743046f);
  p = fmaf(p, a, 0.0889789874f);
  p = fmaf(p, a, -0.2145988016f);
  p = fmaf(p, a, 1.5707963050f);
  const float r = fmaf(-fast_sqrt(1.f - a), p, 1.57079632679f);
  return copysignf(r, x);
}

// Volumetric shadow (DESIGN.md R-dom): transmittance towards one light from its deep opacity map at
// world point pos, the depth behind each texel's nearest hair scaled by beta first (Eq. 7, the depth-comparison fix
// of PAPER.md:138-152). Fragments in front = the cumulative layer count, piecewise linear through the layer ends;
// bilinear over the four texels around the point. The projection and the depth quantisation are R-proj / R8 (the
// same integers as the oracle's); the blend is ordinary fp32.
__device__ __forceinline__ float dom_texel_omega(uint4 c, const uint32_t* D, float d) {
  const float D0 = (float)D[0], D1 = (float)D[1], D2 = (float)D[2], D3 = (float)D[3];
  const float c0 = (float)c.x, c1 = (float)c.y, c2 = (float)c.z, c3 = (float)c.w;
  if (d < D0) return c0 * d / D0;
  if (d < D1) return c0 + c1 * (d - D0) / (D1 - D0);
  if (d < D2) return (c0 + c1) + c2 * (d - D1) / (D2 - D1);
  if (d < D3) return (c0 + c1 + c2) + c3 * (d - D2) / (D3 - D2);
  return c0 + c1 + c2 + c3;
}
__device__ __forceinline__ float dom_transmittance(const DomLight& L, F3 pos, float beta) {
  const Proj q = project_exact(L.cam, pos.x, pos.y, pos.z);
  if (!q.valid) return 1.f;
  const uint32_t dq = quant_depth(fminf(fmaxf(q.zn, 0.f), 1.f));
  const float fx = q.sx - 0.5f, fy = q.sy - 0.5f;
  const float x0 = floorf(fx), y0 = floorf(fy);
  const float wx = fx - x0, wy = fy - y0;
  const int W = (int)L.cam.W, H = (int)L.cam.H;
  float omega = 0.f;
#pragma unroll
  for (int dy = 0; dy < 2; ++dy)
#pragma unroll
    for (int dx = 0; dx < 2; ++dx) {
      const int xi = (int)x0 + dx, yi = (int)y0 + dy;
      if (xi < 0 || yi < 0 || xi >= W || yi >= H) continue;
      const size_t t = (size_t)yi * W + xi;
      const uint32_t z0 = __ldg(&L.z0[t]);
      if (z0 == 0xFFFFFFFFu || dq <= z0) continue;
      const float w = (dx ? wx : 1.f - wx) * (dy ? wy : 1.f - wy);
      omega += w * dom_texel_omega(__ldg(&L.cnt[t]), L.D, beta * (float)(dq - z0));
    }
  return __expf(-L.alpha_s * omega);
}
// beta of Eq. 7 for groom g of the frame being shaded, from the sums k_scan took on the device (R-beta)
__device__ __forceinline__ float groom_beta(const unsigned long long* __restrict__ counters, uint32_t g) {
  const unsigned long long num = __ldg(&counters[CNT_BETA_NUM + g]), den = __ldg(&counters[CNT_BETA_DEN + g]);
  return den ? (float)num / (float)den : 1.f;
}

// the stand-in shading model (R23) at one point: position, unit tangent, strand parameter w, AO
__device__ __forceinline__ F3 shade_model(const GroomDev& g, const CamDev& cam, const ShadeParams& sp, F3 pos, F3 T,
                                          float w, float ao, const DomSet* __restrict__ dom, float beta_lod) {
  const F3 alb = (1.f - w) * f3(g.albedo_root[0], g.albedo_root[1], g.albedo_root[2]) +
                 w * f3(g.albedo_tip[0], g.albedo_tip[1], g.albedo_tip[2]);
  const F3 V = normalize(f3(cam.eye[0], cam.eye[1], cam.eye[2]) - pos);
  F3 rgb = f3(ao * sp.ambient[0] * alb.x, ao * sp.ambient[1] * alb.y, ao * sp.ambient[2] * alb.z);
  const float beta = g.roughness, tilt = g.tilt;
  const float inv2b2 = fast_rcp(2.f * beta * beta);
  const float sin_o = fminf(fmaxf(dot(T, V), -1.f), 1.f);
  const float asin_o = fast_asin(sin_o);
  for (uint32_t li = 0; li < sp.n_lights; ++li) {
    const F3 Lv = f3(sp.light_pos[li][0], sp.light_pos[li][1], sp.light_pos[li][2]) - pos;
    const float d2 = dot(Lv, Lv);
    const float inv_d2 = fast_rcp(d2);
    const F3 om = rsqrtf(d2) * Lv;
    const float sin_i = fminf(fmaxf(dot(T, om), -1.f), 1.f);
    const float cos_i = fast_sqrt(fmaxf(0.f, 1.f - sin_i * sin_i));
    const float th = 0.5f * (fast_asin(sin_i) + asin_o);
    const float a = th + tilt, b = th - 1.5f * tilt;
    const float MR = __expf(-a * a * inv2b2), MT = __expf(-b * b * 0.25f * inv2b2);
    float s = cos_i * inv_d2;
    if (dom && dom->l[li].on) s *= dom_transmittance(dom->l[li], pos, beta_lod);
    rgb.x += sp.light_rgb[li][0] * s * (sp.k_d * alb.x + sp.k_R * MR + sp.k_TRT * MT * alb.x);
    rgb.y += sp.light_rgb[li][1] * s * (sp.k_d * alb.y + sp.k_R * MR + sp.k_TRT * MT * alb.y);
    rgb.z += sp.light_rgb[li][2] * s * (sp.k_d * alb.z + sp.k_R * MR + sp.k_TRT * MT * alb.z);
  }
  return rgb;
}

// O6 for one word: linear RGB of the hit it names
__device__ __forceinline__ F3 shade_word(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec,
                                         const float4* __restrict__ vertices, const CamDev& cam, const ShadeParams& sp,
                                         unsigned long long G, const DomSet* __restrict__ dom,
                                         const unsigned long long* __restrict__ counters) {
  const Loc l = locate_strand(srec, w_sid(G));
  const GroomDev& g = sc->g[l.groom];
  const int j = (int)w_j(G), C = (int)l.C;
  const float t = (float)w_t9(G) * (1.0f / 511.0f);
  const float4* vs = vertices + l.voff;
  const float4 v1 = __ldg(&vs[j]), v2 = __ldg(&vs[j + 1]);
  const float4 v0 = __ldg(&vs[max(j - 1, 0)]), v3 = __ldg(&vs[min(j + 2, C - 1)]);
  const F3 pos = (1.f - t) * f3(v1) + t * f3(v2);
  const float ao = (1.f - t) * v1.w + t * v2.w;
  const F3 Tj = calc_tangent(j, C, f3(v0), f3(v1), f3(v2));
  const F3 Tj1 = calc_tangent(j + 1, C, f3(v1), f3(v2), f3(v3));
  const F3 T = normalize((1.f - t) * Tj + t * Tj1);
  const float w = ((float)j + t) / (float)(C - 1);
  return shade_model(g, cam, sp, pos, T, w, ao, dom, dom ? groom_beta(counters, l.groom) : 1.f);
}

// R-payload: O6 from the paper's payload alone, no vertex read. Position = the point of the
// ray through the pixel centre at the word's depth ("reconstruct it from the depth value")
__device__ __forceinline__ F3 shade_payload(const SceneDev* __restrict__ sc, const CamDev& cam, const ShadeParams& sp,
                                            int x, int y, unsigned long long G, const DomSet* __restrict__ dom,
                                            const unsigned long long* __restrict__ counters) {
  const X3 t = oct_decode_x(pw_ox(G), pw_oy(G));
  const float w = (float)((uint32_t)(G >> 6) & 63u) * (1.0f / 63.0f), ao = (float)((uint32_t)G & 63u) * (1.0f / 63.0f);
  const float zn = (float)w_dq(G) / 16777215.0f;
  const float zv = cam.B / (cam.A - zn);
  const float cx = (((float)x + 0.5f) - cam.half_w) / cam.fpx, cy = (cam.half_h - ((float)y + 0.5f)) / cam.fpx;
  const F3 pos = f3(cam.eye[0] + zv * (cx * cam.r[0] + cy * cam.u[0] + cam.f[0]),
                    cam.eye[1] + zv * (cx * cam.r[1] + cy * cam.u[1] + cam.f[1]),
                    cam.eye[2] + zv * (cx * cam.r[2] + cy * cam.u[2] + cam.f[2]));
  return shade_model(sc->g[sp.pp_groom], cam, sp, pos, f3(t.x, t.y, t.z), w, ao, dom,
                     dom ? groom_beta(counters, sp.pp_groom) : 1.f);
}

template <bool SH>  // SH: deep-opacity shadows on (a kernel of its own: the plain one keeps its 31 registers)
__global__ void __launch_bounds__(256)
k_shade(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec, const float4* __restrict__ vertices,
        CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf, float4* __restrict__ colour,
        const DomSet* __restrict__ dom, const unsigned long long* __restrict__ counters) {
  const size_t n_px = (size_t)cam.W * cam.H;
  const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_px) return;
  const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + p);
  const unsigned long long G = ((unsigned long long)raw.y << 32) | raw.x;
  if (w_none(G)) return;  // colour is only ever read where a centre hit exists
  const F3 rgb = shade_word(sc, srec, vertices, cam, sp, G, SH ? dom : nullptr, counters);
  colour[p] = make_float4(rgb.x, rgb.y, rgb.z, 1.0f);
}

template <bool SH>
__global__ void __launch_bounds__(256)
k_shade_payload(const SceneDev* __restrict__ sc, CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf,
                float4* __restrict__ colour, const DomSet* __restrict__ dom,
                const unsigned long long* __restrict__ counters) {
  const uint32_t x = blockIdx.x * 64u + (threadIdx.x & 63u), y = blockIdx.y * 4u + (threadIdx.x >> 6);
  if (x >= cam.W || y >= cam.H) return;
  const size_t p = (size_t)y * cam.W + x;
  const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + p);
  const unsigned long long G = ((unsigned long long)raw.y << 32) | raw.x;
  if (w_none(G)) return;
  const F3 rgb = shade_payload(sc, cam, sp, (int)x, (int)y, G, SH ? dom : nullptr, counters);
  colour[p] = make_float4(rgb.x, rgb.y, rgb.z, 1.0f);
}

// MSAA-k reference resolve (DESIGN.md R-msaa): mean over the k samples of (shaded hit | background)
template <bool SH>
__global__ void __launch_bounds__(256)
k_resolve_msaa(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec, const float4* __restrict__ vertices,
               CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ samples, uint32_t ms_k,
               const float4* __restrict__ scene_rgb, float4* __restrict__ out, const DomSet* __restrict__ dom,
               const unsigned long long* __restrict__ counters) {
  const size_t n_px = (size_t)cam.W * cam.H;
  const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_px) return;
  F3 acc = f3(0.f, 0.f, 0.f);
  uint32_t n_hit = 0;
  for (uint32_t s = 0; s < ms_k; ++s) {
    const unsigned long long w = __ldg(&samples[(size_t)s * n_px + p]);
    if (w_none(w)) continue;
    acc = acc + shade_word(sc, srec, vertices, cam, sp, w, SH ? dom : nullptr, counters);
    ++n_hit;
  }
  F3 bg = f3(sp.background[0], sp.background[1], sp.background[2]);
  if (scene_rgb) bg = f3(__ldg(&scene_rgb[p]));
  const float inv_k = 1.0f / (float)ms_k, alpha = (float)n_hit * inv_k;
  store_rgba(out, p, make_float4(acc.x * inv_k + (1.f - alpha) * bg.x, acc.y * inv_k + (1.f - alpha) * bg.y,
                                 acc.z * inv_k + (1.f - alpha) * bg.z, alpha), sp.rgb16);
}

void launch_resolve_msaa(const SceneDev* d_scene, const uint2* srec, const float4* vertices, CamDev cam,
                         ShadeParams sp, const unsigned long long* samples, uint32_t ms_k, const float4* scene_rgb,
                         float4* out, const DomSet* dom, const unsigned long long* counters, cudaStream_t st) {
  const size_t n = (size_t)cam.W * cam.H;
  if (sp.shadows && dom)
    k_resolve_msaa<true><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_scene, srec, vertices, cam, sp, samples, ms_k, scene_rgb, out, dom, counters);
  else
    k_resolve_msaa<false><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_scene, srec, vertices, cam, sp, samples, ms_k, scene_rgb, out, nullptr, counters);
}

// R22: unit screen direction of the segment a word names; fixed-order fp32 (decides strip membership)
__device__ __forceinline__ float2 screen_tangent(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec,
                                                 const float4* __restrict__ vertices, const CamDev& cam,
                                                 unsigned long long word) {
  const Loc l = locate_strand(srec, w_sid(word));
  const float4* vs = vertices + l.voff + w_j(word);
  const float4 va = __ldg(vs), vb = __ldg(vs + 1);
  const Proj a = project_exact(cam, va.x, va.y, va.z), b = project_exact(cam, vb.x, vb.y, vb.z);
  const float dx = xsub(b.sx, a.sx), dy = xsub(b.sy, a.sy);
  const float dd = xadd(xmul(dx, dx), xmul(dy, dy));
  if (!(dd >= 1e-12f)) return make_float2(1.f, 0.f);
  const float len = xsqrt(dd);
  return make_float2(xdiv(dx, len), xdiv(dy, len));
}

// R22 for the paper's payload: screen direction of the decoded tangent at the pixel centre. View-space tangent
// (tx, ty, tz), pixel ray (cx, cy, 1): d(sx, sy)/ds is parallel to (tx - cx tz, cy tz - ty) whatever the depth
__device__ __forceinline__ float2 screen_tangent_payload(const CamDev& cam, int x, int y, unsigned long long word) {
  const X3 t = oct_decode_x(pw_ox(word), pw_oy(word));
  const float tx = xdot3(t.x, t.y, t.z, cam.r), ty = xdot3(t.x, t.y, t.z, cam.u), tz = xdot3(t.x, t.y, t.z, cam.f);
  const float cx = xdiv(xsub(xadd((float)x, 0.5f), cam.half_w), cam.fpx);
  const float cy = xdiv(xsub(cam.half_h, xadd((float)y, 0.5f)), cam.fpx);
  const float Sx = xsub(tx, xmul(cx, tz)), Sy = xsub(xmul(cy, tz), ty);
  const float dd = xadd(xmul(Sx, Sx), xmul(Sy, Sy));
  if (!(dd >= 1e-12f)) return make_float2(1.f, 0.f);
  const float len = xsqrt(dd);
  return make_float2(xdiv(Sx, len), xdiv(Sy, len));
}

// ---------------------------------------------------------------------------------------- H7
// Tiled filter. One CTA owns a 32x16 pixel tile:
// (1) the tile + an r-pixel halo goes to shared memory once, in PAIR layout, for the horizontally adjacent pixels
//     a = 2p, b = 2p + 1 of a tile row: s_pa[p] = {x_a, x_b, y_a, y_b}, s_pb[p] = {z_a, z_b, dq_a, dq_b} (colours of
//     centre hits pre-scaled by sqrt(kC), zero elsewhere; dq = 24-bit depth of the centre word, DQ_NONE without a
//     centre hit), s_pk[p] = {k_a, k_b} (k = |scaled colour|^2, read by the accumulations with a colour term only),
//     and s_dq[pixel] = {dq_centre, dq_cons} for the strip loop;
// (2) every hit pixel emits work items: a CENTRE item per centre-hit pixel, compacted in PIXEL ORDER (a warp of a
//     dense tile holds one tile row), and a CONSERVATIVE-SAMPLE item per promoted pixel and per
//     centre-hit pixel with a fly-away strand in front (R21: a second accumulation around the conservative sample,
//     w_color = 1); those are sparse and are dealt by bank class instead;
// (3) item / thread, the warps of the CTA taking item warps from a shared counter. Loop A, Eq. 10,
//     walks the (2r+1)^2 window one PAIR of taps at a time: three loads (two for a conservative-sample item) bring
//     both taps' colour, depth and k, and the arithmetic of the two taps runs in the packed fp32 instructions of
//     sm_100 (FFMA2 / FADD2: fma.rn.f32x2 — two cycles of the FMA pipe like two FFMAs, but ONE issue slot, which is
//     what this loop was short of). Adjacent pixels of a row share their pairs, so the 32 lanes of a row-ordered
//     warp read 16 distinct 16-byte words per LDS.128: two shared-memory cycles instead of four (measured on the
//     B200: the LDS pipe serves 128 distinct bytes per cycle and multicasts for free). The window of a
//     pixel at odd x starts one tap early and the one at even x ends one tap late (pairs are aligned): that tap is
//     masked. Exponent, base 2 and positive so that ex2.approx(-e) is the weight: the quadratic form of Eq. 10 in
//     Horner form over dx, (a dx + B) dx + C with per-row B, C; colour distance |C_P|^2 - 2 C_P.C_Q + |C_Q|^2 with
//     the first term in C and the last read from shared memory. The class test (R20) is the integer compare
//     (d - lo) <= 2 tau (mod 2^32) on the ALU pipe.
//     Loop B, strip hit counts: only lattice points within w_strip of the tangent line can be in the
//     strip, so the loop walks the 2r+1 steps of the tangent's major axis and tests the `strip_nc` (2 for
//     w_strip = 0.5) integer minor offsets that can lie within (w_strip + 0.01) sqrt(2) of the line — a superset;
//     membership itself is Eq. 9 in the oracle's fixed-order fp32 (sqrt_rn(e2) <= w_strip tested as
//     e2 <= strip_e2_max, host-side the largest float whose correctly rounded root is <= w_strip).
// (4) the owning thread combines its pixel's items (R21 blend for a fly-away pixel), composites over the background
//     (R29) and writes out_rgb; pixels without a hit were written at the start.
#define FT_W 32
#ifndef FT_H
#define FT_H 16  // tile rows; FT_W * FT_H / 2 threads per CTA, each owns the pixels (x, y) and (x, y + FT_H / 2)
#endif
#define FT_HH (FT_H / 2)
#define FT_NT (FT_W * FT_HH)
#ifndef FILT_MIN_BLOCKS
#define FILT_MIN_BLOCKS (1024 / FT_NT)  // CTAs per SM the register budget is held to (64 registers per thread)
#endif
#ifndef FILT_DEAL
#define FILT_DEAL 1  // conservative-sample items dealt by bank class (0: packed in pixel order)
#endif
#define DQ_NONE 0x40000000u
#define DQ_OFF 0x80000000u  // as the low end of a depth window: no depth lies within 2 tau above it

__device__ __forceinline__ float fast_ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// packed fp32 (sm_100): both halves in one instruction
__device__ __forceinline__ float2 bc2(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }

// weight of one tap: 2^-e if the tap is of the sample's class (R19 / R20: dd = d - lo <= 2 tau, mod 2^32), else 0; a
// select, never a branch (the lanes of a warp do not diverge)
__device__ __forceinline__ float gated_weight(float e, uint32_t dd, uint32_t tau2) {
  float w;
  asm("{\n\t.reg .pred p;\n\t.reg .f32 n;\n\tsetp.le.u32 p, %2, %3;\n\tneg.f32 n, %1;\n\t"
      "mov.f32 %0, 0f00000000;\n\t@p ex2.approx.ftz.f32 %0, n;\n\t}"
      : "=f"(w)
      : "f"(e), "r"(dd), "r"(tau2));
  return w;
}

// Loop A over the window of one item (one accumulation of Eq. 10, R19-R21). COL: colour term on (centre
// sample) or off (conservative sample: w_color = 1). Positive base-2 exponent
// a dx^2 + b dx dy + c dy^2 + c0 in Horner form over dx. ra / rd: the window's first pair in s_pa / s_pk; u = dx of the
// first tap of a window row (-r, or -r-1 for a pixel at odd x, whose first tap then lies outside the window, as does
// the last tap of a window at even x); (mx, my, mz) = -2 * scaled centre colour; class test (d - lo) <= tau2
template <int R, bool COL>
__device__ __forceinline__ float4 filter_loop_a(const float4* __restrict__ ra, const float2* __restrict__ rd, int HP,
                                                int NP, bool odd, float u, float a, float b, float c, float c0, float mx,
                                                float my, float mz, uint32_t lo, uint32_t tau2) {
  float2 S0 = make_float2(0.f, 0.f), S1 = S0, S2 = S0, Ws = S0;
  float fdy = (float)(-R);
#pragma unroll 1
  for (int dyi = 0; dyi <= 2 * R; ++dyi, ra += HP, rd += HP, fdy += 1.0f) {
    const float B = b * fdy, C = fmaf(c * fdy, fdy, c0);
    float2 dx = make_float2(u, u + 1.0f);
#pragma unroll
    for (int p = 0; p <= R; ++p) {
      const float4 A4 = ra[p], B4 = ra[NP + p];
      const float2 X = make_float2(A4.x, A4.y), Y = make_float2(A4.z, A4.w), Z = make_float2(B4.x, B4.y);
      const uint2 D = make_uint2(__float_as_uint(B4.z), __float_as_uint(B4.w));
      if (p) dx = add2(dx, bc2(2.0f));
      uint32_t Dx = D.x, Dy = D.y;
      if (p == 0) Dx = odd ? DQ_NONE : Dx;  // tap -r-1 of a window at odd x
      if (p == R) Dy = odd ? Dy : DQ_NONE;  // tap r+1 of a window at even x
      float2 e = fma2(fma2(bc2(a), dx, bc2(B)), dx, bc2(C));  // Eq. 10 spatial part (+ |C_P|^2 in c0)
      if (COL) {                                              // Eq. 10 colour part
        e = fma2(bc2(mx), X, e);
        e = fma2(bc2(my), Y, e);
        e = fma2(bc2(mz), Z, e);
        e = add2(e, rd[p]);
      }
      const float2 w = make_float2(gated_weight(e.x, Dx - lo, tau2), gated_weight(e.y, Dy - lo, tau2));  // R19 / R20
      S0 = fma2(w, X, S0);
      S1 = fma2(w, Y, S1);
      S2 = fma2(w, Z, S2);
      Ws = add2(Ws, w);
    }
  }
  return make_float4(S0.x + S0.y, S1.x + S1.y, S2.x + S2.y, Ws.x + Ws.y);
}

// Loop B: strip hit counts by Q's class (R18) around the sample with depth window [lo, lo + tau2] and screen tangent
// (Tx, Ty), in (major, minor) coordinates of the tangent: Eq. 9 is symmetric in x / y and IEEE add / mul commute,
// so the bits are those of the oracle's x / y order. Returns alpha = Hc / (Hc + Ha).
template <int R>
__device__ __forceinline__ float strip_alpha(const uint2* __restrict__ s_dq, int ci, int SW, float Tx, float Ty,
                                             uint32_t lo, uint32_t tau2, const ShadeParams& sp) {
  const bool xmaj = fabsf(Tx) >= fabsf(Ty);
  const float TM = xmaj ? Tx : Ty, TN = xmaj ? Ty : Tx;
  const int strM = xmaj ? 1 : SW, strN = xmaj ? SW : 1;
  const float slope = TN / TM;  // |slope| <= 1; T is a unit vector, so the major part is >= 0.707
  uint32_t Hc = 0, Ha = 0;
  if (sp.strip_nc == 2) {  // w_strip = 0.5: two candidate minor offsets per major step, all unrolled
    // Eq. 9 is point-symmetric — negating (fM, fN) negates every product and sum exactly, the squares are the same
    // bits — and so is the candidate interval, so one membership evaluation serves the taps (s, m) and (-s, -m).
    // (When the interval of step s holds one integer k, the second candidates k + 1 and -k - 1 / -k + 1 all lie
    // outside it: farther than strip_hmax from the line, never in the strip — the same zero either way.)
    {  // s = 0: the pixel itself is in the strip; its neighbour at minor offset 1 is 1 > strip_hmax away
      const uint2 q = s_dq[ci];
      const bool cG = q.x - lo <= tau2, cA = q.y - lo <= tau2;
      Hc += cG ? 1u : 0u;
      Ha += (cA && !cG) ? 1u : 0u;
    }
#pragma unroll
    for (int s = 1; s <= R; ++s) {
      const float fM = (float)s;
      const int m0 = max((int)ceilf(fM * slope - sp.strip_hmax), -R);  // <= R: |s slope| <= R, strip_hmax > 0
      const float pM = xmul(fM, TM);
      const int off0 = s * strM + m0 * strN;
      const bool two = m0 < R;  // m0 + 1 is still a window tap (else its read is clamped and its hit masked)
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const float fN = (float)(m0 + c);
        const float dpar = xadd(pM, xmul(fN, TN));
        const float eM = xsub(fM, xmul(dpar, TM)), eN = xsub(fN, xmul(dpar, TN));
        bool in = xadd(xmul(eM, eM), xmul(eN, eN)) <= sp.strip_e2_max;
        if (c) in = in && two;
        const int off = c ? (two ? off0 + strN : off0) : off0;
#pragma unroll
        for (int sg = 0; sg < 2; ++sg) {
          const uint2 q = s_dq[sg ? ci - off : ci + off];
          const bool cG = q.x - lo <= tau2, cA = q.y - lo <= tau2;
          Hc += (in && cG) ? 1u : 0u;
          Ha += (in && cA && !cG) ? 1u : 0u;
        }
      }
    }
  } else {
#pragma unroll 1
    for (int s = -R; s <= R; ++s) {
      const float fM = (float)s;
      const int m0 = max((int)ceilf(fM * slope - sp.strip_hmax), -R);
      const float pM = xmul(fM, TM);
      for (int c = 0; c < sp.strip_nc; ++c) {
        const int mm = m0 + c;
        if (mm <= R) {
          const float fN = (float)mm;
          const float dpar = xadd(pM, xmul(fN, TN));
          const float eM = xsub(fM, xmul(dpar, TM)), eN = xsub(fN, xmul(dpar, TN));
          const bool in = xadd(xmul(eM, eM), xmul(eN, eN)) <= sp.strip_e2_max;
          const uint2 q = s_dq[ci + s * strM + mm * strN];
          const bool cG = q.x - lo <= tau2, cA = q.y - lo <= tau2;
          Hc += (in && cG) ? 1u : 0u;
          Ha += (in && cA && !cG) ? 1u : 0u;
        }
      }
    }
  }
  return (Hc + Ha) > 0 ? (float)Hc / (float)(Hc + Ha) : 0.f;
}

template <int R>
__global__ void __launch_bounds__(FT_NT, FILT_MIN_BLOCKS)
k_filter(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec, const float4* __restrict__ vertices,
         CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf, const float4* __restrict__ colour,
         const float4* __restrict__ scene_rgb, float4* __restrict__ out) {
  constexpr int SW = FT_W + 2 * R, HP = SW / 2, SH = FT_H + 2 * R, NP = HP * SH, NS = SW * SH;
  extern __shared__ float4 fsm[];
  float4* s_pa = fsm;                                              // [NP] {x_a, x_b, y_a, y_b} of the pixel pair
  float4* s_pb = fsm + NP;                                         // [NP] {z_a, z_b, k_a, k_b}
  float4* s_item = fsm + 2 * NP;                                   // [2 * FT_W * FT_H] item, later its result
  uint2* s_dq = reinterpret_cast<uint2*>(s_item + 2 * FT_W * FT_H);  // [NS] {dq centre, dq conservative}
  float2* s_pk = reinterpret_cast<float2*>(s_dq + NS);             // [NP] {k_a, k_b}
  __shared__ uint32_t s_cc[FT_H + 1][8];  // conservative-sample items per (row, class); then their prefix over rows
  __shared__ uint32_t s_cn[FT_H + 1];     // centre items per row; then their prefix
  __shared__ uint32_t s_next;             // next item warp to take
  const int W = (int)cam.W, H = (int)cam.H;
  const int tid = threadIdx.x, lx = tid & 31, ly = tid >> 5;
  const int x0 = blockIdx.x * FT_W, y0 = blockIdx.y * FT_H;
  // ---- own two pixels (rows ly and ly + FT_H / 2 of the tile)
  unsigned long long G[2], A[2];
  bool inside[2];
  int hit = 0;
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const int px = x0 + lx, py = y0 + ly + FT_HH * k;
    inside[k] = px < W && py < H;
    G[k] = A[k] = HAIR_EMPTY;
    if (inside[k]) {
      const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + (size_t)py * W + px);
      G[k] = ((unsigned long long)raw.y << 32) | raw.x;
      A[k] = ((unsigned long long)raw.w << 32) | raw.z;
    }
    hit |= !w_none(A[k]);  // centre layer is a subset of the conservative one (R10)
  }
  const bool any_hit = __syncthreads_or(hit);
  // pixels without a hit: what the hair is composited over (R29), the constant background or the scene's colour
#pragma unroll
  for (int k = 0; k < 2; ++k)
    if (inside[k] && w_none(A[k])) {
      const size_t p = (size_t)(y0 + ly + FT_HH * k) * W + x0 + lx;
      float4 bg = make_float4(sp.background[0], sp.background[1], sp.background[2], 0.f);
      if (scene_rgb) {
        const float4 b = __ldg(&scene_rgb[p]);
        bg = make_float4(b.x, b.y, b.z, sp.bg_alpha ? b.w : 0.f);
      }
      store_rgba(out, p, bg, sp.rgb16);
    }
  if (!any_hit) return;  // empty tile: background only
  // ---- (1) tile + halo to shared memory, one pixel pair per thread and round
  const float kappa = fmaxf(sqrtf(sp.kC), 1e-15f);
  for (int i = tid; i < NP; i += FT_NT) {
    const int sy = i / HP, pp = i - sy * HP;
    const int gy = y0 + sy - R;
    float c[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
    uint32_t dG[2] = {DQ_NONE, DQ_NONE}, dA[2] = {DQ_NONE, DQ_NONE};
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int gx = x0 + 2 * pp + e - R;
      if (gx >= 0 && gx < W && gy >= 0 && gy < H) {  // samples outside the image do not exist
        const size_t q = (size_t)gy * W + gx;
        const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + q);
        if (!w_none(raw.z, raw.w)) dA[e] = raw.w >> 8;
        if (!w_none(raw.x, raw.y)) {
          dG[e] = raw.y >> 8;
          const float4 cq = __ldg(&colour[q]);
          c[e][0] = kappa * cq.x, c[e][1] = kappa * cq.y, c[e][2] = kappa * cq.z;
          c[e][3] = c[e][0] * c[e][0] + c[e][1] * c[e][1] + c[e][2] * c[e][2];
        }
      }
    }
    s_pa[i] = make_float4(c[0][0], c[1][0], c[0][1], c[1][1]);
    s_pb[i] = make_float4(c[0][2], c[1][2], __uint_as_float(dG[0]), __uint_as_float(dG[1]));
    s_pk[i] = make_float2(c[0][3], c[1][3]);
    reinterpret_cast<uint4*>(s_dq)[i] = make_uint4(dG[0], dA[0], dG[1], dA[1]);
  }
  // ---- (2) work items. Centre items (one per centre-hit pixel) are compacted in PIXEL ORDER: a warp of a dense tile
  // holds one tile row, whose lanes share their pairs. Conservative-sample items (fly-away strand in front of the
  // centre hit, R21, or promoted pixel) are sparse, so they are DEALT BY BANK CLASS instead: the 16-byte
  // bank group a tap read of pixel (x, y) falls on is ((x >> 1) + (HP mod 8) y + const) mod 8, the same constant for
  // every lane, so slot = rank * 8 + class puts at most four different pairs on every bank group of a warp whatever
  // pixels its items sit on. Classes fill unevenly; the few slots left empty are skipped.
  int slot_c[2] = {-1, -1}, slot_a[2] = {-1, -1};
  bool fly[2] = {false, false};
  float2 Tc[2], Ta[2];
  uint32_t balC[2], balA[2];
  const uint32_t lt_mask = (1u << lx) - 1u;
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const bool isCenter = !w_none(G[k]), isCons = !w_none(A[k]);
    Tc[k] = Ta[k] = make_float2(1.f, 0.f);
    if (isCenter) {
      Tc[k] = sp.paper_payload ? screen_tangent_payload(cam, x0 + lx, y0 + ly + FT_HH * k, G[k])
                               : screen_tangent(sc, srec, vertices, cam, G[k]);
      fly[k] = isCons && w_dq(G[k]) >= w_dq(A[k]) && w_dq(G[k]) - w_dq(A[k]) >= sp.taufly_q;  // PAPER.md:175, R21
    }
    const bool isA = fly[k] || (isCons && !isCenter);  // fly-away strand, or promoted pixel: w_color = 1
    if (isA)
      Ta[k] = sp.paper_payload ? screen_tangent_payload(cam, x0 + lx, y0 + ly + FT_HH * k, A[k])
                               : screen_tangent(sc, srec, vertices, cam, A[k]);
    balC[k] = __ballot_sync(0xffffffffu, isCenter);
    balA[k] = __ballot_sync(0xffffffffu, isA);
    if (lx == 0) s_cn[ly + FT_HH * k] = __popc(balC[k]);
  }
  constexpr int KS = HP & 7;  // bank-group step of one tile row
  if (lx < 16) {  // conservative-sample items per (row, class): lane l of warp ly reports k = l >> 3, class = l & 7
    const int rk = lx >> 3, rc = lx & 7, rrow = ly + FT_HH * rk;
    s_cc[rrow][rc] = __popc(balA[rk] & (0x00030003u << (2 * ((rc - KS * rrow) & 7))));
  }
  __syncthreads();
  if (tid < 8) {  // exclusive prefix over the rows, total in row FT_H
    uint32_t t = 0;
#pragma unroll
    for (int r = 0; r < FT_H; ++r) {
      const uint32_t n = s_cc[r][tid];
      s_cc[r][tid] = t;
      t += n;
    }
    s_cc[FT_H][tid] = t;
  } else if (tid == 32) {
    s_next = 0;
    uint32_t t = 0;
#pragma unroll
    for (int r = 0; r < FT_H; ++r) {
      const uint32_t n = s_cn[r];
      s_cn[r] = t;
      t += n;
    }
    s_cn[FT_H] = t;
  }
  __syncthreads();
  uint32_t max_a = 0;
#pragma unroll
  for (int c = 0; c < 8; ++c) max_a = max(max_a, s_cc[FT_H][c]);
  const int n_centre = (int)((s_cn[FT_H] + 31u) & ~31u);  // centre slots, rounded up to whole warps
#if FILT_DEAL
  const int n_item = n_centre + (int)(8u * max_a);
#else
  uint32_t tot_a = 0;
#pragma unroll
  for (int c = 0; c < 8; ++c) tot_a += s_cc[FT_H][c];
  const int n_item = n_centre + (int)tot_a;
#endif
  for (int i = tid; i < n_item; i += FT_NT) s_item[i].w = __uint_as_float(0xFFFFFFFFu);  // empty slot
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const int row = ly + FT_HH * k;
    const uint32_t pix = (uint32_t)(row * FT_W + lx);
    if ((balC[k] >> lx) & 1u) {
      slot_c[k] = (int)(s_cn[row] + __popc(balC[k] & lt_mask));
      s_item[slot_c[k]] = make_float4(Tc[k].x, Tc[k].y, __uint_as_float(w_dq(G[k]) | 0x1000000u), __uint_as_float(pix));
    }
    if ((balA[k] >> lx) & 1u) {
#if FILT_DEAL
      const int cls = ((lx >> 1) + KS * row) & 7;
      const uint32_t same = 0x00030003u << (2 * ((lx >> 1) & 7));  // the four lanes of this row in my class
      slot_a[k] = n_centre + (int)((s_cc[row][cls] + __popc(balA[k] & same & lt_mask)) * 8u) + cls;
#else
      uint32_t before = 0;  // pixel order: items of the rows above, then of the lanes to the left
#pragma unroll
      for (int c = 0; c < 8; ++c) before += s_cc[row][c];
      slot_a[k] = n_centre + (int)(before + __popc(balA[k] & lt_mask));
#endif
      s_item[slot_a[k]] = make_float4(Ta[k].x, Ta[k].y, __uint_as_float(w_dq(A[k])), __uint_as_float(pix));
    }
  }
  __syncthreads();
  // ---- (3) per item (Code 2 PAPER.md:483-515 with DESIGN.md R18-R20)
  const uint32_t tauq = sp.tauz_q, tau2 = 2u * sp.tauz_q;
  const float inv_kappa = 1.0f / kappa;
  // the warps of the CTA take the item warps from a shared counter (centre and conservative-sample warps cost
  // differently, so a fixed deal leaves warps waiting at the barrier)
  for (;;) {
    int it0 = 0;
    if (lx == 0) it0 = (int)atomicAdd(&s_next, 32u);
    it0 = __shfl_sync(0xffffffffu, it0, 0);
    if (it0 >= n_item) break;
    const int it = it0 + lx;
    if (it >= n_item) continue;
    const float4 I = s_item[it];
    const float Tx = I.x, Ty = I.y;
    const uint32_t rm = __float_as_uint(I.z), pix = __float_as_uint(I.w);
    if (pix == 0xFFFFFFFFu) continue;  // empty slot
    const int ix = (int)(pix & 31u), iy = (int)(pix >> 5);
    // R20: class by integer depth compare, |d - ref| <= tau as (unsigned)(d - (ref - tau)) <= 2 tau (mod 2^32);
    // DQ_NONE is farther than tau (<= 2^24) from every depth
    const uint32_t lo = (rm & 0xFFFFFFu) - tauq;
    const int ci = (iy + R) * SW + ix + R;
    // ---- loop A: bilateral sum, positive base-2 exponent as a quadratic form of (dx, dy)
    const float qa = -(sp.kP * Tx * Tx + sp.kQ * Ty * Ty), qb = -2.f * (sp.kP - sp.kQ) * Tx * Ty,
                qc = -(sp.kP * Ty * Ty + sp.kQ * Tx * Tx);
    const float u = -(float)(R + (ix & 1));
    const int rowp = iy * HP + (ix >> 1);
    float4 S;
    // centre items fill whole warps (n_centre is a multiple of 32): no warp mixes the two loops
    if (it - lx < n_centre) {  // centre sample: colour term on; its own tap has weight 1, so no bias is needed
      const float* fa = reinterpret_cast<const float*>(s_pa + (ci >> 1));
      const float cx = fa[ci & 1], cy = fa[2 + (ci & 1)], cz = fa[4 * NP + (ci & 1)];
      const float cp2 = reinterpret_cast<const float*>(s_pk)[ci];
      S = filter_loop_a<R, true>(s_pa + rowp, s_pk + rowp, HP, NP, ix & 1, u, qa, qb, qc, cp2, -2.f * cx, -2.f * cy,
                                 -2.f * cz, lo, tau2);
    } else
      S = filter_loop_a<R, false>(s_pa + rowp, s_pk + rowp, HP, NP, ix & 1, u, qa, qb, qc, -sp.bias_nc, 0.f, 0.f, 0.f,
                                  lo, tau2);
    const float alpha = strip_alpha<R>(s_dq, ci, SW, Tx, Ty, lo, tau2, sp);
    const float inv = S.w > 0.f ? inv_kappa / S.w : 0.f;
    s_item[it] = make_float4(S.x * inv, S.y * inv, S.z * inv, alpha);
  }
  __syncthreads();
  // ---- (4) combine and composite over the background (R29)
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    if (slot_c[k] < 0 && slot_a[k] < 0) continue;  // (pixels without a hit were written at the start)
    float r = 0.f, g = 0.f, b = 0.f, alpha = 0.f;
    if (slot_c[k] >= 0) {
      const float4 a = s_item[slot_c[k]];
      r = a.x, g = a.y, b = a.z, alpha = a.w;
      if (fly[k]) {  // R21
        const float4 f = s_item[slot_a[k]];
        r = f.w * f.x + (1.f - f.w) * a.x;
        g = f.w * f.y + (1.f - f.w) * a.y;
        b = f.w * f.z + (1.f - f.w) * a.z;
        alpha = 1.f;
      }
    } else {
      const float4 a = s_item[slot_a[k]];
      r = a.x, g = a.y, b = a.z, alpha = a.w;
    }
    const size_t p = (size_t)(y0 + ly + FT_HH * k) * W + x0 + lx;
    float4 bg = make_float4(sp.background[0], sp.background[1], sp.background[2], 0.f);
    if (scene_rgb) {
      const float4 s4 = __ldg(&scene_rgb[p]);
      bg = make_float4(s4.x, s4.y, s4.z, sp.bg_alpha ? s4.w : 0.f);
    }
    const float ia = 1.f - alpha;
    store_rgba(out, p, make_float4(alpha * r + ia * bg.x, alpha * g + ia * bg.y, alpha * b + ia * bg.z, alpha + ia * bg.w),
               sp.rgb16);
  }
}

// filter off, or r = 0 (window = the pixel itself): out = centre colour over the background
__global__ void __launch_bounds__(256)
k_filter_passthrough(CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf,
                     const float4* __restrict__ colour, const float4* __restrict__ scene_rgb, float4* __restrict__ out) {
  const size_t n_px = (size_t)cam.W * cam.H;
  const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_px) return;
  const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + p);
  float4 o = make_float4(sp.background[0], sp.background[1], sp.background[2], 0.f);
  if (scene_rgb) {
    const float4 b = __ldg(&scene_rgb[p]);
    o = make_float4(b.x, b.y, b.z, sp.bg_alpha ? b.w : 0.f);
  }
  if (!w_none(raw.x, raw.y)) {
    const float4 c = __ldg(&colour[p]);
    o = make_float4(c.x, c.y, c.z, 1.f);
  }
  store_rgba(out, p, o, sp.rgb16);
}

// hair_stats: non-empty pixels per layer (counters flag only)
__global__ void __launch_bounds__(256)
k_count_pixels(const unsigned long long* __restrict__ gbuf, size_t n_px, unsigned long long* __restrict__ counters) {
  uint32_t nc = 0, na = 0;
  for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n_px; p += (size_t)gridDim.x * blockDim.x) {
    const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + p);
    nc += !w_none(raw.x, raw.y);
    na += !w_none(raw.z, raw.w);
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    nc += __shfl_xor_sync(0xffffffffu, nc, d);
    na += __shfl_xor_sync(0xffffffffu, na, d);
  }
  if ((threadIdx.x & 31) == 0) {
    if (nc) atomicAdd(&counters[CNT_PX_CENTER], (unsigned long long)nc);
    if (na) atomicAdd(&counters[CNT_PX_CONS], (unsigned long long)na);
  }
}

void launch_shade(const SceneDev* d_scene, const uint2* srec, const float4* vertices, CamDev cam,
                  ShadeParams sp, const unsigned long long* gbuf, float4* colour, const DomSet* dom,
                  const unsigned long long* counters, cudaStream_t st) {
  size_t n = (size_t)cam.W * cam.H;
  if (!sp.shadows) dom = nullptr;
  const dim3 gp((cam.W + 63) / 64, (cam.H + 3) / 4);
  const unsigned gs = (unsigned)((n + 255) / 256);
  if (sp.paper_payload) {
    if (dom) k_shade_payload<true><<<gp, 256, 0, st>>>(d_scene, cam, sp, gbuf, colour, dom, counters);
    else k_shade_payload<false><<<gp, 256, 0, st>>>(d_scene, cam, sp, gbuf, colour, nullptr, counters);
    return;
  }
  if (dom) k_shade<true><<<gs, 256, 0, st>>>(d_scene, srec, vertices, cam, sp, gbuf, colour, dom, counters);
  else k_shade<false><<<gs, 256, 0, st>>>(d_scene, srec, vertices, cam, sp, gbuf, colour, nullptr, counters);
}

template <int R>
static void launch_filter_r(const SceneDev* d_scene, const uint2* srec, const float4* vertices, CamDev cam,
                            ShadeParams sp, const unsigned long long* gbuf, const float4* colour,
                            const float4* scene_rgb, float4* out, LaunchState* ls, cudaStream_t st) {
  constexpr int NS = (FT_W + 2 * R) * (FT_H + 2 * R), NP = NS / 2, NI = 2 * FT_W * FT_H;
  // pairs: two float4 + one uint2; strip depths: one uint2 per pixel; items: one float4
  constexpr size_t smem = (size_t)NP * (2 * sizeof(float4) + sizeof(uint2)) + (size_t)NS * sizeof(uint2) +
                          (size_t)NI * sizeof(float4);
  if (!ls->filter_set[R]) {  // once per context (the opt-in is per device)
    raise_dyn_smem(k_filter<R>, smem);
    ls->filter_set[R] = true;
  }
  dim3 grid((cam.W + FT_W - 1) / FT_W, (cam.H + FT_H - 1) / FT_H);
  k_filter<R><<<grid, FT_NT, smem, st>>>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out);
}

int launch_filter(const SceneDev* d_scene, const uint2* srec, const float4* vertices, CamDev cam,
                  ShadeParams sp, const unsigned long long* gbuf, const float4* colour, const float4* scene_rgb,
                  float4* out, unsigned long long* counters, bool count, LaunchState* ls, cudaStream_t st) {
  const size_t n = (size_t)cam.W * cam.H;
  int launches = 1;
  if (count) {
    k_count_pixels<<<148 * 8, 256, 0, st>>>(gbuf, n, counters);
    ++launches;
  }
  if (!sp.filter_on) {
    k_filter_passthrough<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(cam, sp, gbuf, colour, scene_rgb, out);
    return launches;
  }
  switch (sp.r) {
    case 0: launch_filter_r<0>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out, ls, st); break;
    case 1: launch_filter_r<1>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out, ls, st); break;
    case 2: launch_filter_r<2>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out, ls, st); break;
    case 3: launch_filter_r<3>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out, ls, st); break;
    case 4: launch_filter_r<4>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out, ls, st); break;
    case 5: launch_filter_r<5>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out, ls, st); break;
    case 6: launch_filter_r<6>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out, ls, st); break;
    default: launch_filter_r<7>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out, ls, st); break;
  }
  return launches;
}
