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

__global__ void __launch_bounds__(256)
k_shade(const SceneDev* __restrict__ sc, const uint4* __restrict__ table, const float4* __restrict__ vertices,
        CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf, float4* __restrict__ colour) {
  const size_t n_px = (size_t)cam.W * cam.H;
  const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_px) return;
  const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + p);
  const unsigned long long G = ((unsigned long long)raw.y << 32) | raw.x;
  if (G == HAIR_EMPTY) return;  // colour is only ever read where a centre hit exists
  const Loc l = locate_strand(sc, table, w_sid(G));
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
  const F3 alb = (1.f - w) * f3(g.albedo_root[0], g.albedo_root[1], g.albedo_root[2]) +
                 w * f3(g.albedo_tip[0], g.albedo_tip[1], g.albedo_tip[2]);
  const F3 V = normalize(f3(cam.eye[0], cam.eye[1], cam.eye[2]) - pos);
  F3 rgb = f3(ao * sp.ambient[0] * alb.x, ao * sp.ambient[1] * alb.y, ao * sp.ambient[2] * alb.z);
  const float beta = g.roughness, tilt = g.tilt;
  const float inv2b2 = 1.0f / (2.f * beta * beta);
  const float sin_o = fminf(fmaxf(dot(T, V), -1.f), 1.f);
  const float asin_o = asinf(sin_o);
  for (uint32_t li = 0; li < sp.n_lights; ++li) {
    const F3 Lv = f3(sp.light_pos[li][0], sp.light_pos[li][1], sp.light_pos[li][2]) - pos;
    const float d2 = dot(Lv, Lv);
    const float inv_d2 = 1.0f / d2;
    const F3 om = rsqrtf(d2) * Lv;
    const float sin_i = fminf(fmaxf(dot(T, om), -1.f), 1.f);
    const float cos_i = sqrtf(fmaxf(0.f, 1.f - sin_i * sin_i));
    const float th = 0.5f * (asinf(sin_i) + asin_o);
    const float a = th + tilt, b = th - 1.5f * tilt;
    const float MR = __expf(-a * a * inv2b2), MT = __expf(-b * b * 0.25f * inv2b2);
    const float s = cos_i * inv_d2;
    rgb.x += sp.light_rgb[li][0] * s * (sp.k_d * alb.x + sp.k_R * MR + sp.k_TRT * MT * alb.x);
    rgb.y += sp.light_rgb[li][1] * s * (sp.k_d * alb.y + sp.k_R * MR + sp.k_TRT * MT * alb.y);
    rgb.z += sp.light_rgb[li][2] * s * (sp.k_d * alb.z + sp.k_R * MR + sp.k_TRT * MT * alb.z);
  }
  colour[p] = make_float4(rgb.x, rgb.y, rgb.z, 1.0f);
}

// R22: unit screen direction of the segment a word names; fixed-order fp32 (decides strip membership)
__device__ __forceinline__ float2 screen_tangent(const SceneDev* __restrict__ sc, const uint4* __restrict__ table,
                                                 const float4* __restrict__ vertices, const CamDev& cam,
                                                 unsigned long long word) {
  const Loc l = locate_strand(sc, table, w_sid(word));
  const float4* vs = vertices + l.voff + w_j(word);
  const float4 va = __ldg(vs), vb = __ldg(vs + 1);
  const Proj a = project_exact(cam, va.x, va.y, va.z), b = project_exact(cam, vb.x, vb.y, vb.z);
  const float dx = xsub(b.sx, a.sx), dy = xsub(b.sy, a.sy);
  const float dd = xadd(xmul(dx, dx), xmul(dy, dy));
  if (!(dd >= 1e-12f)) return make_float2(1.f, 0.f);
  const float len = xsqrt(dd);
  return make_float2(xdiv(dx, len), xdiv(dy, len));
}

struct Acc {
  float r, g, b, alpha;
};

// One pass over the (2r+1)^2 window around (px, py) for the reference sample (T, dq_ref)
// (Code 2 PAPER.md:483-515 with DESIGN.md R18-R20).
__device__ __forceinline__ Acc accumulate(const ShadeParams& sp, const unsigned long long* __restrict__ gbuf,
                                          const float4* __restrict__ colour, int W, int H, int px, int py,
                                          float2 T, uint32_t dq_ref, bool use_colour, float4 CP) {
  float S0 = 0.f, S1 = 0.f, S2 = 0.f, Wsum = 0.f, emax = -INFINITY;
  uint32_t Hc = 0, Ha = 0;
  const int r = sp.r;
  for (int dy = -r; dy <= r; ++dy) {
    const int qy = py + dy;
    if (qy < 0 || qy >= H) continue;
    for (int dx = -r; dx <= r; ++dx) {
      const int qx = px + dx;
      if (qx < 0 || qx >= W) continue;
      const size_t q = (size_t)qy * W + qx;
      const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + q);
      // R20: class by integer depth compare; an empty word has dq = 0xFFFFFF, never within tau of a hit
      const uint32_t dG = raw.y >> 8, dA = raw.w >> 8;
      const bool cG = (raw.x & raw.y) != 0xFFFFFFFFu && (dG > dq_ref ? dG - dq_ref : dq_ref - dG) <= sp.tauz_q;
      const bool cA = (raw.z & raw.w) != 0xFFFFFFFFu && (dA > dq_ref ? dA - dq_ref : dq_ref - dA) <= sp.tauz_q;
      if (!cG && !cA) continue;
      // Eq. 9, fixed-order fp32
      const float fdx = (float)dx, fdy = (float)dy;
      const float dpar = xadd(xmul(fdx, T.x), xmul(fdy, T.y));
      const float ex = xsub(fdx, xmul(dpar, T.x)), ey = xsub(fdy, xmul(dpar, T.y));
      const float dperp = xsqrt(xadd(xmul(ex, ex), xmul(ey, ey)));
      if (dperp <= sp.w_strip) {
        if (cG) ++Hc;
        else ++Ha;
      }
      if (cG) {  // R19
        float e = -dpar * dpar * sp.inv_sp2 - dperp * dperp * sp.inv_sq2;
        const float4 CQ = __ldg(&colour[q]);
        if (use_colour) {
          const float d0 = CP.x - CQ.x, d1 = CP.y - CQ.y, d2 = CP.z - CQ.z;
          e -= (d0 * d0 + d1 * d1 + d2 * d2) * sp.inv_sc2;  // Eq. 10
        }
        // normalised sum with a running maximum exponent (online softmax): Eq. 10's ratio is unchanged,
        // but weights of e^-90 (5 px across the strand) no longer underflow to denormals / 0
        if (e > emax) {
          const float sc_ = __expf(emax - e);
          S0 *= sc_, S1 *= sc_, S2 *= sc_, Wsum *= sc_;
          emax = e;
        }
        const float w = __expf(e - emax);
        S0 += w * CQ.x;
        S1 += w * CQ.y;
        S2 += w * CQ.z;
        Wsum += w;
      }
    }
  }
  Acc o;
  const float inv = Wsum > 0.f ? 1.0f / Wsum : 0.f;
  o.r = S0 * inv;
  o.g = S1 * inv;
  o.b = S2 * inv;
  o.alpha = (Hc + Ha) > 0 ? (float)Hc / (float)(Hc + Ha) : 0.f;
  return o;
}

template <bool COUNT>
__global__ void __launch_bounds__(256)
k_filter(const SceneDev* __restrict__ sc, const uint4* __restrict__ table, const float4* __restrict__ vertices,
         CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf, const float4* __restrict__ colour,
         float4* __restrict__ out, unsigned long long* __restrict__ counters) {
  const int W = (int)cam.W, H = (int)cam.H;
  const int px = blockIdx.x * 32 + (threadIdx.x & 31), py = blockIdx.y * 8 + (threadIdx.x >> 5);
  const bool inside = px < W && py < H;
  unsigned long long G = HAIR_EMPTY, A = HAIR_EMPTY;
  size_t p = 0;
  if (inside) {
    p = (size_t)py * W + px;
    const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + p);
    G = ((unsigned long long)raw.y << 32) | raw.x;
    A = ((unsigned long long)raw.w << 32) | raw.z;
  }
  const bool isCenter = G != HAIR_EMPTY, isCons = A != HAIR_EMPTY;
  if (COUNT) {
    const uint32_t nc = __popc(__ballot_sync(0xffffffffu, isCenter)), na = __popc(__ballot_sync(0xffffffffu, isCons));
    if ((threadIdx.x & 31) == 0) {
      if (nc) atomicAdd(&counters[CNT_PX_CENTER], (unsigned long long)nc);
      if (na) atomicAdd(&counters[CNT_PX_CONS], (unsigned long long)na);
    }
  }
  if (!inside) return;
  float r = 0.f, g = 0.f, b = 0.f, alpha = 0.f;
  if (!sp.filter_on) {
    if (isCenter) {
      const float4 CP = __ldg(&colour[p]);
      r = CP.x, g = CP.y, b = CP.z, alpha = 1.f;
    }
  } else if (isCenter) {
    const float4 CP = __ldg(&colour[p]);
    const float2 TG = screen_tangent(sc, table, vertices, cam, G);
    Acc a = accumulate(sp, gbuf, colour, W, H, px, py, TG, w_dq(G), true, CP);
    r = a.r, g = a.g, b = a.b, alpha = a.alpha;
    // fly-away strand in front of the centre hit (R21)
    if (isCons && w_dq(G) >= w_dq(A) && w_dq(G) - w_dq(A) >= sp.taufly_q) {
      const float2 TA = screen_tangent(sc, table, vertices, cam, A);
      Acc f = accumulate(sp, gbuf, colour, W, H, px, py, TA, w_dq(A), false, CP);
      r = f.alpha * f.r + (1.f - f.alpha) * a.r;
      g = f.alpha * f.g + (1.f - f.alpha) * a.g;
      b = f.alpha * f.b + (1.f - f.alpha) * a.b;
      alpha = 1.f;
    }
  } else if (isCons) {  // promoted pixel: w_color = 1
    const float2 TA = screen_tangent(sc, table, vertices, cam, A);
    Acc a = accumulate(sp, gbuf, colour, W, H, px, py, TA, w_dq(A), false, make_float4(0.f, 0.f, 0.f, 0.f));
    r = a.r, g = a.g, b = a.b, alpha = a.alpha;
  }
  const float ia = 1.f - alpha;  // R29: composite over the background
  out[p] = make_float4(alpha * r + ia * sp.background[0], alpha * g + ia * sp.background[1],
                       alpha * b + ia * sp.background[2], alpha);
}

void launch_shade(const SceneDev* d_scene, const uint4* table, const float4* vertices, CamDev cam,
                  ShadeParams sp, const unsigned long long* gbuf, float4* colour, cudaStream_t st) {
  size_t n = (size_t)cam.W * cam.H;
  k_shade<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_scene, table, vertices, cam, sp, gbuf, colour);
}

void launch_filter(const SceneDev* d_scene, const uint4* table, const float4* vertices, CamDev cam,
                   ShadeParams sp, const unsigned long long* gbuf, const float4* colour, float4* out,
                   unsigned long long* counters, bool count, cudaStream_t st) {
  dim3 grid((cam.W + 31) / 32, (cam.H + 7) / 8);
  if (count) k_filter<true><<<grid, 256, 0, st>>>(d_scene, table, vertices, cam, sp, gbuf, colour, out, counters);
  else k_filter<false><<<grid, 256, 0, st>>>(d_scene, table, vertices, cam, sp, gbuf, colour, out, counters);
}
