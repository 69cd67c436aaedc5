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

// the stand-in shading model (R23) at one point: position, unit tangent, strand parameter w, AO
__device__ __forceinline__ F3 shade_model(const GroomDev& g, const CamDev& cam, const ShadeParams& sp, F3 pos, F3 T,
                                          float w, float ao) {
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
    const float s = cos_i * inv_d2;
    rgb.x += sp.light_rgb[li][0] * s * (sp.k_d * alb.x + sp.k_R * MR + sp.k_TRT * MT * alb.x);
    rgb.y += sp.light_rgb[li][1] * s * (sp.k_d * alb.y + sp.k_R * MR + sp.k_TRT * MT * alb.y);
    rgb.z += sp.light_rgb[li][2] * s * (sp.k_d * alb.z + sp.k_R * MR + sp.k_TRT * MT * alb.z);
  }
  return rgb;
}

// O6 for one word: linear RGB of the hit it names
__device__ __forceinline__ F3 shade_word(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec,
                                         const float4* __restrict__ vertices, const CamDev& cam, const ShadeParams& sp,
                                         unsigned long long G) {
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
  return shade_model(g, cam, sp, pos, T, w, ao);
}

// R-payload: O6 from the paper's payload alone, no vertex read. Position = the point of the
// ray through the pixel centre at the word's depth ("reconstruct it from the depth value")
__device__ __forceinline__ F3 shade_payload(const SceneDev* __restrict__ sc, const CamDev& cam, const ShadeParams& sp,
                                            int x, int y, unsigned long long G) {
  const X3 t = oct_decode_x(pw_ox(G), pw_oy(G));
  const float w = (float)((uint32_t)(G >> 6) & 63u) * (1.0f / 63.0f), ao = (float)((uint32_t)G & 63u) * (1.0f / 63.0f);
  const float zn = (float)w_dq(G) / 16777215.0f;
  const float zv = cam.B / (cam.A - zn);
  const float cx = (((float)x + 0.5f) - cam.half_w) / cam.fpx, cy = (cam.half_h - ((float)y + 0.5f)) / cam.fpx;
  const F3 pos = f3(cam.eye[0] + zv * (cx * cam.r[0] + cy * cam.u[0] + cam.f[0]),
                    cam.eye[1] + zv * (cx * cam.r[1] + cy * cam.u[1] + cam.f[1]),
                    cam.eye[2] + zv * (cx * cam.r[2] + cy * cam.u[2] + cam.f[2]));
  return shade_model(sc->g[sp.pp_groom], cam, sp, pos, f3(t.x, t.y, t.z), w, ao);
}

__global__ void __launch_bounds__(256)
k_shade(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec, const float4* __restrict__ vertices,
        CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf, float4* __restrict__ colour) {
  const size_t n_px = (size_t)cam.W * cam.H;
  const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_px) return;
  const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + p);
  const unsigned long long G = ((unsigned long long)raw.y << 32) | raw.x;
  if (w_none(G)) return;  // colour is only ever read where a centre hit exists
  const F3 rgb = shade_word(sc, srec, vertices, cam, sp, G);
  colour[p] = make_float4(rgb.x, rgb.y, rgb.z, 1.0f);
}

__global__ void __launch_bounds__(256)
k_shade_payload(const SceneDev* __restrict__ sc, CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf,
                float4* __restrict__ colour) {
  const uint32_t x = blockIdx.x * 64u + (threadIdx.x & 63u), y = blockIdx.y * 4u + (threadIdx.x >> 6);
  if (x >= cam.W || y >= cam.H) return;
  const size_t p = (size_t)y * cam.W + x;
  const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + p);
  const unsigned long long G = ((unsigned long long)raw.y << 32) | raw.x;
  if (w_none(G)) return;
  const F3 rgb = shade_payload(sc, cam, sp, (int)x, (int)y, G);
  colour[p] = make_float4(rgb.x, rgb.y, rgb.z, 1.0f);
}

// MSAA-k reference resolve (DESIGN.md R-msaa): mean over the k samples of (shaded hit | background)
__global__ void __launch_bounds__(256)
k_resolve_msaa(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec, const float4* __restrict__ vertices,
               CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ samples, uint32_t ms_k,
               const float4* __restrict__ scene_rgb, float4* __restrict__ out) {
  const size_t n_px = (size_t)cam.W * cam.H;
  const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n_px) return;
  F3 acc = f3(0.f, 0.f, 0.f);
  uint32_t n_hit = 0;
  for (uint32_t s = 0; s < ms_k; ++s) {
    const unsigned long long w = __ldg(&samples[(size_t)s * n_px + p]);
    if (w_none(w)) continue;
    acc = acc + shade_word(sc, srec, vertices, cam, sp, w);
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
                         float4* out, cudaStream_t st) {
  const size_t n = (size_t)cam.W * cam.H;
  k_resolve_msaa<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_scene, srec, vertices, cam, sp, samples, ms_k, scene_rgb, out);
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
// Tiled filter. One CTA owns a 32x16 pixel tile: (1) the tile + an r-pixel halo of the G-buffer
// (as two 24-bit depths, "none" = DQ_NONE) and of the shaded colour go to shared memory once,
// (2) every hit pixel emits one or two work items (reference tangent, reference depth, colour
// mode; two for a fly-away pixel), compacted through a shared counter so sparse tiles still fill
// their warps, (3) the items are spread over the 256 threads; each item runs two branch-free loops
// over shared memory, (4) the owning thread combines its items and writes out_rgb.
//  loop A, Eq. 10: all (2r+1)^2 taps, one LDS.32 (centre depth) + one LDS.128
//    (colour) per tap; the class test (R20, integer depth compare) becomes a select on the weight,
//    so lanes never diverge. The exponent is the quadratic form a dx^2 + b dx dy + c dy^2 of the
//    window offset (2 FMA per tap), the colour distance is |CP|^2 + |CQ|^2 - 2 CP.CQ with -kC|CQ|^2
//    kept per tile pixel, all pre-multiplied by log2(e) so that one ex2.approx gives the weight.
//  loop B, strip hit counts: only lattice points within w_strip of the tangent line
//    can be in the strip, so instead of testing 121 taps the loop walks the 2r+1 steps of the
//    tangent's major axis and tests the `strip_nc` (2 for w_strip = 0.5) integer minor offsets that
//    can lie within (w_strip + 0.01) sqrt(2) of the line — a superset; membership itself is Eq. 9 in
//    the oracle's fixed-order fp32 (sqrt_rn(e2) <= w_strip tested as e2 <= strip_e2_max, host-side
//    the largest float whose correctly rounded root is <= w_strip; sqrt_rn is monotone).
#define FT_W 32
#define FT_H 16
#ifndef FILT_MIN_BLOCKS
#define FILT_MIN_BLOCKS 4  // CTAs per SM the register budget is held to
#endif
#define DQ_NONE 0x40000000u

__device__ __forceinline__ float fast_ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// Eq. 9 in the oracle's operation order; true iff sqrt_rn(e2) <= w_strip
__device__ __forceinline__ bool in_strip_exact(float fdx, float fdy, float Tx, float Ty, float e2_max) {
  const float dpar = xadd(xmul(fdx, Tx), xmul(fdy, Ty));
  const float ex = xsub(fdx, xmul(dpar, Tx)), ey = xsub(fdy, xmul(dpar, Ty));
  return xadd(xmul(ex, ex), xmul(ey, ey)) <= e2_max;
}

template <int R>
__global__ void __launch_bounds__(256, FILT_MIN_BLOCKS)
k_filter(const SceneDev* __restrict__ sc, const uint2* __restrict__ srec, const float4* __restrict__ vertices,
         CamDev cam, ShadeParams sp, const unsigned long long* __restrict__ gbuf, const float4* __restrict__ colour,
         const float4* __restrict__ scene_rgb, float4* __restrict__ out) {
  constexpr int SW = FT_W + 2 * R, SH = FT_H + 2 * R, NS = SW * SH;
  extern __shared__ float4 fsm[];
  float4* s_col = fsm;                                  // [NS] rgb (zeros where no centre hit), dq of the centre word
  float4* s_item = fsm + NS;                            // [2 * FT_W * FT_H] item, later its result
  uint32_t* s_dqG = reinterpret_cast<uint32_t*>(s_item + 2 * FT_W * FT_H);  // [NS] dq of the centre word
  uint32_t* s_dqA = s_dqG + NS;                                             // [NS] dq of the conservative word
  float* s_k2 = reinterpret_cast<float*>(s_dqA + NS);                       // [NS] -kC |rgb|^2 (Eq. 10 colour term)
  // (the centre depth sits both in s_col.w, where the tap loop gets it with the colour in one LDS.128 — the loop of
  // the conservative-sample items then reads nothing else — and in s_dqG, whose 4-byte stride suits the strip loop)
  __shared__ uint32_t s_cc[2][FT_H + 1][8];  // items per (type, row, class); then their exclusive prefix over rows
  const int W = (int)cam.W, H = (int)cam.H;
  const int tid = threadIdx.x, lx = tid & 31, ly = tid >> 5;
  const int x0 = blockIdx.x * FT_W, y0 = blockIdx.y * FT_H;
  // ---- own two pixels (rows ly and ly + 8 of the tile)
  unsigned long long G[2], A[2];
  bool inside[2];
  int hit = 0;
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const int px = x0 + lx, py = y0 + ly + 8 * k;
    inside[k] = px < W && py < H;
    G[k] = A[k] = HAIR_EMPTY;
    if (inside[k]) {
      const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + (size_t)py * W + px);
      G[k] = ((unsigned long long)raw.y << 32) | raw.x;
      A[k] = ((unsigned long long)raw.w << 32) | raw.z;
    }
    hit |= !w_none(A[k]);  // centre layer is a subset of the conservative one (R10)
  }
  // what the hair is composited over (R29): the constant background, or the scene's colour (R-scene)
  float4 bg[2];
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    bg[k] = make_float4(sp.background[0], sp.background[1], sp.background[2], 0.f);
    if (scene_rgb && inside[k]) {
      const float4 b = __ldg(&scene_rgb[(size_t)(y0 + ly + 8 * k) * W + x0 + lx]);
      bg[k] = make_float4(b.x, b.y, b.z, sp.bg_alpha ? b.w : 0.f);
    }
  }
  if (!__syncthreads_or(hit)) {  // empty tile: background only
#pragma unroll
    for (int k = 0; k < 2; ++k)
      if (inside[k]) store_rgba(out, (size_t)(y0 + ly + 8 * k) * W + x0 + lx, bg[k], sp.rgb16);
    return;
  }
  // ---- (1) tile + halo to shared memory
  for (int i = tid; i < NS; i += 256) {
    const int sy = i / SW, sx = i - sy * SW;
    const int gx = x0 + sx - R, gy = y0 + sy - R;
    uint32_t dG = DQ_NONE, dA = DQ_NONE;
    float4 c4 = make_float4(0.f, 0.f, 0.f, 0.f);
    float k2 = 0.f;
    if (gx >= 0 && gx < W && gy >= 0 && gy < H) {  // samples outside the image do not exist
      const size_t q = (size_t)gy * W + gx;
      const uint4 raw = __ldg(reinterpret_cast<const uint4*>(gbuf) + q);
      if (!w_none(raw.z, raw.w)) dA = raw.w >> 8;
      if (!w_none(raw.x, raw.y)) {
        dG = raw.y >> 8;
        const float4 c = __ldg(&colour[q]);
        c4 = make_float4(c.x, c.y, c.z, 0.f);
        k2 = -sp.kC * (c.x * c.x + c.y * c.y + c.z * c.z);
      }
    }
    c4.w = __uint_as_float(dG);
    s_col[i] = c4;
    s_k2[i] = k2;
    s_dqG[i] = dG;
    s_dqA[i] = dA;
  }
  // ---- (2) work items, compacted by type (all centre items, then all conservative-sample items: all but one warp
  // hold items of one type, which take the tap loop with / without the colour term) and, inside a type, DEALT BY BANK
  // CLASS: the 16-byte bank group a tap read of pixel (x, y) falls on is (x + (SW mod 8) y + const) mod 8, the same
  // constant for every lane, so slot = rank * 8 + class puts eight different bank groups in every quarter warp
  // whatever pixels the items sit on (sparse fly-away / promoted items were 2-way conflicted when merely packed in
  // pixel order). Classes fill unevenly; the few slots left empty are skipped.
  int slot_c[2] = {-1, -1}, slot_a[2] = {-1, -1};
  bool fly[2] = {false, false};
  float2 Tc[2], Ta[2];
  uint32_t bal[4];
  const uint32_t lt_mask = (1u << lx) - 1u;
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const bool isCenter = !w_none(G[k]), isCons = !w_none(A[k]);
    Tc[k] = Ta[k] = make_float2(1.f, 0.f);
    if (isCenter) {
      Tc[k] = sp.paper_payload ? screen_tangent_payload(cam, x0 + lx, y0 + ly + 8 * k, G[k])
                               : screen_tangent(sc, srec, vertices, cam, G[k]);
      fly[k] = isCons && w_dq(G[k]) >= w_dq(A[k]) && w_dq(G[k]) - w_dq(A[k]) >= sp.taufly_q;  // PAPER.md:175, R21
    }
    const bool isA = fly[k] || (isCons && !isCenter);  // fly-away strand, or promoted pixel: w_color = 1
    if (isA)
      Ta[k] = sp.paper_payload ? screen_tangent_payload(cam, x0 + lx, y0 + ly + 8 * k, A[k])
                               : screen_tangent(sc, srec, vertices, cam, A[k]);
    bal[2 * k] = __ballot_sync(0xffffffffu, isCenter);
    bal[2 * k + 1] = __ballot_sync(0xffffffffu, isA);
  }
  constexpr int KS = SW & 7;  // bank-group step of one tile row
  {
    // counts per (type, class, row): lane l of warp ly reports k = l >> 4, type = (l >> 3) & 1, class = l & 7
    const int rk = lx >> 4, rt = (lx >> 3) & 1, rc = lx & 7, rrow = ly + 8 * rk;
    const uint32_t rb = rk ? (rt ? bal[3] : bal[2]) : (rt ? bal[1] : bal[0]);
    s_cc[rt][rrow][rc] = __popc(rb & (0x01010101u << ((rc - KS * rrow) & 7)));
  }
  __syncthreads();
  if (tid < 16) {  // exclusive prefix over the rows, total in row FT_H
    uint32_t t = 0;
#pragma unroll
    for (int r = 0; r < FT_H; ++r) {
      const uint32_t n = s_cc[tid >> 3][r][tid & 7];
      s_cc[tid >> 3][r][tid & 7] = t;
      t += n;
    }
    s_cc[tid >> 3][FT_H][tid & 7] = t;
  }
  __syncthreads();
  uint32_t max_c = 0, max_a = 0;
#pragma unroll
  for (int c = 0; c < 8; ++c) max_c = max(max_c, s_cc[0][FT_H][c]), max_a = max(max_a, s_cc[1][FT_H][c]);
  const int n_centre = (int)((8u * max_c + 31u) & ~31u);  // centre slots, rounded up to whole warps
  const int n_item = n_centre + (int)(8u * max_a);
  for (int i = tid; i < n_item; i += 256) s_item[i].w = __uint_as_float(0xFFFFFFFFu);  // empty slot
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const int row = ly + 8 * k, cls = (lx + KS * row) & 7;
    const uint32_t same = 0x01010101u << (lx & 7);  // the four lanes of this row in my class
    const uint32_t pix = (uint32_t)(row * FT_W + lx);
    const uint32_t before_c = s_cc[0][row][cls], before_a = s_cc[1][row][cls];
    if ((bal[2 * k] >> lx) & 1u) {
      slot_c[k] = (int)((before_c + __popc(bal[2 * k] & same & lt_mask)) * 8u) + cls;
      s_item[slot_c[k]] = make_float4(Tc[k].x, Tc[k].y, __uint_as_float(w_dq(G[k]) | 0x1000000u), __uint_as_float(pix));
    }
    if ((bal[2 * k + 1] >> lx) & 1u) {
      slot_a[k] = n_centre + (int)((before_a + __popc(bal[2 * k + 1] & same & lt_mask)) * 8u) + cls;
      s_item[slot_a[k]] = make_float4(Ta[k].x, Ta[k].y, __uint_as_float(w_dq(A[k])), __uint_as_float(pix));
    }
  }
  __syncthreads();
  // ---- (3) per item (Code 2 PAPER.md:483-515 with DESIGN.md R18-R20)
  const uint32_t tau = sp.tauz_q, tau2 = 2u * sp.tauz_q;
  for (int it = tid; it < n_item; it += 256) {
    const float4 I = s_item[it];
    const float Tx = I.x, Ty = I.y;
    const uint32_t rm = __float_as_uint(I.z), pix = __float_as_uint(I.w);
    if (pix == 0xFFFFFFFFu) continue;  // empty slot of an under-filled bank class
    // R20: class by integer depth compare, |d - ref| <= tau as (unsigned)(d - (ref - tau)) <= 2 tau (mod 2^32);
    // DQ_NONE is farther than tau (<= 2^24) from every depth
    const uint32_t lo = (rm & 0xFFFFFFu) - tau;
    const int ci = ((int)(pix >> 5) + R) * SW + (int)(pix & 31u) + R;
    // ---- loop A: bilateral sum. Exponent (base 2) of the spatial weight as a quadratic form of (dx, dy)
    const float qa = sp.kP * Tx * Tx + sp.kQ * Ty * Ty, qb = 2.f * (sp.kP - sp.kQ) * Tx * Ty,
                qc = sp.kP * Ty * Ty + sp.kQ * Tx * Tx;
    float c2x = 0.f, c2y = 0.f, c2z = 0.f, e0 = sp.bias_nc, m = 0.f;
    if (rm >> 24) {  // centre sample: colour term on; its own tap has weight 1, so no bias is needed
      const float4 CP = s_col[ci];
      c2x = 2.f * sp.kC * CP.x, c2y = 2.f * sp.kC * CP.y, c2z = 2.f * sp.kC * CP.z;
      e0 = s_k2[ci];
      m = 1.f;
    }
    float S0 = 0.f, S1 = 0.f, S2 = 0.f, Wsum = 0.f;
    // items are sorted by type: a warp whose 32 items are all conservative-sample items (no colour term, R21 /
    // PAPER.md:175 w_color = 1) skips the four colour FMAs of every tap
    const int it0 = it - lx;
    if (it0 >= n_centre) {
#pragma unroll 1
      for (int dy = -R; dy <= R; ++dy) {
        const float fdy = (float)dy;
        const float r0 = fmaf(qc * fdy, fdy, e0), r1 = qb * fdy;
        const float4* col_row = s_col + ci + dy * SW;
#pragma unroll
        for (int dx = -R; dx <= R; ++dx) {
          const float4 q = col_row[dx];
          const uint32_t d = __float_as_uint(q.w);
          const float fdx = (float)dx;
          const float e = fmaf(r1, fdx, fmaf(qa, fdx * fdx, r0));  // Eq. 10 spatial part
          const float w = (d - lo <= tau2) ? fast_ex2(e) : 0.f;    // R19: centre-class taps only
          S0 = fmaf(w, q.x, S0);
          S1 = fmaf(w, q.y, S1);
          S2 = fmaf(w, q.z, S2);
          Wsum += w;
        }
      }
    } else {
#pragma unroll 1
      for (int dy = -R; dy <= R; ++dy) {
        const float fdy = (float)dy;
        const float r0 = fmaf(qc * fdy, fdy, e0), r1 = qb * fdy;
        const float* k2_row = s_k2 + ci + dy * SW;
        const float4* col_row = s_col + ci + dy * SW;
#pragma unroll
        for (int dx = -R; dx <= R; ++dx) {
          const float k2 = k2_row[dx];
          const float4 q = col_row[dx];
          const uint32_t d = __float_as_uint(q.w);
          const float fdx = (float)dx;
          float e = fmaf(r1, fdx, fmaf(qa, fdx * fdx, r0));                     // Eq. 10 spatial part
          e = fmaf(c2x, q.x, fmaf(c2y, q.y, fmaf(c2z, q.z, fmaf(m, k2, e))));   // Eq. 10 colour part
          const float w = (d - lo <= tau2) ? fast_ex2(e) : 0.f;                 // R19: centre-class taps only
          S0 = fmaf(w, q.x, S0);
          S1 = fmaf(w, q.y, S1);
          S2 = fmaf(w, q.z, S2);
          Wsum += w;
        }
      }
    }
    // ---- loop B: strip hit counts by Q's class (R18), in (major, minor) coordinates of the tangent: Eq. 9 is
    // symmetric in x / y and IEEE add / mul commute, so the bits are those of the oracle's x / y order
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
        const bool cG = s_dqG[ci] - lo <= tau2, cA = s_dqA[ci] - lo <= tau2;
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
            const int idc = sg ? ci - off : ci + off;
            const bool cG = s_dqG[idc] - lo <= tau2, cA = s_dqA[idc] - lo <= tau2;
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
            const int idx = ci + s * strM + mm * strN;
            const bool cG = s_dqG[idx] - lo <= tau2, cA = s_dqA[idx] - lo <= tau2;
            Hc += (in && cG) ? 1u : 0u;
            Ha += (in && cA && !cG) ? 1u : 0u;
          }
        }
      }
    }
    const float inv = Wsum > 0.f ? 1.0f / Wsum : 0.f;
    const float alpha = (Hc + Ha) > 0 ? (float)Hc / (float)(Hc + Ha) : 0.f;
    s_item[it] = make_float4(S0 * inv, S1 * inv, S2 * inv, alpha);
  }
  __syncthreads();
  // ---- (4) combine and composite over the background (R29)
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    if (!inside[k]) continue;
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
    } else if (slot_a[k] >= 0) {
      const float4 a = s_item[slot_a[k]];
      r = a.x, g = a.y, b = a.z, alpha = a.w;
    }
    const float ia = 1.f - alpha;
    store_rgba(out, (size_t)(y0 + ly + 8 * k) * W + x0 + lx,
               make_float4(alpha * r + ia * bg[k].x, alpha * g + ia * bg[k].y, alpha * b + ia * bg[k].z, alpha + ia * bg[k].w),
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
                  ShadeParams sp, const unsigned long long* gbuf, float4* colour, cudaStream_t st) {
  size_t n = (size_t)cam.W * cam.H;
  if (sp.paper_payload) {
    k_shade_payload<<<dim3((cam.W + 63) / 64, (cam.H + 3) / 4), 256, 0, st>>>(d_scene, cam, sp, gbuf, colour);
    return;
  }
  k_shade<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_scene, srec, vertices, cam, sp, gbuf, colour);
}

template <int R>
static void launch_filter_r(const SceneDev* d_scene, const uint2* srec, const float4* vertices, CamDev cam,
                            ShadeParams sp, const unsigned long long* gbuf, const float4* colour,
                            const float4* scene_rgb, float4* out, LaunchState* ls, cudaStream_t st) {
  constexpr int NS = (FT_W + 2 * R) * (FT_H + 2 * R);
  constexpr size_t smem = (size_t)NS * (sizeof(float4) + 3 * sizeof(uint32_t)) + 2 * FT_W * FT_H * sizeof(float4);
  if (!ls->filter_set[R]) {  // once per context (the opt-in is per device)
    raise_dyn_smem(k_filter<R>, smem);
    ls->filter_set[R] = true;
  }
  dim3 grid((cam.W + FT_W - 1) / FT_W, (cam.H + FT_H - 1) / FT_H);
  k_filter<R><<<grid, 256, smem, st>>>(d_scene, srec, vertices, cam, sp, gbuf, colour, scene_rgb, out);
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
