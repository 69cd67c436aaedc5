// hair_internal.cuh — device-side structs and arithmetic shared by libhair's kernels.
//
// The fp32 "decision" arithmetic of DESIGN.md §3 (projection R-proj, coverage R10, word R7/R8,
// LOD Eq. 1-5, screen tangent R22, strip test Eq. 9) is written with __f*_rn intrinsics: one IEEE
// rounding per operation, never contracted into FMA, whatever the compiler flags. Everything else
// (generation, shading, filter weights) is ordinary fp32 with FMA contraction.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/hair.h"

#define HAIR_EMPTY 0xFFFFFFFFFFFFFFFFull
// R-scene: a word whose 40 payload bits are all ones carries no hair hit (its depth is the scene's, or the far end)
#define HAIR_PAYLOAD_NONE 0xFFFFFFFFFFull
#define RAS_CHUNK 31  // segments a raster warp draws at once (32 vertices, neighbour by shuffle)
#ifndef RAS_GROUP
#define RAS_GROUP 4   // chunks per unit of the raster's device-side work queue
#endif
#ifndef HIZ_TILE
#define HIZ_TILE 16
#endif
// HIZ_TILE: hi-Z tile edge in pixels (k_hiz): a segment's bounding box touches at most 3 x 3 of them
#ifndef HIZ_MIN_VERTS
#define HIZ_MIN_VERTS 3000000u  // frames with fewer vertices after LOD are drawn in one pass
#endif
#ifndef HIZ_CUT
#define HIZ_CUT 0.6f  // bundles whose nearest cage depth lies in the front HIZ_CUT of their instance's range go first
#endif
#define HAIR_ROW 44  // floats per control-point row of the per-bundle table (== 12 mod 32: LDS.128 conflict-free)

struct GroomDev {
  const float* pos;     // [Lv][V][3]
  const float* ao;      // [Lv][V] or nullptr
  const uint32_t* idx;  // [T][3]
  const uint32_t* npt;  // [T]
  const uint32_t* off;  // [T+1] exclusive scan of npt
  const uint32_t* tri_of;  // [N] bundle (root triangle) of each local strand id: the inverse of off
  const float* xform;   // [Q][12] or nullptr
  uint32_t V, Lv, T, Q, N, sid_base, gid_base, c_full;
  uint32_t inst_base;  // index of this groom's first instance among all instances of the scene
  uint32_t spi, seed_h, op_mask, clump_exp, frizz_cells;
  float clump_strength, twist_turns, curl_radius, curl_turns, curl_ramp_w0, frizz_sigma, frizz_ramp_w0;
  float width_world;
  float albedo_root[3], albedo_tip[3], roughness, tilt;
};

struct SceneDev {
  GroomDev g[HAIR_MAX_GROOMS];
  uint32_t n_grooms, n_bi, n_strands_total, pad;
};

struct CamDev {
  float eye[3], r[3], u[3], f[3];
  float near_z, fpx, A, B, half_w, half_h;
  uint32_t W, H;
};

struct LambdaArr {
  float v[HAIR_MAX_GROOMS];
};

struct ShadeParams {
  float light_pos[HAIR_MAX_LIGHTS][3], light_rgb[HAIR_MAX_LIGHTS][3];
  uint32_t n_lights;
  float ambient[3], k_d, k_R, k_TRT, background[3];
  // filter (k_shade_filter.cu): exponents are in base 2
  int r;
  float kP, kQ;        // -log2(e) / sigma_par^2, -log2(e) / sigma_perp^2 (Eq. 10)
  float kC;            // log2(e) / sigma_c^2
  float bias_nc;       // exponent bias of the accumulations without colour term (keeps e^-90 weights normal)
  float strip_hmax;    // (w_strip + 0.01) sqrt(2) + 1e-3: reach of the strip along the tangent's minor axis
  int strip_nc;        // integer minor offsets per major step that can lie within strip_hmax of the line
  float strip_e2_max;  // largest float e2 with sqrt_rn(e2) <= w_strip
  uint32_t tauz_q, taufly_q, filter_on;
  uint32_t bg_alpha;  // R-seq: scene_rgb.w is the alpha accumulated by earlier passes (out.w = a + (1 - a) bg.w)
  float rho_default;  // 0.5 * center_diameter_px
  uint32_t paper_payload;  // R-payload: words carry the paper's payload; pp_groom = the one groom of the pass
  uint32_t pp_groom;
  uint32_t rgb16;  // HAIR_FLAG_RGB16F: the colour output of this pass is half RGBA (8 bytes per pixel)
  uint32_t shadows;  // HAIR_FLAG_SHADOWS and maps exist: lights are scaled by the deep-opacity transmittance
};

// deep opacity maps of the point lights (DESIGN.md R-dom), one per light, in device memory
struct DomLight {
  CamDev cam;
  const uint32_t* z0;  // [res][res] depth of the conservative layer seen from the light, 0xFFFFFFFF = no hair
  const uint4* cnt;    // [res][res] fragments per layer
  uint32_t D[4];       // layer ends in depth steps behind z0
  float alpha_s;
  uint32_t on;
};
struct DomSet {
  DomLight l[HAIR_MAX_LIGHTS];
};

// device counters, one block of 64-bit words (index = enum)
enum {
  CNT_STRANDS = 0,   // sum N_LOD
  CNT_VERTICES,      // sum N_LOD * C
  CNT_SEGMENTS,      // sum N_LOD * (C-1)
  CNT_CULLED,        // bundle-instances with N_LOD == 0
  CNT_WORK_GEN,      // dynamic work counters of the persistent kernels
  CNT_WORK_RASTER,
  CNT_SEG_DRAWN,
  CNT_AT_CENTER,
  CNT_AT_CONS,
  CNT_AT_ISSUED,
  CNT_SEG_LIVE,      // segments that sent at least one atomic (the rest lost every pixel to nearer hair)
  CNT_PX_CENTER,
  CNT_PX_CONS,
  CNT_WORK_RASTER1,  // queue head of the second (far) raster pass
  CNT_HIZ_ON,        // 1: the frame is drawn in two depth-ordered passes with a tile hi-Z between them
  CNT_SEG_HIZ,       // segments dropped by the hi-Z test of the second pass
  CNT_AT_CONS_Y,     // conservative hits of y-major segments (lanes of a warp then sit in different rows)
  CNT_RESET_END,     // k_scan's last tile zeroes [CNT_SEG_DRAWN, CNT_RESET_END) for the kernels behind it
  // Eq. 8: per groom, strands remaining / strands in total over the DRAWN bundle-instances; zeroed by
  // k_lod, accumulated by k_scan (every tile), read by hair_stats
  CNT_BETA_NUM = CNT_RESET_END,
  CNT_BETA_DEN = CNT_BETA_NUM + HAIR_MAX_GROOMS,
  CNT_BETA_MIN = CNT_BETA_DEN + HAIR_MAX_GROOMS,  // float bits of the smallest N_LOD / N of a drawn bundle-instance
  CNT_N
};

// ------------------------------------------------------------------ exact fp32 (one rounding per op)
__device__ __forceinline__ float xmul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float xadd(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float xsub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float xdiv(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ float xsqrt(float a) { return __fsqrt_rn(a); }
__device__ __forceinline__ float xdot3(float ax, float ay, float az, const float* b) {
  return xadd(xadd(xmul(ax, b[0]), xmul(ay, b[1])), xmul(az, b[2]));
}

struct Proj {
  float sx, sy, zn, zv;
  bool valid;
};
// R-proj
__device__ __forceinline__ Proj project_exact(const CamDev& c, float px, float py, float pz) {
  float qx = xsub(px, c.eye[0]), qy = xsub(py, c.eye[1]), qz = xsub(pz, c.eye[2]);
  float xv = xdot3(qx, qy, qz, c.r);
  float yv = xdot3(qx, qy, qz, c.u);
  float zv = xdot3(qx, qy, qz, c.f);
  Proj o;
  o.zv = zv;
  o.valid = zv >= c.near_z;
  float z = o.valid ? zv : 1.0f;
  o.sx = xadd(c.half_w, xdiv(xmul(c.fpx, xv), z));
  o.sy = xsub(c.half_h, xdiv(xmul(c.fpx, yv), z));
  o.zn = xsub(c.A, xdiv(c.B, z));
  return o;
}

// R7/R8 word
__device__ __forceinline__ uint32_t quant_depth(float zn) {
  uint32_t q = (uint32_t)xadd(xmul(zn, 16777215.0f), 0.5f);
  return min(q, 0xFFFFFEu);
}
__device__ __forceinline__ uint32_t quant_t(float t) { return (uint32_t)xadd(xmul(t, 511.0f), 0.5f); }
__device__ __forceinline__ unsigned long long pack_word(float zn, uint32_t sid, uint32_t j, float t) {
  uint32_t hi = (quant_depth(zn) << 8) | (sid >> 16);
  uint32_t lo = (sid << 16) | (j << 9) | quant_t(t);
  return ((unsigned long long)hi << 32) | lo;
}
__device__ __forceinline__ bool w_none(unsigned long long w) { return (w & HAIR_PAYLOAD_NONE) == HAIR_PAYLOAD_NONE; }
__device__ __forceinline__ bool w_none(uint32_t lo, uint32_t hi) { return lo == 0xFFFFFFFFu && (hi & 0xFFu) == 0xFFu; }
__device__ __forceinline__ uint32_t w_dq(unsigned long long w) { return (uint32_t)(w >> 40); }
__device__ __forceinline__ uint32_t w_sid(unsigned long long w) { return (uint32_t)(w >> 16) & 0xFFFFFFu; }
__device__ __forceinline__ uint32_t w_j(unsigned long long w) { return (uint32_t)(w >> 9) & 0x7Fu; }
__device__ __forceinline__ uint32_t w_t9(unsigned long long w) { return (uint32_t)w & 0x1FFu; }

// ------------------------------------------------------------------ the paper's payload (DESIGN.md R-payload)
// [63:40] dq | [39:32] ox8 | [31:24] oy8 | [23:18] u6 | [17:12] v6 | [11:6] w6 | [5:0] ao6. Every
// code is a decision: fp32, one rounding per operation, in the order DESIGN.md states.
struct X3 {
  float x, y, z;
};
__device__ __forceinline__ X3 unit3x(float x, float y, float z) {
  const float dd = xadd(xadd(xmul(x, x), xmul(y, y)), xmul(z, z));
  if (!(dd > 0.f)) return {1.f, 0.f, 0.f};
  const float len = xsqrt(dd);
  return {xdiv(x, len), xdiv(y, len), xdiv(z, len)};
}
// calcTangent on fp32 vertices
__device__ __forceinline__ X3 tangent_x(uint32_t idx, uint32_t count, float4 prev, float4 curr, float4 next) {
  const float4 a = idx + 1 == count ? curr : next;
  const float4 b = idx == 0 ? curr : prev;
  return unit3x(xsub(a.x, b.x), xsub(a.y, b.y), xsub(a.z, b.z));
}
__device__ __forceinline__ uint32_t q8s(float p) {
  return min((uint32_t)xadd(xmul(xadd(xmul(p, 0.5f), 0.5f), 255.f), 0.5f), 255u);
}
__device__ __forceinline__ uint32_t q6(float v) { return min((uint32_t)xadd(xmul(v, 63.f), 0.5f), 63u); }
__device__ __forceinline__ uint32_t uv6(uint32_t a24) { return (a24 * 63u + (1u << 23)) >> 24; }
__device__ __forceinline__ uint32_t oct_encode_x(X3 T) {  // (ox8 << 8) | oy8
  const float s = xadd(xadd(fabsf(T.x), fabsf(T.y)), fabsf(T.z));
  float px = xdiv(T.x, s), py = xdiv(T.y, s);
  if (T.z < 0.f) {
    const float ax = xsub(1.f, fabsf(py)), ay = xsub(1.f, fabsf(px));
    px = px >= 0.f ? ax : -ax;
    py = py >= 0.f ? ay : -ay;
  }
  return (q8s(px) << 8) | q8s(py);
}
__device__ __forceinline__ X3 oct_decode_x(uint32_t ox, uint32_t oy) {
  const float px = xsub(xmul(xdiv((float)ox, 255.f), 2.f), 1.f), py = xsub(xmul(xdiv((float)oy, 255.f), 2.f), 1.f);
  const float z = xsub(xsub(1.f, fabsf(px)), fabsf(py));
  float tx = px, ty = py;
  if (z < 0.f) {
    const float ax = xsub(1.f, fabsf(py)), ay = xsub(1.f, fabsf(px));
    tx = px >= 0.f ? ax : -ax;
    ty = py >= 0.f ? ay : -ay;
  }
  return unit3x(tx, ty, z);
}
__device__ __forceinline__ uint32_t pw_ox(unsigned long long w) { return (uint32_t)(w >> 32) & 0xFFu; }
__device__ __forceinline__ uint32_t pw_oy(unsigned long long w) { return (uint32_t)(w >> 24) & 0xFFu; }

// R26 hash
__device__ __forceinline__ uint32_t pcg(uint32_t v) {
  uint32_t s = v * 747796405u + 2891336453u;
  uint32_t w = ((s >> ((s >> 28) + 4u)) ^ s) * 277803737u;
  return (w >> 22) ^ w;
}

// strand id -> first vertex, control-point count and groom of the strand in this frame's vertex buffer:
// one 8-byte record per strand id, written by k_generate for the strands it generates ({vertex offset,
// C | groom << 8}); one gather instead of the tri_of -> table / off chain when shading and filtering
struct Loc {
  uint32_t voff, C, groom;
};
__device__ __forceinline__ Loc locate_strand(const uint2* __restrict__ srec, uint32_t sid) {
  const uint2 r = __ldg(&srec[sid]);
  Loc l;
  l.voff = r.x;
  l.C = r.y & 0xFFu;
  l.groom = r.y >> 8;
  return l;
}

// The dynamic shared-memory opt-in of a kernel is per device and PROCESS-wide: another context with a smaller table must
// never lower it under a context that needs more (found by test_two_contexts_with_different_table_sizes_in_either_order).
// Ask the driver what is set and only ever raise it.
template <class F>
inline void raise_dyn_smem(F func, size_t bytes) {
  cudaFuncAttributes a;
  if (cudaFuncGetAttributes(&a, func) == cudaSuccess && (size_t)a.maxDynamicSharedSizeBytes >= bytes) return;
  cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// per-context launch state: cudaFuncSetAttribute (dynamic shared memory opt-in) and the occupancy it implies are per
// DEVICE, and a context is bound to one device, so what has been configured lives in hair_ctx — no function statics
struct LaunchState {
  int raster_per_sm[64] = {};      // index = COUNT | MS << 1 | PP << 2 | HZ << 3 | FUSED << 4 | DOM << 5
  size_t raster_smem[64] = {};
  int gen_per_sm = 0;
  size_t gen_smem = 0;
  bool filter_set[8] = {};
};

// ------------------------------------------------------------------ launchers (one per .cu)
// zrange: [2][n_inst][2] u32 (float bits of min / max bundle depth per instance), ping-pong by frame parity;
// grp: two exclusive scans of n_bi + 1 entries (near pass, far pass); two_pass = false draws everything in the first
void launch_lod_scan(const SceneDev* d_scene, uint32_t n_bi, CamDev cam, LambdaArr lam, uint32_t groom_mask,
                     uint4* table, uint32_t* grp, uint4* part, unsigned long long* counters, uint32_t* zrange,
                     uint32_t n_inst, uint32_t parity, bool two_pass, uint32_t* want_two_pass, cudaStream_t st);
void launch_hiz(const unsigned long long* gbuf, uint32_t W, uint32_t H, uint32_t* hiz,
                const unsigned long long* counters, cudaStream_t st);
void launch_generate(const SceneDev* d_scene, uint32_t n_bi, const uint4* table, float4* vertices, uint2* srec,
                     unsigned long long* counters, uint32_t c_max, int n_sm, LaunchState* ls, cudaStream_t st);
void launch_clear(unsigned long long* gbuf, size_t n_pixels, const float* scene_zn, cudaStream_t st);
void launch_reseed(unsigned long long* gbuf, size_t n_pixels, cudaStream_t st);
void launch_raster(const SceneDev* d_scene, uint32_t n_bi, const uint4* table, const uint32_t* grp,
                   const float4* vertices, CamDev cam, float rho_default, unsigned long long* gbuf,
                   unsigned long long* counters, bool count, uint32_t ms_k, bool paper_payload, int pass,
                   const uint32_t* hiz, int n_sm, LaunchState* ls, cudaStream_t st, uint32_t fused_c_max = 0);
// deep opacity map, second step: every conservative hit of the frame's segments under `cam` adds one fragment to the
// layer of its pixel it falls in behind the conservative depth already in gbuf (dom_D: ends of layers 0..2)
void launch_raster_dom(const SceneDev* d_scene, uint32_t n_bi, const uint4* table, const uint32_t* grp,
                       const float4* vertices, CamDev cam, float rho_default, unsigned long long* gbuf,
                       unsigned long long* counters, uint32_t* dom_cnt, uint3 dom_D, int n_sm, LaunchState* ls,
                       cudaStream_t st);
void launch_dom_z0(const unsigned long long* gbuf, size_t n_pixels, uint32_t* z0, cudaStream_t st);
void launch_resolve_msaa(const SceneDev* d_scene, const uint2* srec, const float4* vertices, CamDev cam,
                         ShadeParams sp, const unsigned long long* samples, uint32_t ms_k, const float4* scene_rgb,
                         float4* out, const DomSet* dom, const unsigned long long* counters, cudaStream_t st);
void launch_shade(const SceneDev* d_scene, const uint2* srec, const float4* vertices, CamDev cam,
                  ShadeParams sp, const unsigned long long* gbuf, float4* colour, const DomSet* dom,
                  const unsigned long long* counters, cudaStream_t st);
int launch_filter(const SceneDev* d_scene, const uint2* srec, const float4* vertices, CamDev cam,
                   ShadeParams sp, const unsigned long long* gbuf, const float4* colour, const float4* scene_rgb,
                   float4* out, unsigned long long* counters, bool count, LaunchState* ls, cudaStream_t st);
// hair_mesh_update: a list of copies of 32-bit words done by ONE kernel launch — the staging -> cage apply in front of
// a frame (device to device), and with HAIR_STAGE_DMA=0 also the pinned host -> staging pull over the bus
#define COPY_JOBS_MAX 32
struct CopyJob {
  uint32_t* dst;
  const uint32_t* src;
  size_t n;
};
struct CopyJobs {
  CopyJob j[COPY_JOBS_MAX];
  int n = 0;
};
void launch_copy_jobs(const CopyJobs& jobs, cudaStream_t st);
void launch_atomic_microbench(int mode, unsigned long long* words, unsigned long long n_words,
                              unsigned long long n_ops, uint32_t hot, int n_sm, cudaStream_t st);
// n_steps loads per thread of n_sm * 8 CTAs of 256 threads; sink: one device word nothing is ever written to
void launch_l2_load_microbench(int mode, const unsigned long long* pairs, uint32_t n_pairs, uint32_t pitch,
                               uint32_t n_steps, unsigned long long* sink, int n_sm, cudaStream_t st);
