// k_raster.cu — H4 clear + segment raster (§3.1.2).
//
// Each styled segment is tested against the two coverage predicates of DESIGN.md R9-R11 and every
// hit is resolved with a 64-bit atomic min on depth|strand|segment|t into the
// interleaved two-layer G-buffer ([pixel][0] centre sample, [pixel][1] conservative).
// The predicates and the word are evaluated in the fixed-order fp32 of hair_internal.cuh, so the
// result is bit-identical to the CPU oracle's brute force whatever the enumeration order.
//
// Work distribution: persistent warps fetch one bundle-instance at a time (device-side counter) and
// walk its strand-major vertex run 31 segments per step: lane l loads + projects vertex v0+l once
// (coalesced 16-byte loads) and receives vertex v0+l+1 from lane l+1 by shuffle.
#include "hair_internal.cuh"

#define RAS_WARPS 8

struct Seg {
  float ax, ay, az, bx, by, bz;  // screen endpoints and post-projection depths
  float rho2;
  uint32_t sid, j;
};

// One pixel of one segment: DESIGN.md R10/R11 in fixed-order fp32. Returns 0, 1 (conservative only)
// or 3 (centre + conservative), and the packed word.
__device__ __forceinline__ int cover_pixel(const Seg& s, float dx, float dy, float dd, float ext, float dz,
                                           int x, int y, unsigned long long& word) {
  const float cx = (float)x + 0.5f, cy = (float)y + 0.5f;
  const float ux = xsub(cx, s.ax), uy = xsub(cy, s.ay);
  const float cr = fabsf(xsub(xmul(dx, uy), xmul(dy, ux)));
  if (!(cr <= ext)) return 0;
  float t = 0.f;
  if (dd > 0.f) t = fminf(fmaxf(xdiv(xadd(xmul(ux, dx), xmul(uy, dy)), dd), 0.f), 1.f);
  const float zn = xadd(s.az, xmul(t, dz));
  if (zn < 0.f || zn > 1.f) return 0;
  word = pack_word(zn, s.sid, s.j, t);
  const float ex = xsub(cx, xadd(s.ax, xmul(t, dx))), ey = xsub(cy, xadd(s.ay, xmul(t, dy)));
  const float d2 = xadd(xmul(ex, ex), xmul(ey, ey));
  return d2 <= s.rho2 ? 3 : 1;
}

// read-before-atomic ("reads the existing depth buffer"): words only ever decrease, so
// a stale read can only under-filter, never drop a winner.
template <bool COUNT>
__device__ __forceinline__ void resolve(unsigned long long* p, unsigned long long word, uint32_t& issued) {
  if (word < __ldcg(p)) {
    atomicMin(p, word);
    if (COUNT) ++issued;
  }
}

template <bool COUNT>
__global__ void __launch_bounds__(RAS_WARPS * 32)
k_raster(const SceneDev* __restrict__ sc, uint32_t n_bi, const uint4* __restrict__ table,
         const float4* __restrict__ vertices, CamDev cam, float rho_default, unsigned long long* __restrict__ gbuf,
         unsigned long long* __restrict__ counters) {
  const uint32_t lane = threadIdx.x & 31;
  uint32_t c_center = 0, c_cons = 0, c_drawn = 0, c_issued = 0;
  const float Wm1 = (float)(cam.W - 1), Hm1 = (float)(cam.H - 1);
  for (;;) {
    uint32_t gid = 0;
    if (lane == 0) gid = (uint32_t)atomicAdd(&counters[CNT_WORK_RASTER], 1ull);
    gid = __shfl_sync(0xffffffffu, gid, 0);
    if (gid >= n_bi) break;
    const uint4 e = __ldg(&table[gid]);
    const uint32_t nlod = e.x, C = e.y;
    if (nlod == 0) continue;
    uint32_t gi = 0;
    for (uint32_t k = 1; k < sc->n_grooms; ++k)
      if (gid >= sc->g[k].gid_base) gi = k;
    const GroomDev& g = sc->g[gi];
    const uint32_t rel = gid - g.gid_base;
    const uint32_t q = rel / g.T, t = rel - q * g.T;
    const uint32_t sid0 = g.sid_base + q * g.N + __ldg(&g.off[t]);
    const float width = g.width_world;
    const uint32_t n_v = nlod * C;
    const float4* vin = vertices + e.w;
    for (uint32_t v0 = 0; v0 + 1 < n_v; v0 += 31) {
      const uint32_t v = v0 + lane;
      Proj a;
      a.valid = false;
      a.sx = a.sy = a.zn = a.zv = 0.f;
      if (v < n_v) {
        const float4 p = __ldg(&vin[v]);
        a = project_exact(cam, p.x, p.y, p.z);
      }
      Proj b;
      b.sx = __shfl_down_sync(0xffffffffu, a.sx, 1);
      b.sy = __shfl_down_sync(0xffffffffu, a.sy, 1);
      b.zn = __shfl_down_sync(0xffffffffu, a.zn, 1);
      b.zv = __shfl_down_sync(0xffffffffu, a.zv, 1);
      b.valid = __shfl_down_sync(0xffffffffu, (int)a.valid, 1) != 0;
      const uint32_t k = v / C, j = v - k * C;
      const bool seg = lane < 31 && v + 1 < n_v && j + 1 < C && a.valid && b.valid;  // R12
      if (!seg) continue;
      if (COUNT) ++c_drawn;
      Seg s;
      s.ax = a.sx, s.ay = a.sy, s.az = a.zn, s.bx = b.sx, s.by = b.sy, s.bz = b.zn;
      s.sid = sid0 + k;
      s.j = j;
      float rho = rho_default;
      if (width > 0.f) {  // R9
        const float zm = xmul(0.5f, xadd(a.zv, b.zv));
        const float wpx = fminf(fmaxf(xdiv(xmul(width, cam.fpx), zm), 0.25f), 1.0f);
        rho = xmul(0.5f, wpx);
      }
      s.rho2 = xmul(rho, rho);
      const float dx = xsub(s.bx, s.ax), dy = xsub(s.by, s.ay);
      const float dd = xadd(xmul(dx, dx), xmul(dy, dy));
      const float ext = xmul(0.5f, xadd(fabsf(dx), fabsf(dy)));
      const float dz = xsub(s.bz, s.az);
      // candidate pixels = exactly those whose closed square overlaps the segment's AABB (R10)
      const float fx0 = fmaxf(ceilf(fminf(s.ax, s.bx)) - 1.f, 0.f), fx1 = fminf(floorf(fmaxf(s.ax, s.bx)), Wm1);
      const float fy0 = fmaxf(ceilf(fminf(s.ay, s.by)) - 1.f, 0.f), fy1 = fminf(floorf(fmaxf(s.ay, s.by)), Hm1);
      if (!(fx0 <= fx1) || !(fy0 <= fy1)) continue;
      const int x0 = (int)fx0, x1 = (int)fx1, y0 = (int)fy0, y1 = (int)fy1;
      for (int y = y0; y <= y1; ++y)
        for (int x = x0; x <= x1; ++x) {
          unsigned long long word;
          const int c = cover_pixel(s, dx, dy, dd, ext, dz, x, y, word);
          if (!c) continue;
          unsigned long long* px = gbuf + ((size_t)y * cam.W + x) * 2;
          if (COUNT) ++c_cons;
          resolve<COUNT>(px + 1, word, c_issued);
          if (c & 2) {
            if (COUNT) ++c_center;
            resolve<COUNT>(px, word, c_issued);
          }
        }
    }
  }
  if (COUNT) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
      c_center += __shfl_xor_sync(0xffffffffu, c_center, d);
      c_cons += __shfl_xor_sync(0xffffffffu, c_cons, d);
      c_drawn += __shfl_xor_sync(0xffffffffu, c_drawn, d);
      c_issued += __shfl_xor_sync(0xffffffffu, c_issued, d);
    }
    if (lane == 0) {
      atomicAdd(&counters[CNT_AT_CENTER], (unsigned long long)c_center);
      atomicAdd(&counters[CNT_AT_CONS], (unsigned long long)c_cons);
      atomicAdd(&counters[CNT_SEG_DRAWN], (unsigned long long)c_drawn);
      atomicAdd(&counters[CNT_AT_ISSUED], (unsigned long long)c_issued);
    }
  }
}

// clear both layers to "empty" (all ones): 16 B per pixel, streaming stores
__global__ void __launch_bounds__(256) k_clear(uint4* __restrict__ g, size_t n16) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const uint4 ones = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) g[i] = ones;
}

void launch_clear(unsigned long long* gbuf, size_t n_pixels, cudaStream_t st) {
  size_t blocks = (n_pixels + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  k_clear<<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<uint4*>(gbuf), n_pixels);
}

void launch_raster(const SceneDev* d_scene, uint32_t n_bi, const uint4* table, const float4* vertices,
                   CamDev cam, float rho_default, unsigned long long* gbuf, unsigned long long* counters,
                   bool count, int n_sm, cudaStream_t st) {
  uint32_t grid = (uint32_t)n_sm * 4;
  uint32_t need = (n_bi + RAS_WARPS - 1) / RAS_WARPS;
  if (grid > need) grid = need;
  if (count) k_raster<true><<<grid, RAS_WARPS * 32, 0, st>>>(d_scene, n_bi, table, vertices, cam, rho_default, gbuf, counters);
  else k_raster<false><<<grid, RAS_WARPS * 32, 0, st>>>(d_scene, n_bi, table, vertices, cam, rho_default, gbuf, counters);
}

// ------------------------------------------------------------------ L2-atomic roofline micro-kernels
// 64-bit atomicMin with the result unused (RED.E.MIN.64), the raster's own operation.
__global__ void __launch_bounds__(256) k_atomic_bench(int mode, unsigned long long* __restrict__ words,
                                                      unsigned long long n_words, unsigned long long n_ops,
                                                      uint32_t hot) {
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_ops; i += stride) {
    unsigned long long idx;
    if (mode == 0) idx = i % n_words;                                   // own word, coalesced
    else {
      uint32_t h = pcg((uint32_t)i ^ pcg((uint32_t)(i >> 32) + 0x9E3779B9u));
      unsigned long long r = ((unsigned long long)h << 32) | pcg(h + 1u);
      idx = mode == 1 ? r % n_words : (unsigned long long)(h % hot) * (n_words / hot);  // random / hot set
    }
    atomicMin(&words[idx], (i << 8) | 1ull);
  }
}

void launch_atomic_microbench(int mode, unsigned long long* words, unsigned long long n_words,
                              unsigned long long n_ops, uint32_t hot, int n_sm, cudaStream_t st) {
  k_atomic_bench<<<n_sm * 8, 256, 0, st>>>(mode, words, n_words, n_ops, hot ? hot : 1u);
}
