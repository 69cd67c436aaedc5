// k_lod.cu — H1 LOD / cull and H2 scan (§3.2, Eq. 1-5).
//
// Paper: one thread per bundle writes an indirect-dispatch record. Here: one
// thread per bundle-instance writes {N_LOD, C} into the bundle table, then a single-CTA scan turns
// them into {slot_base, vertex_base} and the device-side totals the later persistent kernels read —
// CUDA's replacement for the indirect dispatch: nothing returns to the host.
#include "hair_internal.cuh"

// Eq. 1, Eq. 4-5; fp32, fixed order (R14).
__device__ __forceinline__ void lod_counts(float L, uint32_t N, float delta, uint32_t Lv, uint32_t c_full,
                                           uint32_t& nlod, uint32_t& C) {
  nlod = 0;
  if (N > 0) {
    float a = xmul(L, xadd((float)N, delta));
    a = fminf(fmaxf(ceilf(a), 1.0f), (float)N);
    nlod = (uint32_t)a;
  }
  uint32_t craw = (uint32_t)floorf(xmul(xsqrt(L), 127.0f));
  craw = max(craw, max(Lv, 3u));
  uint32_t lg = 31u - (uint32_t)__clz((int)(craw - 1u));
  C = min(min((1u << lg) + 1u, 127u), c_full);
}

__global__ void __launch_bounds__(256) k_lod(const SceneDev* __restrict__ sc, uint32_t n_bi, CamDev cam,
                                             LambdaArr lam, uint32_t groom_mask, uint4* __restrict__ table) {
  uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= n_bi) return;
  uint32_t gi = 0;
  for (uint32_t k = 1; k < sc->n_grooms; ++k)
    if (gid >= sc->g[k].gid_base) gi = k;
  const GroomDev& g = sc->g[gi];
  uint32_t rel = gid - g.gid_base;
  uint32_t q = rel / g.T, t = rel - q * g.T;
  uint32_t N = __ldg(&g.npt[t]);
  float lambda = lam.v[gi];
  uint32_t nlod, C;
  if (!(lambda > 0.f)) {  // R14: LOD and culling off
    nlod = N;
    C = g.c_full;
  } else {
    float M[12];
    bool has_m = g.xform != nullptr;
    if (has_m)
      for (int a = 0; a < 12; ++a) M[a] = __ldg(&g.xform[q * 12 + a]);
    uint32_t v[3] = {__ldg(&g.idx[t * 3]), __ldg(&g.idx[t * 3 + 1]), __ldg(&g.idx[t * 3 + 2])};
    float mnx = INFINITY, mny = INFINITY, mxx = -INFINITY, mxy = -INFINITY;
    uint32_t n_valid = 0, n_all = 0;
    for (uint32_t i = 0; i < g.Lv; ++i)
      for (int c = 0; c < 3; ++c) {
        const float* x = g.pos + ((size_t)i * g.V + v[c]) * 3;
        float x0 = __ldg(x), x1 = __ldg(x + 1), x2 = __ldg(x + 2);
        float wx = x0, wy = x1, wz = x2;
        if (has_m) {  // ((m0*x + m1*y) + m2*z) + m3
          wx = xadd(xadd(xadd(xmul(M[0], x0), xmul(M[1], x1)), xmul(M[2], x2)), M[3]);
          wy = xadd(xadd(xadd(xmul(M[4], x0), xmul(M[5], x1)), xmul(M[6], x2)), M[7]);
          wz = xadd(xadd(xadd(xmul(M[8], x0), xmul(M[9], x1)), xmul(M[10], x2)), M[11]);
        }
        Proj p = project_exact(cam, wx, wy, wz);
        ++n_all;
        if (p.valid) {
          ++n_valid;
          mnx = fminf(mnx, p.sx);
          mxx = fmaxf(mxx, p.sx);
          mny = fminf(mny, p.sy);
          mxy = fmaxf(mxy, p.sy);
        }
      }
    bool culled = false;
    float L = 1.f;
    if (n_valid == 0) culled = true;  // R13
    else if (n_valid == n_all) {
      float Wf = (float)cam.W, Hf = (float)cam.H;
      if (mxx < 0.f || mnx > Wf || mxy < 0.f || mny > Hf) culled = true;
      else {
        float dx = xsub(mxx, mnx), dy = xsub(mxy, mny);
        float diag = xsqrt(xadd(xmul(dx, dx), xmul(dy, dy)));
        L = fminf(fmaxf(xmul(xdiv(diag, Hf), lambda), 0.f), 1.f);  // Eq. 2
      }
    }
    if (culled) {
      nlod = 0;
      C = 0;
    } else {
      float delta = (float)(pcg(pcg(g.seed_h + rel) + 0xB0u) >> 8) * (1.0f / 16777216.0f);
      lod_counts(L, N, delta, g.Lv, g.c_full, nlod, C);
      if (nlod == 0) C = 0;
    }
  }
  if (!((groom_mask >> gi) & 1u)) nlod = C = 0;  // R-seq: this groom is not drawn in this pass
  table[gid] = make_uint4(nlod, C, 0u, 0u);
}

// Exclusive scans of N_LOD, N_LOD*C and the raster's work-group count over bundle-instances in
// index order (O1 step 6). One CTA of 1024 threads; each warp owns a contiguous range and
// walks it 32 entries at a time with a shuffle scan and a running carry; the 32 warp totals are
// scanned by warp 0; a second pass adds the warp offsets. Coalesced 16-byte accesses throughout.
__device__ __forceinline__ uint32_t raster_groups(uint32_t n_v) {  // units of RAS_GROUP*RAS_CHUNK segment starts
  return n_v >= 2 ? (n_v - 1 + RAS_GROUP * RAS_CHUNK - 1) / (RAS_GROUP * RAS_CHUNK) : 0u;
}

__global__ void __launch_bounds__(1024) k_scan(uint4* __restrict__ table, uint32_t* __restrict__ grp, uint32_t n_bi,
                                               unsigned long long* __restrict__ counters) {
  __shared__ uint32_t s_slot[32], s_vert[32], s_grp[32], s_cull[32];
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t per_warp = ((n_bi + 31) / 32 + 31) / 32 * 32;  // multiple of 32
  const uint32_t begin = min(warp * per_warp, n_bi), end = min(begin + per_warp, n_bi);
  uint32_t carry_s = 0, carry_v = 0, carry_g = 0, culled = 0;
  for (uint32_t base = begin; base < end; base += 32) {
    uint32_t i = base + lane;
    uint4 e = i < end ? table[i] : make_uint4(0, 0, 0, 0);
    uint32_t s = e.x, v = e.x * e.y, g = raster_groups(v);
    culled += (i < end && e.x == 0) ? 1u : 0u;
    uint32_t is = s, iv = v, ig = g;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      uint32_t a = __shfl_up_sync(0xffffffffu, is, d), b = __shfl_up_sync(0xffffffffu, iv, d),
               c = __shfl_up_sync(0xffffffffu, ig, d);
      if (lane >= d) {
        is += a;
        iv += b;
        ig += c;
      }
    }
    if (i < end) {
      e.z = carry_s + is - s;
      e.w = carry_v + iv - v;
      table[i] = e;
      grp[i] = carry_g + ig - g;
    }
    carry_s += __shfl_sync(0xffffffffu, is, 31);
    carry_v += __shfl_sync(0xffffffffu, iv, 31);
    carry_g += __shfl_sync(0xffffffffu, ig, 31);
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) culled += __shfl_xor_sync(0xffffffffu, culled, d);
  if (lane == 0) {
    s_slot[warp] = carry_s;
    s_vert[warp] = carry_v;
    s_grp[warp] = carry_g;
    s_cull[warp] = culled;
  }
  __syncthreads();
  if (warp == 0) {
    uint32_t s = s_slot[lane], v = s_vert[lane], g = s_grp[lane], c = s_cull[lane];
    uint32_t is = s, iv = v, ig = g;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      uint32_t a = __shfl_up_sync(0xffffffffu, is, d), b = __shfl_up_sync(0xffffffffu, iv, d),
               cc = __shfl_up_sync(0xffffffffu, ig, d);
      if (lane >= d) {
        is += a;
        iv += b;
        ig += cc;
      }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
    s_slot[lane] = is - s;
    s_vert[lane] = iv - v;
    s_grp[lane] = ig - g;
    if (lane == 31) {
      counters[CNT_STRANDS] = is;
      counters[CNT_VERTICES] = iv;
      counters[CNT_SEGMENTS] = iv - is;  // sum N_LOD*(C-1)
      counters[CNT_CULLED] = c;
      counters[CNT_WORK_GEN] = 0;
      counters[CNT_WORK_RASTER] = 0;
      for (int k = CNT_SEG_DRAWN; k < CNT_N; ++k) counters[k] = 0;
      grp[n_bi] = ig;  // total work groups: the raster's queue length
    }
  }
  __syncthreads();
  uint32_t off_s = s_slot[warp], off_v = s_vert[warp], off_g = s_grp[warp];
  if (warp > 0)
    for (uint32_t i = begin + lane; i < end; i += 32) {
      uint4 e = table[i];
      e.z += off_s;
      e.w += off_v;
      table[i] = e;
      grp[i] += off_g;
    }
}

void launch_lod_scan(const SceneDev* d_scene, uint32_t n_bi, CamDev cam, LambdaArr lam, uint32_t groom_mask,
                     uint4* table, uint32_t* grp, unsigned long long* counters, cudaStream_t st) {
  k_lod<<<(n_bi + 255) / 256, 256, 0, st>>>(d_scene, n_bi, cam, lam, groom_mask, table);
  k_scan<<<1, 1024, 0, st>>>(table, grp, n_bi, counters);
}
