// k_lod.cu — H1 LOD / cull and H2 scan (§3.2, Eq. 1-5).
//
// Paper: one thread per bundle writes an indirect-dispatch record. Here: four
// lanes per bundle-instance write {N_LOD, C} into the bundle table (and which of the two raster passes
// draws the bundle), then a tiled scan turns them into {slot_base, vertex_base}, the work-group scans
// of the raster and the device-side totals the later persistent kernels read — CUDA's replacement for
// the indirect dispatch: grid sizes never wait for a device result.
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

__device__ __forceinline__ uint32_t raster_groups(uint32_t n_v) {  // units of RAS_GROUP*RAS_CHUNK segment starts
  return n_v >= 2 ? (n_v - 1 + RAS_GROUP * RAS_CHUNK - 1) / (RAS_GROUP * RAS_CHUNK) : 0u;
}

// Depth order of the raster (k_raster.cu): every bundle-instance also reports its nearest cage depth; the range of
// those depths per instance is accumulated for the NEXT frame (zr_cur) and the range of the PREVIOUS frame (zr_prev)
// decides which of the two raster passes draws the bundle: the front HIZ_CUT of the range first. Order is a
// heuristic only — the resolve is an order-free min — so a stale or empty range (first frame: one pass) is fine.
// Mapping: a CTA of 1024 threads owns a tile of 256 bundle-instances, FOUR lanes per bundle: lane `sub` projects the
// cage layers sub, sub + 4, ... and the quad combines its bounding boxes with two shuffles (min / max are exact, so
// the result does not depend on the split); everything after that is computed by all four, written by lane 0.
__global__ void __launch_bounds__(1024) k_lod(const SceneDev* __restrict__ sc, uint32_t n_bi, CamDev cam,
                                              LambdaArr lam, uint32_t groom_mask, uint4* __restrict__ table,
                                              uint4* __restrict__ part, const uint32_t* __restrict__ zr_prev,
                                              uint32_t* __restrict__ zr_cur, uint32_t two_pass,
                                              unsigned long long* __restrict__ counters) {
  if (blockIdx.x == 0 && threadIdx.x <= 2 * HAIR_MAX_GROOMS)  // Eq. 8 sums restart (k_scan accumulates them)
    counters[CNT_BETA_NUM + threadIdx.x] = threadIdx.x == 2 * HAIR_MAX_GROOMS ? 0x3F800000ull : 0ull;
  const uint32_t sub = threadIdx.x & 3u;
  const uint32_t gid = blockIdx.x * 256u + (threadIdx.x >> 2);
  const bool live = gid < n_bi;
  uint32_t nlod = 0, C = 0, far_pass = 0, gi = 0, rel = 0, N = 0;
  uint32_t inst = 0xFFFFFFFFu;
  float zmin = 3.0e38f, lambda = 0.f;
  float mnx = INFINITY, mny = INFINITY, mxx = -INFINITY, mxy = -INFINITY;
  uint32_t n_valid = 0, n_all = 0;
  // ---- phase 1 (per lane): this lane's layers of the cage
  if (live) {
    for (uint32_t k = 1; k < sc->n_grooms; ++k)
      if (gid >= sc->g[k].gid_base) gi = k;
    const GroomDev& g = sc->g[gi];
    rel = gid - g.gid_base;
    const uint32_t q = rel / g.T, t = rel - q * g.T;
    N = __ldg(&g.npt[t]);
    lambda = lam.v[gi];
    inst = g.inst_base + q;
    const bool lod_on = lambda > 0.f;  // R14: else LOD and culling off, only the ordering key is needed
    float M[12];
    const bool has_m = g.xform != nullptr;
    if (has_m)
      for (int a = 0; a < 12; ++a) M[a] = __ldg(&g.xform[q * 12 + a]);
    const uint32_t v[3] = {__ldg(&g.idx[t * 3]), __ldg(&g.idx[t * 3 + 1]), __ldg(&g.idx[t * 3 + 2])};
    // LOD off: root and tip layer (lanes 0 and 1 of the quad) are enough for an ordering key
    const uint32_t i_begin = lod_on ? sub : (sub == 0 ? 0u : sub == 1 ? g.Lv - 1 : g.Lv), i_step = lod_on ? 4u : g.Lv;
    for (uint32_t i = i_begin; i < g.Lv; i += i_step)
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
        zmin = fminf(zmin, p.zv);
        ++n_all;
        if (p.valid) {
          ++n_valid;
          mnx = fminf(mnx, p.sx);
          mxx = fmaxf(mxx, p.sx);
          mny = fminf(mny, p.sy);
          mxy = fmaxf(mxy, p.sy);
        }
      }
  }
  // ---- phase 2 (converged): the quad's four partial boxes
#pragma unroll
  for (int d = 1; d <= 2; d <<= 1) {
    mnx = fminf(mnx, __shfl_xor_sync(0xffffffffu, mnx, d));
    mny = fminf(mny, __shfl_xor_sync(0xffffffffu, mny, d));
    mxx = fmaxf(mxx, __shfl_xor_sync(0xffffffffu, mxx, d));
    mxy = fmaxf(mxy, __shfl_xor_sync(0xffffffffu, mxy, d));
    zmin = fminf(zmin, __shfl_xor_sync(0xffffffffu, zmin, d));
    n_valid += __shfl_xor_sync(0xffffffffu, n_valid, d);
    n_all += __shfl_xor_sync(0xffffffffu, n_all, d);
  }
  // ---- phase 3 (all four lanes alike, lane 0 writes): Eq. 1-5
  if (live) {
    const GroomDev& g = sc->g[gi];
    if (!(lambda > 0.f)) {  // R14
      nlod = N;
      C = g.c_full;
    } else {
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
      if (!culled) {
        float delta = (float)(pcg(pcg(g.seed_h + rel) + 0xB0u) >> 8) * (1.0f / 16777216.0f);
        lod_counts(L, N, delta, g.Lv, g.c_full, nlod, C);
        if (nlod == 0) C = 0;
      }
    }
    if (!((groom_mask >> gi) & 1u)) nlod = C = 0;  // R-seq: this groom is not drawn in this pass
    if (two_pass) {
      const float z0 = __uint_as_float(__ldg(&zr_prev[inst * 2])), z1 = __uint_as_float(__ldg(&zr_prev[inst * 2 + 1]));
      far_pass = (z1 > z0 && zmin > z0 + HIZ_CUT * (z1 - z0)) ? 1u : 0u;
    }
    if (sub == 0) table[gid] = make_uint4(nlod, C, far_pass, 0u);  // .z: the pass, until k_scan replaces it by the slot base
  }
  {  // depth range per instance for the next frame: positive floats order like their bits
    const uint32_t i0 = __shfl_sync(0xffffffffu, inst, 0);
    const float zc = fmaxf(zmin, 0.f);
    if (__all_sync(0xffffffffu, inst == i0)) {
      float lo = zc, hi = zc;
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) {
        lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, d));
        hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, d));
      }
      if ((threadIdx.x & 31) == 0 && i0 != 0xFFFFFFFFu) {
        atomicMin(&zr_cur[i0 * 2], __float_as_uint(lo));
        atomicMax(&zr_cur[i0 * 2 + 1], __float_as_uint(hi));
      }
    } else if (inst != 0xFFFFFFFFu) {
      atomicMin(&zr_cur[inst * 2], __float_as_uint(zc));
      atomicMax(&zr_cur[inst * 2 + 1], __float_as_uint(zc));
    }
  }
  // sums of this tile of 256 bundle-instances for the scan: strands, vertices, raster work groups, culled
  // part[2 tile] = {strands, vertices, work groups of the near pass, of the far pass}, part[2 tile + 1].x = culled
  if (sub != 0) nlod = C = 0;  // one lane of the quad counts
  const uint32_t ng = raster_groups(nlod * C);
  uint32_t ts = nlod, tv = nlod * C, tg = far_pass ? 0u : ng, tf = far_pass ? ng : 0u,
           tc = (gid < n_bi && nlod == 0 && sub == 0) ? 1u : 0u;
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    ts += __shfl_xor_sync(0xffffffffu, ts, d);
    tv += __shfl_xor_sync(0xffffffffu, tv, d);
    tg += __shfl_xor_sync(0xffffffffu, tg, d);
    tf += __shfl_xor_sync(0xffffffffu, tf, d);
    tc += __shfl_xor_sync(0xffffffffu, tc, d);
  }
  __shared__ uint4 s_w[32];
  __shared__ uint32_t s_c[32];
  if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = make_uint4(ts, tv, tg, tf), s_c[threadIdx.x >> 5] = tc;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint4 a = s_w[0];
    uint32_t cc = s_c[0];
    for (int wv = 1; wv < 32; ++wv) a.x += s_w[wv].x, a.y += s_w[wv].y, a.z += s_w[wv].z, a.w += s_w[wv].w, cc += s_c[wv];
    part[blockIdx.x * 2] = a;
    part[blockIdx.x * 2 + 1] = make_uint4(cc, 0u, 0u, 0u);
  }
}

// Exclusive scans of N_LOD, N_LOD*C and the raster's work-group count over bundle-instances in
// index order (O1 step 6). One CTA of 256 threads per tile of 256 bundle-instances: (1) every CTA sums
// the tile totals k_lod left in `part` for the tiles in front of its own (and the frame's vertex total), (2) a
// shuffle scan per warp plus the 8 warp totals gives the exclusive scan inside the tile, (3) the last tile writes the
// device-side totals and queue lengths. Coalesced 16-byte accesses throughout.

__global__ void __launch_bounds__(256) k_scan(const SceneDev* __restrict__ sc, uint4* __restrict__ table,
                                              uint32_t* __restrict__ grp, uint32_t n_bi,
                                              const uint4* __restrict__ part, unsigned long long* __restrict__ counters,
                                              uint32_t* __restrict__ zr_reset, uint32_t n_inst, uint32_t two_pass,
                                              uint32_t* __restrict__ want_two_pass) {
  __shared__ uint32_t s_a[8][5], s_b[8][4], s_tot[8];
  __shared__ uint32_t s_beta[2 * HAIR_MAX_GROOMS + 1];  // per groom: strands kept, strands in total; min ratio (float bits)
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tile = blockIdx.x;
  if (threadIdx.x <= 2 * HAIR_MAX_GROOMS) s_beta[threadIdx.x] = threadIdx.x == 2 * HAIR_MAX_GROOMS ? 0x3F800000u : 0u;
  uint32_t* grp1 = grp + n_bi + 1;
  // (1) what lies before this tile: sums of the tiles in front of it; and the frame's total of vertices
  uint32_t ps = 0, pv = 0, pg = 0, pf = 0, pc = 0, tot = 0;
  for (uint32_t t = threadIdx.x; t < gridDim.x; t += 256) {
    const uint4 a = __ldg(&part[2 * t]);
    tot += a.y;
    if (t < tile) ps += a.x, pv += a.y, pg += a.z, pf += a.w, pc += __ldg(&part[2 * t + 1]).x;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    ps += __shfl_xor_sync(0xffffffffu, ps, d);
    pv += __shfl_xor_sync(0xffffffffu, pv, d);
    pg += __shfl_xor_sync(0xffffffffu, pg, d);
    pf += __shfl_xor_sync(0xffffffffu, pf, d);
    pc += __shfl_xor_sync(0xffffffffu, pc, d);
    tot += __shfl_xor_sync(0xffffffffu, tot, d);
  }
  if (lane == 0) s_tot[warp] = tot;
  __syncthreads();
  tot = 0;
#pragma unroll
  for (uint32_t wv = 0; wv < 8; ++wv) tot += s_tot[wv];
  // small frames are drawn in one pass: the hi-Z between the passes would cost more than it saves
  // (the host launches the second pass only when the frame before wanted it: want_two_pass is host-mapped memory)
  const bool want = tot >= HIZ_MIN_VERTS;
  const bool two = two_pass != 0u && want;
  // (2) exclusive scan inside the tile: shuffle scan per warp, then the 8 warp totals
  const uint32_t i = tile * 256 + threadIdx.x;
  uint4 e = i < n_bi ? table[i] : make_uint4(0, 0, 0, 0);
  const uint32_t s = e.x, v = e.x * e.y, ng = raster_groups(v);
  // Eq. 8: beta = N_remaining / N_total of each groom over its drawn bundle-instances
  if (s) {
    uint32_t gi = 0;
    for (uint32_t k = 1; k < sc->n_grooms; ++k)
      if (i >= sc->g[k].gid_base) gi = k;
    const GroomDev& gr = sc->g[gi];
    const uint32_t N = __ldg(&gr.npt[(i - gr.gid_base) % gr.T]);
    atomicAdd(&s_beta[gi], s);
    atomicAdd(&s_beta[HAIR_MAX_GROOMS + gi], N);
    atomicMin(&s_beta[2 * HAIR_MAX_GROOMS], __float_as_uint(__fdiv_rn((float)s, (float)N)));  // positive floats order like their bits
  }
  const bool far_pass = two && e.z != 0u;
  const uint32_t g = far_pass ? 0u : ng, f = far_pass ? ng : 0u;
  uint32_t is = s, iv = v, ig = g, jf = f;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t a = __shfl_up_sync(0xffffffffu, is, d), b = __shfl_up_sync(0xffffffffu, iv, d),
             c = __shfl_up_sync(0xffffffffu, ig, d), c1 = __shfl_up_sync(0xffffffffu, jf, d);
    if (lane >= d) {
      is += a;
      iv += b;
      ig += c;
      jf += c1;
    }
  }
  if (!two) pg += pf, pf = 0;  // the tiles in front counted their far bundles apart
  if (lane == 0) s_a[warp][0] = ps, s_a[warp][1] = pv, s_a[warp][2] = pg, s_a[warp][3] = pc, s_a[warp][4] = pf;
  if (lane == 31) s_b[warp][0] = is, s_b[warp][1] = iv, s_b[warp][2] = ig, s_b[warp][3] = jf;
  __syncthreads();
  uint32_t off_s = 0, off_v = 0, off_g = 0, off_f = 0, culled = 0;
#pragma unroll
  for (uint32_t wv = 0; wv < 8; ++wv) {
    off_s += s_a[wv][0], off_v += s_a[wv][1], off_g += s_a[wv][2], culled += s_a[wv][3], off_f += s_a[wv][4];
    if (wv < warp) off_s += s_b[wv][0], off_v += s_b[wv][1], off_g += s_b[wv][2], off_f += s_b[wv][3];
  }
  if (i < n_bi) {
    e.z = off_s + is - s;
    e.w = off_v + iv - v;
    table[i] = e;
    grp[i] = off_g + ig - g;
    grp1[i] = off_f + jf - f;
  }
  // (s_beta is complete: the __syncthreads above follows every thread's atomics)
  if (threadIdx.x < 2 * HAIR_MAX_GROOMS) {
    if (s_beta[threadIdx.x]) atomicAdd(&counters[CNT_BETA_NUM + threadIdx.x], (unsigned long long)s_beta[threadIdx.x]);
  } else if (threadIdx.x == 2 * HAIR_MAX_GROOMS)
    atomicMin(&counters[CNT_BETA_MIN], (unsigned long long)s_beta[2 * HAIR_MAX_GROOMS]);
  // the depth ranges the previous frame left (k_lod has read them) restart for the frame after this one
  if (tile == 0)
    for (uint32_t k = threadIdx.x; k < n_inst; k += 256) zr_reset[2 * k] = 0x7F000000u, zr_reset[2 * k + 1] = 0u;
  // (3) the last tile knows the totals: device-side counts and queue lengths of the frame
  if (tile == gridDim.x - 1 && threadIdx.x == 255) {
    const uint32_t mine_c = __ldg(&part[2 * tile + 1]).x;
    const uint32_t n_s = off_s + is, n_v = off_v + iv, n_g = off_g + ig, n_f = off_f + jf;
    counters[CNT_STRANDS] = n_s;
    counters[CNT_VERTICES] = n_v;
    counters[CNT_SEGMENTS] = n_v - n_s;  // sum N_LOD*(C-1)
    counters[CNT_CULLED] = culled + mine_c;
    counters[CNT_WORK_GEN] = 0;
    counters[CNT_WORK_RASTER] = 0;
    for (int k = CNT_SEG_DRAWN; k < CNT_RESET_END; ++k) counters[k] = 0;
    counters[CNT_HIZ_ON] = (two && n_f > 0) ? 1ull : 0ull;
    grp[n_bi] = n_g;  // total work groups of each pass: the raster's queue lengths
    grp1[n_bi] = n_f;
    *want_two_pass = want ? 1u : 0u;
  }
}

void launch_lod_scan(const SceneDev* d_scene, uint32_t n_bi, CamDev cam, LambdaArr lam, uint32_t groom_mask,
                     uint4* table, uint32_t* grp, uint4* part, unsigned long long* counters, uint32_t* zrange,
                     uint32_t n_inst, uint32_t parity, bool two_pass, uint32_t* want_two_pass, cudaStream_t st) {
  // part: two uint4 per tile of 256 bundle-instances (sums), written by k_lod, read by k_scan
  const uint32_t n_tiles = (n_bi + 255) / 256;
  uint32_t* zr_cur = zrange + (size_t)(parity & 1u) * n_inst * 2;
  uint32_t* zr_prev = zrange + (size_t)((parity + 1u) & 1u) * n_inst * 2;
  k_lod<<<n_tiles, 1024, 0, st>>>(d_scene, n_bi, cam, lam, groom_mask, table, part, zr_prev, zr_cur, two_pass ? 1u : 0u, counters);
  k_scan<<<n_tiles, 256, 0, st>>>(d_scene, table, grp, n_bi, part, counters, zr_prev, n_inst, two_pass ? 1u : 0u, want_two_pass);
}

// hair_mesh_update: every queued copy job in one launch (hair_api.cu flush_updates) — by default the device-to-device
// apply of the staged cages; with HAIR_STAGE_DMA=0 also the pull of the pinned host arrays over the bus. blockIdx.y = job
__global__ void __launch_bounds__(256) k_copy_jobs(CopyJobs jobs) {
  const CopyJob j = jobs.j[blockIdx.y];
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < j.n; i += (size_t)gridDim.x * blockDim.x) j.dst[i] = j.src[i];
}

void launch_copy_jobs(const CopyJobs& jobs, cudaStream_t st) {
  if (jobs.n > 0) k_copy_jobs<<<dim3(32, (unsigned)jobs.n), 256, 0, st>>>(jobs);
}
