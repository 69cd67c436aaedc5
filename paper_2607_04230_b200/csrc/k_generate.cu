// k_generate.cu — H3 strand generation (Code 1 PAPER.md:353-443).
//
// Paper (prior art): one 32-lane workgroup per strand; pass 1 puts the strand's layer data in shared
// memory with neighbour exchange by subgroup shuffles, pass 2 evaluates the styled control points.
// Here (B200): one WARP per BUNDLE-INSTANCE, fetched dynamically by persistent warps.
//   stage 1  lanes = cage layers: load the prism's three edge polylines, Catmull-Rom tangents by
//            __shfl_up/down of the neighbours' points (the paper's pass 1, registers only).
//   stage 2  lanes = control points j: pull layers i(j), i(j)+1 out of the owning lanes with indexed
//            shuffles and evaluate, ONCE PER BUNDLE, the three edge splines E_k(j), their derivatives,
//            the centre curve, the frame edge and every w-dependent styling scalar into a shared
//            per-warp table. The base spline is linear in the root barycentrics
//            (p(b) = sum_k b_k E_k), so no strand ever repeats the Hermite evaluation.
//   stage 3  per strand once (lanes = strands, batches of 32): 3 hashes -> root barycentrics and curl
//            phase, to shared memory. Then a warp iteration covers 4 strands x 8 consecutive control points (fewer
//            strands at a time for small bundles): the four lanes of a control point read the same table row (one
//            shared-memory wavefront per LDS.128), the three-row barycentric blends are packed fp32 (FFMA2), then
//            frame, styling, instance transform, and one 16-byte store per lane (each strand's run of the iteration
//            is 128 contiguous bytes); (strand group, j) advance incrementally, no division per vertex.
// Arithmetic: fp32 with FMA; parity gate = 1e-5 max-abs against the fp64 oracle.
#include "gen_device.cuh"

#define GEN_WARPS 8
#ifndef GEN_MIN_BLOCKS
#define GEN_MIN_BLOCKS 3  // CTAs per SM the register budget is held to
#endif

// (the arithmetic itself lives in gen_device.cuh: gen::build_table, gen::strand_setup, gen::vertex)
__global__ void __launch_bounds__(GEN_WARPS * 32, GEN_MIN_BLOCKS)
k_generate(const SceneDev* __restrict__ sc, uint32_t n_bi, const uint4* __restrict__ table,
           float4* __restrict__ vertices, uint2* __restrict__ strand_rec, unsigned long long* __restrict__ counters,
           uint32_t c_max) {
  extern __shared__ float4 smem4[];
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  // per warp: the bundle table [c_max][HAIR_ROW], then 32 strand records (b1, b2, cos/sin curl phase) + 32 hashes
  const size_t warp_floats = (size_t)c_max * HAIR_ROW + 32 * 5;
  float* tab = reinterpret_cast<float*>(smem4) + (size_t)warp * warp_floats;
  float4* srec = reinterpret_cast<float4*>(tab + (size_t)c_max * HAIR_ROW);
  uint32_t* sbase = reinterpret_cast<uint32_t*>(srec + 32);

  for (;;) {
    // dynamic work fetch: one bundle-instance per warp (the paper's indirect dispatch, device-side)
    uint32_t gid = 0;
    if (lane == 0) gid = (uint32_t)atomicAdd(&counters[CNT_WORK_GEN], 1ull);
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
    const uint32_t ops = g.op_mask;

    // ---- stages 1 + 2: the per-bundle table
    gen::build_table(g, t, C, tab, lane);
    // ---- stage 3: lanes = flattened (strand, control point). One coalesced float4 store each.
    float M[12];
    const bool has_m = g.xform != nullptr;
    if (has_m)
#pragma unroll
      for (int a = 0; a < 12; ++a) M[a] = __ldg(&g.xform[q * 12 + a]);
    const uint32_t off_t = __ldg(&g.off[t]);
    // A warp iteration covers SB strands x (32 / SB) consecutive control points: the lanes of one control point read
    // the same table row (one shared-memory wavefront per LDS.128 for SB = 4 instead of four when every lane has a row
    // of its own), each strand's run is 32 / SB consecutive vertices (128 contiguous bytes for SB = 4). Control points
    // are counted through the groups of SB strands of a batch without a break, so only the batch's last iteration has
    // idle lanes; small bundles take fewer strands at a time.
    const uint32_t sb_log = nlod >= 6 ? 2u : (nlod >= 2 ? 1u : 0u), SB = 1u << sb_log, TB = 32u >> sb_log;
    const uint32_t s_lane = lane & (SB - 1u), t_lane = lane >> sb_log;
    const uint32_t qT = TB / C, rT = TB - qT * C;  // (group, j) of a lane advance by TB control points per iteration
    for (uint32_t k0 = 0; k0 < nlod; k0 += 32) {
      // per strand, once (lanes = strands of this batch): root barycentrics (R6) and the curl phase
      const uint32_t nk = min(32u, nlod - k0);
      if (lane < nk) {
        const gen::Strand s = gen::strand_setup(g, off_t + k0 + lane);
        srec[lane] = make_float4(s.b1, s.b2, s.cphi, s.sphi);
        sbase[lane] = s.base;
        // where shading finds this strand (hair_internal.cuh locate_strand)
        strand_rec[g.sid_base + q * g.N + off_t + k0 + lane] = make_uint2(e.w + (k0 + lane) * C, C | (gi << 8));
      }
      __syncwarp();
      const uint32_t n_t = ((nk + SB - 1u) >> sb_log) * C;  // control points over all groups of the batch
      float4* out = vertices + e.w + (size_t)k0 * C;
      uint32_t gq = t_lane / C, j = t_lane - gq * C;
      for (uint32_t t0 = 0; t0 < n_t; t0 += TB) {
        const uint32_t k = (gq << sb_log) + s_lane;
        if (t0 + t_lane < n_t && k < nk) {
          const float4 sr = srec[k];
          out[k * C + j] = gen::vertex(tab, j, sr.x, sr.y, sr.z, sr.w, sbase[k], ops, has_m ? M : nullptr);
        }
        gq += qT;
        j += rT;
        if (j >= C) {
          j -= C;
          ++gq;
        }
      }
      __syncwarp();
    }
    __syncwarp();
  }
}

void launch_generate(const SceneDev* d_scene, uint32_t n_bi, const uint4* table, float4* vertices, uint2* srec,
                     unsigned long long* counters, uint32_t c_max, int n_sm, LaunchState* ls, cudaStream_t st) {
  size_t smem = (size_t)GEN_WARPS * ((size_t)c_max * HAIR_ROW + 32 * 5) * sizeof(float);
  if (!ls->gen_per_sm || smem != ls->gen_smem) {  // once per context and table size (the opt-in is per device)
    raise_dyn_smem(k_generate, smem);
    int b = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k_generate, GEN_WARPS * 32, smem);
    ls->gen_per_sm = b > 0 ? b : 1;
    ls->gen_smem = smem;
  }
  const int per_sm = ls->gen_per_sm;
  uint32_t grid = (uint32_t)(n_sm * per_sm);
  uint32_t need = (n_bi + GEN_WARPS - 1) / GEN_WARPS;
  if (grid > need) grid = need;
  k_generate<<<grid, GEN_WARPS * 32, smem, st>>>(d_scene, n_bi, table, vertices, srec, counters, c_max);
}
