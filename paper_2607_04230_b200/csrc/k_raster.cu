// k_raster.cu — H4 clear + segment raster (§3.1.2).
//
// Each styled segment is tested against the two coverage predicates of DESIGN.md R9-R11 and every
// hit is resolved with a 64-bit atomic min on depth|strand|segment|t into the
// interleaved two-layer G-buffer ([pixel][0] centre sample, [pixel][1] conservative).
// The predicates and the word are evaluated in the fixed-order fp32 of hair_internal.cuh, so the
// result is bit-identical to the CPU oracle's brute force whatever the enumeration order.
//
// Paper (prior art): each lane walks its own segment with a DDA; "the DDA rasterization stage
// exhibits workload imbalance when threads draw lines of varying lengths".
// Here: a warp takes 31 consecutive segments of a bundle's strand-major vertex run (lane l loads +
// projects vertex v0+l once with a coalesced 16-byte load and gets vertex v0+l+1 from lane l+1 by
// shuffle), publishes one 64-byte record per segment in shared memory, and then spreads the
// (segment, major-axis column) pairs evenly over its lanes: a shuffle scan of the column counts,
// then per 32 tasks one ballot + one REDUX.OR locate every lane's segment. Each task walks the 1-3
// pixels of its column; long and sub-pixel segments cost the same per pixel.
#include "gen_device.cuh"

#ifndef RAS_WARPS
#define RAS_WARPS 8
#endif
#ifndef RAS_MIN_BLOCKS
#define RAS_MIN_BLOCKS 4  // CTAs per SM the register budget is held to (32 of 64 warps; 64 registers, no spills: 715 vs 720 us at 5)
#endif
#define REC_STRIDE 20  // floats per segment record (18 used); 20 mod 32 keeps LDS.128 conflict-free
#define REC_STRIDE_PP 28  // paper payload: + tangents at both ends (6), AO at both ends (2), (u6, v6) bits, C
#define ENUM_EPS 0.015625f  // slack on the minor-axis range of a column: the enumeration must be a superset
#ifndef ROW_BATCH
#define ROW_BATCH 2
#endif
#ifndef GB_LOAD
#define GB_LOAD __ldcg
#endif
// ROW_BATCH: rows of one column whose G-buffer words are requested before any is used

// read-before-atomic ("reads the existing depth buffer"): words only ever decrease, so
// a stale read can only under-filter, never drop a winner.
//
// Work distribution: the unit a warp fetches from the device-side queue is a GROUP of RAS_GROUP
// chunks of RAS_CHUNK segments inside one bundle-instance (k_scan wrote the exclusive scan of the
// group counts, `grp`); the warp finds the bundle of its group with a 32-ary search (one ballot per
// level). Bundles differ 50x in work (strand count after LOD x pixel length), so bundle-sized units
// left a long tail.
// MSAA-k reference mode (MS = true; DESIGN.md R-msaa, "recording samples into multiple layers of a
// uint64 image"): same tasks, but a pixel that passes the conservative predicate is tested at its ms_k sample
// points (closest point to the SAMPLE within the centre radius) and `gbuf` is [ms_k][H][W] words, one layer per
// sample. A reference: plain atomicMin per sample hit, no read-before-atomic.
__constant__ int c_ms_off[4][8][2] = {  // sample offsets from the pixel centre in 1/16 pixel: 1x, 2x, 4x, 8x
    {{0, 0}},
    {{4, 4}, {-4, -4}},
    {{-2, -6}, {6, -2}, {-6, 2}, {2, 6}},
    {{1, -3}, {-1, 3}, {5, 1}, {-3, -5}, {-5, 5}, {-7, -1}, {3, 7}, {7, -7}}};

// Paper payload (PP = true; DESIGN.md R-payload): same tasks and tests; the projecting lane also
// computes calcTangent of its vertex (neighbours by shuffle, one extra load at each end of the chunk) and the
// strand's root codes, the record carries both ends' tangent and AO, and a hit whose depth does not lose builds the
// 40 payload bits (interpolated tangent -> octahedral code, w, AO) in fixed-order fp32 instead of sid | j | t.
// Two depth-ordered passes (HZ = true is the second): k_lod sends the bundles whose nearest cage depth lies in the
// front part of their instance's depth range to the first pass; between the passes k_hiz takes the farthest centre
// depth of every 16 x 16 pixel tile; the second pass drops a segment before any pixel work when its nearest depth
// lies behind that bound in every tile its bounding box touches — every one of its pixels would have failed the
// per-pixel early reject below, so the result is the same G-buffer, bit for bit.
// FUSED ("strand vertices stay in registers"): no vertex buffer. The warp builds the
// per-bundle spline table of its work group in shared memory (gen::build_table, the code k_generate runs) and every
// lane GENERATES the vertex it would have loaded (gen::vertex: same source, same bits). Needs the paper payload (the
// strand-id word is shaded from the vertex buffer). An A/B against the materialised pipeline.
// DOM (deep opacity maps; DESIGN.md R-dom): the frame is a light's view and gbuf already holds its
// resolved G-buffer; every conservative hit adds one fragment to the layer of its pixel it falls in behind the
// pixel's conservative depth (integer compare of 24-bit depths, one RED.ADD.32); nothing is written to gbuf.
template <bool COUNT, bool MS, bool PP, bool HZ, bool FUSED = false, bool DOM = false>
__global__ void __launch_bounds__(RAS_WARPS * 32, FUSED ? 2 : (PP ? 4 : RAS_MIN_BLOCKS))  // payload: 64 registers, no spills
k_raster(const SceneDev* __restrict__ sc, uint32_t n_bi, const uint4* __restrict__ table,
         const uint32_t* __restrict__ grp, const float4* __restrict__ vertices, CamDev cam, float rho_default,
         unsigned long long* __restrict__ gbuf, unsigned long long* __restrict__ counters, uint32_t ms_k,
         uint32_t queue, const uint32_t* __restrict__ hiz, uint32_t c_max, uint32_t* __restrict__ dom_cnt = nullptr,
         uint3 dom_D = make_uint3(0u, 0u, 0u)) {
  static_assert(!FUSED || (PP && !COUNT && !MS), "the fused raster writes the paper payload only");
  static_assert(!DOM || (!COUNT && !MS && !PP && !HZ && !FUSED), "the fragment count is a pass of its own");
  constexpr int RS = PP ? REC_STRIDE_PP : REC_STRIDE;
  __shared__ __align__(16) float s_rec[RAS_WARPS][32][RS];
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float(*rec)[RS] = s_rec[warp];
  uint32_t c_center = 0, c_cons = 0, c_cons_y = 0, c_drawn = 0, c_issued = 0, c_live = 0, c_hiz = 0;
  const int W = (int)cam.W, H = (int)cam.H;
  const int hiz_w = (W + HIZ_TILE - 1) / HIZ_TILE;
  const uint32_t le_mask = 0xFFFFFFFFu >> (31 - lane);
  const uint32_t n_groups = __ldcg(&grp[n_bi]);
  for (;;) {
    uint32_t wi = 0;
    if (lane == 0) wi = (uint32_t)atomicAdd(&counters[queue], 1ull);
    wi = __shfl_sync(0xffffffffu, wi, 0);
    if (wi >= n_groups) break;
    // ---- bundle of this group: largest gid with grp[gid] <= wi (32 pivots per level)
    uint32_t lo = 0, n = n_bi;
    while (n > 1) {
      const uint32_t step = (n + 31) >> 5;
      const uint32_t idx = lo + lane * step;
      const bool le = idx < lo + n && __ldg(&grp[idx]) <= wi;  // non-decreasing => a prefix of the lanes
      const uint32_t cnt = __popc(__ballot_sync(0xffffffffu, le));
      const uint32_t nlo = lo + (cnt - 1) * step;
      n = min(step, lo + n - nlo);
      lo = nlo;
    }
    const uint32_t gid = lo;
    const uint4 e = __ldg(&table[gid]);
    const uint32_t nlod = e.x, C = e.y;
    uint32_t gi = 0;
    for (uint32_t k = 1; k < sc->n_grooms; ++k)
      if (gid >= sc->g[k].gid_base) gi = k;
    const GroomDev& g = sc->g[gi];
    const uint32_t rel = gid - g.gid_base;
    const uint32_t q = rel / g.T, t = rel - q * g.T;
    const uint32_t off_t = __ldg(&g.off[t]);
    const uint32_t sid0 = g.sid_base + q * g.N + off_t;
    const float width = g.width_world;
    const uint32_t n_v = nlod * C;
    const float4* vin = vertices + e.w;
    const uint32_t v_begin = (wi - __ldg(&grp[gid])) * (RAS_GROUP * RAS_CHUNK);
    const uint32_t v_end = min(v_begin + RAS_GROUP * RAS_CHUNK, n_v - 1);  // first vertex of the next group
    float4 p_next = make_float4(0.f, 0.f, 0.f, 0.f);
    float* tab = nullptr;
    float M[12];
    bool has_m = false;
    if constexpr (FUSED) {  // the bundle's spline table, once per work group
      extern __shared__ float4 s_tab[];
      tab = reinterpret_cast<float*>(s_tab) + (size_t)warp * c_max * HAIR_ROW;
      gen::build_table(g, t, C, tab, lane);
      has_m = g.xform != nullptr;
      if (has_m)
#pragma unroll
        for (int a = 0; a < 12; ++a) M[a] = __ldg(&g.xform[q * 12 + a]);
    } else {
      if (v_begin + lane < n_v) p_next = __ldg(&vin[v_begin + lane]);
    }
    for (uint32_t v0 = v_begin; v0 < v_end; v0 += RAS_CHUNK) {
      // ---- project 32 vertices (loaded one chunk ahead, or generated here), neighbour by shuffle
      const uint32_t v = v0 + lane;
      float4 p = p_next;
      gen::Strand S = {};
      if constexpr (FUSED) {
        if (v < n_v) {
          const uint32_t ks = v / C;
          S = gen::strand_setup(g, off_t + ks);
          p = gen::vertex(tab, v - ks * C, S.b1, S.b2, S.cphi, S.sphi, S.base, g.op_mask, has_m ? M : nullptr);
        }
      } else {
        if (v0 + RAS_CHUNK < v_end && v + RAS_CHUNK < n_v) p_next = __ldg(&vin[v + RAS_CHUNK]);
      }
      Proj a;
      a.valid = false;
      a.sx = a.sy = a.zn = a.zv = 0.f;
      if (v < n_v) a = project_exact(cam, p.x, p.y, p.z);
      Proj b;
      b.sx = __shfl_down_sync(0xffffffffu, a.sx, 1);
      b.sy = __shfl_down_sync(0xffffffffu, a.sy, 1);
      b.zn = __shfl_down_sync(0xffffffffu, a.zn, 1);
      b.zv = __shfl_down_sync(0xffffffffu, a.zv, 1);
      b.valid = __shfl_down_sync(0xffffffffu, (int)a.valid, 1) != 0;
      const uint32_t k = v / C, j = v - k * C;
      const bool seg = lane < 31 && v < v_end && j + 1 < C && a.valid && b.valid;  // R12
      if (PP) {  // R-payload: tangent of this vertex, exchanged with the neighbour; AO; the strand's root codes
        float4 pp, pn;
        pp.x = __shfl_up_sync(0xffffffffu, p.x, 1), pp.y = __shfl_up_sync(0xffffffffu, p.y, 1), pp.z = __shfl_up_sync(0xffffffffu, p.z, 1);
        pn.x = __shfl_down_sync(0xffffffffu, p.x, 1), pn.y = __shfl_down_sync(0xffffffffu, p.y, 1), pn.z = __shfl_down_sync(0xffffffffu, p.z, 1);
        pp.w = pn.w = 0.f;
        X3 Tv = {1.f, 0.f, 0.f};
        if (v < n_v) {
          if constexpr (FUSED) {  // the neighbours beyond the chunk's ends: one more vertex on lanes 0 and 31
            const bool e0 = lane == 0 && j > 0, e1 = lane == 31 && j + 1 < C;
            if (e0 || e1) {
              const float4 px = gen::vertex(tab, e0 ? j - 1 : j + 1, S.b1, S.b2, S.cphi, S.sphi, S.base, g.op_mask,
                                            has_m ? M : nullptr);
              if (e0) pp = px;
              else pn = px;
            }
          } else {
            if (lane == 0 && j > 0) pp = __ldg(&vin[v - 1]);
            if (lane == 31 && j + 1 < C) pn = __ldg(&vin[v + 1]);
          }
          Tv = tangent_x(j, C, pp, p, pn);
        }
        const float t1x = __shfl_down_sync(0xffffffffu, Tv.x, 1), t1y = __shfl_down_sync(0xffffffffu, Tv.y, 1),
                    t1z = __shfl_down_sync(0xffffffffu, Tv.z, 1), ao1 = __shfl_down_sync(0xffffffffu, p.w, 1);
        if (seg) {
          uint32_t a1, a2;
          if constexpr (FUSED) {
            a1 = S.a1, a2 = S.a2;
          } else {
            const uint32_t base = pcg(g.seed_h + off_t + k);
            a1 = pcg(base + 1u) >> 8, a2 = pcg(base + 2u) >> 8;
            if (a1 + a2 > 16777216u) {  // R6
              a1 = 16777216u - a1;
              a2 = 16777216u - a2;
            }
          }
          float* rp = rec[lane];
          rp[18] = Tv.x, rp[19] = Tv.y, rp[20] = Tv.z, rp[21] = t1x, rp[22] = t1y, rp[23] = t1z;
          rp[24] = p.w, rp[25] = ao1;
          rp[26] = __uint_as_float((uv6(a1) << 18) | (uv6(a2) << 12));
          rp[27] = __uint_as_float(C);
        }
      }
      // ---- segment record in (major, minor) coordinates; every formula below is symmetric in x/y
      uint32_t n_steps = 0;
      if (seg) {
        if (COUNT) ++c_drawn;
        float rho = rho_default;
        if (width > 0.f) {  // R9
          const float zm = xmul(0.5f, xadd(a.zv, b.zv));
          const float wpx = fminf(fmaxf(xdiv(xmul(width, cam.fpx), zm), 0.25f), 1.0f);
          rho = xmul(0.5f, wpx);
        }
        const float dx = xsub(b.sx, a.sx), dy = xsub(b.sy, a.sy);
        const bool ymajor = fabsf(dy) > fabsf(dx);
        const float aM = ymajor ? a.sy : a.sx, aN = ymajor ? a.sx : a.sy;
        const float bM = ymajor ? b.sy : b.sx, bN = ymajor ? b.sx : b.sy;
        const float dM = ymajor ? dy : dx, dN = ymajor ? dx : dy;
        const float limM = (float)((ymajor ? H : W) - 1), limN = (float)((ymajor ? W : H) - 1);
        // candidate pixels = exactly those whose closed square overlaps the segment's AABB (R10)
        const float fc0 = fmaxf(ceilf(fminf(aM, bM)) - 1.f, 0.f), fc1 = fminf(floorf(fmaxf(aM, bM)), limM);
        const float fr0 = fmaxf(ceilf(fminf(aN, bN)) - 1.f, 0.f), fr1 = fminf(floorf(fmaxf(aN, bN)), limN);
        bool draw = fc0 <= fc1 && fr0 <= fr1;
        // nearest depth any pixel of this segment can store, minus 2 steps for the rounding of R11's lerp
        const uint32_t dqm = quant_depth(fminf(fmaxf(fminf(a.zn, b.zn), 0.f), 1.f));
        const uint32_t dq_lim = dqm > 2u ? dqm - 2u : 0u;
        if (HZ && draw) {  // hi-Z: farthest centre depth over the (at most 3 x 3) tiles of the bounding box
          const int x0 = (int)(ymajor ? fr0 : fc0) / HIZ_TILE, x1 = (int)(ymajor ? fr1 : fc1) / HIZ_TILE;
          const int y0 = (int)(ymajor ? fc0 : fr0) / HIZ_TILE, y1 = (int)(ymajor ? fc1 : fr1) / HIZ_TILE;
          if (x1 - x0 <= 2 && y1 - y0 <= 2) {
            uint32_t zfar = 0;
#pragma unroll
            for (int ty = 0; ty < 3; ++ty)
#pragma unroll
              for (int tx = 0; tx < 3; ++tx)
                zfar = max(zfar, __ldg(&hiz[min(y0 + ty, y1) * hiz_w + min(x0 + tx, x1)]));
            if (dq_lim > zfar) {
              draw = false;
              ++c_hiz;
            }
          }
        }
        if (draw) {
          n_steps = (uint32_t)((int)fc1 - (int)fc0 + 1);
          float4* r4 = reinterpret_cast<float4*>(rec[lane]);
          const float dd = xadd(xmul(dx, dx), xmul(dy, dy));
          r4[0] = make_float4(aM, aN, dM, dN);
          r4[1] = make_float4(dd, xmul(0.5f, xadd(fabsf(dx), fabsf(dy))), a.zn, xsub(b.zn, a.zn));
          // minor coordinate of the line at major coordinate x: icpt + x * slope (enumeration only)
          const float slope = dM != 0.f ? dN / dM : 0.f;
          r4[2] = make_float4(aN - aM * slope, slope, __int_as_float((int)fc0),
                              __uint_as_float(((uint32_t)(int)fr0 << 16) | (uint32_t)(int)fr1));
          rec[lane][17] = xmul(rho, rho);
          r4[3].x = __uint_as_float((ymajor ? 0x80000000u : 0u) | ((sid0 + k) << 7) | j);
          r4[3].w = __uint_as_float(dq_lim);
          if (COUNT) rec[lane][16] = 0.f;
        }
      }
      // ---- spread (segment, column) tasks over the lanes
      const uint32_t n_eff = max(n_steps, 1u);  // empty segments keep one no-op task: starts stay distinct
      uint32_t incl = n_eff;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t up = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += up;
      }
      const uint32_t X = incl - n_eff;
      const uint32_t total = __shfl_sync(0xffffffffu, incl, 31);
      rec[lane][13] = __uint_as_float(X);
      rec[lane][14] = __uint_as_float(n_steps);
      __syncwarp();
      for (uint32_t base = 0; base < total; base += 32) {
        const uint32_t before = __popc(__ballot_sync(0xffffffffu, X < base));
        const uint32_t startbits = __reduce_or_sync(0xffffffffu, (X >= base && X < base + 32) ? 1u << (X - base) : 0u);
        const uint32_t s = before + __popc(startbits & le_mask) - 1;  // owner of task base + lane
        const uint32_t tau = base + lane;
        if (tau >= total) continue;
        const float4* r4 = reinterpret_cast<const float4*>(rec[s]);
        const float4 q3 = r4[3];
        const uint32_t step = tau - __float_as_uint(q3.y);
        if (step >= __float_as_uint(q3.z)) continue;  // the no-op task of an empty segment
        const float4 q0 = r4[0], q1 = r4[1], q2 = r4[2];
        const float aM = q0.x, aN = q0.y, dM = q0.z, dN = q0.w;
        const float dd = q1.x, ext = q1.y, az = q1.z, dz = q1.w;
        const uint32_t key = __float_as_uint(q3.x), dq_min = __float_as_uint(q3.w);
        const bool ymajor = (key >> 31) != 0;
        const int c = __float_as_int(q2.z) + (int)step;
        const int r0 = (int)(__float_as_uint(q2.w) >> 16), r1 = (int)(__float_as_uint(q2.w) & 0xFFFFu);
        // minor-axis extent of the LINE across column [c, c+1], clipped to the rows of the segment's bounding box:
        // a superset of the rows the segment crosses there (the line is monotone; ENUM_EPS covers the rounding)
        const float fc = (float)c;
        const float m0 = fmaf(fc, q2.y, q2.x), m1 = m0 + q2.y;
        const int rlo = max((int)ceilf(fminf(m0, m1) - ENUM_EPS) - 1, r0);
        const int rhi = min((int)floorf(fmaxf(m0, m1) + ENUM_EPS), r1);
        const float cM = fc + 0.5f;
        const float uM = xsub(cM, aM);
        // pixel (c, r) in major/minor order -> index of its word pair (32-bit: W * H <= 2^28); step of one minor step
        const uint32_t pstep = ymajor ? 1u : (uint32_t)W;
        const uint32_t pcol = ymajor ? (uint32_t)c * (uint32_t)W : (uint32_t)c;
        ulonglong2* const gpair = reinterpret_cast<ulonglong2*>(gbuf);
        for (int rb = rlo; rb <= rhi; rb += ROW_BATCH) {
          // pass 1: the cheap half of the conservative predicate (R10), then request the words
          bool ok[ROW_BATCH];
          ulonglong2 cur[ROW_BATCH];
#pragma unroll
          for (int i = 0; i < ROW_BATCH; ++i) {
            const int r = rb + i;
            const float uN = xsub((float)r + 0.5f, aN);
            const float cr = fabsf(xsub(xmul(dM, uN), xmul(dN, uM)));
            ok[i] = r <= rhi && cr <= ext;
            if (!MS && ok[i]) cur[i] = GB_LOAD(gpair + (pcol + (uint32_t)r * pstep));
          }
          if (MS) {  // reference mode: every sample point of the pixels that passed the conservative predicate
            const int pat = ms_k == 8 ? 3 : ms_k == 4 ? 2 : ms_k == 2 ? 1 : 0;
#pragma unroll
            for (int i = 0; i < ROW_BATCH; ++i) {
              if (!ok[i]) continue;
              const int r = rb + i;
              const size_t pix = ymajor ? (size_t)c * W + r : (size_t)r * W + c;
              for (uint32_t smp = 0; smp < ms_k; ++smp) {
                const int ox = c_ms_off[pat][smp][0], oy = c_ms_off[pat][smp][1];
                const float sM = fc + (0.5f + (float)(ymajor ? oy : ox) * 0.0625f);
                const float sN = (float)r + (0.5f + (float)(ymajor ? ox : oy) * 0.0625f);
                const float vM = xsub(sM, aM), vN = xsub(sN, aN);
                float tt = 0.f;
                if (dd > 0.f) tt = fminf(fmaxf(xdiv(xadd(xmul(vM, dM), xmul(vN, dN)), dd), 0.f), 1.f);
                const float zn = xadd(az, xmul(tt, dz));
                if (zn < 0.f || zn > 1.f) continue;
                const float eM = xsub(sM, xadd(aM, xmul(tt, dM))), eN = xsub(sN, xadd(aN, xmul(tt, dN)));
                if (xadd(xmul(eM, eM), xmul(eN, eN)) <= rec[s][17])
                  atomicMin(gbuf + (size_t)smp * W * H + pix, pack_word(zn, (key >> 7) & 0xFFFFFFu, key & 0x7Fu, tt));
              }
            }
            continue;
          }
          // pass 2: closest point, depth, centre predicate, word (R10/R11, fixed-order fp32; x/y-symmetric)
#pragma unroll
          for (int i = 0; i < ROW_BATCH; ++i) {
            if (!ok[i]) continue;
            // early reject: centre word >= conservative word (R10), so a segment that lies entirely behind
            // the pixel's centre hit loses both layers whatever its exact depth at this pixel
            if (!COUNT && !DOM && dq_min > (uint32_t)(cur[i].x >> 40)) continue;
            const int r = rb + i;
            const float cN = (float)r + 0.5f;
            const float uN = xsub(cN, aN);
            float tt = 0.f;
            if (dd > 0.f) tt = fminf(fmaxf(xdiv(xadd(xmul(uM, dM), xmul(uN, dN)), dd), 0.f), 1.f);
            const float zn = xadd(az, xmul(tt, dz));
            if (zn < 0.f || zn > 1.f) continue;
            const float eM = xsub(cM, xadd(aM, xmul(tt, dM))), eN = xsub(cN, xadd(aN, xmul(tt, dN)));
            if (DOM) {  // fragment of the deep opacity map: layer by its depth behind the nearest hair of the pixel
              const uint32_t d = quant_depth(zn) - (uint32_t)(cur[i].y >> 40);
              const uint32_t layer = (d >= dom_D.x ? 1u : 0u) + (d >= dom_D.y ? 1u : 0u) + (d >= dom_D.z ? 1u : 0u);
              const size_t pix = ymajor ? (size_t)c * W + (rb + i) : (size_t)(rb + i) * W + c;
              atomicAdd(dom_cnt + pix * 4 + layer, 1u);
              continue;
            }
            const bool centre = xadd(xmul(eM, eM), xmul(eN, eN)) <= rec[s][17];
            unsigned long long word;
            if (PP) {
              const uint32_t dq = quant_depth(zn);
              word = HAIR_EMPTY;
              // the payload only matters where the depth does not lose outright
              if (COUNT || dq <= (uint32_t)(cur[i].y >> 40) || (centre && dq <= (uint32_t)(cur[i].x >> 40))) {
                const float* rp = rec[s];
                const float omt = xsub(1.f, tt);
                const X3 T = unit3x(xadd(xmul(omt, rp[18]), xmul(tt, rp[21])), xadd(xmul(omt, rp[19]), xmul(tt, rp[22])),
                                    xadd(xmul(omt, rp[20]), xmul(tt, rp[23])));
                const uint32_t oct = oct_encode_x(T);
                const float w = xdiv(xadd((float)(key & 0x7Fu), tt), (float)(__float_as_uint(rp[27]) - 1u));
                const float ao = fminf(fmaxf(xadd(xmul(omt, rp[24]), xmul(tt, rp[25])), 0.f), 1.f);
                const uint32_t lo = ((oct & 0xFFu) << 24) | __float_as_uint(rp[26]) | (q6(w) << 6) | q6(ao);
                word = ((unsigned long long)((dq << 8) | (oct >> 8)) << 32) | lo;
              }
            } else
              word = pack_word(zn, (key >> 7) & 0xFFFFFFu, key & 0x7Fu, tt);
            unsigned long long* px = reinterpret_cast<unsigned long long*>(gpair + (pcol + (uint32_t)r * pstep));
            if (COUNT) {
              ++c_cons;
              c_cons_y += ymajor ? 1u : 0u;
              c_center += centre ? 1u : 0u;
            }
            if (word < cur[i].y) {
              atomicMin(px + 1, word);
              if (COUNT) ++c_issued, rec[s][16] = 1.f;
            }
            if (centre && word < cur[i].x) {
              atomicMin(px, word);
              if (COUNT) ++c_issued, rec[s][16] = 1.f;
            }
          }
        }
      }
      __syncwarp();
      if (COUNT && n_steps && rec[lane][16] != 0.f) ++c_live;
    }
  }
  if (HZ) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) c_hiz += __shfl_xor_sync(0xffffffffu, c_hiz, d);
    if (lane == 0 && c_hiz) atomicAdd(&counters[CNT_SEG_HIZ], (unsigned long long)c_hiz);
  }
  if (COUNT) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
      c_center += __shfl_xor_sync(0xffffffffu, c_center, d);
      c_cons += __shfl_xor_sync(0xffffffffu, c_cons, d);
      c_cons_y += __shfl_xor_sync(0xffffffffu, c_cons_y, d);
      c_drawn += __shfl_xor_sync(0xffffffffu, c_drawn, d);
      c_issued += __shfl_xor_sync(0xffffffffu, c_issued, d);
      c_live += __shfl_xor_sync(0xffffffffu, c_live, d);
    }
    if (lane == 0) {
      atomicAdd(&counters[CNT_AT_CENTER], (unsigned long long)c_center);
      atomicAdd(&counters[CNT_AT_CONS], (unsigned long long)c_cons);
      atomicAdd(&counters[CNT_AT_CONS_Y], (unsigned long long)c_cons_y);
      atomicAdd(&counters[CNT_SEG_DRAWN], (unsigned long long)c_drawn);
      atomicAdd(&counters[CNT_AT_ISSUED], (unsigned long long)c_issued);
      atomicAdd(&counters[CNT_SEG_LIVE], (unsigned long long)c_live);
    }
  }
}

// clear both layers to "no hit": all ones, or (R-scene) the scene's quantised depth (R8) with an all-ones payload,
// which is the paper's pre-existing depth buffer: a hit behind it loses the atomic min
__global__ void __launch_bounds__(256) k_clear(uint4* __restrict__ g, size_t n16, const float* __restrict__ scene_zn) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const uint4 ones = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) {
    uint4 v = ones;
    if (scene_zn) {
      const uint32_t hi = (quant_depth(fminf(fmaxf(__ldg(&scene_zn[i]), 0.f), 1.f)) << 8) | 0xFFu;
      v.y = v.w = hi;
    }
    g[i] = v;
  }
}

// R-seq ("preserving the depth buffer between groom passes"): between two sequential passes both
// layers of a pixel restart at the depth of its centre word (a hit's depth, else the depth kept so far), no hit
__global__ void __launch_bounds__(256) k_reseed(uint4* __restrict__ g, size_t n16) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) {
    const uint32_t hi = g[i].y | 0xFFu;
    g[i] = make_uint4(0xFFFFFFFFu, hi, 0xFFFFFFFFu, hi);
  }
}

void launch_reseed(unsigned long long* gbuf, size_t n_pixels, cudaStream_t st) {
  size_t blocks = (n_pixels + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  k_reseed<<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<uint4*>(gbuf), n_pixels);
}

// farthest centre depth of every HIZ_TILE x HIZ_TILE pixel tile. A warp per tile: lanes 0-15 read the 16 words of
// one tile row, lanes 16-31 those of the next (two coalesced 256-byte runs per load), eight loads cover the tile.
// A pixel without a centre hit keeps the depth it was cleared / seeded with (all ones = never occludes).
__global__ void __launch_bounds__(256) k_hiz(const uint4* __restrict__ g, uint32_t W, uint32_t H,
                                             uint32_t* __restrict__ hiz, const unsigned long long* __restrict__ counters) {
  static_assert(HIZ_TILE == 16, "k_hiz maps 16 lanes to a tile row");
  if (__ldcg(&counters[CNT_HIZ_ON]) == 0ull) return;  // one-pass frame (decided on the device by k_scan)
  const uint32_t tw = (W + HIZ_TILE - 1) / HIZ_TILE, th = (H + HIZ_TILE - 1) / HIZ_TILE;
  const uint32_t tile = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (tile >= tw * th) return;
  const uint32_t ty = tile / tw, tx = tile - ty * tw;
  const uint32_t x = tx * HIZ_TILE + (lane & 15u), y0 = ty * HIZ_TILE + (lane >> 4);
  uint32_t zfar = 0;
  if (x < W) {
#pragma unroll
    for (uint32_t i = 0; i < 8; ++i) {
      const uint32_t y = y0 + 2 * i;
      if (y < H) zfar = max(zfar, __ldcg(reinterpret_cast<const uint32_t*>(g) + ((size_t)y * W + x) * 4 + 1) >> 8);
    }
  }
  zfar = __reduce_max_sync(0xffffffffu, zfar);
  if (lane == 0) hiz[tile] = zfar;
}

void launch_hiz(const unsigned long long* gbuf, uint32_t W, uint32_t H, uint32_t* hiz,
                const unsigned long long* counters, cudaStream_t st) {
  const uint32_t n_tiles = ((W + HIZ_TILE - 1) / HIZ_TILE) * ((H + HIZ_TILE - 1) / HIZ_TILE);
  k_hiz<<<(n_tiles + 7) / 8, 256, 0, st>>>(reinterpret_cast<const uint4*>(gbuf), W, H, hiz, counters);
}

void launch_clear(unsigned long long* gbuf, size_t n_pixels, const float* scene_zn, cudaStream_t st) {
  size_t blocks = (n_pixels + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  k_clear<<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<uint4*>(gbuf), n_pixels, scene_zn);
}

template <bool COUNT, bool MS, bool PP, bool HZ, bool FUSED = false>
static void launch_raster_t(const SceneDev* d_scene, uint32_t n_bi, const uint4* table, const uint32_t* grp,
                            const float4* vertices, CamDev cam, float rho_default, unsigned long long* gbuf,
                            unsigned long long* counters, uint32_t ms_k, uint32_t queue, const uint32_t* hiz, int n_sm,
                            LaunchState* ls, cudaStream_t st, uint32_t c_max = 0) {
  // persistent grid: every CTA slot of the device, the queue feeds them
  const size_t smem = FUSED ? (size_t)RAS_WARPS * c_max * HAIR_ROW * sizeof(float) : 0;  // the warps' spline tables
  constexpr int V = (COUNT ? 1 : 0) | (MS ? 2 : 0) | (PP ? 4 : 0) | (HZ ? 8 : 0) | (FUSED ? 16 : 0);
  if (!ls->raster_per_sm[V] || smem != ls->raster_smem[V]) {  // once per context (= device) and table size
    if (smem) raise_dyn_smem(k_raster<COUNT, MS, PP, HZ, FUSED>, smem);
    int b = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k_raster<COUNT, MS, PP, HZ, FUSED>, RAS_WARPS * 32, smem);
    ls->raster_per_sm[V] = b > 0 ? b : 1;
    ls->raster_smem[V] = smem;
  }
  const int per_sm = ls->raster_per_sm[V];
  k_raster<COUNT, MS, PP, HZ, FUSED><<<(uint32_t)(n_sm * per_sm), RAS_WARPS * 32, smem, st>>>(
      d_scene, n_bi, table, grp, vertices, cam, rho_default, gbuf, counters, ms_k, queue, hiz, c_max);
}

void launch_raster_dom(const SceneDev* d_scene, uint32_t n_bi, const uint4* table, const uint32_t* grp,
                       const float4* vertices, CamDev cam, float rho_default, unsigned long long* gbuf,
                       unsigned long long* counters, uint32_t* dom_cnt, uint3 dom_D, int n_sm, LaunchState* ls,
                       cudaStream_t st) {
  constexpr int V = 32;
  if (!ls->raster_per_sm[V]) {
    int b = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k_raster<false, false, false, false, false, true>, RAS_WARPS * 32, 0);
    ls->raster_per_sm[V] = b > 0 ? b : 1;
  }
  k_raster<false, false, false, false, false, true><<<(uint32_t)(n_sm * ls->raster_per_sm[V]), RAS_WARPS * 32, 0, st>>>(
      d_scene, n_bi, table, grp, vertices, cam, rho_default, gbuf, counters, 0, CNT_WORK_RASTER, nullptr, 0, dom_cnt, dom_D);
}

// z0 of a deep opacity map: the conservative layer's 24-bit depth, 0xFFFFFFFF where the pixel holds no hair
__global__ void __launch_bounds__(256) k_dom_z0(const uint4* __restrict__ g, size_t n, uint32_t* __restrict__ z0) {
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint4 v = __ldg(&g[i]);
    z0[i] = w_none(v.z, v.w) ? 0xFFFFFFFFu : v.w >> 8;
  }
}
void launch_dom_z0(const unsigned long long* gbuf, size_t n_pixels, uint32_t* z0, cudaStream_t st) {
  size_t blocks = (n_pixels + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  k_dom_z0<<<(unsigned)blocks, 256, 0, st>>>(reinterpret_cast<const uint4*>(gbuf), n_pixels, z0);
}

// ms_k = 0: the two-layer G-buffer; ms_k in {1, 2, 4, 8}: gbuf = [ms_k][H][W] sample layers (reference mode).
// pass 0 draws the work groups of grp[0 .. n_bi], pass 1 those of the second scan behind it, with the hi-Z test
void launch_raster(const SceneDev* d_scene, uint32_t n_bi, const uint4* table, const uint32_t* grp,
                   const float4* vertices, CamDev cam, float rho_default, unsigned long long* gbuf,
                   unsigned long long* counters, bool count, uint32_t ms_k, bool paper_payload, int pass,
                   const uint32_t* hiz, int n_sm, LaunchState* ls, cudaStream_t st, uint32_t fused_c_max) {
  const uint32_t* gp = grp + (pass ? (size_t)n_bi + 1 : 0);
  const uint32_t q = pass ? CNT_WORK_RASTER1 : CNT_WORK_RASTER;
#define RAS_ARGS d_scene, n_bi, table, gp, vertices, cam, rho_default, gbuf, counters
  if (fused_c_max && pass) launch_raster_t<false, false, true, true, true>(RAS_ARGS, 0, q, hiz, n_sm, ls, st, fused_c_max);
  else if (fused_c_max) launch_raster_t<false, false, true, false, true>(RAS_ARGS, 0, q, nullptr, n_sm, ls, st, fused_c_max);
  else if (ms_k) launch_raster_t<false, true, false, false>(RAS_ARGS, ms_k, q, nullptr, n_sm, ls, st);
  else if (paper_payload && count) launch_raster_t<true, false, true, false>(RAS_ARGS, 0, q, nullptr, n_sm, ls, st);
  else if (paper_payload && pass) launch_raster_t<false, false, true, true>(RAS_ARGS, 0, q, hiz, n_sm, ls, st);
  else if (paper_payload) launch_raster_t<false, false, true, false>(RAS_ARGS, 0, q, nullptr, n_sm, ls, st);
  else if (count) launch_raster_t<true, false, false, false>(RAS_ARGS, 0, q, nullptr, n_sm, ls, st);
  else if (pass) launch_raster_t<false, false, false, true>(RAS_ARGS, 0, q, hiz, n_sm, ls, st);
  else launch_raster_t<false, false, false, false>(RAS_ARGS, 0, q, nullptr, n_sm, ls, st);
#undef RAS_ARGS
}
