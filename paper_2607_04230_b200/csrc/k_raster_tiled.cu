// k_raster_tiled.cu — H4 as a sort-middle raster: segments binned to 64 x 64 pixel tiles, the tile's two G-buffer
// layers in SHARED memory (HAIR_FLAG_TILED, "hybrid" future work).
//
// Why: k_raster keeps the G-buffer in L2 and pays one 16-byte L2 load per candidate pixel before anything is known
// about its depth (read-before-atomic); measured, it runs AT the L2 pair-load ceiling of its access pattern
// (DESIGN.md 7.5). Here every pixel test is an LDS.128, the resolve is a 64-bit shared-memory atomic min, and — because
// a tile's depth lives next to the warps that draw into it — a two-level hi-Z of the tile (8 x 8 and 16 x 16 pixel
// blocks) is refreshed continuously by the drawing warps themselves and drops occluded segments before any pixel work.
// Depths only ever decrease, so a bound taken from ANY earlier (even racy) snapshot stays valid: no synchronisation.
//
//  k_bin<false>   per segment: count the tiles its candidate-pixel box touches   (near bundles, then far bundles)
//  k_tile_scan    exclusive scan of the tile counts, tile order by work (heaviest first), overflow check
//  k_bin<true>    same walk: claim slots (one atomic per warp and tile) and write 32-byte screen-space records;
//                 near bundles are scattered first, so every tile's list starts with the bundles in front
//  k_raster_tiled persistent CTAs, one tile at a time: init the tile (clear / scene depth / reseed — replaces k_clear),
//                 warps pull batches of 32 records, same (segment, column) tasks and the SAME fixed-order fp32
//                 predicates and words as k_raster => the same G-buffer bit for bit; coalesced 16-byte flush.
#include "hair_internal.cuh"

#define REC_STRIDE 20       // floats per staged segment record, as in k_raster.cu
#define ENUM_EPS 0.015625f  // as in k_raster.cu: slack of the column enumeration (a superset of the covered rows)
#define TR_WARPS 16
#define TR_ROWS 2           // rows of one column whose words are requested before any is used
#define TILE_PX (HAIR_TILE * HAIR_TILE)

// swizzled index of pixel (lx, ly) of the tile: 16-byte pairs, so 8 of them span all 32 banks; XOR-ing the row into the
// low 3 bits of the column puts the 8 lanes of a quarter warp on different bank groups for row walks AND column walks
__device__ __forceinline__ uint32_t tile_idx(uint32_t lx, uint32_t ly) { return ly * HAIR_TILE + (lx ^ (ly & 7u)); }

// ------------------------------------------------------------------------------------------------ binning
// The walk over the vertex buffer is k_raster's: a work group = RAS_GROUP chunks of RAS_CHUNK segments of one
// bundle-instance, lane = vertex, neighbour by shuffle. What is written per (segment, tile) is the projected segment:
// {a.sx, a.sy, b.sx, b.sy} {a.zn, b.zn, key = sid << 7 | j, rho^2}: the raster's predicates need nothing else.
template <bool SCATTER>
__global__ void __launch_bounds__(256)
k_bin(const SceneDev* __restrict__ sc, uint32_t n_bi, const uint4* __restrict__ table, const uint32_t* __restrict__ grp,
      const float4* __restrict__ vertices, CamDev cam, float rho_default, unsigned long long* __restrict__ counters,
      uint32_t queue, uint32_t* __restrict__ tile_count, const uint32_t* __restrict__ tile_base,
      float4* __restrict__ entries, uint32_t cap, uint32_t tiles_x) {
  const uint32_t lane = threadIdx.x & 31;
  const int W = (int)cam.W, H = (int)cam.H;
  const uint32_t n_groups = __ldcg(&grp[n_bi]);
  for (;;) {
    uint32_t wi = 0;
    if (lane == 0) wi = (uint32_t)atomicAdd(&counters[queue], 1ull);
    wi = __shfl_sync(0xffffffffu, wi, 0);
    if (wi >= n_groups) break;
    uint32_t lo = 0, n = n_bi;  // bundle of this group: largest gid with grp[gid] <= wi
    while (n > 1) {
      const uint32_t step = (n + 31) >> 5;
      const uint32_t idx = lo + lane * step;
      const bool le = idx < lo + n && __ldg(&grp[idx]) <= wi;
      const uint32_t cnt = __popc(__ballot_sync(0xffffffffu, le));
      const uint32_t nlo = lo + (cnt - 1) * step;
      n = min(step, lo + n - nlo);
      lo = nlo;
    }
    const uint32_t gid = lo;
    const uint4 e = __ldg(&table[gid]);
    const uint32_t C = e.y, n_v = e.x * e.y;
    uint32_t gi = 0;
    for (uint32_t k = 1; k < sc->n_grooms; ++k)
      if (gid >= sc->g[k].gid_base) gi = k;
    const GroomDev& g = sc->g[gi];
    const uint32_t rel = gid - g.gid_base;
    const uint32_t q = rel / g.T, t = rel - q * g.T;
    const uint32_t sid0 = g.sid_base + q * g.N + __ldg(&g.off[t]);
    const float width = g.width_world;
    const float4* vin = vertices + e.w;
    const uint32_t v_begin = (wi - __ldg(&grp[gid])) * (RAS_GROUP * RAS_CHUNK);
    const uint32_t v_end = min(v_begin + RAS_GROUP * RAS_CHUNK, n_v - 1);
    for (uint32_t v0 = v_begin; v0 < v_end; v0 += RAS_CHUNK) {
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
      const bool seg = lane < 31 && v < v_end && j + 1 < C && a.valid && b.valid;  // R12
      int tx0 = 0, tx1 = -1, ty0 = 0, ty1 = -1;
      if (seg) {  // candidate pixels = those whose closed square overlaps the segment's bounding box (R10)
        const float fx0 = fmaxf(ceilf(fminf(a.sx, b.sx)) - 1.f, 0.f), fx1 = fminf(floorf(fmaxf(a.sx, b.sx)), (float)(W - 1));
        const float fy0 = fmaxf(ceilf(fminf(a.sy, b.sy)) - 1.f, 0.f), fy1 = fminf(floorf(fmaxf(a.sy, b.sy)), (float)(H - 1));
        if (fx0 <= fx1 && fy0 <= fy1) {
          tx0 = (int)fx0 / HAIR_TILE, tx1 = (int)fx1 / HAIR_TILE;
          ty0 = (int)fy0 / HAIR_TILE, ty1 = (int)fy1 / HAIR_TILE;
        }
      }
      const int nx = tx1 - tx0 + 1;
      const uint32_t n_t = tx1 >= tx0 ? (uint32_t)(nx * (ty1 - ty0 + 1)) : 0u;
      float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0;
      if (SCATTER && n_t) {
        float rho = rho_default;
        if (width > 0.f) {  // R9
          const float zm = xmul(0.5f, xadd(a.zv, b.zv));
          rho = xmul(0.5f, fminf(fmaxf(xdiv(xmul(width, cam.fpx), zm), 0.25f), 1.0f));
        }
        r0 = make_float4(a.sx, a.sy, b.sx, b.sy);
        r1 = make_float4(a.zn, b.zn, __uint_as_float(((sid0 + k) << 7) | j), xmul(rho, rho));
      }
      const uint32_t n_max = __reduce_max_sync(0xffffffffu, n_t);
      for (uint32_t it = 0; it < n_max; ++it) {
        const bool on = it < n_t;
        const uint32_t act = __ballot_sync(0xffffffffu, on);
        if (!on) continue;
        const uint32_t tile = (uint32_t)(ty0 + (int)it / nx) * tiles_x + (uint32_t)(tx0 + (int)it % nx);
        const uint32_t peers = __match_any_sync(act, tile);  // one atomic per warp and tile
        const uint32_t leader = __ffs(peers) - 1, rank = __popc(peers & ((1u << lane) - 1u));
        uint32_t slot = 0;
        if (lane == leader) slot = atomicAdd(&tile_count[tile], (uint32_t)__popc(peers));
        if (SCATTER) {
          slot = __shfl_sync(peers, slot, leader) + rank + __ldg(&tile_base[tile]);
          if (slot < cap) {
            entries[2 * (size_t)slot] = r0;
            entries[2 * (size_t)slot + 1] = r1;
          }
        }
      }
    }
  }
}

// Exclusive scan of the tile counts -> tile_base, the counts move to tile_n, tile_count restarts at 0 as the scatter's
// cursor (and once more in k_raster_tiled, as the next frame's counter). Tiles ordered by work, heaviest first (a counting sort on
// log2(count): the persistent raster takes them in this order, so the dense tiles do not end up in the tail).
// One CTA of 1024 threads; n_tiles <= 65 536.
__global__ void __launch_bounds__(1024) k_tile_scan(uint32_t* __restrict__ tile_count, uint32_t* __restrict__ tile_base,
                                                    uint32_t* __restrict__ tile_n, uint32_t* __restrict__ tile_order,
                                                    uint32_t n_tiles, uint32_t cap, unsigned long long* __restrict__ counters) {
  __shared__ uint32_t s_warp[32], s_carry, s_bucket[33], s_cursor[33];
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x < 33) s_bucket[threadIdx.x] = 0;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (uint32_t i0 = 0; i0 < n_tiles; i0 += 1024) {
    const uint32_t i = i0 + threadIdx.x;
    const uint32_t c = i < n_tiles ? tile_count[i] : 0u;
    uint32_t inc = c;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t up = __shfl_up_sync(0xffffffffu, inc, d);
      if (lane >= d) inc += up;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    uint32_t off = s_carry;
    for (uint32_t w = 0; w < warp; ++w) off += s_warp[w];
    if (i < n_tiles) {
      tile_base[i] = off + inc - c;
      tile_n[i] = c;
      tile_count[i] = 0;
      atomicAdd(&s_bucket[c ? 32 - __clz(c) : 0], 1u);  // bucket 0: empty tiles, b: 2^(b-1) <= count < 2^b
    }
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = off + inc;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    uint32_t at = 0;
    for (int b = 32; b >= 0; --b) {
      s_cursor[b] = at;
      at += s_bucket[b];
    }
    counters[CNT_TILE_ENTRIES] = s_carry;
    counters[CNT_TILE_OVERFLOW] = s_carry > cap ? 1ull : 0ull;
  }
  __syncthreads();
  for (uint32_t i = threadIdx.x; i < n_tiles; i += 1024) {
    const uint32_t c = tile_n[i];
    tile_order[atomicAdd(&s_cursor[c ? 32 - __clz(c) : 0], 1u)] = i;
  }
}

// ------------------------------------------------------------------------------------------------ the tile raster
__global__ void __launch_bounds__(TR_WARPS * 32, 2)
k_raster_tiled(CamDev cam, unsigned long long* __restrict__ gbuf, const float* __restrict__ scene_zn, uint32_t reseed,
               unsigned long long* __restrict__ counters, const uint32_t* __restrict__ tile_order,
               const uint32_t* __restrict__ tile_base, const uint32_t* __restrict__ tile_n,
               const float4* __restrict__ entries, uint32_t n_tiles, uint32_t tiles_x, uint32_t cap,
               uint32_t* __restrict__ tile_count) {
  extern __shared__ uint4 tsm[];
  ulonglong2* s_px = reinterpret_cast<ulonglong2*>(tsm);                                     // [64 * 64] word pairs
  float(*s_rec)[32][REC_STRIDE] = reinterpret_cast<float(*)[32][REC_STRIDE]>(tsm + TILE_PX);  // [warps][32][20]
  __shared__ uint32_t s_hz[64 + 16];  // farthest centre depth per 8 x 8 block, then per 16 x 16 block (a valid bound)
  __shared__ uint32_t s_tile, s_next, s_hzc;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  float(*rec)[REC_STRIDE] = s_rec[warp];
  const int W = (int)cam.W, H = (int)cam.H;
  const uint32_t le_mask = 0xFFFFFFFFu >> (31 - lane);
  uint32_t c_hiz = 0;
  for (;;) {
    if (tid == 0) {
      s_tile = (uint32_t)atomicAdd(&counters[CNT_WORK_TILE], 1ull);
      s_next = 0;
      s_hzc = 0;
    }
    __syncthreads();
    if (s_tile >= n_tiles) break;
    const uint32_t tile = __ldg(&tile_order[s_tile]);
    const int x0 = (int)(tile % tiles_x) * HAIR_TILE, y0 = (int)(tile / tiles_x) * HAIR_TILE;
    // ---- the tile starts as k_clear / k_reseed would have left it
    for (uint32_t i = tid; i < TILE_PX; i += TR_WARPS * 32) {
      const uint32_t lx = i & (HAIR_TILE - 1), ly = i / HAIR_TILE;
      const int gx = x0 + (int)lx, gy = y0 + (int)ly;
      uint32_t hi = 0xFFFFFFFFu;
      if (gx < W && gy < H) {
        const size_t p = (size_t)gy * W + gx;
        if (reseed) hi = (uint32_t)(__ldcg(&gbuf[2 * p]) >> 32) | 0xFFu;  // R-seq: depth of the centre word, no hit
        else if (scene_zn) hi = (quant_depth(fminf(fmaxf(__ldg(&scene_zn[p]), 0.f), 1.f)) << 8) | 0xFFu;  // R-scene
      }
      const unsigned long long w = ((unsigned long long)hi << 32) | 0xFFFFFFFFull;
      s_px[tile_idx(lx, ly)] = make_ulonglong2(w, w);
    }
    if (tid < 64 + 16) s_hz[tid] = 0xFFFFFFFFu;
    if (tid == 0) tile_count[tile] = 0;  // the scatter's cursor restarts as the next frame's counter
    __syncthreads();
    const uint32_t n_e = __ldg(&tile_n[tile]), base = __ldg(&tile_base[tile]);
    for (;;) {
      uint32_t b0 = 0;
      if (lane == 0) b0 = atomicAdd(&s_next, 32u);
      b0 = __shfl_sync(0xffffffffu, b0, 0);
      if (b0 >= n_e) break;
      // ---- one record per lane: the setup k_raster does once per segment, clipped to this tile
      const uint32_t ei = b0 + lane;
      uint32_t n_steps = 0;
      if (ei < n_e && base + ei < cap) {
        const float4 q0 = __ldg(&entries[2 * (size_t)(base + ei)]), q1 = __ldg(&entries[2 * (size_t)(base + ei) + 1]);
        const float ax = q0.x, ay = q0.y, bx = q0.z, by = q0.w, azn = q1.x, bzn = q1.y;
        const float dx = xsub(bx, ax), dy = xsub(by, ay);
        const bool ymajor = fabsf(dy) > fabsf(dx);
        const float aM = ymajor ? ay : ax, aN = ymajor ? ax : ay;
        const float bM = ymajor ? by : bx, bN = ymajor ? bx : by;
        const float dM = ymajor ? dy : dx, dN = ymajor ? dx : dy;
        const int tM0 = ymajor ? y0 : x0, tN0 = ymajor ? x0 : y0;
        const float limM = (float)min((ymajor ? H : W) - 1, tM0 + HAIR_TILE - 1);
        const float limN = (float)min((ymajor ? W : H) - 1, tN0 + HAIR_TILE - 1);
        const float fc0 = fmaxf(ceilf(fminf(aM, bM)) - 1.f, (float)tM0), fc1 = fminf(floorf(fmaxf(aM, bM)), limM);
        const float fr0 = fmaxf(ceilf(fminf(aN, bN)) - 1.f, (float)tN0), fr1 = fminf(floorf(fmaxf(aN, bN)), limN);
        bool draw = fc0 <= fc1 && fr0 <= fr1;
        const uint32_t dqm = quant_depth(fminf(fmaxf(fminf(azn, bzn), 0.f), 1.f));
        const uint32_t dq_lim = dqm > 2u ? dqm - 2u : 0u;  // nearest depth a pixel of this segment can store (R11's lerp)
        if (draw) {  // hi-Z of the tile: 3 x 3 blocks of 8 px, else of 16 px, over the clipped box
          const int lx0 = (int)(ymajor ? fr0 : fc0) - x0, lx1 = (int)(ymajor ? fr1 : fc1) - x0;
          const int ly0 = (int)(ymajor ? fc0 : fr0) - y0, ly1 = (int)(ymajor ? fc1 : fr1) - y0;
          int sh = 3, off = 0, pitch = 8;
          if ((lx1 >> 3) - (lx0 >> 3) > 2 || (ly1 >> 3) - (ly0 >> 3) > 2) sh = 4, off = 64, pitch = 4;
          const int bx0 = lx0 >> sh, bx1 = lx1 >> sh, by0 = ly0 >> sh, by1 = ly1 >> sh;
          if (bx1 - bx0 <= 2 && by1 - by0 <= 2) {
            uint32_t zfar = 0;
#pragma unroll
            for (int yy = 0; yy < 3; ++yy)
#pragma unroll
              for (int xx = 0; xx < 3; ++xx) zfar = max(zfar, s_hz[off + min(by0 + yy, by1) * pitch + min(bx0 + xx, bx1)]);
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
          r4[1] = make_float4(dd, xmul(0.5f, xadd(fabsf(dx), fabsf(dy))), azn, xsub(bzn, azn));
          const float slope = dM != 0.f ? dN / dM : 0.f;
          r4[2] = make_float4(aN - aM * slope, slope, __int_as_float((int)fc0),
                              __uint_as_float(((uint32_t)(int)fr0 << 16) | (uint32_t)(int)fr1));
          rec[lane][17] = q1.w;  // rho^2
          r4[3].x = __uint_as_float((ymajor ? 0x80000000u : 0u) | __float_as_uint(q1.z));
          r4[3].w = __uint_as_float(dq_lim);
        }
      }
      // ---- (segment, column) tasks spread over the lanes, as in k_raster
      const uint32_t n_eff = max(n_steps, 1u);
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
      for (uint32_t tb = 0; tb < total; tb += 32) {
        const uint32_t before = __popc(__ballot_sync(0xffffffffu, X < tb));
        const uint32_t startbits = __reduce_or_sync(0xffffffffu, (X >= tb && X < tb + 32) ? 1u << (X - tb) : 0u);
        const uint32_t s = before + __popc(startbits & le_mask) - 1;
        const uint32_t tau = tb + lane;
        if (tau >= total) continue;
        const float4* r4 = reinterpret_cast<const float4*>(rec[s]);
        const float4 q3 = r4[3];
        const uint32_t step = tau - __float_as_uint(q3.y);
        if (step >= __float_as_uint(q3.z)) continue;
        const float4 q0 = r4[0], q1 = r4[1], q2 = r4[2];
        const float aM = q0.x, aN = q0.y, dM = q0.z, dN = q0.w;
        const float dd = q1.x, ext = q1.y, az = q1.z, dz = q1.w;
        const uint32_t key = __float_as_uint(q3.x), dq_min = __float_as_uint(q3.w);
        const bool ymajor = (key >> 31) != 0;
        const int c = __float_as_int(q2.z) + (int)step;
        const int r0 = (int)(__float_as_uint(q2.w) >> 16), r1 = (int)(__float_as_uint(q2.w) & 0xFFFFu);
        const float fc = (float)c;
        const float m0 = fmaf(fc, q2.y, q2.x), m1 = m0 + q2.y;
        const int rlo = max((int)ceilf(fminf(m0, m1) - ENUM_EPS) - 1, r0);
        const int rhi = min((int)floorf(fmaxf(m0, m1) + ENUM_EPS), r1);
        const float cM = fc + 0.5f;
        const float uM = xsub(cM, aM);
        const float rho2 = rec[s][17];
        for (int rb = rlo; rb <= rhi; rb += TR_ROWS) {
          bool ok[TR_ROWS];
          ulonglong2 cur[TR_ROWS];
          uint32_t pidx[TR_ROWS];
#pragma unroll
          for (int i = 0; i < TR_ROWS; ++i) {
            const int r = rb + i;
            const float uN = xsub((float)r + 0.5f, aN);
            const float cr = fabsf(xsub(xmul(dM, uN), xmul(dN, uM)));
            ok[i] = r <= rhi && cr <= ext;  // the cheap half of the conservative predicate (R10)
            pidx[i] = ymajor ? tile_idx((uint32_t)(r - x0), (uint32_t)(c - y0)) : tile_idx((uint32_t)(c - x0), (uint32_t)(r - y0));
            if (ok[i]) cur[i] = s_px[pidx[i]];
          }
#pragma unroll
          for (int i = 0; i < TR_ROWS; ++i) {
            if (!ok[i]) continue;
            if (dq_min > (uint32_t)(cur[i].x >> 40)) continue;  // behind the pixel's centre hit: loses both layers (R10)
            const int r = rb + i;
            const float cN = (float)r + 0.5f;
            const float uN = xsub(cN, aN);
            float tt = 0.f;
            if (dd > 0.f) tt = fminf(fmaxf(xdiv(xadd(xmul(uM, dM), xmul(uN, dN)), dd), 0.f), 1.f);
            const float zn = xadd(az, xmul(tt, dz));
            if (zn < 0.f || zn > 1.f) continue;
            const float eM = xsub(cM, xadd(aM, xmul(tt, dM))), eN = xsub(cN, xadd(aN, xmul(tt, dN)));
            const bool centre = xadd(xmul(eM, eM), xmul(eN, eN)) <= rho2;
            const unsigned long long word = pack_word(zn, (key >> 7) & 0xFFFFFFu, key & 0x7Fu, tt);
            unsigned long long* px = reinterpret_cast<unsigned long long*>(&s_px[pidx[i]]);
            if (word < cur[i].y) atomicMin(px + 1, word);
            if (centre && word < cur[i].x) atomicMin(px, word);
          }
        }
      }
      __syncwarp();
      // ---- refresh the hi-Z of one 16 x 16 block (its four 8 x 8 blocks, then itself); any snapshot is a valid bound
      {
        uint32_t hb = 0;
        if (lane == 0) hb = atomicAdd(&s_hzc, 1u);
        hb = __shfl_sync(0xffffffffu, hb, 0) & 15u;
        const uint32_t bx = (hb & 3u) * 16u, by = (hb >> 2) * 16u;
        const uint32_t px = bx + (lane & 15u), py = by + (lane >> 4);
        uint32_t top = 0, bot = 0;
#pragma unroll
        for (uint32_t k = 0; k < 4; ++k) {
          top = max(top, reinterpret_cast<const uint2*>(&s_px[tile_idx(px, py + 2 * k)])->y >> 8);
          bot = max(bot, reinterpret_cast<const uint2*>(&s_px[tile_idx(px, py + 8 + 2 * k)])->y >> 8);
        }
        const uint32_t half = (lane >> 3) & 1u;  // left / right 8 columns of the block
        const uint32_t m = half ? 0xFF00FF00u : 0x00FF00FFu;
        top = __reduce_max_sync(m, top);
        bot = __reduce_max_sync(m, bot);
        const uint32_t all = __reduce_max_sync(0xffffffffu, max(top, bot));
        if ((lane & 7u) == 0 && lane < 16) {
          const uint32_t b8x = (bx >> 3) + half, b8y = by >> 3;
          s_hz[b8y * 8 + b8x] = top;
          s_hz[(b8y + 1) * 8 + b8x] = bot;
        }
        if (lane == 0) s_hz[64 + (by >> 4) * 4 + (bx >> 4)] = all;
      }
    }
    __syncthreads();
    // ---- flush: one coalesced 16-byte store per pixel
    for (uint32_t i = tid; i < TILE_PX; i += TR_WARPS * 32) {
      const uint32_t lx = i & (HAIR_TILE - 1), ly = i / HAIR_TILE;
      const int gx = x0 + (int)lx, gy = y0 + (int)ly;
      if (gx < W && gy < H) reinterpret_cast<ulonglong2*>(gbuf)[(size_t)gy * W + gx] = s_px[tile_idx(lx, ly)];
    }
    __syncthreads();
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) c_hiz += __shfl_xor_sync(0xffffffffu, c_hiz, d);
  if (lane == 0 && c_hiz) atomicAdd(&counters[CNT_SEG_HIZ], (unsigned long long)c_hiz);
}

// ------------------------------------------------------------------------------------------------ launchers
void launch_bin(bool scatter, const SceneDev* d_scene, uint32_t n_bi, const uint4* table, const uint32_t* grp,
                const float4* vertices, CamDev cam, float rho_default, unsigned long long* counters, int pass,
                TileBufs tb, int n_sm, cudaStream_t st) {
  const uint32_t* gp = grp + (pass ? (size_t)n_bi + 1 : 0);
  const uint32_t q = CNT_WORK_BIN + (scatter ? 2u : 0u) + (pass ? 1u : 0u);
  const uint32_t tiles_x = (cam.W + HAIR_TILE - 1) / HAIR_TILE;
  if (scatter)
    k_bin<true><<<n_sm * 8, 256, 0, st>>>(d_scene, n_bi, table, gp, vertices, cam, rho_default, counters, q, tb.count, tb.base,
                                          tb.entries, tb.cap, tiles_x);
  else
    k_bin<false><<<n_sm * 8, 256, 0, st>>>(d_scene, n_bi, table, gp, vertices, cam, rho_default, counters, q, tb.count, tb.base,
                                           tb.entries, tb.cap, tiles_x);
}

void launch_tile_scan(CamDev cam, TileBufs tb, unsigned long long* counters, cudaStream_t st) {
  const uint32_t n_tiles = ((cam.W + HAIR_TILE - 1) / HAIR_TILE) * ((cam.H + HAIR_TILE - 1) / HAIR_TILE);
  k_tile_scan<<<1, 1024, 0, st>>>(tb.count, tb.base, tb.n, tb.order, n_tiles, tb.cap, counters);
}

void launch_raster_tiled(CamDev cam, unsigned long long* gbuf, const float* scene_zn, bool reseed,
                         unsigned long long* counters, TileBufs tb, int n_sm, LaunchState* ls, cudaStream_t st) {
  const uint32_t tiles_x = (cam.W + HAIR_TILE - 1) / HAIR_TILE, tiles_y = (cam.H + HAIR_TILE - 1) / HAIR_TILE;
  const size_t smem = (size_t)TILE_PX * sizeof(ulonglong2) + (size_t)TR_WARPS * 32 * REC_STRIDE * sizeof(float);
  if (!ls->tiled_per_sm) {  // once per context (the opt-in is per device)
    raise_dyn_smem(k_raster_tiled, smem);
    int b = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k_raster_tiled, TR_WARPS * 32, smem);
    ls->tiled_per_sm = b > 0 ? b : 1;
  }
  uint32_t grid = (uint32_t)(n_sm * ls->tiled_per_sm);
  if (grid > tiles_x * tiles_y) grid = tiles_x * tiles_y;
  k_raster_tiled<<<grid, TR_WARPS * 32, smem, st>>>(cam, gbuf, scene_zn, reseed ? 1u : 0u, counters, tb.order, tb.base, tb.n,
                                                    tb.entries, tiles_x * tiles_y, tiles_x, tb.cap, tb.count);
}
