// k_microbench.cu — roofline denominators measured on the box, in the raster's own operations.
//
//  hair_atomic_microbench   64-bit atomicMin with the result unused (RED.E.MIN.64), the raster's write.
//  hair_l2_load_microbench  16-byte ld.global.cg of one G-buffer word pair, the raster's read-before-atomic
//                           ("reads the existing depth buffer"): every candidate pixel of every segment
//                           costs one such load before anything else is known about it, so the rate at which the
//                           memory system returns them is the ceiling of a raster that keeps its G-buffer in L2.
// Both run over a buffer of the G-buffer's size in the access shapes the raster produces.
#include "hair_internal.cuh"

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

// One 16-byte load per lane and step, L2_MLP independent loads in flight per lane (the raster keeps ROW_BATCH = 2
// per lane and 40 warps per SM). A warp's 32 loads of a step form
//  mode 0  "row":    32 consecutive pairs of one image row (512 contiguous bytes: an x-major segment's columns),
//  mode 1  "column": the same x in 32 consecutive rows (stride pitch * 16 bytes: a y-major segment's columns),
//  mode 2  "random": 32 unrelated pairs (sub-pixel segments scattered over the frame),
//  mode 3 / 4  the column / row walk in a G-buffer laid out in blocks of 2 x 4 pixels,
//  mode 5  "column pairs": the column walk with the two minor-axis neighbours of a row requested together, as a
//          y-major task of the raster does (both loads of a lane fall into one 32-byte sector),
// at a hashed position that changes every step. pitch = pairs per image row.
#define L2_MLP 4
__global__ void __launch_bounds__(256) k_l2_load_bench(int mode, const ulonglong2* __restrict__ pairs, uint32_t n_pairs,
                                                       uint32_t pitch, uint32_t n_steps,
                                                       unsigned long long* __restrict__ sink) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gwarp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const uint32_t rows = n_pairs / pitch;
  unsigned long long acc = 0;
  uint32_t h = pcg(gwarp * 0x9E3779B9u + 17u);
  for (uint32_t s = 0; s < n_steps; s += L2_MLP) {
    ulonglong2 v[L2_MLP];
#pragma unroll
    for (int u = 0; u < L2_MLP; ++u) {
      if (mode != 5 || !(u & 1)) h = pcg(h + (uint32_t)u + 1u);
      uint32_t idx;
      if (mode == 0) idx = h % (n_pairs - 32u) + lane;
      else if (mode == 1) idx = ((h >> 12) % (rows - 32u) + lane) * pitch + (h & 0xFFFu) % pitch;
      else if (mode == 2) idx = pcg(h ^ (lane * 0x85EBCA6Bu)) % n_pairs;
      else if (mode == 5)  // column walk, two horizontally adjacent pairs per lane and row (ROW_BATCH = 2 of a y-major task)
        idx = ((h >> 12) % (rows - 32u) + lane) * pitch + (((h & 0xFFFu) % (pitch - 1u)) & ~1u) + ((uint32_t)u & 1u);
      else {  // the same walks in a layout of 2 x 4-pixel blocks (one 128-byte line = 2 columns x 4 rows)
        uint32_t x, y;
        if (mode == 3) x = (h & 0xFFFu) % pitch, y = (h >> 12) % (rows - 32u) + lane;  // column
        else x = h % (pitch - 32u) + lane, y = (h >> 12) % rows;                        // row
        idx = ((y >> 2) * (pitch >> 1) + (x >> 1)) * 8u + (y & 3u) * 2u + (x & 1u);
        if (idx >= n_pairs) idx = n_pairs - 1u;
      }
      v[u] = __ldcg(&pairs[idx]);
    }
#pragma unroll
    for (int u = 0; u < L2_MLP; ++u) acc += v[u].x ^ v[u].y;
  }
  if (acc == 0x0123456789ABCDEFull) sink[0] = acc;  // keeps the loads alive; never true on a cleared buffer
}

void launch_l2_load_microbench(int mode, const unsigned long long* pairs, uint32_t n_pairs, uint32_t pitch,
                               uint32_t n_steps, unsigned long long* sink, int n_sm, cudaStream_t st) {
  k_l2_load_bench<<<n_sm * 8, 256, 0, st>>>(mode, reinterpret_cast<const ulonglong2*>(pairs), n_pairs, pitch, n_steps, sink);
}
