// k_scan_noalloc.cu — hair_scan_noalloc: H2 scan for callers that must not
// allocate device memory.
//
// Who that is: a renderer that hands all of the GPU's memory to its own pool when it starts and then runs its frame
// loop with nothing left for the CUDA allocator (cudaMalloc fails, or stalls the whole device while it works, in the
// middle of a frame); and a host that forbids allocating calls inside its per-frame section on principle, because
// cudaMalloc / cudaFree synchronise the device. Every other entry point of libhair goes through a hair_ctx, and
// hair_create / hair_mesh_upload / the first hair_render size and cudaMalloc the context's scratch buffers. This one
// needs no context: the caller passes the per-bundle counts and receives the scans, and the one piece of scratch the
// scan needs between its two kernels — the sums of each tile of 256 bundle-instances, which k_lod leaves in the
// context's `part` buffer on the normal path — lives in a fixed array inside the library's device image.
//
// It is the scan of k_lod.cu::k_scan reduced to its two integer scans (slot_base = exclusive scan of N_LOD, vertex_base
// = exclusive scan of N_LOD x C, bundle-instance order); k_lod.cu is not touched and shares nothing with this file.
//
// Rules that follow from the fixed array (also in include/hair.h):
//  - HAIR_SCAN_NOALLOC_MAX bundle-instances at most; 32 KB of device memory per GPU that uses this library, from the
//    moment the library's code is loaded on that GPU until the process exits, whether or not the call is ever made.
//  - One array per device and process, shared by every call: two calls whose kernels can run at the same time on one
//    device (different streams, different host threads) race on it. Calls on one stream are safe back to back.
//  - The array keeps what the last call left in it. Nothing in it has to start at zero: the first kernel of a call
//    rewrites every entry the second kernel of that call reads (tiles 0 .. ceil(n / 256) - 1) and the second reads
//    no entry beyond those, so stale sums of a longer earlier call are never seen.
//  - The first call on a device looks up the array's device address (cudaGetSymbolAddress, which may load the
//    library's device code); make that first call outside any stream capture. Later calls only launch two kernels.
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <mutex>

#include "../../include/hair.h"

namespace {

constexpr uint32_t TILE = 256;  // bundle-instances per CTA, as in k_scan
constexpr uint32_t MAX_TILES = HAIR_SCAN_NOALLOC_MAX / TILE;
constexpr int MAX_DEVICES = 64;
static_assert(HAIR_SCAN_NOALLOC_MAX % TILE == 0, "whole tiles");

// The scratch: {strands, vertices} of every tile. In HOST code this name is only a handle for cudaGetSymbolAddress —
// it is not a device pointer and must never be given to a kernel as one.
static __device__ __align__(256) uint2 g_tile_sums[MAX_TILES];

std::mutex g_setup_mutex;
uint2* g_tile_sums_ptr[MAX_DEVICES] = {};  // device address of g_tile_sums on each device, once looked up
thread_local char g_err[256] = "";

int fail(int code, const char* what, const char* detail) {
  snprintf(g_err, sizeof g_err, "hair_scan_noalloc: %s%s%s", what, detail ? ": " : "", detail ? detail : "");
  return code;
}

// first kernel: the sums of one tile
__global__ void __launch_bounds__(TILE) k_tile_sums_noalloc(const uint2* __restrict__ counts, uint32_t n,
                                                            uint2* __restrict__ tile_sums) {
  __shared__ uint32_t s_s[TILE / 32], s_v[TILE / 32];
  const uint32_t i = blockIdx.x * TILE + threadIdx.x;
  uint32_t s = 0, v = 0;
  if (i < n) {
    const uint2 e = __ldg(&counts[i]);
    s = e.x;
    v = e.x * e.y;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    s += __shfl_xor_sync(0xffffffffu, s, d);
    v += __shfl_xor_sync(0xffffffffu, v, d);
  }
  if ((threadIdx.x & 31) == 0) s_s[threadIdx.x >> 5] = s, s_v[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t a = 0, b = 0;
#pragma unroll
    for (uint32_t w = 0; w < TILE / 32; ++w) a += s_s[w], b += s_v[w];
    tile_sums[blockIdx.x] = make_uint2(a, b);
  }
}

// second kernel: what lies in front of the tile (sums of the tiles before it) + the exclusive scan inside the tile
__global__ void __launch_bounds__(TILE) k_scan_noalloc(const uint2* __restrict__ counts, uint32_t n,
                                                       const uint2* __restrict__ tile_sums, uint2* __restrict__ bases,
                                                       uint32_t* __restrict__ totals) {
  __shared__ uint32_t s_front[TILE / 32][2], s_incl[TILE / 32][2];
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tile = blockIdx.x;
  uint32_t ps = 0, pv = 0;
  for (uint32_t t = threadIdx.x; t < tile; t += TILE) {
    const uint2 a = tile_sums[t];  // written by the kernel before this one: a plain load, not the read-only path
    ps += a.x;
    pv += a.y;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    ps += __shfl_xor_sync(0xffffffffu, ps, d);
    pv += __shfl_xor_sync(0xffffffffu, pv, d);
  }
  const uint32_t i = tile * TILE + threadIdx.x;
  uint32_t s = 0, v = 0;
  if (i < n) {
    const uint2 e = __ldg(&counts[i]);
    s = e.x;
    v = e.x * e.y;
  }
  uint32_t is = s, iv = v;  // inclusive scan over the warp
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t a = __shfl_up_sync(0xffffffffu, is, d), b = __shfl_up_sync(0xffffffffu, iv, d);
    if (lane >= d) is += a, iv += b;
  }
  if (lane == 0) s_front[warp][0] = ps, s_front[warp][1] = pv;
  if (lane == 31) s_incl[warp][0] = is, s_incl[warp][1] = iv;
  __syncthreads();
  uint32_t off_s = 0, off_v = 0;
#pragma unroll
  for (uint32_t w = 0; w < TILE / 32; ++w) {
    off_s += s_front[w][0], off_v += s_front[w][1];
    if (w < warp) off_s += s_incl[w][0], off_v += s_incl[w][1];
  }
  if (i < n) bases[i] = make_uint2(off_s + is - s, off_v + iv - v);
  if (tile == gridDim.x - 1 && threadIdx.x == TILE - 1) totals[0] = off_s + is, totals[1] = off_v + iv;
}

}  // namespace

extern "C" const char* hair_scan_noalloc_error(void) { return g_err; }

extern "C" int hair_scan_noalloc(int cuda_device, void* cuda_stream, const uint32_t* dev_counts, uint32_t n,
                                 uint32_t* dev_bases, uint32_t* dev_totals) {
  g_err[0] = 0;
  // argument checks first: they touch neither CUDA nor the GPU
  if (n > HAIR_SCAN_NOALLOC_MAX) {
    char d[128];
    snprintf(d, sizeof d, "n = %u bundle-instances, the fixed scratch array holds at most HAIR_SCAN_NOALLOC_MAX = %u",
             n, (unsigned)HAIR_SCAN_NOALLOC_MAX);
    return fail(HAIR_E_INVALID_ARG, "size beyond the maximum", d);
  }
  if (!dev_totals || (n > 0 && (!dev_counts || !dev_bases))) return fail(HAIR_E_INVALID_ARG, "null pointer", nullptr);
  if (((uintptr_t)dev_counts | (uintptr_t)dev_bases) & 7u)
    return fail(HAIR_E_INVALID_ARG, "dev_counts and dev_bases must be 8-byte aligned", nullptr);
  if (cuda_device < 0 || cuda_device >= MAX_DEVICES) return fail(HAIR_E_INVALID_ARG, "cuda_device out of range", nullptr);
  cudaError_t e = cudaSetDevice(cuda_device);
  if (e != cudaSuccess) return fail(HAIR_E_CUDA, "cudaSetDevice", cudaGetErrorString(e));
  // set-up, once per device, with that device current: the device address behind the symbol
  uint2* tile_sums = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_tile_sums_ptr[cuda_device]) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_tile_sums);
      if (e != cudaSuccess || !p) return fail(HAIR_E_CUDA, "cudaGetSymbolAddress(g_tile_sums)", cudaGetErrorString(e));
      g_tile_sums_ptr[cuda_device] = (uint2*)p;
    }
    tile_sums = g_tile_sums_ptr[cuda_device];
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const uint32_t n_tiles = n ? (n + TILE - 1) / TILE : 1u;  // n == 0: one empty tile writes the zero totals
  k_tile_sums_noalloc<<<n_tiles, TILE, 0, st>>>((const uint2*)dev_counts, n, tile_sums);
  k_scan_noalloc<<<n_tiles, TILE, 0, st>>>((const uint2*)dev_counts, n, tile_sums, (uint2*)dev_bases, dev_totals);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(HAIR_E_CUDA, "kernel launch", cudaGetErrorString(e));
  return HAIR_OK;
}
