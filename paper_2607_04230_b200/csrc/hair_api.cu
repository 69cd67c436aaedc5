// hair_api.cu — host side of libhair: the C ABI of include/hair.h, the frame scheduler and
// device-buffer ownership. No torch, no exceptions across the boundary.
//
// hair_render enqueues a fixed kernel sequence on the caller's stream:
//   k_lod -> k_scan -> k_generate -> k_clear -> k_raster -> k_shade -> k_filter
// Grid sizes never depend on device results: the LOD-dependent stages are persistent kernels
// that read their work counts from device memory (the CUDA form of the paper's indirect
// dispatch), so no stage waits for the host.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "hair_internal.cuh"

namespace {

struct GroomHost {
  float *pos = nullptr, *ao = nullptr, *xform = nullptr;
  float *pos_stage = nullptr, *ao_stage = nullptr;  // hair_mesh_update from pinned memory lands here first
  uint32_t *idx = nullptr, *npt = nullptr, *off = nullptr, *tri_of = nullptr;
  size_t pos_bytes = 0, ao_bytes = 0;
};

enum { EV_BEGIN = 0, EV_LOD, EV_GEN, EV_CLEAR, EV_RASTER, EV_SHADE, EV_FILTER, EV_N };
const int EV_RING = 64;  // stage timings of up to 64 frames are averaged by hair_stats without a sync in between

}  // namespace

#ifndef HAIR_STAGE_DMA
#define HAIR_STAGE_DMA 1  // hair_mesh_update staging by the copy engine on the second stream (0: by one SM copy kernel)
#endif
struct hair_ctx {
  int device = 0;
  int n_sm = 148;
  cudaStream_t stream = nullptr;
  std::string err;
  SceneDev scene;  // host mirror
  SceneDev* d_scene = nullptr;
  bool scene_dirty = true;
  std::vector<GroomHost> grooms;
  hair_render_params prm;
  // scratch
  uint4* d_table = nullptr;
  uint4* d_part = nullptr;    // [2 ceil(n_bi / 256)] tile sums between k_lod and k_scan
  uint32_t* d_grp = nullptr;  // [2][n_bi + 1] exclusive scans of the work groups of the near and the far raster pass
  uint32_t* d_zrange = nullptr;  // [2][n_inst][2] min / max bundle depth per instance, ping-pong by frame parity
  uint32_t n_inst = 0, zrange_cap = 0, frame_no = 0;
  uint32_t* h_want = nullptr;  // host-mapped: 1 if the last scanned frame was big enough for two raster passes
  uint32_t* d_want = nullptr;  // its device alias (written by k_scan)
  uint32_t* d_hiz = nullptr;  // [ceil(h / 16)][ceil(w / 16)] farthest centre depth per tile between the passes
  size_t hiz_cap = 0;
  // hair_mesh_update from pinned memory: host -> staging copies (cudaMemcpyAsync on aux_stream, i.e. the copy engine,
  // beside the frame before; one SM copy kernel instead with HAIR_STAGE_DMA=0) and staging -> cage copies (one kernel
  // on the stream, in front of the next frame)
  CopyJobs jobs, jobs_apply;
  cudaEvent_t ev_staged = nullptr, ev_applied = nullptr;
  bool applied_once = false;
  size_t table_cap = 0;
  uint2* d_srec = nullptr;  // per strand id: {vertex offset, C | groom << 8} of this frame (k_generate)
  size_t srec_cap = 0;
  float4* d_vertices = nullptr;
  size_t vertex_cap = 0;
  size_t vertex_need = 0;
  float4* d_colour = nullptr;
  size_t colour_cap = 0;
  float4* d_target2 = nullptr;  // hair_render_sequential: second render target of the ping-pong
  size_t target2_cap = 0;
  unsigned long long* d_counters = nullptr;
  unsigned long long* d_sink = nullptr;  // one word the load micro-benchmark may (never does) write
  unsigned long long* h_counters = nullptr;  // pinned
  uint32_t c_max = 0;
  LaunchState ls;  // what this context has configured on its device (opt-in shared memory, occupancy)
  // owned outputs for hair_render_to_host(_async): HAIR_HOST_SLOTS frames in flight
  unsigned long long* d_own_gbuf[HAIR_HOST_SLOTS] = {};
  float* d_own_rgb[HAIR_HOST_SLOTS] = {};
  size_t own_px = 0;
  cudaStream_t copy_stream = nullptr;
  cudaStream_t aux_stream = nullptr;  // the G-buffer clear runs here, beside LOD / scan / generate
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  cudaEvent_t ev_rendered[HAIR_HOST_SLOTS] = {}, ev_copied[HAIR_HOST_SLOTS] = {};
  bool slot_used[HAIR_HOST_SLOTS] = {};
  int next_slot = 0;
  cudaEvent_t ev[EV_RING][EV_N] = {};
  uint32_t ev_frames = 0;  // timed frames since the last hair_stats
  // deep opacity maps (hair_shadow_build): per light z0 + layer counts, the light view's G-buffer (scratch), the
  // device copy of the lights' cameras and map pointers
  DomSet dom;  // host mirror
  DomSet* d_dom = nullptr;
  uint32_t* d_dom_z0[HAIR_MAX_LIGHTS] = {};
  uint4* d_dom_cnt[HAIR_MAX_LIGHTS] = {};
  unsigned long long* d_dom_gbuf = nullptr;
  size_t dom_px = 0;
  bool dom_on = false;
  bool timed = false, counted = false, last_two_pass = false;
  uint32_t last_w = 0, last_h = 0, launches = 0;
  CamDev last_cam;
};

namespace {

int fail(hair_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
#define CK(call)                                                                                  \
  do {                                                                                            \
    cudaError_t e_ = (call);                                                                      \
    if (e_ != cudaSuccess)                                                                        \
      return fail(c, e_ == cudaErrorMemoryAllocation ? HAIR_E_OUT_OF_MEMORY : HAIR_E_CUDA,        \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                            \
  } while (0)

uint32_t pcg_host(uint32_t v) {
  uint32_t s = v * 747796405u + 2891336453u;
  uint32_t w = ((s >> ((s >> 28) + 4u)) ^ s) * 277803737u;
  return (w >> 22) ^ w;
}

CamDev make_cam(const hair_camera* cam, uint32_t w, uint32_t h) {
  CamDev k;
  for (int i = 0; i < 3; ++i) {
    k.eye[i] = cam->eye[i];
    k.r[i] = cam->right[i];
    k.u[i] = cam->up[i];
    k.f[i] = cam->forward[i];
  }
  k.near_z = cam->near_z;
  k.W = w;
  k.H = h;
  // R-proj: constants in double, rounded once to float
  double fpx = (0.5 * (double)h) / std::tan(0.5 * (double)cam->vfov_y);
  double fn = (double)cam->far_z - (double)cam->near_z;
  k.fpx = (float)fpx;
  k.A = (float)((double)cam->far_z / fn);
  k.B = (float)((double)cam->far_z * (double)cam->near_z / fn);
  k.half_w = 0.5f * (float)w;
  k.half_h = 0.5f * (float)h;
  return k;
}

ShadeParams make_shade(const hair_render_params& p) {
  ShadeParams s;
  memset(&s, 0, sizeof(s));
  memcpy(s.light_pos, p.light_pos, sizeof(s.light_pos));
  memcpy(s.light_rgb, p.light_rgb, sizeof(s.light_rgb));
  s.n_lights = p.n_lights > HAIR_MAX_LIGHTS ? HAIR_MAX_LIGHTS : p.n_lights;
  for (int i = 0; i < 3; ++i) {
    s.ambient[i] = p.ambient_rgb[i];
    s.background[i] = p.background_rgb[i];
  }
  s.k_d = p.k_d;
  s.k_R = p.k_R;
  s.k_TRT = p.k_TRT;
  s.r = p.filter_radius;
  const double L2E = 1.4426950408889634;
  double sp = (double)p.filter_radius * (double)p.s_par, sq = (double)p.filter_radius * (double)p.s_perp;
  s.kP = sp > 0 ? (float)(-L2E / (sp * sp)) : 0.f;  // Eq. 10, sigma = r * s
  s.kQ = sq > 0 ? (float)(-L2E / (sq * sq)) : 0.f;
  s.kC = (float)(L2E / ((double)p.sigma_c * (double)p.sigma_c));
  const double e_min = ((double)s.kP + (double)s.kQ) * 2.0 * p.filter_radius * p.filter_radius;  // window corner
  s.bias_nc = (float)std::fmin(std::fmax(-0.5 * e_min, 0.0), 60.0);
  {  // loop B of k_filter: candidates m in [ceil(y* - hmax), ceil(y* - hmax) + nc - 1] cover every integer within hmax of y*
    const double hmax = ((double)p.w_strip + 0.01) * 1.41421357 + 1e-3;
    s.strip_hmax = (float)hmax;
    const double nc = std::floor(2.0 * hmax) + 1.0;
    s.strip_nc = !(p.w_strip >= 0.f) ? 0 : (nc > 2.0 * p.filter_radius + 1.0 ? 2 * p.filter_radius + 1 : (int)nc);
  }
  if (!(p.w_strip >= 0.f)) s.strip_e2_max = -1.f;  // Eq. 9 distance is never negative
  else if (p.w_strip > 1e6f) s.strip_e2_max = 3.0e38f;
  else {  // sqrt_rn(e2) <= w_strip  <=>  e2 <= strip_e2_max (sqrt_rn is monotone; host sqrtf is IEEE)
    float c = (float)((double)p.w_strip * (double)p.w_strip);
    while (std::sqrt(c) <= p.w_strip) c = std::nextafter(c, INFINITY);
    while (c > 0.f && std::sqrt(c) > p.w_strip) c = std::nextafter(c, -INFINITY);
    s.strip_e2_max = c;
  }
  // R20: integer thresholds (depth differences never exceed 2^24 - 2, so clamping changes nothing)
  s.tauz_q = (uint32_t)std::fmin(std::floor((double)p.tau_z * 16777215.0 + 0.5), 16777215.0);
  s.taufly_q = (uint32_t)std::floor((double)p.tau_fly * 16777215.0 + 0.5);
  s.filter_on = (p.flags & HAIR_FLAG_FILTER) ? 1u : 0u;
  s.rho_default = 0.5f * p.center_diameter_px;
  return s;
}

template <class T>
int upload(hair_ctx* c, T** dst, const T* src, size_t n) {
  CK(cudaMalloc((void**)dst, n * sizeof(T)));
  CK(cudaMemcpy(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice));
  return HAIR_OK;
}

void free_groom(GroomHost& g) {
  cudaFree(g.pos);
  cudaFree(g.ao);
  cudaFree(g.xform);
  cudaFree(g.idx);
  cudaFree(g.npt);
  cudaFree(g.off);
  cudaFree(g.tri_of);
  cudaFree(g.pos_stage);
  cudaFree(g.ao_stage);
  g = GroomHost();
}

int ensure_scratch(hair_ctx* c, uint32_t w, uint32_t h) {
  if (c->scene.n_bi > c->table_cap) {
    cudaFree(c->d_table);
    cudaFree(c->d_grp);
    cudaFree(c->d_part);
    c->d_part = nullptr;
    c->d_table = nullptr;
    c->d_grp = nullptr;
    c->table_cap = 0;
    CK(cudaMalloc((void**)&c->d_table, (size_t)c->scene.n_bi * sizeof(uint4)));
    CK(cudaMalloc((void**)&c->d_grp, 2 * ((size_t)c->scene.n_bi + 1) * sizeof(uint32_t)));
    CK(cudaMalloc((void**)&c->d_part, 2 * ((size_t)c->scene.n_bi / 256 + 1) * sizeof(uint4)));
    c->table_cap = c->scene.n_bi;
  }
  if (c->scene.n_strands_total > c->srec_cap) {
    cudaFree(c->d_srec);
    c->d_srec = nullptr;
    c->srec_cap = 0;
    CK(cudaMalloc((void**)&c->d_srec, (size_t)c->scene.n_strands_total * sizeof(uint2)));
    c->srec_cap = c->scene.n_strands_total;
  }
  if (c->vertex_need > c->vertex_cap) {
    cudaFree(c->d_vertices);
    c->d_vertices = nullptr;
    CK(cudaMalloc((void**)&c->d_vertices, (c->vertex_need + 32) * sizeof(float4)));
    c->vertex_cap = c->vertex_need;
  }
  if (c->n_inst > c->zrange_cap) {  // empty ranges: min = a huge float, max = 0 (the first frame then draws in one pass)
    cudaFree(c->d_zrange);
    c->d_zrange = nullptr;
    c->zrange_cap = 0;
    CK(cudaMalloc((void**)&c->d_zrange, (size_t)c->n_inst * 4 * sizeof(uint32_t)));
    std::vector<uint32_t> init((size_t)c->n_inst * 4);
    for (size_t i = 0; i < init.size(); ++i) init[i] = (i & 1) ? 0u : 0x7F000000u;
    CK(cudaMemcpyAsync(c->d_zrange, init.data(), init.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    c->zrange_cap = c->n_inst;
  }
  const size_t n_hiz = (size_t)((w + HIZ_TILE - 1) / HIZ_TILE) * ((h + HIZ_TILE - 1) / HIZ_TILE);
  if (n_hiz > c->hiz_cap) {
    cudaFree(c->d_hiz);
    c->d_hiz = nullptr;
    c->hiz_cap = 0;
    CK(cudaMalloc((void**)&c->d_hiz, n_hiz * sizeof(uint32_t)));
    c->hiz_cap = n_hiz;
  }
  size_t px = (size_t)w * h;
  if (px > c->colour_cap) {
    cudaFree(c->d_colour);
    c->d_colour = nullptr;
    CK(cudaMalloc((void**)&c->d_colour, px * sizeof(float4)));
    c->colour_cap = px;
  }
  if (c->scene_dirty) {
    CK(cudaMemcpyAsync(c->d_scene, &c->scene, sizeof(SceneDev), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));  // host mirror may change after return
    c->scene_dirty = false;
  }
  return HAIR_OK;
}

// hair_mesh_update's queued pinned-memory copies: one kernel for all of them, on the context's stream
void flush_updates(hair_ctx* c) {
  if (!c->jobs.n) return;
  // the bus transfer runs on the second stream — beside whatever the stream is still busy with (the frame before, when
  // the host runs ahead) — once the staging buffers' previous content has been applied; only the device-to-device apply
  // is in front of the next frame. The transfer itself is left to the host-to-device copy engine: an SM copy kernel
  // pulling the cages over the bus (HAIR_STAGE_DMA=0) has to find CTA slots beside the frame's persistent kernels and
  // measured 1.55 ms per pipelined frame against 1.45 ms (the device-to-host copy of the image, which bounds it)
  if (c->applied_once) cudaStreamWaitEvent(c->aux_stream, c->ev_applied, 0);
#if HAIR_STAGE_DMA
  for (int i = 0; i < c->jobs.n; ++i)
    cudaMemcpyAsync(c->jobs.j[i].dst, c->jobs.j[i].src, c->jobs.j[i].n * 4, cudaMemcpyDefault, c->aux_stream);
#else
  launch_copy_jobs(c->jobs, c->aux_stream);
#endif
  cudaEventRecord(c->ev_staged, c->aux_stream);
  cudaStreamWaitEvent(c->stream, c->ev_staged, 0);
  launch_copy_jobs(c->jobs_apply, c->stream);
  cudaEventRecord(c->ev_applied, c->stream);
  c->applied_once = true;
  c->jobs.n = c->jobs_apply.n = 0;
}

// what one pass draws into: R-scene (scene_zn, scene_rgb) and R-seq (grooms of this pass, depth kept in the
// G-buffer from the pass before, alpha accumulated so far in scene_rgb.w)
struct PassOpts {
  const float* scene_zn = nullptr;
  const float* scene_rgb = nullptr;
  uint32_t groom_mask = 0xFFFFFFFFu;
  bool reseed = false;
  bool bg_alpha = false;
  uint32_t ms_k = 0;  // R-msaa: gbuf is [ms_k][h][w] sample layers, resolve instead of shade + filter
  bool final_target = true;  // false: an intermediate target of the sequential passes (stays float under HAIR_FLAG_RGB16F)
};

int render_impl(hair_ctx* c, const hair_camera* cam, uint32_t w, uint32_t h, const float* lam, uint32_t n_lam,
                uint32_t stage_mask, bool front, unsigned long long* gbuf, float* rgb, const PassOpts& po = PassOpts()) {
  const float *scene_zn = po.scene_zn, *scene_rgb = po.scene_rgb;
  if (!c) return HAIR_E_INVALID_ARG;
  if (!cam || !gbuf || !rgb || w == 0 || h == 0 || w > 16384 || h > 16384)
    return fail(c, HAIR_E_INVALID_ARG, "hair_render: null argument or bad resolution");
  if (((uintptr_t)gbuf & 15) || ((uintptr_t)rgb & 15) || ((uintptr_t)scene_rgb & 15) || ((uintptr_t)scene_zn & 3))
    return fail(c, HAIR_E_INVALID_ARG, "hair_render: outputs and scene_rgb must be 16-byte aligned");
  if (!(cam->far_z > cam->near_z) || !(cam->near_z > 0.f) || !(cam->vfov_y > 0.f))
    return fail(c, HAIR_E_INVALID_ARG, "hair_render: bad camera");
  if (front && !(n_lam == 1 || n_lam == c->scene.n_grooms || (n_lam == 0 && lam == nullptr)))
    return fail(c, HAIR_E_INVALID_ARG, "hair_render: n_lambda must be 0, 1 or the number of grooms");
  if (front && n_lam > 0 && lam == nullptr) return fail(c, HAIR_E_INVALID_ARG, "hair_render: lod_lambda is NULL but n_lambda > 0");
  CK(cudaSetDevice(c->device));
  flush_updates(c);
  int rc = ensure_scratch(c, w, h);
  if (rc) return rc;
  const CamDev k = make_cam(cam, w, h);
  ShadeParams sp = make_shade(c->prm);
  sp.bg_alpha = po.bg_alpha ? 1u : 0u;
  sp.rgb16 = ((c->prm.flags & HAIR_FLAG_RGB16F) && po.final_target) ? 1u : 0u;
  sp.shadows = ((c->prm.flags & HAIR_FLAG_SHADOWS) && c->dom_on) ? 1u : 0u;
  // R-payload: the paper's word names no groom, so a pass draws exactly one
  const bool pp = (c->prm.flags & HAIR_FLAG_PAPER_PAYLOAD) != 0;
  sp.paper_payload = pp ? 1u : 0u;
  sp.pp_groom = 0;
  if (pp) {
    if (po.ms_k) return fail(c, HAIR_E_INVALID_ARG, "hair_render_msaa: HAIR_FLAG_PAPER_PAYLOAD is not available in the MSAA reference mode");
    const uint32_t all = c->scene.n_grooms >= 32 ? 0xFFFFFFFFu : ((1u << c->scene.n_grooms) - 1u);
    const uint32_t active = po.groom_mask & c->prm.groom_mask & all;
    if (active == 0 || (active & (active - 1u)))
      return fail(c, HAIR_E_INVALID_ARG, "HAIR_FLAG_PAPER_PAYLOAD: exactly one groom per pass (groom_mask, or hair_render_sequential)");
    while (!((active >> sp.pp_groom) & 1u)) ++sp.pp_groom;
  }
  // the raster generates its own vertices (no vertex buffer); only the paper payload shades without one
  const bool fused = (c->prm.flags & HAIR_FLAG_FUSED) != 0;
  if (fused && (!pp || (c->prm.flags & HAIR_FLAG_COUNTERS)))
    return fail(c, HAIR_E_INVALID_ARG, "HAIR_FLAG_FUSED needs HAIR_FLAG_PAPER_PAYLOAD and no HAIR_FLAG_COUNTERS");
  if (fused && !front) return fail(c, HAIR_E_INVALID_ARG, "hair_render_stages: not with HAIR_FLAG_FUSED");
  const bool timed = (c->prm.flags & HAIR_FLAG_STAGE_TIMING) != 0;
  const bool count = (c->prm.flags & HAIR_FLAG_COUNTERS) != 0;
  const uint32_t n_bi = c->scene.n_bi;
  cudaStream_t st = c->stream;
  uint32_t launches = 0;
  // two depth-ordered raster passes with a tile hi-Z between them (k_raster.cu); the counted and the reference
  // rasters visit every hit, so they draw in one pass
  // and small frames too: k_scan reports through host-mapped memory whether the frame it scanned was big enough,
  // and the next frame launches the hi-Z and the second pass only then (no empty launches, no host sync)
  const bool two_pass = front && !count && !po.ms_k && !(c->prm.flags & HAIR_FLAG_SINGLE_PASS) &&
                        *(volatile uint32_t*)c->h_want != 0u;
  cudaEvent_t* evs = c->ev[c->ev_frames % EV_RING];
  auto mark = [&](int e) {
    if (timed) cudaEventRecord(evs[e], st);
  };
  mark(EV_BEGIN);
  // The clear of the G-buffer does not depend on LOD / scan / generate: it runs beside them on the context's second
  // stream (forked after everything already enqueued on `st`, joined before the raster). ms_clear then reads ~0.
  const bool fork_clear = front && n_bi && (stage_mask & 1u);
  auto clear_on = [&](cudaStream_t cs) -> int {
    if (po.ms_k) CK(cudaMemsetAsync(gbuf, 0xFF, (size_t)w * h * po.ms_k * sizeof(unsigned long long), cs));
    else if (po.reseed) launch_reseed(gbuf, (size_t)w * h, cs);
    else launch_clear(gbuf, (size_t)w * h, scene_zn, cs);
    return HAIR_OK;
  };
  if (fork_clear) {
    CK(cudaEventRecord(c->ev_fork, st));
    CK(cudaStreamWaitEvent(c->aux_stream, c->ev_fork, 0));
    rc = clear_on(c->aux_stream);
    if (rc) return rc;
    CK(cudaEventRecord(c->ev_join, c->aux_stream));
    ++launches;
  }
  if (front && !n_bi) CK(cudaMemsetAsync(c->d_counters, 0, CNT_N * sizeof(unsigned long long), st));
  if (front && n_bi) {
    LambdaArr la;
    for (uint32_t i = 0; i < HAIR_MAX_GROOMS; ++i) la.v[i] = n_lam == 0 ? 0.f : lam[n_lam == 1 ? 0 : (i < n_lam ? i : 0)];
    launch_lod_scan(c->d_scene, n_bi, k, la, po.groom_mask & c->prm.groom_mask, c->d_table, c->d_grp, c->d_part,
                    c->d_counters, c->d_zrange, c->n_inst, c->frame_no++, two_pass, c->d_want, st);
    launches += 2;
  }
  mark(EV_LOD);
  if (front && n_bi && !fused) {
    launch_generate(c->d_scene, n_bi, c->d_table, c->d_vertices, c->d_srec, c->d_counters, c->c_max, c->n_sm, &c->ls, st);
    ++launches;
  }
  mark(EV_GEN);
  if (fork_clear) CK(cudaStreamWaitEvent(st, c->ev_join, 0));
  else if (stage_mask & 1u) {
    rc = clear_on(st);
    if (rc) return rc;
    ++launches;
  }
  mark(EV_CLEAR);
  if ((stage_mask & 1u) && n_bi) {
    if (!front) {  // the table (and its pass split) is the last frame's: restart both queues
      CK(cudaMemsetAsync(c->d_counters + CNT_WORK_RASTER, 0, sizeof(unsigned long long), st));
      CK(cudaMemsetAsync(c->d_counters + CNT_WORK_RASTER1, 0, sizeof(unsigned long long), st));
    }
    launch_raster(c->d_scene, n_bi, c->d_table, c->d_grp, c->d_vertices, k, sp.rho_default, gbuf, c->d_counters,
                  count && !po.ms_k, po.ms_k, pp, 0, nullptr, c->n_sm, &c->ls, st, fused ? c->c_max : 0u);
    ++launches;
    if (two_pass || (!front && c->last_two_pass)) {
      launch_hiz(gbuf, w, h, c->d_hiz, c->d_counters, st);
      launch_raster(c->d_scene, n_bi, c->d_table, c->d_grp, c->d_vertices, k, sp.rho_default, gbuf, c->d_counters,
                    false, 0, pp, 1, c->d_hiz, c->n_sm, &c->ls, st, fused ? c->c_max : 0u);
      launches += 2;
    }
  }
  mark(EV_RASTER);
  if (po.ms_k) {
    launch_resolve_msaa(c->d_scene, c->d_srec, c->d_vertices, k, sp, gbuf, po.ms_k, (const float4*)scene_rgb,
                        (float4*)rgb, c->d_dom, c->d_counters, st);
    ++launches;
  }
  if ((stage_mask & 2u) && !po.ms_k) {
    launch_shade(c->d_scene, c->d_srec, c->d_vertices, k, sp, gbuf, c->d_colour, c->d_dom, c->d_counters, st);
    ++launches;
  }
  mark(EV_SHADE);
  if ((stage_mask & 4u) && !po.ms_k) {
    launches += launch_filter(c->d_scene, c->d_srec, c->d_vertices, k, sp, gbuf, c->d_colour,
                              (const float4*)scene_rgb, (float4*)rgb, c->d_counters, count, &c->ls, st);
  }
  mark(EV_FILTER);
  CK(cudaGetLastError());
  c->timed = timed;
  if (timed) ++c->ev_frames;
  c->counted = count;
  if (front) c->last_two_pass = two_pass;
  c->last_w = w;
  c->last_h = h;
  c->launches = launches;
  c->last_cam = k;
  return HAIR_OK;
}

}  // namespace

extern "C" {

int hair_create(hair_ctx** out, int cuda_device, void* cuda_stream) {
  if (!out) return HAIR_E_INVALID_ARG;
  *out = nullptr;
  int n = 0;
  if (cudaGetDeviceCount(&n) != cudaSuccess || cuda_device < 0 || cuda_device >= n) return HAIR_E_CUDA;
  hair_ctx* c = new hair_ctx();
  c->device = cuda_device;
  c->stream = (cudaStream_t)cuda_stream;
  memset(&c->scene, 0, sizeof(c->scene));
  hair_default_render_params(&c->prm);
  bool ok = cudaSetDevice(cuda_device) == cudaSuccess &&
            cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, cuda_device) == cudaSuccess &&
            cudaMalloc((void**)&c->d_scene, sizeof(SceneDev)) == cudaSuccess &&
            cudaMalloc((void**)&c->d_counters, CNT_N * sizeof(unsigned long long)) == cudaSuccess &&
            cudaMalloc((void**)&c->d_sink, sizeof(unsigned long long)) == cudaSuccess &&
            cudaMemset(c->d_counters, 0, CNT_N * sizeof(unsigned long long)) == cudaSuccess &&
            cudaMallocHost((void**)&c->h_counters, CNT_N * sizeof(unsigned long long)) == cudaSuccess &&
            cudaHostAlloc((void**)&c->h_want, sizeof(uint32_t), cudaHostAllocMapped) == cudaSuccess &&
            cudaHostGetDevicePointer((void**)&c->d_want, c->h_want, 0) == cudaSuccess;
  if (ok) *c->h_want = 0u;
  for (int f = 0; ok && f < EV_RING; ++f)
    for (int i = 0; ok && i < EV_N; ++i) ok = cudaEventCreate(&c->ev[f][i]) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) == cudaSuccess &&
       cudaStreamCreateWithFlags(&c->aux_stream, cudaStreamNonBlocking) == cudaSuccess &&
       cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) == cudaSuccess &&
       cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) == cudaSuccess &&
       cudaEventCreateWithFlags(&c->ev_staged, cudaEventDisableTiming) == cudaSuccess &&
       cudaEventCreateWithFlags(&c->ev_applied, cudaEventDisableTiming) == cudaSuccess;
  for (int k = 0; ok && k < HAIR_HOST_SLOTS; ++k)
    ok = cudaEventCreateWithFlags(&c->ev_rendered[k], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->ev_copied[k], cudaEventDisableTiming) == cudaSuccess;
  if (!ok) {
    hair_destroy(c);
    return HAIR_E_CUDA;
  }
  *out = c;
  return HAIR_OK;
}

void hair_destroy(hair_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->device);
  c->jobs.n = c->jobs_apply.n = 0;  // queued cage updates are dropped, not read: their host arrays may be gone already
  cudaStreamSynchronize(c->stream);
  cudaStreamSynchronize(c->aux_stream);
  for (auto& g : c->grooms) free_groom(g);
  cudaFree(c->d_scene);
  cudaFree(c->d_table);
  cudaFree(c->d_grp);
  cudaFree(c->d_part);
  cudaFree(c->d_vertices);
  cudaFree(c->d_srec);
  cudaFree(c->d_colour);
  cudaFree(c->d_target2);
  cudaFree(c->d_zrange);
  cudaFree(c->d_hiz);
  cudaFree(c->d_counters);
  cudaFree(c->d_sink);
  cudaFree(c->d_dom);
  cudaFree(c->d_dom_gbuf);
  for (int l = 0; l < HAIR_MAX_LIGHTS; ++l) {
    cudaFree(c->d_dom_z0[l]);
    cudaFree(c->d_dom_cnt[l]);
  }
  if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);
  for (int k = 0; k < HAIR_HOST_SLOTS; ++k) {
    cudaFree(c->d_own_gbuf[k]);
    cudaFree(c->d_own_rgb[k]);
    if (c->ev_rendered[k]) cudaEventDestroy(c->ev_rendered[k]);
    if (c->ev_copied[k]) cudaEventDestroy(c->ev_copied[k]);
  }
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->aux_stream) {
    cudaStreamSynchronize(c->aux_stream);
    cudaStreamDestroy(c->aux_stream);
  }
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_join) cudaEventDestroy(c->ev_join);
  if (c->ev_staged) cudaEventDestroy(c->ev_staged);
  if (c->ev_applied) cudaEventDestroy(c->ev_applied);
  if (c->h_counters) cudaFreeHost(c->h_counters);
  if (c->h_want) cudaFreeHost(c->h_want);
  for (int f = 0; f < EV_RING; ++f)
    for (int i = 0; i < EV_N; ++i)
      if (c->ev[f][i]) cudaEventDestroy(c->ev[f][i]);
  delete c;
}

const char* hair_last_error(const hair_ctx* c) { return c ? c->err.c_str() : "null context"; }

void hair_default_render_params(hair_render_params* p) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->center_diameter_px = 0.5f;
  p->filter_radius = 5;
  p->s_par = 0.5f;
  p->s_perp = 0.15f;
  p->sigma_c = 0.9f;
  p->tau_z = 1.45e-3f;
  p->tau_fly = 5e-4f;
  p->w_strip = 0.5f;
  p->n_lights = 0;
  p->ambient_rgb[0] = p->ambient_rgb[1] = p->ambient_rgb[2] = 0.15f;
  p->k_d = 0.4f;
  p->k_R = 0.25f;
  p->k_TRT = 0.5f;
  p->flags = HAIR_FLAG_FILTER;
  p->groom_mask = 0xFFFFFFFFu;
}

int hair_set_render_params(hair_ctx* c, const hair_render_params* p) {
  if (!c || !p) return HAIR_E_INVALID_ARG;
  if (p->filter_radius < 0 || p->filter_radius > 7) return fail(c, HAIR_E_INVALID_ARG, "filter_radius must be 0..7");
  if (p->n_lights > HAIR_MAX_LIGHTS) return fail(c, HAIR_E_INVALID_ARG, "too many lights");
  if (!(p->center_diameter_px > 0.f) || p->center_diameter_px > 1.f)
    return fail(c, HAIR_E_INVALID_ARG, "center_diameter_px must be in (0, 1] (centre layer inside conservative)");
  if (!(p->sigma_c > 0.f)) return fail(c, HAIR_E_INVALID_ARG, "sigma_c must be positive");
  c->prm = *p;
  return HAIR_OK;
}

int hair_mesh_upload(hair_ctx* c, const hair_cage* cage, const hair_roots* roots, const hair_style* st,
                     int* out_groom_id) {
  if (!c) return HAIR_E_INVALID_ARG;
  if (!cage || !roots || !st || !cage->pos || !roots->idx || !roots->strands_per_tri)
    return fail(c, HAIR_E_INVALID_ARG, "hair_mesh_upload: null argument");
  if (cage->n_layers < 2 || cage->n_layers > 32 || cage->n_verts == 0 || roots->n_tris == 0 || st->spi == 0)
    return fail(c, HAIR_E_INVALID_ARG, "hair_mesh_upload: need 2..32 layers, >= 1 triangle, spi >= 1");
  if (c->scene.n_grooms >= HAIR_MAX_GROOMS) return fail(c, HAIR_E_TOO_MANY_GROOMS, "too many grooms");
  const uint32_t c_full = (cage->n_layers - 1) * st->spi + 1;
  if (c_full > 127) return fail(c, HAIR_E_TOO_MANY_CPS, "C_full = (n_layers-1)*spi+1 exceeds 127");
  const uint32_t T = roots->n_tris, Q = st->n_instances ? st->n_instances : 1;
  for (size_t i = 0; i < (size_t)T * 3; ++i)
    if (roots->idx[i] >= cage->n_verts) return fail(c, HAIR_E_INVALID_ARG, "triangle index out of range");
  std::vector<uint32_t> off(T + 1);
  uint64_t acc = 0;
  for (uint32_t t = 0; t < T; ++t) {
    off[t] = (uint32_t)acc;
    acc += roots->strands_per_tri[t];
  }
  off[T] = (uint32_t)acc;
  const uint64_t N = acc;
  const uint32_t gi = c->scene.n_grooms;
  uint32_t sid_base = 0, gid_base = 0;
  if (gi > 0) {
    const GroomDev& p = c->scene.g[gi - 1];
    sid_base = p.sid_base + p.N * p.Q;
    gid_base = p.gid_base + p.T * p.Q;
  }
  if (N == 0) return fail(c, HAIR_E_INVALID_ARG, "groom has no strands");
  if ((uint64_t)sid_base + N * Q >= (1ull << 24)) return fail(c, HAIR_E_TOO_MANY_STRANDS, "more than 2^24 strand ids");
  if ((uint64_t)c->vertex_need + N * Q * c_full >= (1ull << 32)) return fail(c, HAIR_E_TOO_MANY_STRANDS, "vertex index overflow");
  CK(cudaSetDevice(c->device));
  GroomHost gh;
  GroomDev gd;
  memset(&gd, 0, sizeof(gd));
  gh.pos_bytes = (size_t)cage->n_layers * cage->n_verts * 3 * sizeof(float);
  gh.ao_bytes = (size_t)cage->n_layers * cage->n_verts * sizeof(float);
  int rc = upload(c, &gh.pos, cage->pos, (size_t)cage->n_layers * cage->n_verts * 3);
  if (!rc && cage->ao) rc = upload(c, &gh.ao, cage->ao, (size_t)cage->n_layers * cage->n_verts);
  if (!rc) rc = upload(c, &gh.idx, roots->idx, (size_t)T * 3);
  if (!rc) rc = upload(c, &gh.npt, roots->strands_per_tri, (size_t)T);
  if (!rc) rc = upload(c, &gh.off, off.data(), (size_t)T + 1);
  if (!rc) {
    std::vector<uint32_t> tri_of((size_t)N);
    for (uint32_t t = 0; t < T; ++t)
      for (uint32_t i = off[t]; i < off[t + 1]; ++i) tri_of[i] = t;
    rc = upload(c, &gh.tri_of, tri_of.data(), (size_t)N);
  }
  if (!rc && st->instance_xform) rc = upload(c, &gh.xform, st->instance_xform, (size_t)Q * 12);
  if (rc) {
    free_groom(gh);
    return rc;
  }
  gd.pos = gh.pos;
  gd.ao = gh.ao;
  gd.idx = gh.idx;
  gd.npt = gh.npt;
  gd.off = gh.off;
  gd.tri_of = gh.tri_of;
  gd.xform = gh.xform;
  gd.V = cage->n_verts;
  gd.Lv = cage->n_layers;
  gd.T = T;
  gd.Q = Q;
  gd.N = (uint32_t)N;
  gd.sid_base = sid_base;
  gd.gid_base = gid_base;
  gd.inst_base = c->n_inst;
  gd.c_full = c_full;
  gd.spi = st->spi;
  gd.seed_h = pcg_host(st->seed);
  gd.op_mask = st->op_mask;
  gd.clump_exp = st->clump_exp;
  gd.frizz_cells = st->frizz_cells;
  gd.clump_strength = st->clump_strength;
  gd.twist_turns = st->twist_turns;
  gd.curl_radius = st->curl_radius;
  gd.curl_turns = st->curl_turns;
  gd.curl_ramp_w0 = st->curl_ramp_w0;
  gd.frizz_sigma = st->frizz_sigma;
  gd.frizz_ramp_w0 = st->frizz_ramp_w0;
  gd.width_world = st->width_world;
  for (int i = 0; i < 3; ++i) {
    gd.albedo_root[i] = st->albedo_root[i];
    gd.albedo_tip[i] = st->albedo_tip[i];
  }
  gd.roughness = st->roughness;
  gd.tilt = st->tilt;
  c->scene.g[gi] = gd;
  c->scene.n_grooms = gi + 1;
  c->scene.n_bi = gid_base + T * Q;
  c->scene.n_strands_total = sid_base + (uint32_t)N * Q;
  c->n_inst += Q;
  c->vertex_need += (size_t)N * Q * c_full;
  if (c_full > c->c_max) c->c_max = c_full;
  c->grooms.push_back(gh);
  c->scene_dirty = true;
  if (out_groom_id) *out_groom_id = (int)gi;
  return HAIR_OK;
}

int hair_mesh_update(hair_ctx* c, int groom_id, const hair_cage* cage) {
  if (!c) return HAIR_E_INVALID_ARG;
  if (groom_id < 0 || (uint32_t)groom_id >= c->scene.n_grooms || !cage || !cage->pos)
    return fail(c, HAIR_E_INVALID_ARG, "hair_mesh_update: bad groom or cage");
  const GroomDev& gd = c->scene.g[groom_id];
  if (cage->n_layers != gd.Lv || cage->n_verts != gd.V) return fail(c, HAIR_E_INVALID_ARG, "hair_mesh_update: size mismatch");
  GroomHost& gh = c->grooms[groom_id];
  // Pinned host memory: the update is only QUEUED here. flush_updates, called by the next hair_render* / hair_stats /
  // hair_shadow_build, sends every queued array to a per-groom staging buffer with the copy engine on the second
  // stream (HAIR_STAGE_DMA=1; beside whatever the main stream is still running) and then applies staging -> cage with
  // one device-to-device kernel on the main stream in front of the frame. So the host arrays are read AFTER that later
  // call is issued and must stay valid until its frame has completed. Ten small cudaMemcpyAsync per frame on the main
  // stream (five grooms x positions, AO), each a bus round trip of its own while the previous frame's 66-133 MB image is
  // on its way to the host, held the next frame's kernels back by 0.6 ms (2.11 against 1.51 ms per pipelined frame).
  // Pageable memory: the queue is flushed (call order of updates is kept) and the copy is a cudaMemcpyAsync here.
  auto put = [&](float* dst, float** stage, const float* src, size_t bytes) -> int {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, src) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer) {
      if (!*stage) CK(cudaMalloc((void**)stage, bytes));
      if (c->jobs.n == COPY_JOBS_MAX) flush_updates(c);
      c->jobs.j[c->jobs.n++] = CopyJob{(uint32_t*)*stage, (const uint32_t*)at.devicePointer, bytes / 4};
      c->jobs_apply.j[c->jobs_apply.n++] = CopyJob{(uint32_t*)dst, (const uint32_t*)*stage, bytes / 4};
      return HAIR_OK;
    }
    cudaGetLastError();  // (an unregistered pointer may leave an error behind on old drivers)
    flush_updates(c);  // updates queued earlier go first: the newest data of a groom is the one that stays
    CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, c->stream));
    return HAIR_OK;
  };
  int rc = put(gh.pos, &gh.pos_stage, cage->pos, gh.pos_bytes);
  if (rc) return rc;
  if (cage->ao && gh.ao) rc = put(gh.ao, &gh.ao_stage, cage->ao, gh.ao_bytes);
  return rc;
}

int hair_mesh_clear(hair_ctx* c) {
  if (!c) return HAIR_E_INVALID_ARG;
  c->jobs.n = c->jobs_apply.n = 0;  // queued updates of the grooms being removed are dropped, their host arrays not read
  cudaStreamSynchronize(c->stream);
  cudaStreamSynchronize(c->aux_stream);  // (staging copies of an earlier flush write into buffers free_groom releases)
  for (auto& g : c->grooms) free_groom(g);
  c->grooms.clear();
  memset(&c->scene, 0, sizeof(c->scene));
  c->vertex_need = 0;
  c->c_max = 0;
  c->n_inst = 0;
  c->zrange_cap = 0;  // the per-instance depth ranges of the two-pass split restart empty (one pass on the next frame)
  c->frame_no = 0;
  if (c->h_want) *c->h_want = 0u;
  c->last_two_pass = false;
  c->scene_dirty = true;
  c->dom_on = false;  // the maps were built from the grooms just removed
  return HAIR_OK;
}

int hair_render(hair_ctx* c, const hair_camera* cam, uint32_t w, uint32_t h, const float* lam, uint32_t n_lam,
                uint64_t* out_gbuffer, float* out_rgb) {
  return render_impl(c, cam, w, h, lam, n_lam, 7u, true, (unsigned long long*)out_gbuffer, out_rgb);
}

int hair_render_scene(hair_ctx* c, const hair_camera* cam, uint32_t w, uint32_t h, const float* lam, uint32_t n_lam,
                      const float* scene_zn, const float* scene_rgb, uint64_t* out_gbuffer, float* out_rgb) {
  PassOpts po;
  po.scene_zn = scene_zn;
  po.scene_rgb = scene_rgb;
  return render_impl(c, cam, w, h, lam, n_lam, 7u, true, (unsigned long long*)out_gbuffer, out_rgb, po);
}

int hair_render_msaa(hair_ctx* c, const hair_camera* cam, uint32_t w, uint32_t h, const float* lam, uint32_t n_lam,
                     uint32_t k, uint64_t* out_samples, float* out_rgb) {
  if (!c) return HAIR_E_INVALID_ARG;
  if (k != 1 && k != 2 && k != 4 && k != 8) return fail(c, HAIR_E_INVALID_ARG, "hair_render_msaa: k must be 1, 2, 4 or 8");
  PassOpts po;
  po.ms_k = k;
  return render_impl(c, cam, w, h, lam, n_lam, 7u, true, (unsigned long long*)out_samples, out_rgb, po);
}

int hair_render_sequential(hair_ctx* c, const hair_camera* cam, uint32_t w, uint32_t h, const float* lam,
                           uint32_t n_lam, const float* scene_zn, const float* scene_rgb, uint64_t* out_gbuffer,
                           float* out_rgb) {
  if (!c) return HAIR_E_INVALID_ARG;
  const uint32_t n = c->scene.n_grooms;
  if (n <= 1) return hair_render_scene(c, cam, w, h, lam, n_lam, scene_zn, scene_rgb, out_gbuffer, out_rgb);
  CK(cudaSetDevice(c->device));
  const size_t px = (size_t)w * h;
  if (px > c->target2_cap) {  // the second render target of the ping-pong
    cudaFree(c->d_target2);
    c->d_target2 = nullptr;
    c->target2_cap = 0;
    CK(cudaMalloc((void**)&c->d_target2, px * sizeof(float4)));
    c->target2_cap = px;
  }
  uint32_t launches = 0;
  const float* target_in = scene_rgb;
  uint32_t n_pass = 0, i_pass = 0;
  for (uint32_t g = 0; g < n; ++g) n_pass += (c->prm.groom_mask >> g) & 1u;
  if (n_pass <= 1) return hair_render_scene(c, cam, w, h, lam, n_lam, scene_zn, scene_rgb, out_gbuffer, out_rgb);
  for (uint32_t g = 0; g < n; ++g) {
    if (!((c->prm.groom_mask >> g) & 1u)) continue;
    // the last pass must land in out_rgb: passes alternate between the two targets, counted from the end
    float* target_out = ((n_pass - 1 - i_pass) & 1u) ? (float*)c->d_target2 : out_rgb;
    PassOpts po;
    po.scene_zn = i_pass == 0 ? scene_zn : nullptr;
    po.scene_rgb = target_in;
    po.groom_mask = 1u << g;
    po.reseed = i_pass > 0;
    po.bg_alpha = i_pass > 0;
    ++i_pass;
    po.final_target = i_pass == n_pass;
    int rc = render_impl(c, cam, w, h, lam, n_lam, 7u, true, (unsigned long long*)out_gbuffer, target_out, po);
    if (rc) return rc;
    launches += c->launches;
    target_in = target_out;
  }
  c->launches = launches;
  return HAIR_OK;
}

int hair_render_stages(hair_ctx* c, const hair_camera* cam, uint32_t w, uint32_t h, uint32_t stage_mask,
                       uint64_t* out_gbuffer, float* out_rgb) {
  return render_impl(c, cam, w, h, nullptr, 0, stage_mask & 7u, false, (unsigned long long*)out_gbuffer, out_rgb);
}

int hair_render_to_host_async(hair_ctx* c, const hair_camera* cam, uint32_t w, uint32_t h, const float* lam,
                              uint32_t n_lam, uint64_t* host_gbuffer, float* host_rgb, int* out_slot) {
  if (!c) return HAIR_E_INVALID_ARG;
  if (!host_rgb) return fail(c, HAIR_E_INVALID_ARG, "hair_render_to_host: host_rgb is required");
  CK(cudaSetDevice(c->device));
  const size_t px = (size_t)w * h;
  if (px > c->own_px) {
    CK(cudaStreamSynchronize(c->copy_stream));  // copies out of the old buffers
    CK(cudaStreamSynchronize(c->stream));
    for (int k = 0; k < HAIR_HOST_SLOTS; ++k) {
      cudaFree(c->d_own_gbuf[k]);
      cudaFree(c->d_own_rgb[k]);
      c->d_own_gbuf[k] = nullptr;
      c->d_own_rgb[k] = nullptr;
      c->slot_used[k] = false;
    }
    c->own_px = 0;
    for (int k = 0; k < HAIR_HOST_SLOTS; ++k) {
      CK(cudaMalloc((void**)&c->d_own_gbuf[k], px * 16));
      CK(cudaMalloc((void**)&c->d_own_rgb[k], px * 16));
    }
    c->own_px = px;
  }
  const int k = c->next_slot;
  // the slot's previous copies must have left before its buffers are overwritten (stream-ordered, no host wait)
  if (c->slot_used[k]) CK(cudaStreamWaitEvent(c->stream, c->ev_copied[k], 0));
  int rc = render_impl(c, cam, w, h, lam, n_lam, 7u, true, c->d_own_gbuf[k], c->d_own_rgb[k]);
  if (rc) return rc;
  CK(cudaEventRecord(c->ev_rendered[k], c->stream));
  CK(cudaStreamWaitEvent(c->copy_stream, c->ev_rendered[k], 0));
  CK(cudaMemcpyAsync(host_rgb, c->d_own_rgb[k], px * ((c->prm.flags & HAIR_FLAG_RGB16F) ? 8 : 16), cudaMemcpyDeviceToHost,
                     c->copy_stream));
  if (host_gbuffer) CK(cudaMemcpyAsync(host_gbuffer, c->d_own_gbuf[k], px * 16, cudaMemcpyDeviceToHost, c->copy_stream));
  CK(cudaEventRecord(c->ev_copied[k], c->copy_stream));
  c->slot_used[k] = true;
  c->next_slot = (k + 1) % HAIR_HOST_SLOTS;
  if (out_slot) *out_slot = k;
  return HAIR_OK;
}

int hair_host_wait(hair_ctx* c, int slot) {
  if (!c) return HAIR_E_INVALID_ARG;
  if (slot >= HAIR_HOST_SLOTS) return fail(c, HAIR_E_INVALID_ARG, "hair_host_wait: no such slot");
  CK(cudaSetDevice(c->device));
  for (int k = 0; k < HAIR_HOST_SLOTS; ++k)
    if ((slot < 0 || slot == k) && c->slot_used[k]) CK(cudaEventSynchronize(c->ev_copied[k]));
  return HAIR_OK;
}

int hair_render_to_host(hair_ctx* c, const hair_camera* cam, uint32_t w, uint32_t h, const float* lam,
                        uint32_t n_lam, uint64_t* host_gbuffer, float* host_rgb) {
  int slot = -1;
  int rc = hair_render_to_host_async(c, cam, w, h, lam, n_lam, host_gbuffer, host_rgb, &slot);
  if (rc) return rc;
  rc = hair_host_wait(c, slot);
  if (rc) return rc;
  CK(cudaStreamSynchronize(c->stream));
  return HAIR_OK;
}

// PAPER.md:192 / DESIGN.md R-dom: one light view per light through LOD (off) -> generate -> clear -> raster (the
// conservative layer is z0), then the same segments once more, every conservative hit counted into its layer
int hair_shadow_build(hair_ctx* c, const hair_shadow_params* p) {
  if (!c) return HAIR_E_INVALID_ARG;
  if (!p || p->n_lights == 0 || p->n_lights > HAIR_MAX_LIGHTS || p->res < 16 || p->res > 8192 || !(p->layer_d1 > 0.f) ||
      !(p->alpha_s >= 0.f))
    return fail(c, HAIR_E_INVALID_ARG, "hair_shadow_build: bad parameters");
  if (!c->scene.n_bi) return fail(c, HAIR_E_INVALID_ARG, "hair_shadow_build: no groom uploaded");
  CK(cudaSetDevice(c->device));
  const uint32_t S = p->res;
  const size_t px = (size_t)S * S;
  if (px != c->dom_px) {
    for (int l = 0; l < HAIR_MAX_LIGHTS; ++l) {
      cudaFree(c->d_dom_z0[l]);
      cudaFree(c->d_dom_cnt[l]);
      c->d_dom_z0[l] = nullptr;
      c->d_dom_cnt[l] = nullptr;
    }
    cudaFree(c->d_dom_gbuf);
    c->d_dom_gbuf = nullptr;
    c->dom_px = 0;
    CK(cudaMalloc((void**)&c->d_dom_gbuf, px * 2 * sizeof(unsigned long long)));
    c->dom_px = px;
  }
  if (!c->d_dom) CK(cudaMalloc((void**)&c->d_dom, sizeof(DomSet)));
  c->dom_on = false;
  memset(&c->dom, 0, sizeof(c->dom));
  const double d1 = std::floor((double)p->layer_d1 * 16777215.0 + 0.5);
  const uint32_t D1 = (uint32_t)std::fmin(std::fmax(d1, 1.0), 1000000.0);
  const hair_render_params saved = c->prm;
  c->prm.flags = HAIR_FLAG_SINGLE_PASS;  // plain strand-id words, one raster pass, no timing
  c->prm.groom_mask = 0xFFFFFFFFu;
  int rc = HAIR_OK;
  for (uint32_t l = 0; l < p->n_lights && rc == HAIR_OK; ++l) {
    if (!c->d_dom_z0[l]) {
      if (cudaMalloc((void**)&c->d_dom_z0[l], px * sizeof(uint32_t)) != cudaSuccess ||
          cudaMalloc((void**)&c->d_dom_cnt[l], px * sizeof(uint4)) != cudaSuccess) {
        rc = fail(c, HAIR_E_OUT_OF_MEMORY, "hair_shadow_build: out of device memory");
        break;
      }
    }
    const float lam0 = 0.f;  // the maps are built from the full groom
    rc = render_impl(c, &p->cam[l], S, S, &lam0, 1, 1u, true, c->d_dom_gbuf, (float*)c->d_dom_gbuf);
    if (rc) break;
    DomLight& L = c->dom.l[l];
    L.cam = c->last_cam;
    L.z0 = c->d_dom_z0[l];
    L.cnt = c->d_dom_cnt[l];
    L.D[0] = D1, L.D[1] = 3u * D1, L.D[2] = 7u * D1, L.D[3] = 15u * D1;
    L.alpha_s = p->alpha_s;
    L.on = 1u;
    cudaMemsetAsync(c->d_dom_cnt[l], 0, px * sizeof(uint4), c->stream);
    cudaMemsetAsync(c->d_counters + CNT_WORK_RASTER, 0, sizeof(unsigned long long), c->stream);
    launch_raster_dom(c->d_scene, c->scene.n_bi, c->d_table, c->d_grp, c->d_vertices, L.cam, 0.5f * c->prm.center_diameter_px,
                      c->d_dom_gbuf, c->d_counters, reinterpret_cast<uint32_t*>(c->d_dom_cnt[l]),
                      make_uint3(L.D[0], L.D[1], L.D[2]), c->n_sm, &c->ls, c->stream);
    launch_dom_z0(c->d_dom_gbuf, px, c->d_dom_z0[l], c->stream);
  }
  c->prm = saved;
  if (rc) return rc;
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(c->d_dom, &c->dom, sizeof(DomSet), cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));  // the host mirror may change after return
  c->dom_on = true;
  return HAIR_OK;
}

int hair_shadow_clear(hair_ctx* c) {
  if (!c) return HAIR_E_INVALID_ARG;
  c->dom_on = false;
  return HAIR_OK;
}

int hair_debug_shadow(hair_ctx* c, uint32_t light, const uint32_t** dev_z0, const uint32_t** dev_cnt, uint32_t out_D[4]) {
  if (!c) return HAIR_E_INVALID_ARG;
  if (!c->dom_on || light >= HAIR_MAX_LIGHTS || !c->dom.l[light].on)
    return fail(c, HAIR_E_INVALID_ARG, "hair_debug_shadow: no map for this light");
  if (dev_z0) *dev_z0 = c->d_dom_z0[light];
  if (dev_cnt) *dev_cnt = reinterpret_cast<const uint32_t*>(c->d_dom_cnt[light]);
  if (out_D)
    for (int i = 0; i < 4; ++i) out_D[i] = c->dom.l[light].D[i];
  return HAIR_OK;
}

int hair_stats(hair_ctx* c, hair_stats_t* out) {
  if (!c || !out) return HAIR_E_INVALID_ARG;
  memset(out, 0, sizeof(*out));
  CK(cudaSetDevice(c->device));
  flush_updates(c);
  CK(cudaMemcpyAsync(c->h_counters, c->d_counters, CNT_N * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  const unsigned long long* k = c->h_counters;
  out->n_grooms = c->scene.n_grooms;
  out->n_bundles = c->scene.n_bi;
  out->n_bundles_culled = (uint32_t)k[CNT_CULLED];
  out->n_strands_total = c->scene.n_strands_total;
  out->n_strands_lod = (uint32_t)k[CNT_STRANDS];
  out->n_vertices = (uint32_t)k[CNT_VERTICES];
  out->n_segments = (uint32_t)k[CNT_SEGMENTS];
  out->gpu_launches = c->launches;
  out->two_pass = (uint32_t)k[CNT_HIZ_ON];
  out->n_segments_hiz_culled = (uint32_t)k[CNT_SEG_HIZ];
  out->beta_mean = c->scene.n_strands_total ? (float)((double)k[CNT_STRANDS] / (double)c->scene.n_strands_total) : 1.f;
  // Eq. 8: per-groom beta from the device-side sums of the frame's scan, delta = -log(beta)
  out->beta_min = 1.f;
  for (uint32_t g = 0; g < HAIR_MAX_GROOMS; ++g) {
    const unsigned long long num = k[CNT_BETA_NUM + g], den = k[CNT_BETA_DEN + g];
    const double b = (g < c->scene.n_grooms && den) ? (double)num / (double)den : 1.0;
    out->beta_groom[g] = (float)b;
    out->delta_groom[g] = (float)-std::log(b);
  }
  if (c->scene.n_bi) {
    const uint32_t bits = (uint32_t)k[CNT_BETA_MIN];
    memcpy(&out->beta_min, &bits, sizeof(float));
  }
  if (c->counted) {
    out->n_segments_drawn = (uint32_t)k[CNT_SEG_DRAWN];
    out->n_atomics_center = k[CNT_AT_CENTER];
    out->n_atomics_cons = k[CNT_AT_CONS];
    out->n_atomics_issued = k[CNT_AT_ISSUED];
    out->n_atomics_cons_ymajor = k[CNT_AT_CONS_Y];
    out->n_segments_live = (uint32_t)k[CNT_SEG_LIVE];
    out->n_pixels_center = (uint32_t)k[CNT_PX_CENTER];
    out->n_pixels_cons = (uint32_t)k[CNT_PX_CONS];
  }
  if (c->timed && c->ev_frames) {  // mean over the timed frames since the last call (at most EV_RING)
    float* dst[6] = {&out->ms_lod, &out->ms_generate, &out->ms_clear, &out->ms_raster, &out->ms_shade, &out->ms_filter};
    const uint32_t n = c->ev_frames < (uint32_t)EV_RING ? c->ev_frames : (uint32_t)EV_RING;
    for (uint32_t f = 0; f < n; ++f) {
      cudaEvent_t* evs = c->ev[(c->ev_frames - 1 - f) % EV_RING];
      float ms = 0.f;
      for (int i = 0; i < 6; ++i) {
        cudaEventElapsedTime(&ms, evs[i], evs[i + 1]);
        *dst[i] += ms / (float)n;
      }
      cudaEventElapsedTime(&ms, evs[EV_BEGIN], evs[EV_FILTER]);
      out->ms_total += ms / (float)n;
    }
    out->n_timed_frames = n;
    c->ev_frames = 0;
  }
  return HAIR_OK;
}

int hair_debug_buffers(hair_ctx* c, const float** v, const uint32_t** t, const float** col) {
  if (!c) return HAIR_E_INVALID_ARG;
  if (v) *v = (const float*)c->d_vertices;
  if (t) *t = (const uint32_t*)c->d_table;
  if (col) *col = (const float*)c->d_colour;
  return HAIR_OK;
}

int hair_debug_set_vertices(hair_ctx* c, const float* dev_src, uint32_t n) {
  if (!c || !dev_src) return HAIR_E_INVALID_ARG;
  if ((size_t)n > c->vertex_cap) return fail(c, HAIR_E_INVALID_ARG, "hair_debug_set_vertices: too many vertices");
  CK(cudaMemcpyAsync(c->d_vertices, dev_src, (size_t)n * sizeof(float4), cudaMemcpyDeviceToDevice, c->stream));
  return HAIR_OK;
}

void hair_abi_sizes(uint32_t out[7]) {
  out[0] = sizeof(hair_cage);
  out[1] = sizeof(hair_roots);
  out[2] = sizeof(hair_style);
  out[3] = sizeof(hair_camera);
  out[4] = sizeof(hair_render_params);
  out[5] = sizeof(hair_stats_t);
  out[6] = sizeof(hair_shadow_params);
}

int hair_atomic_microbench(hair_ctx* c, int mode, uint64_t* dev_words, uint64_t n_words, uint64_t n_ops,
                           uint32_t hot_words, float* out_ms) {
  if (!c || !dev_words || !out_ms || n_words == 0 || mode < 0 || mode > 2) return HAIR_E_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  cudaEvent_t a, b;
  CK(cudaEventCreate(&a));
  CK(cudaEventCreate(&b));
  CK(cudaMemsetAsync(dev_words, 0xFF, n_words * 8, c->stream));
  CK(cudaEventRecord(a, c->stream));
  launch_atomic_microbench(mode, (unsigned long long*)dev_words, n_words, n_ops, hot_words, c->n_sm, c->stream);
  CK(cudaEventRecord(b, c->stream));
  CK(cudaEventSynchronize(b));
  CK(cudaEventElapsedTime(out_ms, a, b));
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  CK(cudaGetLastError());
  return HAIR_OK;
}

int hair_l2_load_microbench(hair_ctx* c, int mode, const uint64_t* dev_pairs, uint64_t n_pairs, uint32_t pitch,
                            uint32_t n_steps, uint64_t* out_loads, float* out_ms) {
  if (!c || !dev_pairs || !out_ms || !out_loads || mode < 0 || mode > 5 || pitch < 64 || n_pairs < 64ull * pitch ||
      n_pairs >= (1ull << 32) || n_steps == 0 || (n_steps & 3u))
    return HAIR_E_INVALID_ARG;
  CK(cudaSetDevice(c->device));
  cudaEvent_t a, b;
  CK(cudaEventCreate(&a));
  CK(cudaEventCreate(&b));
  CK(cudaEventRecord(a, c->stream));
  // the sink is never written (the kernel's guard is false for any real buffer): the counters' last word serves
  launch_l2_load_microbench(mode, (const unsigned long long*)dev_pairs, (uint32_t)n_pairs, pitch, n_steps,
                            c->d_sink, c->n_sm, c->stream);
  CK(cudaEventRecord(b, c->stream));
  CK(cudaEventSynchronize(b));
  CK(cudaEventElapsedTime(out_ms, a, b));
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  CK(cudaGetLastError());
  *out_loads = (uint64_t)c->n_sm * 8ull * 256ull * n_steps;
  return HAIR_OK;
}

}  // extern "C"
