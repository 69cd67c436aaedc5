/* hair.h — C ABI of libhair: the deferred hair pipeline of arxiv/paper_2607_04230 on one B200.
 *
 * The calls follow the paper's statement of the problem (Fig. 2, §3):
 * inputs are a hair mesh (cage of prism layers + root triangles), a styling function
 * and a camera; outputs are the 64-bit compressed G-buffer and the
 * filtered, alpha-composited colour. Everything between runs in hand-written
 * CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *  - Every function returns HAIR_OK (0) or a negative HAIR_E_* code; hair_last_error() gives text.
 *  - "host" pointers are read during the call and may be freed after it returns (the library
 *    copies). "DEVICE" pointers are caller-owned CUDA allocations on the context's device.
 *  - All work is enqueued on the CUDA stream given to hair_create (the caller's, e.g. torch's
 *    current stream). hair_render never synchronises and waits for no device result: grid sizes come from
 *    device-side counters; the one thing the host looks at is a host-mapped word in which the scan of the frame
 *    BEFORE said whether that frame was big enough for two raster passes (HAIR_FLAG_SINGLE_PASS), read without
 *    waiting — a stale value changes the launch count of this frame, never its result.
 *  - A context is not thread-safe. No global state.
 *  - Arithmetic contract (operation order of the fp32 decisions, bit layout): DESIGN.md §3.
 */
#ifndef HAIR_H
#define HAIR_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define HAIR_OK 0
#define HAIR_E_INVALID_ARG (-1)
#define HAIR_E_CUDA (-2)
#define HAIR_E_OUT_OF_MEMORY (-3)
#define HAIR_E_TOO_MANY_STRANDS (-4) /* sum of strands x instances >= 2^24 (24-bit strand id) */
#define HAIR_E_TOO_MANY_CPS (-5)     /* C_full = (n_layers-1)*spi + 1 > 127 (7-bit segment index) */
#define HAIR_E_TOO_MANY_GROOMS (-6)  /* > HAIR_MAX_GROOMS */
#define HAIR_MAX_GROOMS 16
#define HAIR_MAX_LIGHTS 4

/* styling operators, applied in this order (R24) */
#define HAIR_OP_CLUMP 1u
#define HAIR_OP_TWIST 2u
#define HAIR_OP_CURL 4u
#define HAIR_OP_FRIZZ 8u

/* render flags */
#define HAIR_FLAG_FILTER 1u       /* run the reconstruction filter; else pass centre colour */
#define HAIR_FLAG_COUNTERS 2u     /* count predicate-true hits (algorithmic atomics) in hair_stats; slower */
#define HAIR_FLAG_STAGE_TIMING 4u /* record CUDA events around each stage for hair_stats.ms_* */
/* The paper's self-contained G-buffer word ("G-buffer compression"; DESIGN.md R-payload) instead of
 * depth24|strand24|segment7|t9:
 *   [63:40] depth24 | [39:32] ox8 | [31:24] oy8 | [23:18] u6 | [17:12] v6 | [11:6] w6 | [5:0] ao6
 * octahedral code of the interpolated calcTangent (2 x uint8), root coordinates u, v, strand parameter w and
 * ambient occlusion (4 x uint6). Shading then reads no vertex: position from the depth at the pixel centre
 * (PAPER.md:90), tangent from the code, shading parameters from w; the filter's screen tangent is the projected
 * decoded tangent. The word names no groom, so exactly ONE groom may be drawn per pass (groom_mask selecting one
 * groom with hair_render / hair_render_scene, or hair_render_sequential, the paper's groom-by-groom path
 * PAPER.md:208): otherwise HAIR_E_INVALID_ARG. Not available with hair_render_msaa. */
#define HAIR_FLAG_PAPER_PAYLOAD 8u
/* Draw the frame in ONE raster pass. Default: large frames are drawn in two depth-ordered passes with a tile
 * hi-Z between them, which drops occluded segments of the second pass before any pixel work; the G-buffer is the
 * same bit for bit (the resolve is an order-free min). For A/B measurements. */
#define HAIR_FLAG_SINGLE_PASS 16u
/* Fused generation + raster (the paper's own arrangement: "strand vertices stay in
 * registers"): no vertex buffer is written; the raster's warps build the bundle's spline table and generate the
 * vertices they draw (the very code k_generate runs, so the words equal the materialised frame's bit for bit).
 * Requires HAIR_FLAG_PAPER_PAYLOAD (the strand-id word is shaded from the vertex buffer): otherwise
 * HAIR_E_INVALID_ARG. The debug vertex buffer is not valid after such a frame. An A/B against the default pipeline. */
#define HAIR_FLAG_FUSED 32u

/* (bit 64u was HAIR_FLAG_TILED, a tile-binned raster A/B that lost 2.7x and was removed in round 3: DESIGN.md 7.1b) */

/* Half-precision colour output: out_rgb / host_rgb of every render call is [height][width][4] IEEE binary16 (8 bytes per
 * pixel; the buffer still 16-byte aligned) instead of float, written by the filter itself (round to nearest; absolute error <= 2^-11 of
 * the value's binade, i.e. < 1e-3 for |v| < 2, < 2e-3 for |v| < 4). Halves the device->host copy of
 * hair_render_to_host(_async), which PCIe bounds. scene_rgb stays float. */
#define HAIR_FLAG_RGB16F 128u

/* Volumetric shadows (§3.4 "Volumetric shadows are computed using deep-opacity maps ..., which we query
 * using the depth-correction described in Section 3.2"; DESIGN.md R-dom): the shading of every hair_render* call
 * scales the contribution of light l by the transmittance towards it, looked up in the deep opacity map that
 * hair_shadow_build made for that light, at the depth-corrected depth d_eff = beta_g d (Eq. 7) of the groom being
 * shaded. Lights without a map are unshadowed. */
#define HAIR_FLAG_SHADOWS 256u

typedef struct hair_ctx hair_ctx; /* opaque; owns all device scratch */

/* Creates a context on `cuda_device` that enqueues on `cuda_stream` (a cudaStream_t; NULL = the
 * legacy default stream). The stream stays owned by the caller and must outlive the context. */
int hair_create(hair_ctx** out, int cuda_device, void* cuda_stream);
void hair_destroy(hair_ctx*);
const char* hair_last_error(const hair_ctx*);

/* Hair mesh: bundles = triangular prisms over root triangles (R1). */
typedef struct {
  uint32_t n_verts;  /* cage vertices per layer */
  uint32_t n_layers; /* Lv: vertex layers, root layer first, tip last; 2 <= Lv <= 32 */
  const float* pos;  /* host, [n_layers][n_verts][3], groom-local space */
  const float* ao;   /* host, [n_layers][n_verts] baked ambient occlusion, or NULL (= 1) */
} hair_cage;

typedef struct {
  uint32_t n_tris;                 /* bundles */
  const uint32_t* idx;             /* host, [n_tris][3] indices into n_verts */
  const uint32_t* strands_per_tri; /* host, [n_tris]: N of Eq. 1 per bundle */
} hair_roots;

typedef struct {
  uint32_t spi;  /* control points per layer interval: C_full = (Lv-1)*spi + 1 */
  uint32_t seed; /* hash seed (R26) */
  uint32_t op_mask, clump_exp, frizz_cells;
  float clump_strength, twist_turns;
  float curl_radius, curl_turns, curl_ramp_w0;
  float frizz_sigma, frizz_ramp_w0;
  float width_world; /* > 0: centre radius from projected width (R9); 0: center_diameter_px */
  float albedo_root[3], albedo_tip[3], roughness, tilt;
  uint32_t n_instances;        /* >= 1 */
  const float* instance_xform; /* host, [n_instances][12] row-major 3x4 [R|t], or NULL = identity */
} hair_style;

/* Appends a groom. Copies everything to the device (synchronously) and sizes the scratch buffers
 * for the worst case (LOD off). Strand ids are assigned in upload order (DESIGN.md §3 "sid"). */
int hair_mesh_upload(hair_ctx*, const hair_cage*, const hair_roots*, const hair_style*, int* out_groom_id);
/* Replaces positions / AO of an uploaded groom (animated cage). Same sizes.
 * From PINNED host memory the call only queues the update; nothing is read yet. The next hair_render* / hair_stats /
 * hair_shadow_build call sends every queued array to a staging buffer on the device with the copy engine
 * (cudaMemcpyAsync on the context's second stream, so the bus transfer can run beside the frame before) and then
 * copies staging -> cage with one device-to-device kernel on the context's stream in front of its own work. The host
 * arrays are therefore read AFTER that later call has been issued: they must stay valid and unchanged until its work
 * has completed (e.g. until hair_host_wait of that frame, or a hair_stats). hair_mesh_clear and hair_destroy drop
 * updates still queued without reading them.
 * From pageable memory the copy is a cudaMemcpyAsync on the context's stream inside this call (updates queued before
 * it are sent first, so the updates of a groom take effect in call order); the array may be freed when it returns. */
int hair_mesh_update(hair_ctx*, int groom_id, const hair_cage*);
/* Removes all grooms (buffers are kept), so that another hair mesh can be uploaded into the same context;
 * the counterpart of hair_mesh_upload in north_star's boundary. */
int hair_mesh_clear(hair_ctx*);

typedef struct {
  float eye[3], right[3], up[3], forward[3]; /* orthonormal; +forward = increasing depth */
  float vfov_y, near_z, far_z;               /* radians; depth range of the 24-bit depth */
} hair_camera;

typedef struct {
  float center_diameter_px; /* PAPER.md:74 "configurable diameter"; default 0.5 */
  int32_t filter_radius;    /* r of PAPER.md:160; 0..7, default 5 */
  float s_par, s_perp;      /* sigma_par = r*s_par, sigma_perp = r*s_perp */
  float sigma_c;            /* 0.9 */
  float tau_z, tau_fly;     /* 1.45e-3, 5e-4 in normalised depth */
  float w_strip;            /* 0.5 px */
  float light_pos[HAIR_MAX_LIGHTS][3], light_rgb[HAIR_MAX_LIGHTS][3];
  uint32_t n_lights;
  float ambient_rgb[3], k_d, k_R, k_TRT, background_rgb[3];
  uint32_t flags; /* HAIR_FLAG_* */
  uint32_t groom_mask; /* bit g set = groom g (upload order) is drawn; default all ones. Grooms left out get
                          N_LOD = 0 in the LOD pass, so the frame is exactly the frame of the remaining grooms
                          (strand ids in the words stay global). */
} hair_render_params;

void hair_default_render_params(hair_render_params* out);
int hair_set_render_params(hair_ctx*, const hair_render_params*);

/* One frame: LOD -> scan -> generate -> clear+raster -> shade -> filter, all on the stream.
 *  lod_lambda  host, per groom (n_lambda == n_grooms) or one value for all (n_lambda == 1);
 *              <= 0 switches LOD and culling off for that groom (R14)
 *  out_gbuffer DEVICE, [height][width][2] uint64, 16-byte aligned: [..][0] centre-sample layer,
 *              [..][1] conservative layer; word = depth24|strand24|segment7|t9,
 *              empty = all ones. Cleared by the call.
 *  out_rgb     DEVICE, [height][width][4] float, 16-byte aligned: linear rgb composited over the
 *              background, alpha in .w (R29). */
int hair_render(hair_ctx*, const hair_camera*, uint32_t width, uint32_t height, const float* lod_lambda,
                uint32_t n_lambda, uint64_t* out_gbuffer, float* out_rgb);

/* hair_render into an existing scene (DESIGN.md R-scene; "reads the existing depth buffer ... blended
 * into the main render target", 208-210 "keeping depth"):
 *  scene_zn   DEVICE, [height][width] float, normalised depth zn = A - B / z_view in [0, 1] of what is already in
 *             the frame (clamped), or NULL. Both layers of every pixel start at its 24-bit quantisation with an
 *             all-ones payload, so a hair hit behind the scene loses the atomic min; a hit at the same quantised
 *             depth wins. In out_gbuffer a word whose low 40 bits are all ones means "no hair hit" (its depth bits
 *             are the scene's; without a scene such words are all ones as in hair_render).
 *  scene_rgb  DEVICE, [height][width][4] float, 16-byte aligned (.w ignored), or NULL: what the hair is composited
 *             over instead of background_rgb. out_rgb.w is the hair's alpha alone. */
int hair_render_scene(hair_ctx*, const hair_camera*, uint32_t width, uint32_t height, const float* lod_lambda,
                      uint32_t n_lambda, const float* scene_zn, const float* scene_rgb, uint64_t* out_gbuffer,
                      float* out_rgb);

/* MSAA-k REFERENCE mode (DESIGN.md R-msaa; "recording samples into multiple layers of a uint64 image
 * and resolving them later ... only as a reference"): k in {1, 2, 4, 8} sample points per pixel (the standard
 * multisample patterns), one atomic-min layer per sample; a sample is hit when the segment meets the pixel's closed
 * square and passes within the centre radius of the sample point. No filter: out_rgb = mean over the samples of
 * (shaded hit | background), .w = hit samples / k.
 *  out_samples DEVICE, [k][height][width] uint64, 16-byte aligned, cleared by the call (empty = all ones). */
int hair_render_msaa(hair_ctx*, const hair_camera*, uint32_t width, uint32_t height, const float* lod_lambda,
                     uint32_t n_lambda, uint32_t k, uint64_t* out_samples, float* out_rgb);

/* The paper's multi-groom path (DESIGN.md R-seq): the grooms one after the other in upload
 * order, each through the whole pipeline on its own (LOD .. filter), its filtered result blended over the target
 * so far, the depth of its centre layer kept so that later grooms are rejected behind it. hair_render, by
 * contrast, resolves all grooms in one G-buffer and filters once (R15). Arguments as hair_render_scene.
 * After the call out_gbuffer holds the LAST pass: that groom's words, elsewhere "no hit" words carrying the depth
 * kept from all passes; out_rgb.w = the accumulated alpha 1 - prod(1 - alpha_g). hair_stats then reports the last
 * pass's counts, gpu_launches of all passes, and stage times averaged per PASS. Uses one more width x height x
 * 16-byte buffer inside the context (allocated on first use). */
int hair_render_sequential(hair_ctx*, const hair_camera*, uint32_t width, uint32_t height, const float* lod_lambda,
                           uint32_t n_lambda, const float* scene_zn, const float* scene_rgb, uint64_t* out_gbuffer,
                           float* out_rgb);

/* Same frame, results copied to HOST memory (pinned for full speed) inside the call:
 * host_rgb [h][w][4] float is required, host_gbuffer [h][w][2] may be NULL. Synchronises the stream. */
int hair_render_to_host(hair_ctx*, const hair_camera*, uint32_t width, uint32_t height,
                        const float* lod_lambda, uint32_t n_lambda, uint64_t* host_gbuffer, float* host_rgb);

/* Pipelined form of hair_render_to_host: enqueues the frame on the context's stream and the device->host
 * copies on the context's own copy stream, then returns without waiting, so the copies of frame i overlap the
 * kernels of frame i+1. Results live in one of HAIR_HOST_SLOTS device buffer pairs owned by the context; a
 * slot is reused (stream-ordered, no host wait) once its previous copies are done. *out_slot receives the
 * slot; host_rgb / host_gbuffer must stay valid and unread until hair_host_wait(ctx, slot) returns.
 * Use a different host buffer for each frame in flight. */
#define HAIR_HOST_SLOTS 2
int hair_render_to_host_async(hair_ctx*, const hair_camera*, uint32_t width, uint32_t height,
                              const float* lod_lambda, uint32_t n_lambda, uint64_t* host_gbuffer, float* host_rgb,
                              int* out_slot);
/* Blocks until the copies of `slot` (0..HAIR_HOST_SLOTS-1), or of every slot (slot < 0), have finished. (Host-side
 * completion of hair_render_to_host_async; not an operation of the paper — the e2e measurement of SURVEY.md §8d needs it.) */
int hair_host_wait(hair_ctx*, int slot);

/* Deep opacity maps (Yuksel and Keyser 2008, named by PAPER.md:192; the paper gives no more, DESIGN.md R-dom states
 * the reading). For each light l < n_lights, from the light's camera cam[l] (eye = the light's position; the caller
 * frames the scene, e.g. a look-at camera) at res x res:
 *   z0(u, v)     24-bit depth (the G-buffer's quantisation, R8) of the nearest hair touching light pixel (u, v): the
 *                conservative layer of a G-buffer rendered from the light, 0xFFFFFFFF where no hair is;
 *   cnt(u, v, k) number of (segment, pixel) conservative hits of that pixel in layer k behind z0; layer k spans
 *                [D[k-1], D[k]) depth steps with D[-1] = 0, D[k] = round(layer_d1 * 16777215) * (2^(k+1) - 1) for
 *                k = 0..2; layer 3 is open-ended and is taken to end at D[3] when looked up.
 * Built from the FULL grooms (LOD off), as PAPER.md:140 has it ("previously computed depth maps ... recomputing
 * them is computationally expensive"): this is what makes the depth-comparison fix necessary when a frame thins
 * the groom. Lookup (in the shading of a frame rendered with HAIR_FLAG_SHADOWS): world point p -> light pixel and
 * depth dq; per texel d = max(dq - z0, 0), d_eff = beta_g * d (Eq. 7; beta_g = hair_stats_t.beta_groom of the frame
 * being rendered, taken on the device), fragments in front = the cumulative count, piecewise linear through the
 * layer ends; bilinear over the four texels around p (texel centres at integer + 1/2; empty texels contribute 0);
 * transmittance = exp(-alpha_s * fragments in front) (Eq. 6).
 * The call runs the grooms through LOD (off) -> generate -> clear -> raster -> fragment count once per light on the
 * context's stream, overwriting the context's vertex buffer and table (render a frame afterwards before using the
 * debug accessors for it), and keeps 20 bytes per texel and light. Grooms uploaded or updated later need a rebuild. */
typedef struct {
  hair_camera cam[HAIR_MAX_LIGHTS];
  uint32_t n_lights; /* maps to build: lights 0 .. n_lights-1 of the render params in force when frames are shaded */
  uint32_t res;      /* 16 .. 8192 */
  float layer_d1;    /* thickness of the first layer in normalised depth of the light's camera, > 0 */
  float alpha_s;     /* opacity one fragment adds, >= 0 */
} hair_shadow_params;
int hair_shadow_build(hair_ctx*, const hair_shadow_params*);
/* Drops the maps (shading is unshadowed again). */
int hair_shadow_clear(hair_ctx*);
/* Parity access: DEVICE pointers to light l's z0 [res][res] uint32 and cnt [res][res][4] uint32, and the four
 * layer ends. */
int hair_debug_shadow(hair_ctx*, uint32_t light, const uint32_t** dev_z0, const uint32_t** dev_cnt, uint32_t out_D[4]);

typedef struct {
  uint32_t n_grooms, n_bundles, n_bundles_culled;
  uint32_t n_strands_total, n_strands_lod;
  uint32_t n_vertices, n_segments;
  uint32_t n_segments_drawn;               /* both endpoints in front of the near plane (counters flag) */
  uint32_t n_segments_live;                /* segments that won at least one pixel test when drawn (counters flag) */
  uint64_t n_atomics_center, n_atomics_cons; /* predicate-true hits before any filtering (counters flag) */
  uint64_t n_atomics_issued;               /* atomics actually sent to L2 (counters flag) */
  uint64_t n_atomics_cons_ymajor;          /* conservative hits of y-major segments: neighbouring lanes of a raster warp
                                              then sit in neighbouring ROWS of the G-buffer (counters flag) */
  uint32_t n_pixels_center, n_pixels_cons; /* non-empty pixels after the frame (counters flag) */
  /* stage-timing flag: mean over the frames rendered since the previous hair_stats (last 64 at most) */
  float ms_lod, ms_generate, ms_clear, ms_raster, ms_shade, ms_filter, ms_total;
  uint32_t n_timed_frames;
  float beta_mean; /* strands after LOD / strands uploaded, over all grooms (frustum-culled bundles count as removed) */
  /* Depth-comparison fix (Eq. 6-8; DESIGN.md R-beta), for the consumer of a depth / opacity map
   * that was built from the full groom: beta_groom[g] = N_remaining / N_total of groom g over its DRAWN
   * bundle-instances (N_LOD > 0), 1 if none; delta_groom[g] = -ln beta (Eq. 8): a depth d into the groom is to be
   * tested at d exp(-delta) (the additive shift -delta in log depth, Eq. 7); beta_min = the most thinned drawn
   * bundle-instance's N_LOD / N. Sums are taken on the device by the scan of every frame. */
  float beta_min;
  float beta_groom[HAIR_MAX_GROOMS], delta_groom[HAIR_MAX_GROOMS];
  uint32_t gpu_launches; /* kernels launched by the last hair_render */
  uint32_t two_pass;              /* 1: the last frame was drawn in two depth-ordered raster passes */
  uint32_t n_segments_hiz_culled; /* segments of the second pass dropped by the tile hi-Z test before any pixel work */
} hair_stats_t;
/* hair_stats() of north_star's boundary: synchronises the stream and reads the device counters of the
 * last frame — the LOD pass's strand / vertex totals, the per-groom beta and delta of the
 * depth-comparison fix (Eq. 8), the raster's hit counts and the stage times.
 * hair_stats_t holds every field SURVEY §8(b) lists, in another order and with more. ms_clear reads ~0: the clear runs
 * on the context's second stream beside LOD / scan / generate and is not bracketed by events. */
int hair_stats(hair_ctx*, hair_stats_t* out);

/* Debug / parity access to the intermediates of the last frame (DEVICE pointers, owned by the context). Replaces
 * SURVEY.md §8(b)'s hair_debug_vertices(ctx, &verts, &table): same two buffers plus the shaded colour buffer:
 * vertices float4[n_vertices] = (x, y, z, ao); table uint4[n_bundles] = {N_LOD, C, slot_base,
 * vertex_base}; colour float4[h][w] = shaded rgb of centre-hit pixels (undefined elsewhere). */
int hair_debug_buffers(hair_ctx*, const float** dev_vertices, const uint32_t** dev_table, const float** dev_colour);
/* Stage-wise parity: run only H4..H7 of a frame on caller-supplied intermediates.
 *  stage_mask bit0 = clear+raster (from the context's vertex buffer), bit1 = shade, bit2 = filter.
 *  If bit0 is clear, out_gbuffer is taken as input. */
int hair_render_stages(hair_ctx*, const hair_camera*, uint32_t width, uint32_t height, uint32_t stage_mask,
                       uint64_t* out_gbuffer, float* out_rgb);
/* Overwrites the context's vertex buffer of the last frame (DEVICE src, n float4) — lets a test feed
 * the raster with vertices of its choice. n must equal the last frame's n_vertices. */
int hair_debug_set_vertices(hair_ctx*, const float* dev_src, uint32_t n);

/* MEASUREMENT TOOLING, not part of the render path (bench.py measures its roofline denominators with the two calls
 * below in the same run as the frame).
 * L2-atomic roofline denominators: 64-bit atomicMin (RED.MIN.64) micro-kernels over a
 * DEVICE buffer of n_words uint64.
 *  mode 0: each thread its own word, coalesced;  mode 1: hashed uniformly random word per op;
 *  mode 2: all ops into `hot_words` words (contention floor).
 * Enqueues `n_ops` atomics; returns the elapsed milliseconds (CUDA events; synchronises). */
int hair_atomic_microbench(hair_ctx*, int mode, uint64_t* dev_words, uint64_t n_words, uint64_t n_ops,
                           uint32_t hot_words, float* out_ms);

/* L2-load roofline denominator for the raster's read-before-atomic ("reads the existing depth buffer";
 * SURVEY.md §8d): 16-byte ld.global.cg of word pairs over a DEVICE buffer of n_pairs pairs laid out as image rows
 * of `pitch` pairs (n_pairs >= 64 * pitch, pitch >= 64). A warp's 32 loads of one step are
 *  mode 0: 32 consecutive pairs of a row;  mode 1: one column over 32 consecutive rows;  mode 2: 32 random pairs;
 *  mode 3 / 4: the column / row walk in a layout of 2 x 4-pixel blocks (an experiment);
 *  mode 5: the column walk with the two horizontally adjacent pairs of a row requested together by each lane, the
 *          shape of a y-major raster task (two loads per sector).
 * Every thread of n_SM * 8 CTAs of 256 threads issues `n_steps` loads (a multiple of 4). Writes the total number of
 * loads to *out_loads and the elapsed milliseconds (CUDA events; synchronises) to *out_ms. The buffer is only read. */
int hair_l2_load_microbench(hair_ctx*, int mode, const uint64_t* dev_pairs, uint64_t n_pairs, uint32_t pitch,
                            uint32_t n_steps, uint64_t* out_loads, float* out_ms);

/* The H2 scan (per-bundle LOD records -> where each bundle's strands and vertices go) as a
 * call that allocates nothing, for callers that cannot let a library cudaMalloc: an engine that gave all device
 * memory to its own pool at start-up (an allocation in the frame loop fails or stalls the device), or a host whose
 * per-frame code may not make synchronising calls, which cudaMalloc / cudaFree are. It takes no hair_ctx (creating
 * one, uploading a groom and the first render all allocate) and calls no cudaMalloc, cudaFree or allocating library
 * routine; the tile sums it needs between its two kernels sit in a fixed 32 KB array inside the library's device
 * code, which every GPU that loads this library holds until the process exits.
 *  cuda_device  device of the pointers and the stream; made current and left current, as by the other calls
 *  cuda_stream  a cudaStream_t of that device (NULL = legacy default stream); the two kernels are enqueued on it and
 *               the call returns without waiting
 *  dev_counts   DEVICE, [n][2] uint32, 8-byte aligned: {N_LOD, C} of every bundle-instance in index order (columns
 *               .x, .y of the bundle table, Eq. 1 and Eq. 4-5); only read
 *  n            bundle-instances, 0 <= n <= HAIR_SCAN_NOALLOC_MAX; more returns HAIR_E_INVALID_ARG before anything
 *               is launched (the array cannot grow), with the limit in hair_scan_noalloc_error()
 *  dev_bases    DEVICE, [n][2] uint32, 8-byte aligned, written: {slot_base, vertex_base} = exclusive sums of N_LOD
 *               and of N_LOD * C over the bundle-instances in front (columns .z, .w of the bundle table), mod 2^32
 *  dev_totals   DEVICE, [2] uint32, written: {sum N_LOD, sum N_LOD * C} (hair_stats_t.n_strands_lod, .n_vertices)
 * Must not overlap other calls on the same device: all calls of a process share the one array per device, so two
 * whose kernels can run concurrently (two streams, two threads) race; back to back on one stream is fine. The array
 * keeps the previous call's sums; every call rewrites all the entries it reads, so nothing needs clearing. The first
 * call on a device also looks up the array's device address (cudaGetSymbolAddress): make that call before any
 * stream capture begins. Returns HAIR_OK, HAIR_E_INVALID_ARG (size, null or misaligned pointer, device number) or
 * HAIR_E_CUDA; hair_scan_noalloc_error() gives the text of the calling thread's last failure ("" after success). */
#define HAIR_SCAN_NOALLOC_MAX (1u << 20)
int hair_scan_noalloc(int cuda_device, void* cuda_stream, const uint32_t* dev_counts, uint32_t n,
                      uint32_t* dev_bases, uint32_t* dev_totals);
const char* hair_scan_noalloc_error(void);

/* sizeof of {hair_cage, hair_roots, hair_style, hair_camera, hair_render_params, hair_stats_t, hair_shadow_params},
 * so a foreign-language binding can check its struct layouts without a GPU. */
void hair_abi_sizes(uint32_t out[7]);

#ifdef __cplusplus
}
#endif
#endif
