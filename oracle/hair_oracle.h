/* hair_oracle.h — C interface of the CPU ORACLE.
 *
 * TEST INFRASTRUCTURE ONLY. This is the plain, slow, single-threaded CPU
 * restatement of what the deferred hair pipeline of arxiv/paper_2607_04230
 * computes (§3.1-3.4, Eq. 1-5, Eq. 9-10, Code 1, Code 2), written from
 * the paper and from the readings listed in DESIGN.md §3. Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it. It shares no code, header, table or helper with the CUDA library
 * (include/hair.h, paper_2607_04230_b200/csrc); the struct layouts below are the
 * oracle's own.
 *
 * Precision. Generation (O2), shading (O6) and the filter's weights (O7) are
 * fp64. Every place where floating point decides an integer — LOD counts (O1),
 * the two coverage predicates and the packed word (O4), the filter's sample
 * classification (O7) — is fp32, one rounding per operation, no FMA contraction
 * (built with -ffp-contract=off), in the operation order DESIGN.md §3 states,
 * because the CUDA path takes the same decisions in fp32.
 *
 * Pins (tests/test_oracle_*.py): see DESIGN.md §4. Unpinned against the paper:
 * the hash constants and the stand-in shading model (the paper prints neither).
 */
#ifndef HAIR_ORACLE_H
#define HAIR_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  uint32_t spi, seed, op_mask, clump_exp, frizz_cells;
  float clump_strength, twist_turns;
  float curl_radius, curl_turns, curl_ramp_w0;
  float frizz_sigma, frizz_ramp_w0;
  float width_world;
  float albedo_root[3], albedo_tip[3], roughness, tilt;
} orc_style;

typedef struct {
  uint32_t n_verts, n_layers, n_tris, n_instances; /* n_instances >= 1 */
  const float* pos;                /* [n_layers][n_verts][3] */
  const float* ao;                 /* [n_layers][n_verts] or NULL (= 1) */
  const uint32_t* idx;             /* [n_tris][3] */
  const uint32_t* strands_per_tri; /* [n_tris] */
  const float* xform;              /* [n_instances][12] row-major 3x4, or NULL (identity) */
  orc_style style;
} orc_groom;

typedef struct {
  float eye[3], right[3], up[3], forward[3];
  float vfov_y, near_z, far_z;
  uint32_t width, height;
} orc_camera;

typedef struct {
  float center_diameter_px;
  int32_t filter_radius;
  float s_par, s_perp, sigma_c, tau_z, tau_fly, w_strip;
  float light_pos[4][3], light_rgb[4][3];
  uint32_t n_lights;
  float ambient_rgb[3], k_d, k_R, k_TRT, background_rgb[3];
  uint32_t filter_on;
} orc_params;

/* op_mask bits */
#define ORC_OP_CLUMP 1u
#define ORC_OP_TWIST 2u
#define ORC_OP_CURL 4u
#define ORC_OP_FRIZZ 8u

typedef struct orc_frame orc_frame;

/* ---- small pure functions (pins) ---- */
uint32_t orc_pcg(uint32_t v);
uint32_t orc_hash3(uint32_t seed, uint32_t id, uint32_t stream);
/* Eq. 1 + Eq. 4-5 for one bundle given L: out[0]=N_LOD, out[1]=C_raw, out[2]=C */
void orc_lod_counts(float L, uint32_t N, float delta, uint32_t n_layers, uint32_t c_full,
                    uint32_t out[3]);
void orc_calc_tangent(int idx, int count, const double prev[3], const double curr[3],
                      const double next[3], double out[3]);
uint64_t orc_pack(float zn, uint32_t sid, uint32_t j, float t);
void orc_unpack(uint64_t w, uint32_t out[4]); /* dq, sid, j, t9 */
/* coverage of ONE screen-space segment on a w x h grid: cover[y*w+x] bit0 = conservative,
 * bit1 = centre; tq[y*w+x] = closest-point parameter t (fp32). */
/* per-sample coverage of one screen-space segment in MSAA-k mode (R-msaa): cover[k][h][w] in {0, 1}, tq likewise */
int orc_segment_cover_msaa(const float a[2], const float b[2], float rho, uint32_t w, uint32_t h, uint32_t k,
                           uint8_t* cover, float* tq);
void orc_segment_cover(const float a[2], const float b[2], float rho, uint32_t w, uint32_t h,
                       uint8_t* cover, float* tq);
/* project one world point: out = sx, sy, zn, zv; returns valid */
int orc_project(const orc_camera* cam, const float p[3], float out[4]);

/* ---- frame pipeline ---- */
orc_frame* orc_frame_create(void);
void orc_frame_destroy(orc_frame*);
int orc_frame_add_groom(orc_frame*, const orc_groom*); /* copies; returns groom id */

/* O1 + scans. lambda: per groom (n_lambda = 1 broadcasts); <= 0 => LOD off. */
int orc_frame_lod(orc_frame*, const orc_camera*, const float* lambda, uint32_t n_lambda);
uint32_t orc_frame_n_bundles(const orc_frame*);      /* bundle-instances over all grooms */
uint32_t orc_frame_n_strands_total(const orc_frame*);
uint32_t orc_frame_n_strands(const orc_frame*);      /* after LOD */
uint64_t orc_frame_n_vertices(const orc_frame*);
/* table[gid] = {N_LOD, C, slot_base, vertex_base}; L[gid] = LOD selection value (-1 = culled/off) */
void orc_frame_get_table(const orc_frame*, uint32_t* table4, float* L);
/* replace the table (e.g. by the CUDA path's, for stage-wise parity). Recomputes nothing else. */
int orc_frame_set_table(orc_frame*, const uint32_t* table4, uint32_t n);

/* Depth-comparison fix (§3.2.3, Eq. 6-8; DESIGN.md R-beta), from the current table:
 *  beta[g]  = N_remaining / N_total of groom g = sum N_LOD / sum N over its bundle-instances that are drawn
 *             (N_LOD > 0; frustum-culled bundles are outside the view, not stochastically thinned); 1 if none
 *  delta[g] = -ln beta[g]                                                            (Eq. 8)
 *  *beta_min = min over all drawn bundle-instances of N_LOD / N (the most thinned bundle); 1 if none.
 * beta, delta: one double per groom. */
void orc_frame_beta(const orc_frame*, double* beta, double* delta, double* beta_min);
/* Eq. 7-8: a depth d INTO the groom (optical-depth axis, sigma * d), tested after stochastic thinning to the fraction
 * beta = exp(-delta): the additive shift -delta in log-depth space, ln d_eff = ln d - delta, i.e. d_eff = d exp(-delta) */
double orc_depth_fix(double d, double delta);

/* Deep opacity maps of the point lights ("Volumetric shadows are computed using deep-opacity maps ...,
 * which we query using the depth-correction described in Section 3.2"; DESIGN.md R-dom). The paper gives no more
 * than the name, so this follows the published technique as restated in hair_oracle.cpp: per light pixel the depth
 * z0 of the nearest hair (the conservative layer of a G-buffer rendered from the light, orc_frame_raster with the
 * light's camera, which must have run before) and, in layers behind it, the number of hair fragments.
 *  D[3]  ends of layers 0..2 in 24-bit depth steps behind z0 (layer 3 is open-ended)
 *  z0    out, [h][w]: 24-bit depth, 0xFFFFFFFF = no hair;  cnt  out, [h][w][4] fragments per layer.
 * Pins: tests/test_oracle_shadow.py. */
int orc_frame_dom_count(orc_frame*, const orc_camera* light_cam, const orc_params*, const uint32_t D[3], uint32_t* z0,
                        uint32_t* cnt);
/* Transmittance exp(-alpha_s * fragments in front) towards the light at world point p: fragment count piecewise
 * linear in the depth behind z0 through the layer ends D[0..3] (constant beyond D[3]), that depth scaled by beta
 * first (Eq. 7, d_eff = beta d: the depth-comparison fix), bilinear over the four texels around the point. */
double orc_dom_transmittance(const orc_camera* light_cam, const uint32_t* z0, const uint32_t* cnt, const uint32_t D[4],
                             double alpha_s, double beta, const float p[3]);
/* O6 then scales light `light`'s contribution by that transmittance (cam == NULL switches it off). The arrays stay
 * the caller's. beta: per groom, of the frame being shaded (orc_frame_beta). */
int orc_frame_set_dom(orc_frame*, uint32_t light, const orc_camera* light_cam, const uint32_t* z0, const uint32_t* cnt,
                      const uint32_t D[4], double alpha_s);
void orc_frame_set_dom_beta(orc_frame*, const double* beta, uint32_t n);

/* O2: vertices for the current table. fp64 result, and its fp32 rounding. */
int orc_frame_generate(orc_frame*);
void orc_frame_get_vertices_f64(const orc_frame*, double* xyz_ao);
void orc_frame_get_vertices_f32(const orc_frame*, float* xyz_ao);
int orc_frame_set_vertices_f32(orc_frame*, const float* xyz_ao, uint64_t n);
/* one unstyled/styled strand in groom-local space, fp64, for closed-form pins:
 * out[C][4] (x,y,z,ao), tan[C][3] base tangents (may be NULL) */
int orc_strand(const orc_frame*, uint32_t groom, uint32_t id_local, uint32_t C, double* out,
               double* base_tan);
/* root barycentrics (fp64 exact multiples of 2^-24) and bundle of a strand */
int orc_root(const orc_frame*, uint32_t groom, uint32_t id_local, double b[3], uint32_t* tri);

/* O4: raster the current fp32 vertices with the current table. gbuffer [H][W][2] (0 = centre, 1 = cons).
 * order: optional permutation of strand slots (NULL = natural) — result must not depend on it.
 * counts[0] = centre atomics (predicate-true hits), counts[1] = conservative, counts[2] = segments
 * with both endpoints valid. */
int orc_frame_raster(orc_frame*, const orc_camera*, const orc_params*, const uint32_t* order,
                     uint64_t counts[3]);
void orc_frame_get_gbuffer(const orc_frame*, uint64_t* out);
int orc_frame_set_gbuffer(orc_frame*, const uint64_t* in, uint32_t w, uint32_t h);
/* R-scene: optional scene the hair is drawn into. zn[h][w] in [0, 1] (NULL: none) seeds both layers
 * of every pixel with depth = quant(zn), payload = all ones ("no hair hit"): a hit behind it loses the atomic
 * min ("reads the existing depth buffer", 208-210 "keeping depth"). rgb[h][w][3] (NULL: the constant
 * background) is what O7 composites over ("blended into the main render target"). */
int orc_frame_set_scene(orc_frame*, const float* zn, const float* rgb, uint32_t w, uint32_t h);
/* R-seq ("each groom is processed sequentially ... blended into the render target
 * before the next ... preserving the depth buffer between groom passes"): state of ONE pass. groom_mask: bit g set
 * = groom g is drawn in this pass (O1 gives the others N_LOD = 0); dq[h][w]: the depth kept so far as 24-bit
 * integers (NULL: none; takes precedence over the scene's zn); alpha[h][w]: the alpha accumulated so far (NULL: 0),
 * O7 writes out.w = a + (1 - a) alpha. Reset with (0xFFFFFFFF, NULL, NULL, 0, 0). */
int orc_frame_set_pass(orc_frame*, uint32_t groom_mask, const uint32_t* dq, const float* alpha, uint32_t w, uint32_t h);
/* Restrict the pixel loops of O4, O6 (grown by 7 px) and O7 to [x0, x1) x [y0, y1). Pixels are independent in
 * all three, so values inside the window equal those of the full-frame run: a way to SAMPLE a full-size frame
 * (the raster's hit counts then cover the window only). Default / reset: 0, 0, 1 << 30, 1 << 30. */
void orc_frame_set_window(orc_frame*, int x0, int y0, int x1, int y1);

/* MSAA-k reference mode (DESIGN.md R-msaa; "recording samples into multiple layers of a uint64 image
 * and resolving them later ... only as a reference"). k in {1, 2, 4, 8}: sample s of a pixel sits at the standard
 * multisample offset; layer s = atomic min over the hits at that sample: the segment meets the pixel's closed
 * square (R10) and passes within the centre radius (R9) of the SAMPLE point; depth / parameter at the closest
 * point to the sample (R11); word as O4. ms[k][H][W]. Resolve: out = mean over samples of (shaded hit | background),
 * alpha = hit samples / k. */
int orc_frame_raster_msaa(orc_frame*, const orc_camera*, const orc_params*, uint32_t k);
void orc_frame_get_msaa(const orc_frame*, uint64_t* out);
int orc_frame_set_msaa(orc_frame*, const uint64_t* in, uint32_t k, uint32_t w, uint32_t h);
int orc_frame_resolve_msaa(orc_frame*, const orc_camera*, const orc_params*);

/* R-payload ("G-buffer compression"): mode 1 makes O4 write the paper's self-contained
 * word [63:40] dq | [39:32] ox8 | [31:24] oy8 | [23:18] u6 | [17:12] v6 | [11:6] w6 | [5:0] ao6 (octahedral tangent
 * 2 x uint8; root coordinates u, v, strand parameter w and ambient occlusion 4 x uint6) instead of
 * strand id | segment | t, and O6 shade from the word alone: position from the depth at the pixel centre
 * (PAPER.md:90), tangent from the octahedral code, shading parameters from w, AO from the word; the screen tangent
 * O7 uses is the projected direction of the decoded tangent. The word names no groom, so O6 needs exactly one
 * groom in the pass mask (the paper shades groom by groom): else orc_frame_shade returns -4.
 * Mode 0 (default) is the strand-id payload. MSAA mode ignores it. */
void orc_frame_set_payload_mode(orc_frame*, int mode);
/* pure functions of the payload, fp32 fixed order (pins): octahedral code of a unit vector / unit vector of a code;
 * the 40 payload bits of a hit at parameter t on segment j of a strand v[C][4] (x, y, z, ao) with folded 24-bit
 * root coordinates a1, a2 (R6); fields of a word: dq, ox8, oy8, u6, v6, w6, ao6 */
void orc_oct_encode(const float T[3], uint32_t out[2]);
void orc_oct_decode(uint32_t ox, uint32_t oy, float out[3]);
uint64_t orc_payload40(const float* v, int j, int C, float t, uint32_t a1, uint32_t a2);
void orc_unpack_payload(uint64_t w, uint32_t out[7]);

/* O6: colour[H][W][3] fp64 (0 where no centre hit); tangents[H][W][4] fp32 = (T_G.xy, T_A.xy) */
int orc_frame_shade(orc_frame*, const orc_camera*, const orc_params*);
void orc_frame_get_colour(const orc_frame*, double* rgb);
void orc_frame_get_tangents(const orc_frame*, float* t4);
/* O7: out[H][W][4] fp64 (rgb premultiplied-composited over background, alpha) */
int orc_frame_filter(orc_frame*, const orc_camera*, const orc_params*);
void orc_frame_get_out(const orc_frame*, double* rgba);

#ifdef __cplusplus
}
#endif
#endif
