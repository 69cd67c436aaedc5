// hair_oracle.cpp — CPU ORACLE of the deferred hair pipeline (arxiv/paper_2607_04230).
//
// TEST INFRASTRUCTURE ONLY (see hair_oracle.h). Plain, slow, single-threaded, obviously
// correct. No blocking, no fusion, no reordering beyond what the paper / DESIGN.md §3
// state. Build: g++ -std=c++17 -O2 -ffp-contract=off -fno-fast-math -shared -fPIC.
//
// Stage map (DESIGN.md §3 numbering; PAPER.md = /root/reference/PAPER.md):
//   O1 LOD            PAPER.md:102-136  §3.2, Eq. 1-5
//   O2 generation     PAPER.md:50, 62-64 §2 / §3.1.1, Code 1
//   O3 calcTangent    PAPER.md:353-359  Code 1 lines 1-4
//   O4 raster+resolve PAPER.md:66-96    §3.1.2 (two layers PAPER.md:68-74, atomic min PAPER.md:85)
//   O6 shading        PAPER.md:188-196  §3.4 (stand-in model, R23: parity unpinned vs paper)
//   O7 filter         PAPER.md:154-176  §3.3, Eq. 9-10, Code 2
//   O4p/O6p paper payload PAPER.md:78-96 §3.1.2 "G-buffer compression" (DESIGN.md R-payload): the word carries
//                     octahedral tangent 2 x uint8 + u, v, w, AO 4 x uint6 instead of strand id | segment | t;
//                     shading reconstructs the position from the depth and reads everything else from the word
#include "hair_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

namespace {

const uint64_t EMPTY = ~0ull;
// DESIGN.md R-scene: a word whose 40 payload bits are all ones carries no hair hit; its depth bits are the
// scene's depth at the pixel (the far end, all ones, without a scene). Real hits never have strand id 2^24 - 1.
const uint64_t PAYLOAD_NONE = (1ull << 40) - 1;
inline bool none(uint64_t w) { return (w & PAYLOAD_NONE) == PAYLOAD_NONE; }
const double PI = 3.14159265358979323846;

// ---------------------------------------------------------------- hash (R26)
// PAPER.md:369-371 "PCG rand(b.strandIndex); uv = rand.next2()". Stateless form:
// the 32-bit PCG output permutation RXS-M-XS applied to an LCG step, keyed
// (seed, id, stream): hash = pcg(pcg(pcg(seed) + id) + stream).
inline uint32_t pcg(uint32_t v) {
  uint32_t s = v * 747796405u + 2891336453u;
  uint32_t w = ((s >> ((s >> 28) + 4u)) ^ s) * 277803737u;
  return (w >> 22) ^ w;
}
inline uint32_t hash3(uint32_t seed, uint32_t id, uint32_t stream) {
  return pcg(pcg(pcg(seed) + id) + stream);
}
inline uint32_t u24(uint32_t h) { return h >> 8; }                 // 24-bit integer
inline double u01(uint32_t h) { return double(h >> 8) / 16777216.0; }  // exact in fp32 and fp64

enum : uint32_t { ST_ROOT1 = 1, ST_ROOT2 = 2, ST_CURL = 3, ST_FRIZZ = 16, ST_LOD = 0xB0 };

struct V3 {
  double x, y, z;
};
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
inline V3 normalize(V3 a) {
  double l = std::sqrt(dot(a, a));
  return l > 0 ? (1.0 / l) * a : V3{0, 0, 0};
}

// ---------------------------------------------------------------- O3 calcTangent
// PAPER.md:353-359, verbatim semantics.
inline V3 calcTangent(int idx, int count, V3 prev, V3 curr, V3 next) {
  if (idx == 0) return normalize(next - curr);               // Root
  else if (idx == count - 1) return normalize(curr - prev);  // Tip
  else return normalize(next - prev);
}

// ---------------------------------------------------------------- word (R7, R8)
// [63:40] dq | [39:16] sid | [15:9] j | [8:0] t9. fp32, one rounding per op.
inline uint32_t quant_depth(float zn) {
  float s = zn * 16777215.0f;
  s = s + 0.5f;
  uint32_t q = (uint32_t)s;
  return std::min<uint32_t>(q, 0xFFFFFEu);
}
inline uint32_t quant_t(float t) {
  float s = t * 511.0f;
  s = s + 0.5f;
  return (uint32_t)s;
}
inline uint64_t pack(float zn, uint32_t sid, uint32_t j, float t) {
  return (uint64_t(quant_depth(zn)) << 40) | (uint64_t(sid & 0xFFFFFFu) << 16) |
         (uint64_t(j & 0x7Fu) << 9) | uint64_t(quant_t(t) & 0x1FFu);
}
inline uint32_t w_dq(uint64_t w) { return uint32_t(w >> 40); }
inline uint32_t w_sid(uint64_t w) { return uint32_t(w >> 16) & 0xFFFFFFu; }
inline uint32_t w_j(uint64_t w) { return uint32_t(w >> 9) & 0x7Fu; }
inline uint32_t w_t9(uint64_t w) { return uint32_t(w) & 0x1FFu; }

// ---------------------------------------------------------------- paper payload (R-payload)
// [63:40] dq | [39:32] ox8 | [31:24] oy8 | [23:18] u6 | [17:12] v6 | [11:6] w6 | [5:0] ao6: "24 bits are used for
// depth", "octahedral unit vector encoding" of the tangent, "uvw styling coordinates", ambient occlusion, "all
// float values except for depth are quantized as either uint8 or uint6" — 2 x 8 + 4 x 6 is the only such split
// that fills the 40 bits. Every code is a decision taken in fp32, one rounding per operation, in this order.
struct F3 {
  float x, y, z;
};
inline F3 unit3f(float x, float y, float z) {
  float dd = x * x;
  float e = y * y;
  dd = dd + e;
  e = z * z;
  dd = dd + e;
  if (!(dd > 0.f)) return {1.f, 0.f, 0.f};
  float len = std::sqrt(dd);
  return {x / len, y / len, z / len};
}
// calcTangent on fp32 vertices
inline F3 tangent_f32(int idx, int count, const float* prev, const float* curr, const float* next) {
  const float *a, *b;
  if (idx == 0) a = next, b = curr;                // Root
  else if (idx == count - 1) a = curr, b = prev;   // Tip
  else a = next, b = prev;
  return unit3f(a[0] - b[0], a[1] - b[1], a[2] - b[2]);
}
inline uint32_t q8s(float p) {  // [-1, 1] -> uint8
  float h = p * 0.5f;
  h = h + 0.5f;
  h = h * 255.f;
  h = h + 0.5f;
  return std::min<uint32_t>(uint32_t(h), 255u);
}
inline uint32_t q6(float v) {  // [0, 1] -> uint6
  float h = v * 63.f;
  h = h + 0.5f;
  return std::min<uint32_t>(uint32_t(h), 63u);
}
// octahedral encoding of a unit vector: project on |x| + |y| + |z| = 1, fold the lower hemisphere outwards
inline void oct_encode(F3 T, uint32_t& ox, uint32_t& oy) {
  float s = std::fabs(T.x) + std::fabs(T.y);
  s = s + std::fabs(T.z);
  float px = T.x / s, py = T.y / s;
  if (T.z < 0.f) {
    float ax = 1.f - std::fabs(py), ay = 1.f - std::fabs(px);
    px = px >= 0.f ? ax : -ax;
    py = py >= 0.f ? ay : -ay;
  }
  ox = q8s(px);
  oy = q8s(py);
}
inline F3 oct_decode(uint32_t ox, uint32_t oy) {
  float px = float(ox) / 255.f;
  px = px * 2.f;
  px = px - 1.f;
  float py = float(oy) / 255.f;
  py = py * 2.f;
  py = py - 1.f;
  float z = 1.f - std::fabs(px);
  z = z - std::fabs(py);
  float tx = px, ty = py;
  if (z < 0.f) {
    float ax = 1.f - std::fabs(py), ay = 1.f - std::fabs(px);
    tx = px >= 0.f ? ax : -ax;
    ty = py >= 0.f ? ay : -ay;
  }
  return unit3f(tx, ty, z);
}
inline uint32_t uv6(uint32_t a24) { return (a24 * 63u + (1u << 23)) >> 24; }  // round(a * 2^-24 * 63), integers
// the 40 payload bits of a hit on segment j (of C control points) at parameter t. v = the strand's fp32 vertices
// (x, y, z, ao) x C; a1, a2 = the strand's folded 24-bit root coordinates (R6).
inline uint64_t payload40(const float* v, int j, int C, float t, uint32_t a1, uint32_t a2) {
  auto P = [&](int i) { return v + 4 * std::min(std::max(i, 0), C - 1); };
  F3 Tj = tangent_f32(j, C, P(j - 1), P(j), P(j + 1));
  F3 Tj1 = tangent_f32(j + 1, C, P(j), P(j + 1), P(j + 2));
  float omt = 1.f - t;
  float x = omt * Tj.x, y = omt * Tj.y, z = omt * Tj.z;
  float x1 = t * Tj1.x, y1 = t * Tj1.y, z1 = t * Tj1.z;
  F3 T = unit3f(x + x1, y + y1, z + z1);
  uint32_t ox, oy;
  oct_encode(T, ox, oy);
  float w = float(j) + t;
  w = w / float(C - 1);
  float ao = omt * P(j)[3];
  float ao1 = t * P(j + 1)[3];
  ao = ao + ao1;
  ao = std::min(std::max(ao, 0.f), 1.f);
  return (uint64_t(ox) << 32) | (uint64_t(oy) << 24) | (uint64_t(uv6(a1)) << 18) | (uint64_t(uv6(a2)) << 12) |
         (uint64_t(q6(w)) << 6) | uint64_t(q6(ao));
}

// ---------------------------------------------------------------- camera (R-proj)
struct Cam {
  float eye[3], r[3], u[3], f[3];
  float near_z, fpx, A, B, half_w, half_h;
  uint32_t W, H;
};
Cam make_cam(const orc_camera* c) {
  Cam k;
  for (int i = 0; i < 3; ++i) {
    k.eye[i] = c->eye[i];
    k.r[i] = c->right[i];
    k.u[i] = c->up[i];
    k.f[i] = c->forward[i];
  }
  k.near_z = c->near_z;
  k.W = c->width;
  k.H = c->height;
  // constants computed once in double, rounded to float
  double fpx = (0.5 * double(c->height)) / std::tan(0.5 * double(c->vfov_y));
  double fn = double(c->far_z) - double(c->near_z);
  k.fpx = float(fpx);
  k.A = float(double(c->far_z) / fn);
  k.B = float(double(c->far_z) * double(c->near_z) / fn);
  k.half_w = 0.5f * float(c->width);
  k.half_h = 0.5f * float(c->height);
  return k;
}
struct Proj {
  float sx, sy, zn, zv;
  bool valid;
};
// fp32, fixed operation order: dot(a,b) = (a.x*b.x + a.y*b.y) + a.z*b.z
inline float dot3f(float ax, float ay, float az, const float* b) {
  float s = ax * b[0];
  float t = ay * b[1];
  s = s + t;
  t = az * b[2];
  return s + t;
}
inline Proj project(const Cam& k, float px, float py, float pz) {
  float qx = px - k.eye[0], qy = py - k.eye[1], qz = pz - k.eye[2];
  float xv = dot3f(qx, qy, qz, k.r);
  float yv = dot3f(qx, qy, qz, k.u);
  float zv = dot3f(qx, qy, qz, k.f);
  Proj o;
  o.zv = zv;
  o.valid = zv >= k.near_z;
  if (!o.valid) {
    o.sx = o.sy = o.zn = 0.f;
    return o;
  }
  float a = k.fpx * xv;
  a = a / zv;
  o.sx = k.half_w + a;
  float b = k.fpx * yv;
  b = b / zv;
  o.sy = k.half_h - b;
  float c = k.B / zv;
  o.zn = k.A - c;
  return o;
}

// ---------------------------------------------------------------- scene
struct Groom {
  uint32_t V, Lv, T, Q;
  std::vector<float> pos, ao, xform;
  std::vector<uint32_t> idx, npt, off;  // off = exclusive scan of npt (size T+1)
  orc_style st;
  uint32_t N;         // strands per instance
  uint32_t sid_base;  // first stable strand id
  uint32_t gid_base;  // first bundle-instance index
  uint32_t c_full;
  const float* X(uint32_t layer, uint32_t v) const { return &pos[(size_t(layer) * V + v) * 3]; }
  double AO(uint32_t layer, uint32_t v) const { return ao.empty() ? 1.0 : double(ao[size_t(layer) * V + v]); }
};

struct Entry {
  uint32_t nlod, C, slot_base, vertex_base;
};

}  // namespace

struct orc_frame {
  std::vector<Groom> grooms;
  std::vector<Entry> table;
  std::vector<float> L;
  uint32_t n_strands = 0;
  uint64_t n_vertices = 0;
  std::vector<double> v64;
  std::vector<float> v32;
  uint32_t W = 0, H = 0;
  std::vector<uint64_t> gbuf;
  std::vector<double> colour;
  std::vector<float> tang;
  std::vector<double> out;
  // Pixel window [wx0, wx1) x [wy0, wy1) the pixel loops of O4/O6/O7 are restricted to (default: the whole
  // image). Pixels are independent in all three stages, so every value inside the window is the value of the
  // full-frame run; this only lets a test sample a full-size frame in seconds. O6 covers the window grown by
  // the largest filter radius (7), which is what O7 reads.
  int wx0 = 0, wy0 = 0, wx1 = 1 << 30, wy1 = 1 << 30;
  // optional scene behind / in front of the hair (R-scene): depth zn in [0, 1] per pixel and the colour the hair
  // is composited over ("reads the existing depth buffer ... blended into the main render target")
  std::vector<float> scene_zn;   // [H][W] or empty
  std::vector<float> scene_rgb;  // [H][W][3] or empty
  // sequential per-groom passes (DESIGN.md R-seq): the depth kept from the passes before,
  // already quantised (takes precedence over scene_zn), the alpha accumulated so far, and the grooms of this pass
  std::vector<uint64_t> ms;         // MSAA-k reference: [k][H][W] words (R-msaa)
  uint32_t ms_k = 0;
  std::vector<uint32_t> scene_dq;   // [H][W] or empty
  std::vector<float> scene_alpha;   // [H][W] or empty
  uint32_t groom_mask = 0xFFFFFFFFu;
  int payload_mode = 0;  // 0: strand id | segment | t (R7); 1: the paper's payload (R-payload)
  // deep opacity maps of the point lights (DESIGN.md R-dom), set by orc_frame_set_dom: O6 then scales
  // light l's contribution by the transmittance towards it. Not owned: the caller keeps the arrays alive.
  struct Dom {
    bool on = false;
    orc_camera cam;
    const uint32_t* z0 = nullptr;   // [res][res] depth of the conservative layer seen from the light, 0xFFFFFFFF = none
    const uint32_t* cnt = nullptr;  // [res][res][4] fragments per layer
    uint32_t D[4];                  // layer ends, in depth steps behind z0
    double alpha_s = 0.0;
  } dom[4];
  double dom_beta[16] = {1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1, 1};  // Eq. 7: per groom, of the frame being shaded
};

namespace {

// exclusive scans over bundle-instances in index order (O1 step 6)
void rescan(orc_frame* f) {
  uint32_t slot = 0;
  uint64_t vtx = 0;
  for (auto& e : f->table) {
    e.slot_base = slot;
    e.vertex_base = uint32_t(vtx);
    slot += e.nlod;
    vtx += uint64_t(e.nlod) * e.C;
  }
  f->n_strands = slot;
  f->n_vertices = vtx;
}

// Eq. 1 and Eq. 4-5, fp32. R14: C = min(C, C_full),
// C_raw = max(C_raw, 3).
void lod_counts(float L, uint32_t N, float delta, uint32_t Lv, uint32_t c_full, uint32_t out[3]) {
  uint32_t nlod = 0;
  if (N > 0) {
    float a = float(N) + delta;
    a = L * a;
    a = std::ceil(a);
    a = std::min(std::max(a, 1.0f), float(N));
    nlod = uint32_t(a);
  }
  float s = std::sqrt(L);
  s = s * 127.0f;
  s = std::floor(s);
  uint32_t craw = uint32_t(s);
  craw = std::max(craw, std::max(Lv, 3u));
  uint32_t lg = 31u - uint32_t(__builtin_clz(craw - 1u));  // floor(log2(craw-1)), craw >= 3
  uint32_t C = std::min((1u << lg) + 1u, 127u);
  C = std::min(C, c_full);
  out[0] = nlod;
  out[1] = craw;
  out[2] = C;
}

// ---------------------------------------------------------------- O2 generation (fp64)
struct Base {
  V3 p, T;     // position and unit tangent of the base spline
  double ao;   // R25
  uint32_t i;  // interval
  double t;
};

struct StrandCtx {
  const Groom* g;
  uint32_t tri;
  std::vector<V3> P, m, Pc, mc;  // strand's and centre curve's layer points / Catmull-Rom tangents
  std::vector<double> AOl;
};

void layer_points(const Groom& g, uint32_t tri, const double b[3], std::vector<V3>& P,
                  std::vector<V3>& m, std::vector<double>* AOl) {
  const uint32_t* v = &g.idx[size_t(tri) * 3];
  P.resize(g.Lv);
  m.resize(g.Lv);
  if (AOl) AOl->resize(g.Lv);
  for (uint32_t i = 0; i < g.Lv; ++i) {
    const float *x0 = g.X(i, v[0]), *x1 = g.X(i, v[1]), *x2 = g.X(i, v[2]);
    // R1: barycentric interpolation inside the prism layer (paper: bilinear in a quad)
    P[i] = {b[0] * x0[0] + b[1] * x1[0] + b[2] * x2[0], b[0] * x0[1] + b[1] * x1[1] + b[2] * x2[1],
            b[0] * x0[2] + b[1] * x1[2] + b[2] * x2[2]};
    if (AOl) (*AOl)[i] = b[0] * g.AO(i, v[0]) + b[1] * g.AO(i, v[1]) + b[2] * g.AO(i, v[2]);
  }
  // R4: finite-difference (Catmull-Rom) tangents, one-sided at the ends (Code 1 pass 1)
  for (uint32_t i = 0; i < g.Lv; ++i) {
    if (i == 0) m[i] = P[1] - P[0];
    else if (i == g.Lv - 1) m[i] = P[i] - P[i - 1];
    else m[i] = 0.5 * (P[i + 1] - P[i - 1]);
  }
}

// R5: control point j of C, uniform in w; layer i at w = i/(Lv-1); integer index arithmetic.
inline void cp_param(uint32_t j, uint32_t C, uint32_t Lv, uint32_t& i, double& t, double& w) {
  uint32_t num = j * (Lv - 1), den = C - 1;
  i = std::min(num / den, Lv - 2);
  t = double(num - i * den) / double(den);
  w = double(j) / double(den);
}

// cubic Hermite between layers i and i+1
inline void hermite(const std::vector<V3>& P, const std::vector<V3>& m, uint32_t i, double t, V3& p,
                    V3& T) {
  double t2 = t * t, t3 = t2 * t;
  double h00 = 2 * t3 - 3 * t2 + 1, h10 = t3 - 2 * t2 + t, h01 = -2 * t3 + 3 * t2, h11 = t3 - t2;
  p = h00 * P[i] + h10 * m[i] + h01 * P[i + 1] + h11 * m[i + 1];
  double d00 = 6 * t2 - 6 * t, d10 = 3 * t2 - 4 * t + 1, d01 = -6 * t2 + 6 * t, d11 = 3 * t2 - 2 * t;
  T = normalize(d00 * P[i] + d10 * m[i] + d01 * P[i + 1] + d11 * m[i + 1]);
}

// root barycentrics (R6): fold map on 24-bit integers, so that fp32 and fp64 agree exactly
void root_a24(const Groom& g, uint32_t id_local, uint32_t& a1, uint32_t& a2) {
  a1 = u24(hash3(g.st.seed, id_local, ST_ROOT1));
  a2 = u24(hash3(g.st.seed, id_local, ST_ROOT2));
  if (a1 + a2 > 16777216u) {
    a1 = 16777216u - a1;
    a2 = 16777216u - a2;
  }
}
void root_bary(const Groom& g, uint32_t id_local, double b[3]) {
  uint32_t a1, a2;
  root_a24(g, id_local, a1, a2);
  b[1] = double(a1) / 16777216.0;
  b[2] = double(a2) / 16777216.0;
  b[0] = (1.0 - b[1]) - b[2];
}

uint32_t tri_of(const Groom& g, uint32_t id_local) {
  return uint32_t(std::upper_bound(g.off.begin(), g.off.end(), id_local) - g.off.begin()) - 1u;
}

// frizz lattice value (R24): one hash per (node, channel); the sum of its four bytes is a discrete
// Irwin-Hall(4) variable with mean 510 and variance 4*(256^2-1)/12 = 21845: unit variance, no
// transcendental.
double frizz_lattice(const Groom& g, uint32_t id_local, uint32_t n, uint32_t ch) {
  uint32_t h = hash3(g.st.seed, id_local, ST_FRIZZ + 2u * n + ch);
  uint32_t s = (h & 255u) + ((h >> 8) & 255u) + ((h >> 16) & 255u) + (h >> 24);
  return (double(s) - 510.0) / std::sqrt(21845.0);
}

// one strand, groom-local space, C control points: out[C][4], base_tan[C][3]
void strand_local(const Groom& g, uint32_t id_local, uint32_t C, double* out, double* base_tan) {
  const orc_style& st = g.st;
  uint32_t tri = tri_of(g, id_local);
  double b[3];
  root_bary(g, id_local, b);
  std::vector<V3> P, m, Pc, mc;
  std::vector<double> AOl;
  layer_points(g, tri, b, P, m, &AOl);
  const double third[3] = {1.0 / 3.0, 1.0 / 3.0, 1.0 / 3.0};
  layer_points(g, tri, third, Pc, mc, nullptr);
  const uint32_t* v = &g.idx[size_t(tri) * 3];
  double curl_u = u01(hash3(st.seed, id_local, ST_CURL));
  for (uint32_t j = 0; j < C; ++j) {
    uint32_t i;
    double t, w;
    cp_param(j, C, g.Lv, i, t, w);
    V3 p, T, c, Tc;
    hermite(P, m, i, t, p, T);
    hermite(Pc, mc, i, t, c, Tc);
    double ao = (1 - t) * AOl[i] + t * AOl[i + 1];
    ao = std::min(std::max(ao, 0.0), 1.0);
    // frame from the cage edge v0->v1, orthogonalised against the UNSTYLED base tangent
    const float *e0a = g.X(i, v[0]), *e0b = g.X(i, v[1]), *e1a = g.X(i + 1, v[0]), *e1b = g.X(i + 1, v[1]);
    V3 E0 = {double(e0b[0]) - e0a[0], double(e0b[1]) - e0a[1], double(e0b[2]) - e0a[2]};
    V3 E1 = {double(e1b[0]) - e1a[0], double(e1b[1]) - e1a[1], double(e1b[2]) - e1a[2]};
    V3 E = (1 - t) * E0 + t * E1;
    V3 Nn = E - dot(E, T) * T;
    if (dot(Nn, Nn) < 1e-20) {  // degenerate: least-aligned coordinate axis
      double ax = std::fabs(T.x), ay = std::fabs(T.y), az = std::fabs(T.z);
      V3 a = (ax <= ay && ax <= az) ? V3{1, 0, 0} : (ay <= az ? V3{0, 1, 0} : V3{0, 0, 1});
      Nn = a - dot(a, T) * T;
    }
    V3 N = normalize(Nn);
    V3 B = cross(T, N);
    // styling, fixed order clump -> twist -> curl -> frizz (R24)
    if (st.op_mask & ORC_OP_CLUMP) {
      double we = 1.0;
      for (uint32_t e = 0; e < st.clump_exp; ++e) we *= w;
      p = p + (double(st.clump_strength) * we) * (c - p);
    }
    if (st.op_mask & ORC_OP_TWIST) {
      double th = 2.0 * PI * double(st.twist_turns) * w;
      double cs = std::cos(th), sn = std::sin(th);
      V3 d = p - c;  // Rodrigues rotation of d about Tc
      V3 dr = cs * d + sn * cross(Tc, d) + (dot(Tc, d) * (1.0 - cs)) * Tc;
      p = c + dr;
    }
    if (st.op_mask & ORC_OP_CURL) {
      double th = 2.0 * PI * (double(st.curl_turns) * w + curl_u);
      double a = st.curl_ramp_w0 > 0 ? std::min(w / double(st.curl_ramp_w0), 1.0) : 1.0;
      p = p + (double(st.curl_radius) * a) * (std::cos(th) * N + std::sin(th) * B);
    }
    if (st.op_mask & ORC_OP_FRIZZ) {
      uint32_t cells = std::max(st.frizz_cells, 1u);
      // x = w*cells = (j*cells)/(C-1), cell index and fraction in integers (exact)
      uint32_t xn = j * cells, den = C - 1;
      uint32_t c0 = std::min(xn / den, cells - 1u);
      double fr = double(xn - c0 * den) / double(den);
      double s = fr * fr * (3.0 - 2.0 * fr);
      double n0 = (1 - s) * frizz_lattice(g, id_local, c0, 0) + s * frizz_lattice(g, id_local, c0 + 1, 0);
      double n1 = (1 - s) * frizz_lattice(g, id_local, c0, 1) + s * frizz_lattice(g, id_local, c0 + 1, 1);
      double env = st.frizz_ramp_w0 > 0 ? std::min(w / double(st.frizz_ramp_w0), 1.0) : 1.0;
      p = p + (double(st.frizz_sigma) * env) * (n0 * N + n1 * B);
    }
    out[j * 4 + 0] = p.x;
    out[j * 4 + 1] = p.y;
    out[j * 4 + 2] = p.z;
    out[j * 4 + 3] = ao;
    if (base_tan) {
      base_tan[j * 3 + 0] = T.x;
      base_tan[j * 3 + 1] = T.y;
      base_tan[j * 3 + 2] = T.z;
    }
  }
}

// ---------------------------------------------------------------- sid -> vertices
struct Loc {
  bool ok;
  uint64_t voff;
  uint32_t C;
};
Loc locate(const orc_frame* f, uint32_t sid) {
  for (const Groom& g : f->grooms) {
    uint32_t n = g.N * g.Q;
    if (sid >= g.sid_base && sid < g.sid_base + n) {
      uint32_t rel = sid - g.sid_base;
      uint32_t q = rel / g.N, id_local = rel % g.N;
      uint32_t tri = tri_of(g, id_local);
      uint32_t k = id_local - g.off[tri];
      const Entry& e = f->table[g.gid_base + q * g.T + tri];
      if (k >= e.nlod) return {false, 0, 0};
      return {true, uint64_t(e.vertex_base) + uint64_t(k) * e.C, e.C};
    }
  }
  return {false, 0, 0};
}

inline V3 vtx(const orc_frame* f, uint64_t i) {
  return {double(f->v32[i * 4]), double(f->v32[i * 4 + 1]), double(f->v32[i * 4 + 2])};
}

// screen tangent of the segment a word names (R22), fp32 fixed order
void screen_tangent(const orc_frame* f, const Cam& k, uint64_t word, float T[2]) {
  T[0] = 1.f;
  T[1] = 0.f;
  Loc l = locate(f, w_sid(word));
  if (!l.ok) return;
  uint64_t i0 = l.voff + w_j(word);
  Proj a = project(k, f->v32[i0 * 4], f->v32[i0 * 4 + 1], f->v32[i0 * 4 + 2]);
  Proj b = project(k, f->v32[i0 * 4 + 4], f->v32[i0 * 4 + 5], f->v32[i0 * 4 + 6]);
  float dx = b.sx - a.sx, dy = b.sy - a.sy;
  float dd = dx * dx;
  float e = dy * dy;
  dd = dd + e;
  if (!(dd >= 1e-12f)) return;
  float len = std::sqrt(dd);
  T[0] = dx / len;
  T[1] = dy / len;
}

}  // namespace

// =====================================================================================
extern "C" {

uint32_t orc_pcg(uint32_t v) { return pcg(v); }
uint32_t orc_hash3(uint32_t seed, uint32_t id, uint32_t stream) { return hash3(seed, id, stream); }
void orc_lod_counts(float L, uint32_t N, float delta, uint32_t n_layers, uint32_t c_full,
                    uint32_t out[3]) {
  lod_counts(L, N, delta, n_layers, c_full, out);
}
void orc_calc_tangent(int idx, int count, const double prev[3], const double curr[3],
                      const double next[3], double out[3]) {
  V3 t = calcTangent(idx, count, {prev[0], prev[1], prev[2]}, {curr[0], curr[1], curr[2]},
                     {next[0], next[1], next[2]});
  out[0] = t.x;
  out[1] = t.y;
  out[2] = t.z;
}
uint64_t orc_pack(float zn, uint32_t sid, uint32_t j, float t) { return pack(zn, sid, j, t); }
void orc_unpack(uint64_t w, uint32_t out[4]) {
  out[0] = w_dq(w);
  out[1] = w_sid(w);
  out[2] = w_j(w);
  out[3] = w_t9(w);
}
void orc_frame_set_payload_mode(orc_frame* f, int mode) { f->payload_mode = mode ? 1 : 0; }
void orc_oct_encode(const float T[3], uint32_t out[2]) { oct_encode({T[0], T[1], T[2]}, out[0], out[1]); }
void orc_oct_decode(uint32_t ox, uint32_t oy, float out[3]) {
  F3 t = oct_decode(ox, oy);
  out[0] = t.x, out[1] = t.y, out[2] = t.z;
}
uint64_t orc_payload40(const float* v, int j, int C, float t, uint32_t a1, uint32_t a2) {
  return payload40(v, j, C, t, a1, a2);
}
void orc_unpack_payload(uint64_t w, uint32_t out[7]) {
  out[0] = w_dq(w);
  out[1] = uint32_t(w >> 32) & 0xFFu;
  out[2] = uint32_t(w >> 24) & 0xFFu;
  out[3] = uint32_t(w >> 18) & 63u;
  out[4] = uint32_t(w >> 12) & 63u;
  out[5] = uint32_t(w >> 6) & 63u;
  out[6] = uint32_t(w) & 63u;
}
int orc_project(const orc_camera* cam, const float p[3], float out[4]) {
  Cam k = make_cam(cam);
  Proj r = project(k, p[0], p[1], p[2]);
  out[0] = r.sx;
  out[1] = r.sy;
  out[2] = r.zn;
  out[3] = r.zv;
  return r.valid ? 1 : 0;
}

// O4 coverage of one segment at one pixel (fp32, fixed order). Returns bit0 = conservative,
// bit1 = centre (R9-R11; centre requires conservative, so centre ⊂ conservative exactly).
static inline int cover_px(float ax, float ay, float bx, float by, float rho2, int x, int y, float& t_out) {
  float dx = bx - ax, dy = by - ay;
  float dd = dx * dx;
  {
    float e = dy * dy;
    dd = dd + e;
  }
  float cx = float(x) + 0.5f, cy = float(y) + 0.5f;
  float ux = cx - ax, uy = cy - ay;
  float t = 0.f;
  if (dd > 0.f) {
    float n = ux * dx;
    float e = uy * dy;
    n = n + e;
    t = n / dd;
    t = std::min(std::max(t, 0.0f), 1.0f);
  }
  t_out = t;
  // conservative: closed segment meets closed pixel square (R10)
  float mnx = std::min(ax, bx), mxx = std::max(ax, bx), mny = std::min(ay, by), mxy = std::max(ay, by);
  bool box = mnx <= float(x + 1) && mxx >= float(x) && mny <= float(y + 1) && mxy >= float(y);
  float c1 = dx * uy;
  float c2 = dy * ux;
  float cr = std::fabs(c1 - c2);
  float ext = std::fabs(dx) + std::fabs(dy);
  ext = 0.5f * ext;
  bool cons = box && cr <= ext;
  if (!cons) return 0;
  // centre: closest point on the segment within rho of the pixel centre (R9)
  float qx = t * dx;
  qx = ax + qx;
  float qy = t * dy;
  qy = ay + qy;
  float ex = cx - qx, ey = cy - qy;
  float d2 = ex * ex;
  {
    float e = ey * ey;
    d2 = d2 + e;
  }
  return (d2 <= rho2) ? 3 : 1;
}

// R-msaa: sample positions inside the pixel, in 1/16 pixel from the pixel centre (the standard 2x / 4x / 8x
// multisample patterns; 1x = the pixel centre). The paper names no pattern.
static const int MS_OFF[4][8][2] = {
    {{0, 0}},
    {{4, 4}, {-4, -4}},
    {{-2, -6}, {6, -2}, {-6, 2}, {2, 6}},
    {{1, -3}, {-1, 3}, {5, 1}, {-3, -5}, {-5, 5}, {-7, -1}, {3, 7}, {7, -7}}};
static inline const int (*ms_pattern(uint32_t k))[2] { return k == 1 ? MS_OFF[0] : k == 2 ? MS_OFF[1] : k == 4 ? MS_OFF[2] : k == 8 ? MS_OFF[3] : nullptr; }

// One sample point of pixel (x, y) at offset (ox, oy)/16 from the centre: hit iff the segment meets the pixel's
// closed square (R10, as the conservative layer) and passes within rho of the sample point (R9 moved to the sample).
// fp32, fixed order, the arithmetic of cover_px with the sample point in place of the pixel centre.
static inline bool sample_hit(float ax, float ay, float bx, float by, float rho2, int x, int y, int ox, int oy, float& t_out) {
  float dx = bx - ax, dy = by - ay;
  float dd = dx * dx;
  {
    float e = dy * dy;
    dd = dd + e;
  }
  // conservative test at the pixel centre
  float cx = float(x) + 0.5f, cy = float(y) + 0.5f;
  float ux = cx - ax, uy = cy - ay;
  float mnx = std::min(ax, bx), mxx = std::max(ax, bx), mny = std::min(ay, by), mxy = std::max(ay, by);
  bool box = mnx <= float(x + 1) && mxx >= float(x) && mny <= float(y + 1) && mxy >= float(y);
  float c1 = dx * uy;
  float c2 = dy * ux;
  float cr = std::fabs(c1 - c2);
  float ext = std::fabs(dx) + std::fabs(dy);
  ext = 0.5f * ext;
  if (!(box && cr <= ext)) return false;
  // closest point to the sample (sample coordinates are exact: multiples of 1/16)
  float sx = float(x) + (0.5f + float(ox) * 0.0625f), sy = float(y) + (0.5f + float(oy) * 0.0625f);
  float vx = sx - ax, vy = sy - ay;
  float t = 0.f;
  if (dd > 0.f) {
    float n = vx * dx;
    float e = vy * dy;
    n = n + e;
    t = n / dd;
    t = std::min(std::max(t, 0.0f), 1.0f);
  }
  t_out = t;
  float qx = t * dx;
  qx = ax + qx;
  float qy = t * dy;
  qy = ay + qy;
  float ex = sx - qx, ey = sy - qy;
  float d2 = ex * ex;
  {
    float e = ey * ey;
    d2 = d2 + e;
  }
  return d2 <= rho2;
}

void orc_segment_cover(const float a[2], const float b[2], float rho, uint32_t w, uint32_t h,
                       uint8_t* cover, float* tq) {
  float rho2 = rho * rho;
  for (uint32_t y = 0; y < h; ++y)
    for (uint32_t x = 0; x < w; ++x) {
      float t;
      cover[y * w + x] = uint8_t(cover_px(a[0], a[1], b[0], b[1], rho2, int(x), int(y), t));
      if (tq) tq[y * w + x] = t;
    }
}

int orc_segment_cover_msaa(const float a[2], const float b[2], float rho, uint32_t w, uint32_t h, uint32_t k,
                           uint8_t* cover, float* tq) {
  const int (*pat)[2] = ms_pattern(k);
  if (!pat) return -4;
  float rho2 = rho * rho;
  for (uint32_t s = 0; s < k; ++s)
    for (uint32_t y = 0; y < h; ++y)
      for (uint32_t x = 0; x < w; ++x) {
        float t = 0.f;
        cover[(s * h + y) * w + x] = sample_hit(a[0], a[1], b[0], b[1], rho2, int(x), int(y), pat[s][0], pat[s][1], t) ? 1 : 0;
        if (tq) tq[(s * h + y) * w + x] = t;
      }
  return 0;
}

orc_frame* orc_frame_create(void) { return new orc_frame(); }
void orc_frame_destroy(orc_frame* f) { delete f; }

int orc_frame_add_groom(orc_frame* f, const orc_groom* in) {
  if (!in || in->n_layers < 2 || in->n_tris == 0 || in->style.spi == 0) return -1;
  Groom g;
  g.V = in->n_verts;
  g.Lv = in->n_layers;
  g.T = in->n_tris;
  g.Q = std::max(in->n_instances, 1u);
  g.pos.assign(in->pos, in->pos + size_t(g.Lv) * g.V * 3);
  if (in->ao) g.ao.assign(in->ao, in->ao + size_t(g.Lv) * g.V);
  g.idx.assign(in->idx, in->idx + size_t(g.T) * 3);
  g.npt.assign(in->strands_per_tri, in->strands_per_tri + g.T);
  if (in->xform) g.xform.assign(in->xform, in->xform + size_t(g.Q) * 12);
  g.st = in->style;
  g.off.resize(g.T + 1);
  uint32_t acc = 0;
  for (uint32_t t = 0; t < g.T; ++t) {
    g.off[t] = acc;
    acc += g.npt[t];
  }
  g.off[g.T] = acc;
  g.N = acc;
  g.c_full = (g.Lv - 1) * g.st.spi + 1;  // PAPER.md:406 (Code 1 line 29)
  if (g.c_full > 127) return -2;
  if (f->grooms.empty()) {
    g.sid_base = 0;
    g.gid_base = 0;
  } else {
    const Groom& p = f->grooms.back();
    g.sid_base = p.sid_base + p.N * p.Q;
    g.gid_base = p.gid_base + p.T * p.Q;
  }
  if (uint64_t(g.sid_base) + uint64_t(g.N) * g.Q >= (1ull << 24)) return -3;
  f->grooms.push_back(std::move(g));
  return int(f->grooms.size()) - 1;
}

// ------------------------------------------------------------------ O1
int orc_frame_lod(orc_frame* f, const orc_camera* cam, const float* lambda, uint32_t n_lambda) {
  Cam k = make_cam(cam);
  f->table.clear();
  f->L.clear();
  float Wf = float(k.W), Hf = float(k.H);
  for (size_t gi = 0; gi < f->grooms.size(); ++gi) {
    const Groom& g = f->grooms[gi];
    float lam = n_lambda == 0 ? 0.f : lambda[n_lambda == 1 ? 0 : gi];
    for (uint32_t q = 0; q < g.Q; ++q)
      for (uint32_t t = 0; t < g.T; ++t) {
        Entry e{0, 0, 0, 0};
        uint32_t N = g.npt[t];
        float Lsel = -1.f;
        if (!(lam > 0.f)) {  // R14: LOD and culling off
          e.nlod = N;
          e.C = g.c_full;
        } else {
          // project each layer's vertices, one AABB over all layers (Eq. 3)
          float mnx = INFINITY, mny = INFINITY, mxx = -INFINITY, mxy = -INFINITY;
          uint32_t n_valid = 0, n_all = 0;
          const float* M = g.xform.empty() ? nullptr : &g.xform[size_t(q) * 12];
          for (uint32_t i = 0; i < g.Lv; ++i)
            for (int c = 0; c < 3; ++c) {
              const float* x = g.X(i, g.idx[size_t(t) * 3 + c]);
              float wx = x[0], wy = x[1], wz = x[2];
              if (M) {  // ((m0*x + m1*y) + m2*z) + m3, fp32
                float r[3];
                for (int a = 0; a < 3; ++a) {
                  float s = M[a * 4 + 0] * x[0];
                  float u = M[a * 4 + 1] * x[1];
                  s = s + u;
                  u = M[a * 4 + 2] * x[2];
                  s = s + u;
                  r[a] = s + M[a * 4 + 3];
                }
                wx = r[0];
                wy = r[1];
                wz = r[2];
              }
              Proj p = project(k, wx, wy, wz);
              ++n_all;
              if (p.valid) {
                ++n_valid;
                mnx = std::min(mnx, p.sx);
                mxx = std::max(mxx, p.sx);
                mny = std::min(mny, p.sy);
                mxy = std::max(mxy, p.sy);
              }
            }
          bool culled = false;
          if (n_valid == 0) culled = true;  // R13: all behind the near plane
          else if (n_valid < n_all) Lsel = 1.f;  // R13: some behind => full detail
          else {
            if (mxx < 0.f || mnx > Wf || mxy < 0.f || mny > Hf) culled = true;
            else {
              float dx = mxx - mnx, dy = mxy - mny;
              float dd = dx * dx;
              float ee = dy * dy;
              dd = dd + ee;
              float diag = std::sqrt(dd);
              float r = diag / Hf;  // Eq. 2, R_y = H
              r = r * lam;
              Lsel = std::min(std::max(r, 0.0f), 1.0f);
            }
          }
          if (culled) {
            e.nlod = 0;
            e.C = 0;
          } else {
            float delta = float(u01(hash3(g.st.seed, q * g.T + t, ST_LOD)));
            uint32_t o[3];
            lod_counts(Lsel, N, delta, g.Lv, g.c_full, o);
            e.nlod = o[0];
            e.C = o[0] ? o[2] : 0;
          }
        }
        if (!((f->groom_mask >> (&g - &f->grooms[0])) & 1u)) e.nlod = e.C = 0;  // R-seq: not in this pass
        f->table.push_back(e);
        f->L.push_back(Lsel);
      }
  }
  rescan(f);
  return 0;
}

uint32_t orc_frame_n_bundles(const orc_frame* f) {
  uint32_t n = 0;
  for (const Groom& g : f->grooms) n += g.T * g.Q;
  return n;
}
uint32_t orc_frame_n_strands_total(const orc_frame* f) {
  uint32_t n = 0;
  for (const Groom& g : f->grooms) n += g.N * g.Q;
  return n;
}
// Eq. 6-8: beta = N_remaining / N_total, delta = -log(beta)
void orc_frame_beta(const orc_frame* f, double* beta, double* delta, double* beta_min) {
  size_t gid = 0;
  double bmin = 1.0;
  for (size_t gi = 0; gi < f->grooms.size(); ++gi) {
    const Groom& g = f->grooms[gi];
    uint64_t remaining = 0, total = 0;
    for (uint32_t q = 0; q < g.Q; ++q)
      for (uint32_t t = 0; t < g.T; ++t, ++gid) {
        const uint32_t nlod = f->table[gid].nlod, N = g.npt[t];
        if (nlod == 0) continue;  // not drawn: frustum-culled, masked, or an empty bundle
        remaining += nlod;
        total += N;
        bmin = std::min(bmin, double(nlod) / double(N));
      }
    const double b = total ? double(remaining) / double(total) : 1.0;
    if (beta) beta[gi] = b;
    if (delta) delta[gi] = -std::log(b);  // Eq. 8
  }
  if (beta_min) *beta_min = bmin;
}
// Eq. 7: V'(d) = exp(-sigma (beta d)): thinning to the fraction beta = traversing the depth beta d = d exp(-delta)
double orc_depth_fix(double d, double delta) { return d * std::exp(-delta); }

uint32_t orc_frame_n_strands(const orc_frame* f) { return f->n_strands; }
uint64_t orc_frame_n_vertices(const orc_frame* f) { return f->n_vertices; }
void orc_frame_get_table(const orc_frame* f, uint32_t* t4, float* L) {
  for (size_t i = 0; i < f->table.size(); ++i) {
    if (t4) {
      t4[i * 4 + 0] = f->table[i].nlod;
      t4[i * 4 + 1] = f->table[i].C;
      t4[i * 4 + 2] = f->table[i].slot_base;
      t4[i * 4 + 3] = f->table[i].vertex_base;
    }
    if (L) L[i] = f->L[i];
  }
}
int orc_frame_set_table(orc_frame* f, const uint32_t* t4, uint32_t n) {
  if (n != orc_frame_n_bundles(f)) return -1;
  f->table.resize(n);
  f->L.assign(n, -1.f);
  for (uint32_t i = 0; i < n; ++i) f->table[i] = {t4[i * 4], t4[i * 4 + 1], 0, 0};
  rescan(f);
  for (uint32_t i = 0; i < n; ++i)
    if (f->table[i].nlod && (f->table[i].slot_base != t4[i * 4 + 2] || f->table[i].vertex_base != t4[i * 4 + 3]))
      return -2;  // the supplied scans disagree with the definition
  return 0;
}

// ------------------------------------------------------------------ O2
int orc_frame_generate(orc_frame* f) {
  f->v64.assign(size_t(f->n_vertices) * 4, 0.0);
  std::vector<double> loc;
  for (const Groom& g : f->grooms)
    for (uint32_t q = 0; q < g.Q; ++q)
      for (uint32_t t = 0; t < g.T; ++t) {
        const Entry& e = f->table[g.gid_base + q * g.T + t];
        if (e.nlod == 0) continue;
        loc.resize(size_t(e.C) * 4);
        const float* M = g.xform.empty() ? nullptr : &g.xform[size_t(q) * 12];
        for (uint32_t k = 0; k < e.nlod; ++k) {  // R27: surviving strands = local indices k < N_LOD
          strand_local(g, g.off[t] + k, e.C, loc.data(), nullptr);
          double* o = &f->v64[(size_t(e.vertex_base) + size_t(k) * e.C) * 4];
          for (uint32_t j = 0; j < e.C; ++j) {
            double x = loc[j * 4], y = loc[j * 4 + 1], z = loc[j * 4 + 2];
            if (M) {  // instance transform applied last (DESIGN.md R-inst)
              double wx = double(M[0]) * x + double(M[1]) * y + double(M[2]) * z + double(M[3]);
              double wy = double(M[4]) * x + double(M[5]) * y + double(M[6]) * z + double(M[7]);
              double wz = double(M[8]) * x + double(M[9]) * y + double(M[10]) * z + double(M[11]);
              x = wx;
              y = wy;
              z = wz;
            }
            o[j * 4 + 0] = x;
            o[j * 4 + 1] = y;
            o[j * 4 + 2] = z;
            o[j * 4 + 3] = loc[j * 4 + 3];
          }
        }
      }
  f->v32.resize(f->v64.size());
  for (size_t i = 0; i < f->v64.size(); ++i) f->v32[i] = float(f->v64[i]);
  return 0;
}
void orc_frame_get_vertices_f64(const orc_frame* f, double* o) {
  std::memcpy(o, f->v64.data(), f->v64.size() * sizeof(double));
}
void orc_frame_get_vertices_f32(const orc_frame* f, float* o) {
  std::memcpy(o, f->v32.data(), f->v32.size() * sizeof(float));
}
int orc_frame_set_vertices_f32(orc_frame* f, const float* v, uint64_t n) {
  if (n != f->n_vertices) return -1;
  f->v32.assign(v, v + size_t(n) * 4);
  return 0;
}
int orc_strand(const orc_frame* f, uint32_t groom, uint32_t id_local, uint32_t C, double* out,
               double* base_tan) {
  if (groom >= f->grooms.size() || id_local >= f->grooms[groom].N || C < 2) return -1;
  strand_local(f->grooms[groom], id_local, C, out, base_tan);
  return 0;
}
int orc_root(const orc_frame* f, uint32_t groom, uint32_t id_local, double b[3], uint32_t* tri) {
  if (groom >= f->grooms.size() || id_local >= f->grooms[groom].N) return -1;
  root_bary(f->grooms[groom], id_local, b);
  if (tri) *tri = tri_of(f->grooms[groom], id_local);
  return 0;
}

// ------------------------------------------------------------------ O4 (+ O5: the min IS the resolve)
// Enumerates every (segment, pixel) hit of the frame's vertices under camera k in strand order (`order`: optional
// permutation of the strands): fn(strand, j, x, y, cover bits (1 = conservative, 2 = centre), zn, t). The coverage
// arithmetic of R9-R12 lives here, once, for the G-buffer resolve and for the deep-opacity-map fragment count.
}  // extern "C"
namespace {
struct StrandDir {
  uint64_t voff;
  uint32_t C, sid;
  float width;
  uint32_t a1, a2;  // R-payload: the strand's root coordinates (u, v)
};
template <class Fn>
uint64_t for_each_hit(const orc_frame* f, const Cam& k, const orc_params* prm, const uint32_t* order, Fn&& fn) {
  uint64_t n_seg = 0;
  // strand directory in slot order
  std::vector<StrandDir> dir;
  dir.reserve(f->n_strands);
  for (const Groom& g : f->grooms)
    for (uint32_t q = 0; q < g.Q; ++q)
      for (uint32_t t = 0; t < g.T; ++t) {
        const Entry& e = f->table[g.gid_base + q * g.T + t];
        for (uint32_t kk = 0; kk < e.nlod; ++kk) {
          uint32_t a1 = 0, a2 = 0;
          if (f->payload_mode) root_a24(g, g.off[t] + kk, a1, a2);
          dir.push_back({uint64_t(e.vertex_base) + uint64_t(kk) * e.C, e.C,
                         g.sid_base + q * g.N + g.off[t] + kk, g.st.width_world, a1, a2});
        }
      }
  for (size_t si = 0; si < dir.size(); ++si) {
    const StrandDir& s = dir[order ? order[si] : si];
    for (uint32_t j = 0; j + 1 < s.C; ++j) {
      const float* va = &f->v32[(s.voff + j) * 4];
      const float* vb = va + 4;
      Proj a = project(k, va[0], va[1], va[2]);
      Proj b = project(k, vb[0], vb[1], vb[2]);
      if (!a.valid || !b.valid) continue;  // R12
      ++n_seg;
      // centre radius (R9)
      float rho;
      if (s.width > 0.f) {
        float zm = a.zv + b.zv;
        zm = 0.5f * zm;
        float wpx = s.width * k.fpx;
        wpx = wpx / zm;
        wpx = std::min(std::max(wpx, 0.25f), 1.0f);
        rho = 0.5f * wpx;
      } else
        rho = 0.5f * prm->center_diameter_px;
      float rho2 = rho * rho;
      float mnx = std::min(a.sx, b.sx), mxx = std::max(a.sx, b.sx);
      float mny = std::min(a.sy, b.sy), mxy = std::max(a.sy, b.sy);
      // candidate pixels: [floor(min)-1, floor(max)+1] clipped to the viewport
      float fx0 = std::max(std::floor(mnx) - 1.f, 0.f), fx1 = std::min(std::floor(mxx) + 1.f, float(k.W) - 1.f);
      float fy0 = std::max(std::floor(mny) - 1.f, 0.f), fy1 = std::min(std::floor(mxy) + 1.f, float(k.H) - 1.f);
      if (!(fx0 <= fx1) || !(fy0 <= fy1)) continue;
      int x0 = std::max(int(fx0), f->wx0), x1 = std::min(int(fx1), f->wx1 - 1);
      int y0 = std::max(int(fy0), f->wy0), y1 = std::min(int(fy1), f->wy1 - 1);
      float dz = b.zn - a.zn;
      for (int y = y0; y <= y1; ++y)
        for (int x = x0; x <= x1; ++x) {
          float t;
          int c = cover_px(a.sx, a.sy, b.sx, b.sy, rho2, x, y, t);
          if (!c) continue;
          float zn = t * dz;  // R11: depth at the closest point, linear in screen space
          zn = a.zn + zn;
          if (zn < 0.f || zn > 1.f) continue;
          fn(s, j, x, y, c, zn, t);
        }
    }
  }
  return n_seg;
}
}  // namespace
extern "C" {

int orc_frame_raster(orc_frame* f, const orc_camera* cam, const orc_params* prm,
                     const uint32_t* order, uint64_t counts[3]) {
  Cam k = make_cam(cam);
  f->W = k.W;
  f->H = k.H;
  f->gbuf.assign(size_t(k.W) * k.H * 2, EMPTY);
  if (!f->scene_zn.empty()) {  // R-scene: both layers start at the scene's quantised depth (R8), payload = none
    if (f->scene_zn.size() != size_t(k.W) * k.H) return -3;
    for (size_t p = 0; p < size_t(k.W) * k.H; ++p) {
      float zn = std::min(std::max(f->scene_zn[p], 0.f), 1.f);
      uint64_t seed = (uint64_t(quant_depth(zn)) << 40) | PAYLOAD_NONE;
      f->gbuf[p * 2] = f->gbuf[p * 2 + 1] = seed;
    }
  }
  if (!f->scene_dq.empty()) {  // R-seq: depth kept from the previous passes, as the 24-bit integers themselves
    if (f->scene_dq.size() != size_t(k.W) * k.H) return -3;
    for (size_t p = 0; p < size_t(k.W) * k.H; ++p)
      f->gbuf[p * 2] = f->gbuf[p * 2 + 1] = (uint64_t(f->scene_dq[p] & 0xFFFFFFu) << 40) | PAYLOAD_NONE;
  }
  if (f->v32.size() != size_t(f->n_vertices) * 4) return -1;
  uint64_t n_center = 0, n_cons = 0;
  const uint64_t n_seg = for_each_hit(f, k, prm, order, [&](const StrandDir& s, uint32_t j, int x, int y, int c, float zn, float t) {
    uint64_t w = pack(zn, s.sid, j, t);
    if (f->payload_mode)  // R-payload: same depth bits, the paper's 40 payload bits
      w = (uint64_t(quant_depth(zn)) << 40) | payload40(&f->v32[s.voff * 4], int(j), int(s.C), t, s.a1, s.a2);
    uint64_t* px = &f->gbuf[(size_t(y) * k.W + x) * 2];
    ++n_cons;
    px[1] = std::min(px[1], w);  // PAPER.md:85 atomic min, depth in the high bits
    if (c & 2) {
      ++n_center;
      px[0] = std::min(px[0], w);
    }
  });
  if (counts) {
    counts[0] = n_center;
    counts[1] = n_cons;
    counts[2] = n_seg;
  }
  return 0;
}

// ------------------------------------------------------------------ deep opacity maps (DESIGN.md R-dom)
// The paper names the technique (Yuksel and Keyser 2008) and no more. As restated here, for one light camera:
//  z0(u, v)     = depth of the nearest hair that touches light pixel (u, v): the conservative layer of the frame's
//                 G-buffer rendered from the light, as its 24-bit integer (0xFFFFFFFF where nothing is hit);
//  cnt(u, v, k) = number of (segment, pixel) conservative hits of that pixel whose depth lies in layer k behind z0,
//                 layer k = [D[k-1], D[k]) depth steps (D[-1] = 0, the last layer is open-ended).
// orc_frame_raster under the same camera must have run before (it leaves z0 in the frame's G-buffer).
int orc_frame_dom_count(orc_frame* f, const orc_camera* cam, const orc_params* prm, const uint32_t D[3],
                        uint32_t* z0, uint32_t* cnt) {
  Cam k = make_cam(cam);
  if (f->W != k.W || f->H != k.H || f->gbuf.size() != size_t(k.W) * k.H * 2) return -1;
  if (f->v32.size() != size_t(f->n_vertices) * 4) return -1;
  const size_t n_px = size_t(k.W) * k.H;
  for (size_t p = 0; p < n_px; ++p) z0[p] = none(f->gbuf[p * 2 + 1]) ? 0xFFFFFFFFu : w_dq(f->gbuf[p * 2 + 1]);
  std::memset(cnt, 0, n_px * 4 * sizeof(uint32_t));
  for_each_hit(f, k, prm, nullptr, [&](const StrandDir&, uint32_t, int x, int y, int, float zn, float) {
    const size_t p = size_t(y) * k.W + x;
    const uint32_t d = quant_depth(zn) - z0[p];  // >= 0: z0 is the minimum over these very hits
    const int layer = (d >= D[0]) + (d >= D[1]) + (d >= D[2]);
    ++cnt[p * 4 + layer];
  });
  return 0;
}

// Optical depth seen from ONE texel at `d` depth steps behind its z0: the cumulative fragment count, piecewise linear
// through (0, 0), (D0, c0), (D1, c0 + c1), (D2, c0 + c1 + c2), (D3, c0 + .. + c3), constant beyond (the open last
// layer is taken to end at D3).
static double dom_texel_omega(const uint32_t* cnt4, const uint32_t D[4], double d) {
  if (!(d > 0.0)) return 0.0;
  double lo = 0.0, acc = 0.0;
  for (int kk = 0; kk < 4; ++kk) {
    const double hi = double(D[kk]);
    if (d < hi) return acc + double(cnt4[kk]) * (d - lo) / (hi - lo);
    acc += double(cnt4[kk]);
    lo = hi;
  }
  return acc;
}

// Transmittance towards the light of the map at world point p (Eq. 6: V = exp(-sigma d), with sigma d = alpha_s times
// the fragment count in front of the point). The point's depth behind each texel's z0 is scaled by beta before the
// lookup (Eq. 7: d_eff = beta d, the depth-comparison fix of PAPER.md:138-152). The four texels around the point are
// blended bilinearly (texel centres at integer + 1/2); a texel without hair, or outside the map, contributes 0.
double orc_dom_transmittance(const orc_camera* cam, const uint32_t* z0, const uint32_t* cnt, const uint32_t D[4],
                             double alpha_s, double beta, const float p[3]) {
  Cam k = make_cam(cam);
  Proj q = project(k, p[0], p[1], p[2]);
  if (!q.valid) return 1.0;
  const float zc = std::min(std::max(q.zn, 0.f), 1.f);
  const uint32_t dq = quant_depth(zc);
  const double fx = double(q.sx) - 0.5, fy = double(q.sy) - 0.5;
  const double x0 = std::floor(fx), y0 = std::floor(fy);
  const double wx = fx - x0, wy = fy - y0;
  double omega = 0.0;
  for (int dy = 0; dy < 2; ++dy)
    for (int dx = 0; dx < 2; ++dx) {
      const double xi = x0 + dx, yi = y0 + dy;
      if (xi < 0 || yi < 0 || xi >= double(k.W) || yi >= double(k.H)) continue;
      const size_t t = size_t(yi) * k.W + size_t(xi);
      if (z0[t] == 0xFFFFFFFFu || dq <= z0[t]) continue;
      const double w = (dx ? wx : 1.0 - wx) * (dy ? wy : 1.0 - wy);
      omega += w * dom_texel_omega(&cnt[t * 4], D, beta * double(dq - z0[t]));
    }
  return std::exp(-alpha_s * omega);
}

int orc_frame_set_dom(orc_frame* f, uint32_t light, const orc_camera* cam, const uint32_t* z0, const uint32_t* cnt,
                      const uint32_t D[4], double alpha_s) {
  if (light >= 4) return -1;
  orc_frame::Dom& d = f->dom[light];
  d.on = cam != nullptr;
  if (!d.on) return 0;
  d.cam = *cam;
  d.z0 = z0;
  d.cnt = cnt;
  for (int i = 0; i < 4; ++i) d.D[i] = D[i];
  d.alpha_s = alpha_s;
  return 0;
}
void orc_frame_set_dom_beta(orc_frame* f, const double* beta, uint32_t n) {
  for (uint32_t g = 0; g < 16; ++g) f->dom_beta[g] = g < n ? beta[g] : 1.0;
}

void orc_frame_get_gbuffer(const orc_frame* f, uint64_t* o) {
  std::memcpy(o, f->gbuf.data(), f->gbuf.size() * sizeof(uint64_t));
}
int orc_frame_set_scene(orc_frame* f, const float* zn, const float* rgb, uint32_t w, uint32_t h) {
  f->scene_zn.clear();
  f->scene_rgb.clear();
  if (zn) f->scene_zn.assign(zn, zn + size_t(w) * h);
  if (rgb) f->scene_rgb.assign(rgb, rgb + size_t(w) * h * 3);
  return 0;
}
int orc_frame_set_pass(orc_frame* f, uint32_t groom_mask, const uint32_t* dq, const float* alpha, uint32_t w, uint32_t h) {
  f->groom_mask = groom_mask;
  f->scene_dq.clear();
  f->scene_alpha.clear();
  if (dq) f->scene_dq.assign(dq, dq + size_t(w) * h);
  if (alpha) f->scene_alpha.assign(alpha, alpha + size_t(w) * h);
  return 0;
}
void orc_frame_set_window(orc_frame* f, int x0, int y0, int x1, int y1) {
  f->wx0 = x0, f->wy0 = y0, f->wx1 = x1, f->wy1 = y1;
}
int orc_frame_set_gbuffer(orc_frame* f, const uint64_t* in, uint32_t w, uint32_t h) {
  f->W = w;
  f->H = h;
  f->gbuf.assign(in, in + size_t(w) * h * 2);
  return 0;
}

static bool shade_word(const orc_frame* f, const Cam& k, const orc_params* prm, uint64_t G, double rgb[3]);

// ------------------------------------------------------------------ MSAA-k reference (R-msaa)
// "recording samples into multiple layers of a uint64 image and resolving them later": k sample layers, each the
// atomic min over the hits at its sample point. Same strand directory, projection, centre radius and word as O4.
int orc_frame_raster_msaa(orc_frame* f, const orc_camera* cam, const orc_params* prm, uint32_t ksamp) {
  const int (*pat)[2] = ms_pattern(ksamp);
  if (!pat) return -4;
  Cam k = make_cam(cam);
  f->W = k.W;
  f->H = k.H;
  const size_t np = size_t(k.W) * k.H;
  f->ms.assign(np * ksamp, EMPTY);
  f->ms_k = ksamp;
  if (f->v32.size() != size_t(f->n_vertices) * 4) return -1;
  for (const Groom& g : f->grooms)
    for (uint32_t q = 0; q < g.Q; ++q)
      for (uint32_t t = 0; t < g.T; ++t) {
        const Entry& e = f->table[g.gid_base + q * g.T + t];
        for (uint32_t kk = 0; kk < e.nlod; ++kk) {
          const uint64_t voff = uint64_t(e.vertex_base) + uint64_t(kk) * e.C;
          const uint32_t sid = g.sid_base + q * g.N + g.off[t] + kk;
          for (uint32_t j = 0; j + 1 < e.C; ++j) {
            const float* va = &f->v32[(voff + j) * 4];
            const float* vb = va + 4;
            Proj a = project(k, va[0], va[1], va[2]);
            Proj b = project(k, vb[0], vb[1], vb[2]);
            if (!a.valid || !b.valid) continue;  // R12
            float rho;
            if (g.st.width_world > 0.f) {  // R9
              float zm = a.zv + b.zv;
              zm = 0.5f * zm;
              float wpx = g.st.width_world * k.fpx;
              wpx = wpx / zm;
              wpx = std::min(std::max(wpx, 0.25f), 1.0f);
              rho = 0.5f * wpx;
            } else
              rho = 0.5f * prm->center_diameter_px;
            float rho2 = rho * rho;
            float mnx = std::min(a.sx, b.sx), mxx = std::max(a.sx, b.sx);
            float mny = std::min(a.sy, b.sy), mxy = std::max(a.sy, b.sy);
            float fx0 = std::max(std::floor(mnx) - 1.f, 0.f), fx1 = std::min(std::floor(mxx) + 1.f, float(k.W) - 1.f);
            float fy0 = std::max(std::floor(mny) - 1.f, 0.f), fy1 = std::min(std::floor(mxy) + 1.f, float(k.H) - 1.f);
            if (!(fx0 <= fx1) || !(fy0 <= fy1)) continue;
            int x0 = std::max(int(fx0), f->wx0), x1 = std::min(int(fx1), f->wx1 - 1);
            int y0 = std::max(int(fy0), f->wy0), y1 = std::min(int(fy1), f->wy1 - 1);
            float dz = b.zn - a.zn;
            for (int y = y0; y <= y1; ++y)
              for (int x = x0; x <= x1; ++x)
                for (uint32_t s = 0; s < ksamp; ++s) {
                  float tt;
                  if (!sample_hit(a.sx, a.sy, b.sx, b.sy, rho2, x, y, pat[s][0], pat[s][1], tt)) continue;
                  float zn = tt * dz;
                  zn = a.zn + zn;
                  if (zn < 0.f || zn > 1.f) continue;
                  uint64_t w = pack(zn, sid, j, tt);
                  uint64_t* px = &f->ms[(size_t(s) * k.H + y) * k.W + x];
                  *px = std::min(*px, w);
                }
          }
        }
      }
  return 0;
}
void orc_frame_get_msaa(const orc_frame* f, uint64_t* o) { std::memcpy(o, f->ms.data(), f->ms.size() * sizeof(uint64_t)); }
int orc_frame_set_msaa(orc_frame* f, const uint64_t* in, uint32_t ksamp, uint32_t w, uint32_t h) {
  f->W = w;
  f->H = h;
  f->ms_k = ksamp;
  f->ms.assign(in, in + size_t(w) * h * ksamp);
  return 0;
}
// resolve: every sample with a hit is shaded (O6 of its word), samples without one show the background;
// out = mean over the k samples, alpha = hit samples / k
int orc_frame_resolve_msaa(orc_frame* f, const orc_camera* cam, const orc_params* prm) {
  Cam k = make_cam(cam);
  if (f->W != k.W || f->H != k.H || !f->ms_k) return -1;
  const size_t np = size_t(k.W) * k.H;
  f->out.assign(np * 4, 0.0);
  for (int y = std::max(f->wy0, 0); y < std::min(f->wy1, int(k.H)); ++y)
    for (int x = std::max(f->wx0, 0); x < std::min(f->wx1, int(k.W)); ++x) {
      const size_t p = size_t(y) * k.W + x;
      double acc[3] = {0, 0, 0};
      uint32_t n_hit = 0;
      for (uint32_t s = 0; s < f->ms_k; ++s) {
        uint64_t w = f->ms[size_t(s) * np + p];
        if (none(w)) continue;
        double rgb[3];
        if (!shade_word(f, k, prm, w, rgb)) return -2;
        for (int c = 0; c < 3; ++c) acc[c] += rgb[c];
        ++n_hit;
      }
      double alpha = double(n_hit) / double(f->ms_k);
      for (int c = 0; c < 3; ++c) {
        double bg = f->scene_rgb.empty() ? double(prm->background_rgb[c]) : double(f->scene_rgb[p * 3 + c]);
        f->out[p * 4 + c] = acc[c] / double(f->ms_k) + (1 - alpha) * bg;
      }
      f->out[p * 4 + 3] = alpha;
    }
  return 0;
}

// ------------------------------------------------------------------ O6
// O6 for one word: the shaded linear RGB of the hit it names (stand-in model, R23). Returns false if the strand
// id does not resolve.
// the stand-in shading model (R23) at one point: position, unit tangent, strand parameter w, ambient occlusion
static void shade_model(const orc_frame* f, const Groom* g, const Cam& k, const orc_params* prm, V3 pos, V3 T, double w,
                        double ao, double rgb[3]) {
  V3 eye = {double(k.eye[0]), double(k.eye[1]), double(k.eye[2])};
  double alb[3];
  for (int c = 0; c < 3; ++c)
    alb[c] = (1 - w) * double(g->st.albedo_root[c]) + w * double(g->st.albedo_tip[c]);
  V3 Vd = normalize(eye - pos);
  for (int c = 0; c < 3; ++c) rgb[c] = ao * double(prm->ambient_rgb[c]) * alb[c];
  double beta = double(g->st.roughness), tilt = double(g->st.tilt);
  for (uint32_t li = 0; li < prm->n_lights; ++li) {
    V3 lp = {double(prm->light_pos[li][0]), double(prm->light_pos[li][1]), double(prm->light_pos[li][2])};
    V3 Lv = lp - pos;
    double d2 = dot(Lv, Lv);
    V3 om = (1.0 / std::sqrt(d2)) * Lv;
    double sin_i = std::min(std::max(dot(T, om), -1.0), 1.0);
    double sin_o = std::min(std::max(dot(T, Vd), -1.0), 1.0);
    double cos_i = std::sqrt(std::max(0.0, 1.0 - sin_i * sin_i));
    double th = 0.5 * (std::asin(sin_i) + std::asin(sin_o));
    double MR = std::exp(-(th + tilt) * (th + tilt) / (2.0 * beta * beta));
    double MT = std::exp(-(th - 1.5 * tilt) * (th - 1.5 * tilt) / (8.0 * beta * beta));
    // volumetric shadow (R-dom): transmittance towards light li from its deep opacity map, looked up
    // with the depth-comparison fix of the groom being shaded (Eq. 7)
    double Tl = 1.0;
    if (li < 4 && f->dom[li].on) {
      const float pf[3] = {float(pos.x), float(pos.y), float(pos.z)};
      const orc_frame::Dom& dm = f->dom[li];
      Tl = orc_dom_transmittance(&dm.cam, dm.z0, dm.cnt, dm.D, dm.alpha_s, f->dom_beta[g - f->grooms.data()], pf);
    }
    for (int c = 0; c < 3; ++c) {
      double E = Tl * double(prm->light_rgb[li][c]) / d2;
      rgb[c] += E * cos_i * (double(prm->k_d) * alb[c] + double(prm->k_R) * MR + double(prm->k_TRT) * MT * alb[c]);
    }
  }
}

static bool shade_word(const orc_frame* f, const Cam& k, const orc_params* prm, uint64_t G, double rgb[3]) {
  Loc l = locate(f, w_sid(G));
  if (!l.ok) return false;
  const Groom* g = nullptr;
  for (const Groom& gg : f->grooms)
    if (w_sid(G) >= gg.sid_base && w_sid(G) < gg.sid_base + gg.N * gg.Q) g = &gg;
  int j = int(w_j(G)), C = int(l.C);
  double t = double(w_t9(G)) / 511.0;
  auto V = [&](int i) { return vtx(f, l.voff + uint64_t(std::min(std::max(i, 0), C - 1))); };
  V3 pos = (1 - t) * V(j) + t * V(j + 1);
  double ao = (1 - t) * double(f->v32[(l.voff + j) * 4 + 3]) + t * double(f->v32[(l.voff + j + 1) * 4 + 3]);
  // O3 tangents on the styled polyline, interpolated along the segment
  V3 Tj = calcTangent(j, C, V(j - 1), V(j), V(j + 1));
  V3 Tj1 = calcTangent(j + 1, C, V(j), V(j + 1), V(j + 2));
  V3 T = normalize((1 - t) * Tj + t * Tj1);
  double w = (double(j) + t) / double(C - 1);
  shade_model(f, g, k, prm, pos, T, w, ao, rgb);
  return true;
}

// R-payload ("reconstruct it from the depth value ... a specific sample location within the pixel"):
// the view-space point on the ray through the centre of pixel (x, y) at the word's depth
static V3 position_from_depth(const Cam& k, int x, int y, uint32_t dq) {
  double zn = double(dq) / 16777215.0;
  double zv = double(k.B) / (double(k.A) - zn);
  double cx = ((double(x) + 0.5) - double(k.half_w)) / double(k.fpx);
  double cy = (double(k.half_h) - (double(y) + 0.5)) / double(k.fpx);
  V3 p;
  p.x = double(k.eye[0]) + zv * (cx * double(k.r[0]) + cy * double(k.u[0]) + double(k.f[0]));
  p.y = double(k.eye[1]) + zv * (cx * double(k.r[1]) + cy * double(k.u[1]) + double(k.f[1]));
  p.z = double(k.eye[2]) + zv * (cx * double(k.r[2]) + cy * double(k.u[2]) + double(k.f[2]));
  return p;
}
// O6 from the paper's payload alone: no vertex is read
static void shade_payload(const orc_frame* f, const Groom* g, const Cam& k, const orc_params* prm, int x, int y,
                          uint64_t G, double rgb[3]) {
  F3 Tf = oct_decode(uint32_t(G >> 32) & 0xFFu, uint32_t(G >> 24) & 0xFFu);
  V3 T = {double(Tf.x), double(Tf.y), double(Tf.z)};
  double w = double(uint32_t(G >> 6) & 63u) / 63.0, ao = double(uint32_t(G) & 63u) / 63.0;
  shade_model(f, g, k, prm, position_from_depth(k, x, y, w_dq(G)), T, w, ao, rgb);
}
// R22 for the paper's payload: screen direction of the decoded tangent at the pixel centre. With view-space
// tangent (tx, ty, tz) and the pixel's ray (cx, cy, 1), d(sx, sy)/ds is parallel to (tx - cx tz, cy tz - ty),
// whatever the depth. fp32 fixed order (decides the strip membership).
static void screen_tangent_payload(const Cam& k, int x, int y, uint64_t word, float T[2]) {
  T[0] = 1.f;
  T[1] = 0.f;
  F3 t = oct_decode(uint32_t(word >> 32) & 0xFFu, uint32_t(word >> 24) & 0xFFu);
  float tx = dot3f(t.x, t.y, t.z, k.r), ty = dot3f(t.x, t.y, t.z, k.u), tz = dot3f(t.x, t.y, t.z, k.f);
  float cx = float(x) + 0.5f;
  cx = cx - k.half_w;
  cx = cx / k.fpx;
  float cy = float(y) + 0.5f;
  cy = k.half_h - cy;
  cy = cy / k.fpx;
  float a = cx * tz;
  float Sx = tx - a;
  float b = cy * tz;
  float Sy = b - ty;
  float dd = Sx * Sx;
  float e = Sy * Sy;
  dd = dd + e;
  if (!(dd >= 1e-12f)) return;
  float len = std::sqrt(dd);
  T[0] = Sx / len;
  T[1] = Sy / len;
}
// the one groom a payload pass draws (the payload names no groom: the paper shades groom by groom)
static const Groom* payload_groom(const orc_frame* f) {
  const Groom* g = nullptr;
  for (size_t i = 0; i < f->grooms.size(); ++i)
    if ((f->groom_mask >> i) & 1u) {
      if (g) return nullptr;
      g = &f->grooms[i];
    }
  return g;
}

int orc_frame_shade(orc_frame* f, const orc_camera* cam, const orc_params* prm) {
  Cam k = make_cam(cam);
  if (f->W != k.W || f->H != k.H) return -1;
  size_t np = size_t(k.W) * k.H;
  f->colour.assign(np * 3, 0.0);
  f->tang.assign(np * 4, 0.f);
  const int sx0 = std::max(f->wx0 - 7, 0), sx1 = std::min(f->wx1 < (1 << 30) ? f->wx1 + 7 : f->wx1, int(k.W));
  const int sy0 = std::max(f->wy0 - 7, 0), sy1 = std::min(f->wy1 < (1 << 30) ? f->wy1 + 7 : f->wy1, int(k.H));
  const Groom* pg = f->payload_mode ? payload_groom(f) : nullptr;
  for (int sy = sy0; sy < sy1; ++sy)
  for (int sx = sx0; sx < sx1; ++sx) {
    const size_t p = size_t(sy) * k.W + sx;
    uint64_t G = f->gbuf[p * 2], A = f->gbuf[p * 2 + 1];
    double rgb[3];
    if (f->payload_mode) {  // R-payload: everything comes from the word and the pixel position
      if (!pg) return -4;
      if (!none(A)) screen_tangent_payload(k, sx, sy, A, &f->tang[p * 4 + 2]);
      if (none(G)) continue;
      screen_tangent_payload(k, sx, sy, G, &f->tang[p * 4]);
      shade_payload(f, pg, k, prm, sx, sy, G, rgb);
      for (int c = 0; c < 3; ++c) f->colour[p * 3 + c] = rgb[c];
      continue;
    }
    if (!none(A)) screen_tangent(f, k, A, &f->tang[p * 4 + 2]);
    if (none(G)) continue;
    screen_tangent(f, k, G, &f->tang[p * 4]);
    if (!shade_word(f, k, prm, G, rgb)) return -2;
    for (int c = 0; c < 3; ++c) f->colour[p * 3 + c] = rgb[c];
  }
  return 0;
}
void orc_frame_get_colour(const orc_frame* f, double* o) {
  std::memcpy(o, f->colour.data(), f->colour.size() * sizeof(double));
}
void orc_frame_get_tangents(const orc_frame* f, float* o) {
  std::memcpy(o, f->tang.data(), f->tang.size() * sizeof(float));
}

// ------------------------------------------------------------------ O7
namespace {
struct AccOut {
  double C[3];
  double alpha;
};
AccOut accumulate(const orc_frame* f, const orc_params* prm, int W, int H, int px, int py, float Tx,
                  float Ty, uint32_t dq_ref, bool use_colour, const double* CP, uint32_t tauz_q) {
  int r = prm->filter_radius;
  double sp = double(r) * double(prm->s_par), sq = double(r) * double(prm->s_perp);
  double inv_sp2 = sp > 0 ? 1.0 / (sp * sp) : 0.0, inv_sq2 = sq > 0 ? 1.0 / (sq * sq) : 0.0;
  double inv_sc2 = 1.0 / (double(prm->sigma_c) * double(prm->sigma_c));
  double S[3] = {0, 0, 0}, Wsum = 0, Hc = 0, Ha = 0;
  for (int dy = -r; dy <= r; ++dy)
    for (int dx = -r; dx <= r; ++dx) {
      int qx = px + dx, qy = py + dy;
      if (qx < 0 || qy < 0 || qx >= W || qy >= H) continue;  // PAPER.md:489 bounds check
      size_t q = size_t(qy) * W + qx;
      uint64_t GQ = f->gbuf[q * 2], AQ = f->gbuf[q * 2 + 1];
      // R20: class of Q by a depth test on the quantised depths (integers)
      auto close = [&](uint64_t w) {
        uint32_t d = w_dq(w);
        uint32_t diff = d > dq_ref ? d - dq_ref : dq_ref - d;
        return diff <= tauz_q;  // PAPER.md:169 threshold 1.45e-3
      };
      int cls = 0;  // 1 = centre, 2 = cons-only
      if (!none(GQ) && close(GQ)) cls = 1;
      else if (!none(AQ) && close(AQ)) cls = 2;
      if (!cls) continue;
      // Eq. 9, fp32 fixed order (decides the strip membership)
      float fdx = float(dx), fdy = float(dy);
      float a = fdx * Tx;
      float b = fdy * Ty;
      float dpar = a + b;
      float ex = dpar * Tx;
      ex = fdx - ex;
      float ey = dpar * Ty;
      ey = fdy - ey;
      float e2 = ex * ex;
      {
        float e3 = ey * ey;
        e2 = e2 + e3;
      }
      float dperp = std::sqrt(e2);
      if (dperp <= prm->w_strip) {  // PAPER.md:176, 498-503; R18: Q's class
        if (cls == 1) Hc += 1;
        else Ha += 1;
      }
      if (cls == 1) {  // R19: only centre-class neighbours carry colour
        double w = std::exp(-double(dpar) * double(dpar) * inv_sp2 - double(dperp) * double(dperp) * inv_sq2);
        if (use_colour) {
          double d2 = 0;
          for (int c = 0; c < 3; ++c) {
            double d = CP[c] - f->colour[q * 3 + c];
            d2 += d * d;
          }
          w *= std::exp(-d2 * inv_sc2);  // Eq. 10
        }
        for (int c = 0; c < 3; ++c) S[c] += w * f->colour[q * 3 + c];
        Wsum += w;
      }
    }
  AccOut o;
  for (int c = 0; c < 3; ++c) o.C[c] = Wsum > 0 ? S[c] / Wsum : 0.0;
  o.alpha = (Hc + Ha) > 0 ? Hc / (Hc + Ha) : 0.0;
  return o;
}
}  // namespace

int orc_frame_filter(orc_frame* f, const orc_camera* cam, const orc_params* prm) {
  int W = int(cam->width), H = int(cam->height);
  if (f->W != uint32_t(W) || f->H != uint32_t(H)) return -1;
  size_t np = size_t(W) * H;
  if (f->colour.size() != np * 3) return -2;
  f->out.assign(np * 4, 0.0);
  uint32_t tauz_q = uint32_t(std::floor(double(prm->tau_z) * 16777215.0 + 0.5));
  uint32_t taufly_q = uint32_t(std::floor(double(prm->tau_fly) * 16777215.0 + 0.5));
  double bg[3] = {double(prm->background_rgb[0]), double(prm->background_rgb[1]), double(prm->background_rgb[2])};
  for (int py = std::max(f->wy0, 0); py < std::min(f->wy1, H); ++py)
    for (int px = std::max(f->wx0, 0); px < std::min(f->wx1, W); ++px) {
      size_t p = size_t(py) * W + px;
      uint64_t G = f->gbuf[p * 2], A = f->gbuf[p * 2 + 1];
      bool isCenter = !none(G), isCons = !none(A);
      if (!f->scene_rgb.empty())
        for (int c = 0; c < 3; ++c) bg[c] = double(f->scene_rgb[p * 3 + c]);
      double C[3] = {0, 0, 0}, alpha = 0;
      const double* CP = &f->colour[p * 3];
      if (!prm->filter_on) {
        if (isCenter) {
          for (int c = 0; c < 3; ++c) C[c] = CP[c];
          alpha = 1;
        }
      } else if (isCenter || isCons) {
        const float* TG = &f->tang[p * 4];
        const float* TA = &f->tang[p * 4 + 2];
        if (isCenter) {
          AccOut a = accumulate(f, prm, W, H, px, py, TG[0], TG[1], w_dq(G), true, CP, tauz_q);
          for (int c = 0; c < 3; ++c) C[c] = a.C[c];
          alpha = a.alpha;
          // fly-away strand in front of the centre hit (R21)
          if (isCons && w_dq(G) - w_dq(A) >= taufly_q && w_dq(G) >= w_dq(A)) {
            AccOut b = accumulate(f, prm, W, H, px, py, TA[0], TA[1], w_dq(A), false, CP, tauz_q);
            for (int c = 0; c < 3; ++c) C[c] = b.alpha * b.C[c] + (1 - b.alpha) * a.C[c];
            alpha = 1;
          }
        } else {  // promoted pixel: w_color = 1
          AccOut a = accumulate(f, prm, W, H, px, py, TA[0], TA[1], w_dq(A), false, CP, tauz_q);
          for (int c = 0; c < 3; ++c) C[c] = a.C[c];
          alpha = a.alpha;
        }
      }
      for (int c = 0; c < 3; ++c) f->out[p * 4 + c] = alpha * C[c] + (1 - alpha) * bg[c];  // R29
      // alpha of everything drawn so far: "over" (R-seq); without earlier passes this is alpha itself
      double a_bg = f->scene_alpha.empty() ? 0.0 : double(f->scene_alpha[p]);
      f->out[p * 4 + 3] = alpha + (1 - alpha) * a_bg;
    }
  return 0;
}
void orc_frame_get_out(const orc_frame* f, double* o) {
  std::memcpy(o, f->out.data(), f->out.size() * sizeof(double));
}

}  // extern "C"
