"""CPU oracle of the deferred hair pipeline — TEST INFRASTRUCTURE ONLY.

ctypes front end of ``hair_oracle.cpp`` (see ``hair_oracle.h`` for what it is and what pins
it). Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package. It imports nothing from the CUDA package
and the CUDA package imports nothing from here; scene descriptions reach both sides as plain
dicts of numpy arrays (``paper_2607_04230_b200.synth``), which hold no pipeline arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = [os.path.join(_HERE, "hair_oracle.cpp"), os.path.join(_HERE, "hair_oracle.h")]


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (no FMA contraction: the fp32 decisions must round per op)."""
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
           "-Wall", "-o", _SO, _SRC[0]]
    subprocess.check_call(cmd)
    return _SO


class Style(C.Structure):
    _fields_ = [("spi", C.c_uint32), ("seed", C.c_uint32), ("op_mask", C.c_uint32),
                ("clump_exp", C.c_uint32), ("frizz_cells", C.c_uint32),
                ("clump_strength", C.c_float), ("twist_turns", C.c_float),
                ("curl_radius", C.c_float), ("curl_turns", C.c_float), ("curl_ramp_w0", C.c_float),
                ("frizz_sigma", C.c_float), ("frizz_ramp_w0", C.c_float),
                ("width_world", C.c_float),
                ("albedo_root", C.c_float * 3), ("albedo_tip", C.c_float * 3),
                ("roughness", C.c_float), ("tilt", C.c_float)]


class Groom(C.Structure):
    _fields_ = [("n_verts", C.c_uint32), ("n_layers", C.c_uint32), ("n_tris", C.c_uint32),
                ("n_instances", C.c_uint32),
                ("pos", C.c_void_p), ("ao", C.c_void_p), ("idx", C.c_void_p),
                ("strands_per_tri", C.c_void_p), ("xform", C.c_void_p), ("style", Style)]


class Camera(C.Structure):
    _fields_ = [("eye", C.c_float * 3), ("right", C.c_float * 3), ("up", C.c_float * 3),
                ("forward", C.c_float * 3), ("vfov_y", C.c_float), ("near_z", C.c_float),
                ("far_z", C.c_float), ("width", C.c_uint32), ("height", C.c_uint32)]


class Params(C.Structure):
    _fields_ = [("center_diameter_px", C.c_float), ("filter_radius", C.c_int32),
                ("s_par", C.c_float), ("s_perp", C.c_float), ("sigma_c", C.c_float),
                ("tau_z", C.c_float), ("tau_fly", C.c_float), ("w_strip", C.c_float),
                ("light_pos", (C.c_float * 3) * 4), ("light_rgb", (C.c_float * 3) * 4),
                ("n_lights", C.c_uint32), ("ambient_rgb", C.c_float * 3),
                ("k_d", C.c_float), ("k_R", C.c_float), ("k_TRT", C.c_float),
                ("background_rgb", C.c_float * 3), ("filter_on", C.c_uint32)]


OP_BITS = {"clump": 1, "twist": 2, "curl": 4, "frizz": 8}
_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        vp, u32, u64, f32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_float
        L.orc_pcg.restype = u32
        L.orc_pcg.argtypes = [u32]
        L.orc_hash3.restype = u32
        L.orc_hash3.argtypes = [u32, u32, u32]
        L.orc_lod_counts.restype = None
        L.orc_lod_counts.argtypes = [f32, u32, f32, u32, u32, vp]
        L.orc_calc_tangent.restype = None
        L.orc_calc_tangent.argtypes = [C.c_int, C.c_int, vp, vp, vp, vp]
        L.orc_pack.restype = u64
        L.orc_pack.argtypes = [f32, u32, u32, f32]
        L.orc_unpack.restype = None
        L.orc_unpack.argtypes = [u64, vp]
        L.orc_segment_cover_msaa.argtypes = [vp, vp, f32, u32, u32, u32, vp, vp]
        L.orc_segment_cover.restype = None
        L.orc_segment_cover.argtypes = [vp, vp, f32, u32, u32, vp, vp]
        L.orc_project.restype = C.c_int
        L.orc_project.argtypes = [vp, vp, vp]
        L.orc_frame_create.restype = vp
        L.orc_frame_destroy.argtypes = [vp]
        L.orc_frame_add_groom.argtypes = [vp, vp]
        L.orc_frame_lod.argtypes = [vp, vp, vp, u32]
        for n in ("n_bundles", "n_strands_total", "n_strands"):
            getattr(L, "orc_frame_" + n).restype = u32
            getattr(L, "orc_frame_" + n).argtypes = [vp]
        L.orc_frame_n_vertices.restype = u64
        L.orc_frame_n_vertices.argtypes = [vp]
        L.orc_frame_get_table.argtypes = [vp, vp, vp]
        L.orc_frame_set_table.argtypes = [vp, vp, u32]
        L.orc_frame_generate.argtypes = [vp]
        L.orc_frame_beta.restype = None
        L.orc_frame_beta.argtypes = [vp, vp, vp, vp]
        L.orc_depth_fix.restype = C.c_double
        L.orc_depth_fix.argtypes = [C.c_double, C.c_double]
        L.orc_frame_dom_count.restype = C.c_int
        L.orc_frame_dom_count.argtypes = [vp, vp, vp, vp, vp, vp]
        L.orc_dom_transmittance.restype = C.c_double
        L.orc_dom_transmittance.argtypes = [vp, vp, vp, vp, C.c_double, C.c_double, vp]
        L.orc_frame_set_dom.restype = C.c_int
        L.orc_frame_set_dom.argtypes = [vp, C.c_uint32, vp, vp, vp, vp, C.c_double]
        L.orc_frame_set_dom_beta.restype = None
        L.orc_frame_set_dom_beta.argtypes = [vp, vp, C.c_uint32]
        L.orc_frame_get_vertices_f64.argtypes = [vp, vp]
        L.orc_frame_get_vertices_f32.argtypes = [vp, vp]
        L.orc_frame_set_vertices_f32.argtypes = [vp, vp, u64]
        L.orc_strand.argtypes = [vp, u32, u32, u32, vp, vp]
        L.orc_root.argtypes = [vp, u32, u32, vp, vp]
        L.orc_frame_raster.argtypes = [vp, vp, vp, vp, vp]
        L.orc_frame_get_gbuffer.argtypes = [vp, vp]
        L.orc_frame_set_gbuffer.argtypes = [vp, vp, u32, u32]
        L.orc_frame_set_scene.argtypes = [vp, vp, vp, u32, u32]
        L.orc_frame_set_pass.argtypes = [vp, u32, vp, vp, u32, u32]
        L.orc_frame_set_window.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int]
        L.orc_frame_set_window.restype = None
        L.orc_frame_raster_msaa.argtypes = [vp, vp, vp, u32]
        L.orc_frame_get_msaa.argtypes = [vp, vp]
        L.orc_frame_get_msaa.restype = None
        L.orc_frame_set_msaa.argtypes = [vp, vp, u32, u32, u32]
        L.orc_frame_resolve_msaa.argtypes = [vp, vp, vp]
        L.orc_frame_shade.argtypes = [vp, vp, vp]
        L.orc_frame_get_colour.argtypes = [vp, vp]
        L.orc_frame_get_tangents.argtypes = [vp, vp]
        L.orc_frame_filter.argtypes = [vp, vp, vp]
        L.orc_frame_get_out.argtypes = [vp, vp]
        L.orc_frame_set_payload_mode.restype = None
        L.orc_frame_set_payload_mode.argtypes = [vp, C.c_int]
        L.orc_oct_encode.restype = None
        L.orc_oct_encode.argtypes = [vp, vp]
        L.orc_oct_decode.restype = None
        L.orc_oct_decode.argtypes = [u32, u32, vp]
        L.orc_payload40.restype = u64
        L.orc_payload40.argtypes = [vp, C.c_int, C.c_int, f32, u32, u32]
        L.orc_unpack_payload.restype = None
        L.orc_unpack_payload.argtypes = [u64, vp]
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def make_style(d: dict) -> Style:
    s = Style()
    s.spi = d["spi"]
    s.seed = d["seed"]
    s.op_mask = sum(OP_BITS[o] for o in d.get("ops", ()))
    s.clump_exp = d.get("clump_exp", 1)
    s.frizz_cells = d.get("frizz_cells", 8)
    for k in ("clump_strength", "twist_turns", "curl_radius", "curl_turns", "curl_ramp_w0",
              "frizz_sigma", "frizz_ramp_w0", "width_world"):
        setattr(s, k, float(d.get(k, 0.0)))
    s.albedo_root[:] = d.get("albedo_root", (0.3, 0.2, 0.1))
    s.albedo_tip[:] = d.get("albedo_tip", (0.6, 0.45, 0.3))
    s.roughness = d.get("roughness", 0.3)
    s.tilt = d.get("tilt", -0.05)
    return s


def make_camera(d: dict) -> Camera:
    c = Camera()
    c.eye[:] = d["eye"]
    c.right[:] = d["right"]
    c.up[:] = d["up"]
    c.forward[:] = d["forward"]
    c.vfov_y, c.near_z, c.far_z = d["vfov_y"], d["near_z"], d["far_z"]
    c.width, c.height = d["width"], d["height"]
    return c


def make_params(d: dict) -> Params:
    p = Params()
    p.center_diameter_px = d.get("center_diameter_px", 0.5)
    p.filter_radius = d.get("filter_radius", 5)
    p.s_par, p.s_perp = d.get("s_par", 0.5), d.get("s_perp", 0.15)
    p.sigma_c, p.tau_z, p.tau_fly = d.get("sigma_c", 0.9), d.get("tau_z", 1.45e-3), d.get("tau_fly", 5e-4)
    p.w_strip = d.get("w_strip", 0.5)
    lights = d.get("lights", [])
    p.n_lights = len(lights)
    for i, (pos, rgb) in enumerate(lights):
        p.light_pos[i][:] = pos
        p.light_rgb[i][:] = rgb
    p.ambient_rgb[:] = d.get("ambient_rgb", (0.15, 0.15, 0.15))
    p.k_d, p.k_R, p.k_TRT = d.get("k_d", 0.4), d.get("k_R", 0.25), d.get("k_TRT", 0.5)
    p.background_rgb[:] = d.get("background_rgb", (0.0, 0.0, 0.0))
    p.filter_on = 1 if d.get("filter_on", True) else 0
    return p


def oct_encode(T):
    """R-payload: (ox8, oy8) of a unit vector, fp32 fixed order."""
    T = np.ascontiguousarray(T, dtype=np.float32)
    out = np.zeros(2, np.uint32)
    lib().orc_oct_encode(_ptr(T), _ptr(out))
    return int(out[0]), int(out[1])


def oct_decode(ox: int, oy: int):
    out = np.zeros(3, np.float32)
    lib().orc_oct_decode(int(ox), int(oy), _ptr(out))
    return out


def payload40(v, j: int, t: float, a1: int, a2: int) -> int:
    """R-payload: the 40 payload bits of a hit at parameter t on segment j of the strand v [C][4] float32."""
    v = np.ascontiguousarray(v, dtype=np.float32).reshape(-1, 4)
    return int(lib().orc_payload40(_ptr(v), int(j), v.shape[0], float(t), int(a1), int(a2)))


def unpack_payload(words):
    """fields of paper-payload words: dict of arrays dq, ox, oy, u6, v6, w6, ao6 (pure bit slicing)."""
    w = np.asarray(words, dtype=np.uint64)
    f = lambda sh, m: ((w >> np.uint64(sh)) & np.uint64(m)).astype(np.uint32)
    return {"dq": f(40, 0xFFFFFF), "ox": f(32, 0xFF), "oy": f(24, 0xFF), "u6": f(18, 63), "v6": f(12, 63),
            "w6": f(6, 63), "ao6": f(0, 63)}


class Frame:
    """One scene + one frame of oracle state (table, vertices, G-buffer, colour, output)."""

    def set_payload_mode(self, on: bool) -> None:
        """R-payload: O4 writes / O6 reads the paper's self-contained payload (see hair_oracle.h)."""
        self.L.orc_frame_set_payload_mode(self.h, 1 if on else 0)

    def __init__(self, grooms: list[dict]):
        self.L = lib()
        self.h = C.c_void_p(self.L.orc_frame_create())
        self._keep = []
        self._n_grooms = 0
        for g in grooms:
            self.add_groom(g)

    def __del__(self):
        if getattr(self, "h", None):
            self.L.orc_frame_destroy(self.h)
            self.h = None

    def add_groom(self, g: dict) -> int:
        pos = np.ascontiguousarray(g["pos"], dtype=np.float32)
        idx = np.ascontiguousarray(g["idx"], dtype=np.uint32)
        npt = np.ascontiguousarray(g["strands_per_tri"], dtype=np.uint32)
        ao = None if g.get("ao") is None else np.ascontiguousarray(g["ao"], dtype=np.float32)
        xf = None if g.get("xform") is None else np.ascontiguousarray(g["xform"], dtype=np.float32).reshape(-1, 12)
        G = Groom()
        G.n_layers, G.n_verts = pos.shape[0], pos.shape[1]
        G.n_tris = idx.shape[0]
        G.n_instances = 1 if xf is None else xf.shape[0]
        G.pos, G.idx, G.strands_per_tri = _ptr(pos), _ptr(idx), _ptr(npt)
        G.ao = None if ao is None else _ptr(ao)
        G.xform = None if xf is None else _ptr(xf)
        G.style = make_style(g["style"])
        r = self.L.orc_frame_add_groom(self.h, C.byref(G))
        if r < 0:
            raise ValueError(f"orc_frame_add_groom failed: {r}")
        self._n_grooms += 1
        return r

    # ---- O1
    def lod(self, cam: dict, lam) -> None:
        lam = np.atleast_1d(np.asarray(lam, dtype=np.float32))
        c = make_camera(cam)
        assert self.L.orc_frame_lod(self.h, C.byref(c), _ptr(lam), len(lam)) == 0

    @property
    def n_bundles(self):
        return self.L.orc_frame_n_bundles(self.h)

    @property
    def n_strands_total(self):
        return self.L.orc_frame_n_strands_total(self.h)

    @property
    def n_strands(self):
        return self.L.orc_frame_n_strands(self.h)

    @property
    def n_vertices(self):
        return self.L.orc_frame_n_vertices(self.h)

    def table(self):
        t = np.zeros((self.n_bundles, 4), np.uint32)
        l = np.zeros(self.n_bundles, np.float32)
        self.L.orc_frame_get_table(self.h, _ptr(t), _ptr(l))
        return t, l

    def set_table(self, t4) -> None:
        t4 = np.ascontiguousarray(t4, dtype=np.uint32)
        r = self.L.orc_frame_set_table(self.h, _ptr(t4), t4.shape[0])
        if r != 0:
            raise ValueError(f"orc_frame_set_table: {r}")

    def beta(self):
        """Eq. 6-8 from the current table: (beta per groom, delta = -ln beta per groom, beta_min over drawn bundles)."""
        b, d, m = np.zeros(self._n_grooms), np.zeros(self._n_grooms), C.c_double(1.0)
        self.L.orc_frame_beta(self.h, _ptr(b), _ptr(d), C.byref(m))
        return b, d, m.value

    # ---- O2
    def generate(self) -> None:
        assert self.L.orc_frame_generate(self.h) == 0

    def vertices_f64(self):
        v = np.zeros((self.n_vertices, 4), np.float64)
        self.L.orc_frame_get_vertices_f64(self.h, _ptr(v))
        return v

    def vertices_f32(self):
        v = np.zeros((self.n_vertices, 4), np.float32)
        self.L.orc_frame_get_vertices_f32(self.h, _ptr(v))
        return v

    def set_vertices_f32(self, v) -> None:
        v = np.ascontiguousarray(v, dtype=np.float32).reshape(-1, 4)
        r = self.L.orc_frame_set_vertices_f32(self.h, _ptr(v), v.shape[0])
        if r != 0:
            raise ValueError(f"orc_frame_set_vertices_f32: {r}")

    def strand(self, groom: int, id_local: int, n_cp: int):
        out = np.zeros((n_cp, 4), np.float64)
        tan = np.zeros((n_cp, 3), np.float64)
        assert self.L.orc_strand(self.h, groom, id_local, n_cp, _ptr(out), _ptr(tan)) == 0
        return out, tan

    def root(self, groom: int, id_local: int):
        b = np.zeros(3, np.float64)
        tri = C.c_uint32(0)
        assert self.L.orc_root(self.h, groom, id_local, _ptr(b), C.byref(tri)) == 0
        return b, tri.value

    # ---- O4
    def raster(self, cam: dict, prm: dict, order=None):
        c, p = make_camera(cam), make_params(prm)
        counts = np.zeros(3, np.uint64)
        o = None if order is None else np.ascontiguousarray(order, dtype=np.uint32)
        r = self.L.orc_frame_raster(self.h, C.byref(c), C.byref(p), None if o is None else _ptr(o), _ptr(counts))
        assert r == 0, r
        self._wh = (cam["width"], cam["height"])
        return {"center": int(counts[0]), "cons": int(counts[1]), "segments": int(counts[2])}

    def gbuffer(self):
        w, h = self._wh
        g = np.zeros((h, w, 2), np.uint64)
        self.L.orc_frame_get_gbuffer(self.h, _ptr(g))
        return g

    def set_gbuffer(self, g) -> None:
        g = np.ascontiguousarray(g, dtype=np.uint64)
        h, w = g.shape[:2]
        self._wh = (w, h)
        self.L.orc_frame_set_gbuffer(self.h, _ptr(g), w, h)

    def set_scene(self, zn=None, rgb=None) -> None:
        """R-scene: zn [h][w] float32 in [0, 1] seeds the depth of both layers; rgb [h][w][3] is composited over."""
        self._scene = (None if zn is None else np.ascontiguousarray(zn, dtype=np.float32),
                       None if rgb is None else np.ascontiguousarray(rgb, dtype=np.float32))
        a = self._scene[0] if self._scene[0] is not None else self._scene[1]
        h, w = (0, 0) if a is None else a.shape[:2]
        self.L.orc_frame_set_scene(self.h, None if self._scene[0] is None else _ptr(self._scene[0]),
                                   None if self._scene[1] is None else _ptr(self._scene[1]), w, h)

    def set_pass(self, groom_mask: int = 0xFFFFFFFF, dq=None, alpha=None) -> None:
        """R-seq: the state of one sequential pass (see hair_oracle.h); no arguments = reset."""
        self._pass = (None if dq is None else np.ascontiguousarray(dq, dtype=np.uint32),
                      None if alpha is None else np.ascontiguousarray(alpha, dtype=np.float32))
        a = self._pass[0] if self._pass[0] is not None else self._pass[1]
        h, w = (0, 0) if a is None else a.shape[:2]
        self.L.orc_frame_set_pass(self.h, groom_mask & 0xFFFFFFFF, None if self._pass[0] is None else _ptr(self._pass[0]),
                                  None if self._pass[1] is None else _ptr(self._pass[1]), w, h)

    def render_sequential(self, cam: dict, prm: dict, lam, scene_zn=None, scene_rgb=None):
        """PAPER.md:208-210, DESIGN.md R-seq: the grooms one after the other, each through O1-O7 on its own, its
        result blended over the target so far, the centre layer's depth kept for the next pass. Returns
        (out [h][w][4], G-buffer of the last pass, kept depth [h][w] uint32)."""
        h, w = cam["height"], cam["width"]
        bgc = np.asarray(prm.get("background_rgb", (0.0, 0.0, 0.0)), dtype=np.float32)
        target = (np.broadcast_to(bgc, (h, w, 3)).copy() if scene_rgb is None
                  else np.ascontiguousarray(scene_rgb, dtype=np.float32)[..., :3].copy())
        alpha = np.zeros((h, w), np.float32)
        if scene_zn is None:
            dq = np.full((h, w), 0xFFFFFF, np.uint32)
        else:  # R8 quantisation of the scene's depth, in fp32
            z = np.clip(np.asarray(scene_zn, np.float32), np.float32(0), np.float32(1))
            dq = np.minimum((z * np.float32(16777215.0) + np.float32(0.5)).astype(np.float32).astype(np.uint32),
                            np.uint32(0xFFFFFE))
        out = np.concatenate([target.astype(np.float64), np.zeros((h, w, 1))], -1)
        g = None
        for gi in range(self._n_grooms):
            self.set_pass(1 << gi, dq, alpha)
            self.set_scene(None, target)
            self.lod(cam, lam)
            self.generate()
            self.set_vertices_f32(self.vertices_f32())
            self.raster(cam, prm)
            self.shade(cam, prm)
            out = self.filter(cam, prm)
            g = self.gbuffer()
            dq = (g[..., 0] >> np.uint64(40)).astype(np.uint32)  # centre layer: hit depth, else the depth kept so far
            # the next pass composites over this pass's result (fp32 target, as the render target is)
            target = out[..., :3].astype(np.float32)
            alpha = out[..., 3].astype(np.float32)
        self.set_pass()
        self.set_scene(None, None)
        return out, g, dq

    def set_window(self, x0: int = 0, y0: int = 0, x1: int = 1 << 30, y1: int = 1 << 30) -> None:
        """Sample a full-size frame: O4 / O6 / O7 only visit pixels of [x0, x1) x [y0, y1) (O6 grown by 7 px)."""
        self.L.orc_frame_set_window(self.h, int(x0), int(y0), int(x1), int(y1))

    # ---- MSAA-k reference (R-msaa)
    def raster_msaa(self, cam: dict, prm: dict, k: int):
        c, p = make_camera(cam), make_params(prm)
        r = self.L.orc_frame_raster_msaa(self.h, C.byref(c), C.byref(p), int(k))
        if r:
            raise ValueError(f"orc_frame_raster_msaa failed: {r}")
        self._wh = (cam["width"], cam["height"])
        self._ms_k = int(k)
        ms = np.empty((int(k), cam["height"], cam["width"]), dtype=np.uint64)
        self.L.orc_frame_get_msaa(self.h, _ptr(ms))
        return ms

    def set_msaa(self, ms) -> None:
        ms = np.ascontiguousarray(ms, dtype=np.uint64)
        k, h, w = ms.shape
        self._wh = (w, h)
        self._ms_k = k
        self.L.orc_frame_set_msaa(self.h, _ptr(ms), k, w, h)

    def resolve_msaa(self, cam: dict, prm: dict):
        c, p = make_camera(cam), make_params(prm)
        r = self.L.orc_frame_resolve_msaa(self.h, C.byref(c), C.byref(p))
        if r:
            raise ValueError(f"orc_frame_resolve_msaa failed: {r}")
        out = np.empty((cam["height"], cam["width"], 4), dtype=np.float64)
        self.L.orc_frame_get_out(self.h, _ptr(out))
        return out

    # ---- deep opacity maps (DESIGN.md R-dom)
    def dom_build(self, light_cam: dict, prm: dict, D3):
        """z0 [h][w] uint32 and fragment counts [h][w][4] uint32 of the frame's CURRENT vertices seen from `light_cam`
        (runs O4 with that camera first). D3: ends of layers 0..2 in depth steps."""
        self.raster(light_cam, prm)
        c, p = make_camera(light_cam), make_params(prm)
        w, h = light_cam["width"], light_cam["height"]
        z0 = np.zeros((h, w), np.uint32)
        cnt = np.zeros((h, w, 4), np.uint32)
        D = np.ascontiguousarray(D3, dtype=np.uint32)
        r = self.L.orc_frame_dom_count(self.h, C.byref(c), C.byref(p), _ptr(D), _ptr(z0), _ptr(cnt))
        assert r == 0, r
        return z0, cnt

    def set_dom(self, light: int, light_cam, z0=None, cnt=None, D4=None, alpha_s: float = 0.0) -> None:
        """O6 scales light `light` by the transmittance of this map (light_cam None: off)."""
        if not hasattr(self, "_dom"):
            self._dom = {}
        if light_cam is None:
            self.L.orc_frame_set_dom(self.h, light, None, None, None, None, 0.0)
            self._dom.pop(light, None)
            return
        c = make_camera(light_cam)
        z0 = np.ascontiguousarray(z0, dtype=np.uint32)
        cnt = np.ascontiguousarray(cnt, dtype=np.uint32)
        D = np.ascontiguousarray(D4, dtype=np.uint32)
        self._dom[light] = (c, z0, cnt, D)  # the C side keeps the pointers
        r = self.L.orc_frame_set_dom(self.h, light, C.byref(c), _ptr(z0), _ptr(cnt), _ptr(D), float(alpha_s))
        assert r == 0, r

    def set_dom_beta(self, beta) -> None:
        b = np.ascontiguousarray(beta, dtype=np.float64)
        self.L.orc_frame_set_dom_beta(self.h, _ptr(b), b.size)

    # ---- O6 / O7
    def shade(self, cam: dict, prm: dict):
        c, p = make_camera(cam), make_params(prm)
        r = self.L.orc_frame_shade(self.h, C.byref(c), C.byref(p))
        assert r == 0, r
        w, h = self._wh
        col = np.zeros((h, w, 3), np.float64)
        self.L.orc_frame_get_colour(self.h, _ptr(col))
        return col

    def tangents(self):
        w, h = self._wh
        t = np.zeros((h, w, 4), np.float32)
        self.L.orc_frame_get_tangents(self.h, _ptr(t))
        return t

    def filter(self, cam: dict, prm: dict):
        c, p = make_camera(cam), make_params(prm)
        r = self.L.orc_frame_filter(self.h, C.byref(c), C.byref(p))
        assert r == 0, r
        w, h = self._wh
        out = np.zeros((h, w, 4), np.float64)
        self.L.orc_frame_get_out(self.h, _ptr(out))
        return out

    def render(self, cam: dict, prm: dict, lam=0.0):
        """All of O1-O7, pure oracle."""
        self.lod(cam, lam)
        self.generate()
        self.raster(cam, prm)
        self.shade(cam, prm)
        return self.filter(cam, prm)


# small pure functions ---------------------------------------------------------------------
def pcg(v: int) -> int:
    return lib().orc_pcg(v & 0xFFFFFFFF)


def hash3(seed: int, i: int, stream: int) -> int:
    return lib().orc_hash3(seed, i, stream)


def dom_transmittance(light_cam: dict, z0, cnt, D4, alpha_s: float, beta: float, p) -> float:
    """Transmittance towards the light of the deep opacity map (z0, cnt) at world point p (see hair_oracle.h)."""
    c = make_camera(light_cam)
    z0 = np.ascontiguousarray(z0, dtype=np.uint32)
    cnt = np.ascontiguousarray(cnt, dtype=np.uint32)
    D = np.ascontiguousarray(D4, dtype=np.uint32)
    pp = np.ascontiguousarray(p, dtype=np.float32)
    return float(lib().orc_dom_transmittance(C.byref(c), _ptr(z0), _ptr(cnt), _ptr(D), float(alpha_s), float(beta), _ptr(pp)))


def depth_fix(d: float, delta: float) -> float:
    """Eq. 7-8: the depth a thinned groom is tested at, d exp(-delta)."""
    return float(lib().orc_depth_fix(float(d), float(delta)))


def lod_counts(L: float, N: int, delta: float, n_layers: int, c_full: int):
    o = np.zeros(3, np.uint32)
    lib().orc_lod_counts(L, N, delta, n_layers, c_full, _ptr(o))
    return int(o[0]), int(o[1]), int(o[2])


def calc_tangent(idx, count, prev, curr, nxt):
    a = [np.ascontiguousarray(x, dtype=np.float64) for x in (prev, curr, nxt)]
    o = np.zeros(3, np.float64)
    lib().orc_calc_tangent(idx, count, _ptr(a[0]), _ptr(a[1]), _ptr(a[2]), _ptr(o))
    return o


def pack(zn, sid, j, t) -> int:
    return lib().orc_pack(zn, sid, j, t)


def unpack(w: int):
    o = np.zeros(4, np.uint32)
    lib().orc_unpack(C.c_uint64(int(w)), _ptr(o))
    return tuple(int(x) for x in o)


def segment_cover(a, b, rho, w, h):
    a = np.ascontiguousarray(a, dtype=np.float32)
    b = np.ascontiguousarray(b, dtype=np.float32)
    cover = np.zeros((h, w), np.uint8)
    tq = np.zeros((h, w), np.float32)
    lib().orc_segment_cover(_ptr(a), _ptr(b), rho, w, h, _ptr(cover), _ptr(tq))
    return cover, tq


MSAA_OFFSETS = {  # sample offsets from the pixel centre in 1/16 pixel (R-msaa), restated for the tests
    1: [(0, 0)], 2: [(4, 4), (-4, -4)], 4: [(-2, -6), (6, -2), (-6, 2), (2, 6)],
    8: [(1, -3), (-1, 3), (5, 1), (-3, -5), (-5, 5), (-7, -1), (3, 7), (7, -7)]}


def segment_cover_msaa(a, b, rho, w, h, k):
    a = np.ascontiguousarray(a, dtype=np.float32)
    b = np.ascontiguousarray(b, dtype=np.float32)
    cover = np.zeros((k, h, w), np.uint8)
    tq = np.zeros((k, h, w), np.float32)
    r = lib().orc_segment_cover_msaa(_ptr(a), _ptr(b), rho, w, h, k, _ptr(cover), _ptr(tq))
    if r:
        raise ValueError(f"unsupported sample count {k}")
    return cover, tq


def project(cam: dict, p):
    c = make_camera(cam)
    p = np.ascontiguousarray(p, dtype=np.float32)
    o = np.zeros(4, np.float32)
    v = lib().orc_project(C.byref(c), _ptr(p), _ptr(o))
    return o, bool(v)
