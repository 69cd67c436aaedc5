"""Thin ctypes binding of libhair (include/hair.h). Argument marshalling only — every step of the
path runs in the library's CUDA kernels. torch supplies device memory and the stream.

There is no CPU fallback: `load()` raises if the shared library is missing, and `Hair(...)` raises
if no CUDA device is visible.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "csrc", "libhair.so")

OP_BITS = {"clump": 1, "twist": 2, "curl": 4, "frizz": 8}
FLAG_FILTER, FLAG_COUNTERS, FLAG_STAGE_TIMING, FLAG_PAPER_PAYLOAD, FLAG_SINGLE_PASS, FLAG_FUSED, FLAG_RGB16F = 1, 2, 4, 8, 16, 32, 128
FLAG_SHADOWS = 256
EMPTY = 0xFFFFFFFFFFFFFFFF

EXPORTS = ["hair_create", "hair_destroy", "hair_last_error", "hair_default_render_params",
           "hair_set_render_params", "hair_mesh_upload", "hair_mesh_update", "hair_mesh_clear",
           "hair_render", "hair_render_scene", "hair_render_sequential", "hair_render_msaa", "hair_render_to_host", "hair_render_to_host_async", "hair_host_wait", "hair_render_stages", "hair_stats",
           "hair_debug_buffers", "hair_debug_set_vertices", "hair_atomic_microbench", "hair_l2_load_microbench", "hair_abi_sizes",
           "hair_shadow_build", "hair_shadow_clear", "hair_debug_shadow",
           "hair_scan_noalloc", "hair_scan_noalloc_error"]
SCAN_NOALLOC_MAX = 1 << 20


class HairError(RuntimeError):
    pass


class hair_cage(C.Structure):
    _fields_ = [("n_verts", C.c_uint32), ("n_layers", C.c_uint32), ("pos", C.c_void_p), ("ao", C.c_void_p)]


class hair_roots(C.Structure):
    _fields_ = [("n_tris", C.c_uint32), ("idx", C.c_void_p), ("strands_per_tri", C.c_void_p)]


class hair_style(C.Structure):
    _fields_ = [("spi", C.c_uint32), ("seed", C.c_uint32), ("op_mask", C.c_uint32),
                ("clump_exp", C.c_uint32), ("frizz_cells", C.c_uint32),
                ("clump_strength", C.c_float), ("twist_turns", C.c_float),
                ("curl_radius", C.c_float), ("curl_turns", C.c_float), ("curl_ramp_w0", C.c_float),
                ("frizz_sigma", C.c_float), ("frizz_ramp_w0", C.c_float), ("width_world", C.c_float),
                ("albedo_root", C.c_float * 3), ("albedo_tip", C.c_float * 3),
                ("roughness", C.c_float), ("tilt", C.c_float),
                ("n_instances", C.c_uint32), ("instance_xform", C.c_void_p)]


class hair_camera(C.Structure):
    _fields_ = [("eye", C.c_float * 3), ("right", C.c_float * 3), ("up", C.c_float * 3),
                ("forward", C.c_float * 3), ("vfov_y", C.c_float), ("near_z", C.c_float), ("far_z", C.c_float)]


class hair_shadow_params(C.Structure):
    _fields_ = [("cam", hair_camera * 4), ("n_lights", C.c_uint32), ("res", C.c_uint32), ("layer_d1", C.c_float),
                ("alpha_s", C.c_float)]


class hair_render_params(C.Structure):
    _fields_ = [("center_diameter_px", C.c_float), ("filter_radius", C.c_int32),
                ("s_par", C.c_float), ("s_perp", C.c_float), ("sigma_c", C.c_float),
                ("tau_z", C.c_float), ("tau_fly", C.c_float), ("w_strip", C.c_float),
                ("light_pos", (C.c_float * 3) * 4), ("light_rgb", (C.c_float * 3) * 4),
                ("n_lights", C.c_uint32), ("ambient_rgb", C.c_float * 3),
                ("k_d", C.c_float), ("k_R", C.c_float), ("k_TRT", C.c_float),
                ("background_rgb", C.c_float * 3), ("flags", C.c_uint32), ("groom_mask", C.c_uint32)]


class hair_stats_t(C.Structure):
    _fields_ = [("n_grooms", C.c_uint32), ("n_bundles", C.c_uint32), ("n_bundles_culled", C.c_uint32),
                ("n_strands_total", C.c_uint32), ("n_strands_lod", C.c_uint32),
                ("n_vertices", C.c_uint32), ("n_segments", C.c_uint32), ("n_segments_drawn", C.c_uint32),
                ("n_segments_live", C.c_uint32),
                ("n_atomics_center", C.c_uint64), ("n_atomics_cons", C.c_uint64), ("n_atomics_issued", C.c_uint64),
                ("n_atomics_cons_ymajor", C.c_uint64),
                ("n_pixels_center", C.c_uint32), ("n_pixels_cons", C.c_uint32),
                ("ms_lod", C.c_float), ("ms_generate", C.c_float), ("ms_clear", C.c_float),
                ("ms_raster", C.c_float), ("ms_shade", C.c_float), ("ms_filter", C.c_float),
                ("ms_total", C.c_float), ("n_timed_frames", C.c_uint32), ("beta_mean", C.c_float),
                ("beta_min", C.c_float), ("beta_groom", C.c_float * 16), ("delta_groom", C.c_float * 16),
                ("gpu_launches", C.c_uint32),
                ("two_pass", C.c_uint32), ("n_segments_hiz_culled", C.c_uint32)]

    def as_dict(self):
        return {k: (list(getattr(self, k)) if k in ("beta_groom", "delta_groom") else getattr(self, k)) for k, _ in self._fields_}


_lib = None


def load():
    """dlopen libhair.so and declare the prototypes. Raises HairError if it is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(SO_PATH):
        raise HairError(f"{SO_PATH} is missing: run `python -m paper_2607_04230_b200.build` "
                        "(there is no CPU fallback)")
    L = C.CDLL(SO_PATH)
    vp, u32, u64p = C.c_void_p, C.c_uint32, C.c_void_p
    L.hair_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    L.hair_destroy.argtypes = [vp]
    L.hair_destroy.restype = None
    L.hair_last_error.argtypes = [vp]
    L.hair_last_error.restype = C.c_char_p
    L.hair_default_render_params.argtypes = [C.POINTER(hair_render_params)]
    L.hair_default_render_params.restype = None
    L.hair_set_render_params.argtypes = [vp, C.POINTER(hair_render_params)]
    L.hair_mesh_upload.argtypes = [vp, C.POINTER(hair_cage), C.POINTER(hair_roots), C.POINTER(hair_style), C.POINTER(C.c_int)]
    L.hair_mesh_update.argtypes = [vp, C.c_int, C.POINTER(hair_cage)]
    L.hair_mesh_clear.argtypes = [vp]
    L.hair_render.argtypes = [vp, C.POINTER(hair_camera), u32, u32, vp, u32, u64p, vp]
    L.hair_render_scene.argtypes = [vp, C.POINTER(hair_camera), u32, u32, vp, u32, vp, vp, u64p, vp]
    L.hair_render_sequential.argtypes = [vp, C.POINTER(hair_camera), u32, u32, vp, u32, vp, vp, u64p, vp]
    L.hair_render_msaa.argtypes = [vp, C.POINTER(hair_camera), u32, u32, vp, u32, u32, u64p, vp]
    L.hair_render_to_host.argtypes = [vp, C.POINTER(hair_camera), u32, u32, vp, u32, u64p, vp]
    L.hair_render_to_host_async.argtypes = [vp, C.POINTER(hair_camera), u32, u32, vp, u32, u64p, vp, C.POINTER(C.c_int)]
    L.hair_host_wait.argtypes = [vp, C.c_int]
    L.hair_render_stages.argtypes = [vp, C.POINTER(hair_camera), u32, u32, u32, u64p, vp]
    L.hair_stats.argtypes = [vp, C.POINTER(hair_stats_t)]
    L.hair_debug_buffers.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    L.hair_debug_set_vertices.argtypes = [vp, vp, u32]
    L.hair_atomic_microbench.argtypes = [vp, C.c_int, vp, C.c_uint64, C.c_uint64, u32, C.POINTER(C.c_float)]
    L.hair_l2_load_microbench.argtypes = [vp, C.c_int, vp, C.c_uint64, u32, u32, C.POINTER(C.c_uint64), C.POINTER(C.c_float)]
    L.hair_shadow_build.argtypes = [vp, C.POINTER(hair_shadow_params)]
    L.hair_shadow_clear.argtypes = [vp]
    L.hair_debug_shadow.argtypes = [vp, u32, C.POINTER(vp), C.POINTER(vp), C.POINTER(u32 * 4)]
    L.hair_scan_noalloc.argtypes = [C.c_int, vp, vp, u32, vp, vp]
    L.hair_scan_noalloc_error.argtypes = []
    L.hair_scan_noalloc_error.restype = C.c_char_p
    L.hair_abi_sizes.argtypes = [C.POINTER(C.c_uint32 * 7)]
    L.hair_abi_sizes.restype = None
    sizes = (C.c_uint32 * 7)()
    L.hair_abi_sizes(C.byref(sizes))
    mine = [C.sizeof(t) for t in (hair_cage, hair_roots, hair_style, hair_camera, hair_render_params, hair_stats_t,
                                    hair_shadow_params)]
    if list(sizes) != mine:
        raise HairError(f"struct layout mismatch between binding.py {mine} and libhair {list(sizes)}")
    _lib = L
    return L


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def make_camera(d: dict) -> hair_camera:
    c = hair_camera()
    c.eye[:] = d["eye"]
    c.right[:] = d["right"]
    c.up[:] = d["up"]
    c.forward[:] = d["forward"]
    c.vfov_y, c.near_z, c.far_z = d["vfov_y"], d["near_z"], d["far_z"]
    return c


def make_params(d: dict, flags: int | None = None) -> hair_render_params:
    p = hair_render_params()
    load().hair_default_render_params(C.byref(p))
    for k in ("center_diameter_px", "filter_radius", "s_par", "s_perp", "sigma_c", "tau_z", "tau_fly",
              "w_strip", "k_d", "k_R", "k_TRT"):
        if k in d:
            setattr(p, k, d[k])
    lights = d.get("lights", [])
    p.n_lights = len(lights)
    for i, (pos, rgb) in enumerate(lights):
        p.light_pos[i][:] = pos
        p.light_rgb[i][:] = rgb
    if "ambient_rgb" in d:
        p.ambient_rgb[:] = d["ambient_rgb"]
    if "background_rgb" in d:
        p.background_rgb[:] = d["background_rgb"]
    f = FLAG_FILTER if d.get("filter_on", True) else 0
    p.flags = f | (flags or 0)
    p.groom_mask = int(d.get("groom_mask", 0xFFFFFFFF)) & 0xFFFFFFFF
    return p


class Hair:
    """One libhair context bound to torch's current CUDA stream."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise HairError("no CUDA device: libhair has no CPU fallback")
        self.torch = torch
        self.L = load()
        self.device = device
        torch.cuda.set_device(device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(device)
        self.h = C.c_void_p()
        self._check(self.L.hair_create(C.byref(self.h), device, C.c_void_p(self.stream.cuda_stream)), "hair_create")
        self.n_grooms = 0
        self._res = None
        self._pending_updates = []  # [event or None, arrays] of mesh_update calls whose host arrays may still be read

    def close(self):
        if getattr(self, "h", None) and self.h.value:
            self.L.hair_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, what: str):
        if rc != 0:
            msg = self.L.hair_last_error(self.h).decode() if self.h.value else ""
            raise HairError(f"{what} failed ({rc}): {msg}")

    # ---- hair_mesh_upload(cage, root triangles, styling params)
    def mesh_upload(self, g: dict) -> int:
        pos = np.ascontiguousarray(g["pos"], dtype=np.float32)
        idx = np.ascontiguousarray(g["idx"], dtype=np.uint32)
        npt = np.ascontiguousarray(g["strands_per_tri"], dtype=np.uint32)
        ao = None if g.get("ao") is None else np.ascontiguousarray(g["ao"], dtype=np.float32)
        xf = None if g.get("xform") is None else np.ascontiguousarray(g["xform"], dtype=np.float32).reshape(-1, 12)
        cage = hair_cage(pos.shape[1], pos.shape[0], _ptr(pos), None if ao is None else _ptr(ao))
        roots = hair_roots(idx.shape[0], _ptr(idx), _ptr(npt))
        d = g["style"]
        st = hair_style()
        st.spi, st.seed = d["spi"], d["seed"]
        st.op_mask = sum(OP_BITS[o] for o in d.get("ops", ()))
        st.clump_exp, st.frizz_cells = d.get("clump_exp", 1), d.get("frizz_cells", 8)
        for k in ("clump_strength", "twist_turns", "curl_radius", "curl_turns", "curl_ramp_w0",
                  "frizz_sigma", "frizz_ramp_w0", "width_world"):
            setattr(st, k, float(d.get(k, 0.0)))
        st.albedo_root[:] = d.get("albedo_root", (0.3, 0.2, 0.1))
        st.albedo_tip[:] = d.get("albedo_tip", (0.6, 0.45, 0.3))
        st.roughness, st.tilt = d.get("roughness", 0.3), d.get("tilt", -0.05)
        st.n_instances = 1 if xf is None else xf.shape[0]
        st.instance_xform = None if xf is None else _ptr(xf)
        gid = C.c_int(-1)
        self._check(self.L.hair_mesh_upload(self.h, C.byref(cage), C.byref(roots), C.byref(st), C.byref(gid)),
                    "hair_mesh_upload")
        self.n_grooms += 1
        return gid.value

    def mesh_update(self, groom_id: int, pos_pinned, ao_pinned=None):
        """pos_pinned / ao_pinned: torch CPU tensors (pinned for an async copy) or numpy arrays.

        Lifetime: from pinned memory the library only queues the update and reads the arrays when the NEXT render /
        stats / shadow_build is issued, finishing when that frame completes (include/hair.h). The binding therefore
        keeps a reference to the arrays until an event recorded behind that frame has completed, so a temporary
        (`torch.from_numpy(a).pin_memory()`) cannot be handed back to torch's pinned-memory cache and reused while the
        copy is still to come. The CONTENTS are the caller's to leave alone until then."""
        def hp(x):
            return C.c_void_p(x.data_ptr()) if hasattr(x, "data_ptr") else _ptr(x)
        shp = pos_pinned.shape
        cage = hair_cage(shp[1], shp[0], hp(pos_pinned), None if ao_pinned is None else hp(ao_pinned))
        self._check(self.L.hair_mesh_update(self.h, groom_id, C.byref(cage)), "hair_mesh_update")
        self._pending_updates.append([None, (pos_pinned, ao_pinned)])

    def _updates_issued(self):
        """Called after a call that flushed the queued updates onto the stream: mark them with an event behind that
        work, and let go of the arrays of updates whose event has completed."""
        ev = None
        for p in self._pending_updates:
            if p[0] is None:
                if ev is None:
                    ev = self.torch.cuda.Event()
                    ev.record(self.stream)
                p[0] = ev
        self._pending_updates = [p for p in self._pending_updates if not p[0].query()]

    def mesh_clear(self):
        self._check(self.L.hair_mesh_clear(self.h), "hair_mesh_clear")
        self.n_grooms = 0
        self._pending_updates = []  # the library dropped what was queued and synchronised its streams

    def set_render_params(self, prm: dict, flags: int = 0):
        p = make_params(prm, flags)
        self._check(self.L.hair_set_render_params(self.h, C.byref(p)), "hair_set_render_params")

    def alloc_outputs(self, width: int, height: int, rgb16: bool = False):
        """Device outputs of one frame; rgb16: the half-precision colour buffer HAIR_FLAG_RGB16F writes."""
        t = self.torch
        dev = f"cuda:{self.device}"
        gb = t.empty((height, width, 2), dtype=t.int64, device=dev)  # uint64 words, viewed as int64
        rgb = t.empty((height, width, 4), dtype=t.float16 if rgb16 else t.float32, device=dev)
        return gb, rgb

    # ---- hair_render(camera, resolution, lod_lambda, out_gbuffer, out_rgb)
    def render(self, cam: dict, lam, out_gbuffer=None, out_rgb=None):
        w, h = cam["width"], cam["height"]
        if out_gbuffer is None or out_rgb is None:
            out_gbuffer, out_rgb = self.alloc_outputs(w, h)
        lam = np.atleast_1d(np.asarray(lam, dtype=np.float32))
        c = make_camera(cam)
        self._check(self.L.hair_render(self.h, C.byref(c), w, h, _ptr(lam), len(lam),
                                       C.c_void_p(out_gbuffer.data_ptr()), C.c_void_p(out_rgb.data_ptr())), "hair_render")
        self._updates_issued()
        self._res = (w, h)
        return out_gbuffer, out_rgb

    def render_msaa(self, cam: dict, lam, k: int):
        """hair_render_msaa: returns (samples int64 [k][h][w] device tensor, out_rgb float32 [h][w][4])."""
        import torch
        w, h = cam["width"], cam["height"]
        samples = torch.empty((int(k), h, w), dtype=torch.int64, device=f"cuda:{self.device}")
        out_rgb = torch.empty((h, w, 4), dtype=torch.float32, device=f"cuda:{self.device}")
        lam = np.atleast_1d(np.asarray(lam, dtype=np.float32))
        c = make_camera(cam)
        self._check(self.L.hair_render_msaa(self.h, C.byref(c), w, h, _ptr(lam), len(lam), int(k),
                                            C.c_void_p(samples.data_ptr()), C.c_void_p(out_rgb.data_ptr())), "hair_render_msaa")
        self._updates_issued()
        self._res = (w, h)
        return samples, out_rgb

    def render_sequential(self, cam: dict, lam, scene_zn=None, scene_rgb=None, out_gbuffer=None, out_rgb=None):
        """hair_render_sequential: the grooms one after the other; arguments as render_scene."""
        return self.render_scene(cam, lam, scene_zn, scene_rgb, out_gbuffer, out_rgb, _fn="hair_render_sequential")

    def render_scene(self, cam: dict, lam, scene_zn=None, scene_rgb=None, out_gbuffer=None, out_rgb=None,
                     _fn="hair_render_scene"):
        """hair_render_scene: scene_zn float32 [h][w], scene_rgb float32 [h][w][4] device tensors (or None)."""
        w, h = cam["width"], cam["height"]
        if out_gbuffer is None or out_rgb is None:
            out_gbuffer, out_rgb = self.alloc_outputs(w, h)
        lam = np.atleast_1d(np.asarray(lam, dtype=np.float32))
        c = make_camera(cam)
        self._check(getattr(self.L, _fn)(self.h, C.byref(c), w, h, _ptr(lam), len(lam),
                                             None if scene_zn is None else C.c_void_p(scene_zn.data_ptr()),
                                             None if scene_rgb is None else C.c_void_p(scene_rgb.data_ptr()),
                                             C.c_void_p(out_gbuffer.data_ptr()), C.c_void_p(out_rgb.data_ptr())),
                    _fn)
        self._updates_issued()
        self._res = (w, h)
        return out_gbuffer, out_rgb

    def render_to_host(self, cam: dict, lam, host_rgb, host_gbuffer=None):
        w, h = cam["width"], cam["height"]
        lam = np.atleast_1d(np.asarray(lam, dtype=np.float32))
        c = make_camera(cam)
        self._check(self.L.hair_render_to_host(self.h, C.byref(c), w, h, _ptr(lam), len(lam),
                                               None if host_gbuffer is None else C.c_void_p(host_gbuffer.data_ptr()),
                                               C.c_void_p(host_rgb.data_ptr())), "hair_render_to_host")
        self._updates_issued()
        self._res = (w, h)

    def render_to_host_async(self, cam: dict, lam, host_rgb, host_gbuffer=None) -> int:
        """Enqueue the frame and its device->host copies; returns the slot to pass to host_wait."""
        w, h = cam["width"], cam["height"]
        lam = np.atleast_1d(np.asarray(lam, dtype=np.float32))
        c = make_camera(cam)
        slot = C.c_int(-1)
        self._check(self.L.hair_render_to_host_async(self.h, C.byref(c), w, h, _ptr(lam), len(lam),
                                                     None if host_gbuffer is None else C.c_void_p(host_gbuffer.data_ptr()),
                                                     C.c_void_p(host_rgb.data_ptr()), C.byref(slot)), "hair_render_to_host_async")
        self._updates_issued()
        self._res = (w, h)
        return slot.value

    def host_wait(self, slot: int = -1):
        self._check(self.L.hair_host_wait(self.h, int(slot)), "hair_host_wait")

    def render_stages(self, cam: dict, stage_mask: int, gbuffer, out_rgb):
        w, h = cam["width"], cam["height"]
        c = make_camera(cam)
        self._check(self.L.hair_render_stages(self.h, C.byref(c), w, h, stage_mask, C.c_void_p(gbuffer.data_ptr()),
                                              C.c_void_p(out_rgb.data_ptr())), "hair_render_stages")

    # ---- hair_stats()
    def stats(self) -> dict:
        s = hair_stats_t()
        self._check(self.L.hair_stats(self.h, C.byref(s)), "hair_stats")
        self._updates_issued()
        return s.as_dict()

    # ---- debug / parity
    def _wrap(self, ptr: int, shape, dtype):
        """A torch tensor aliasing library-owned device memory (valid until the next upload/render)."""
        t = self.torch
        n = int(np.prod(shape))
        if n == 0:
            return t.empty(shape, dtype=dtype, device=f"cuda:{self.device}")
        itemsize = t.empty((), dtype=dtype).element_size()

        class _Holder:
            pass
        hd = _Holder()
        hd.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": {t.float32: "<f4", t.int32: "<i4"}[dtype],
                                       "data": (ptr, False), "version": 2, "strides": None}
        del itemsize
        return t.as_tensor(hd, device=f"cuda:{self.device}")

    def debug_vertices(self):
        s = self.stats()
        v, tb, col = C.c_void_p(), C.c_void_p(), C.c_void_p()
        self._check(self.L.hair_debug_buffers(self.h, C.byref(v), C.byref(tb), C.byref(col)), "hair_debug_buffers")
        return self._wrap(v.value, (s["n_vertices"], 4), self.torch.float32).clone()

    def debug_table(self):
        s = self.stats()
        v, tb, col = C.c_void_p(), C.c_void_p(), C.c_void_p()
        self._check(self.L.hair_debug_buffers(self.h, C.byref(v), C.byref(tb), C.byref(col)), "hair_debug_buffers")
        return self._wrap(tb.value, (s["n_bundles"], 4), self.torch.int32).clone()

    def debug_colour(self):
        w, h = self._res
        v, tb, col = C.c_void_p(), C.c_void_p(), C.c_void_p()
        self._check(self.L.hair_debug_buffers(self.h, C.byref(v), C.byref(tb), C.byref(col)), "hair_debug_buffers")
        return self._wrap(col.value, (h, w, 4), self.torch.float32).clone()

    def debug_set_vertices(self, v):
        v = v.contiguous()
        self._check(self.L.hair_debug_set_vertices(self.h, C.c_void_p(v.data_ptr()), v.shape[0]), "hair_debug_set_vertices")

    def shadow_build(self, light_cams: list, layer_d1: float, alpha_s: float) -> None:
        """hair_shadow_build: one deep opacity map per camera of `light_cams` (dicts with width == height == res)."""
        p = hair_shadow_params()
        p.n_lights, p.res = len(light_cams), int(light_cams[0]["width"])
        p.layer_d1, p.alpha_s = float(layer_d1), float(alpha_s)
        for i, lc in enumerate(light_cams):
            assert lc["width"] == lc["height"] == p.res
            p.cam[i] = make_camera(lc)
        self._check(self.L.hair_shadow_build(self.h, C.byref(p)), "hair_shadow_build")
        self._updates_issued()
        self._shadow_res = p.res

    def shadow_clear(self) -> None:
        self._check(self.L.hair_shadow_clear(self.h), "hair_shadow_clear")

    def debug_shadow(self, light: int):
        """(z0 [res][res], cnt [res][res][4], D[4]) of light `light`'s map: int32 device tensors (bit patterns of uint32)."""
        z0, cnt, D = C.c_void_p(), C.c_void_p(), (C.c_uint32 * 4)()
        self._check(self.L.hair_debug_shadow(self.h, light, C.byref(z0), C.byref(cnt), C.byref(D)), "hair_debug_shadow")
        r = self._shadow_res
        return (self._wrap(z0.value, (r, r), self.torch.int32).clone(), self._wrap(cnt.value, (r, r, 4), self.torch.int32).clone(),
                [int(x) for x in D])

    def atomic_microbench(self, mode: int, words, n_ops: int, hot_words: int = 1024) -> float:
        ms = C.c_float(0)
        self._check(self.L.hair_atomic_microbench(self.h, mode, C.c_void_p(words.data_ptr()), words.numel(), n_ops,
                                                  hot_words, C.byref(ms)), "hair_atomic_microbench")
        return ms.value

    def l2_load_microbench(self, mode: int, pairs, pitch: int, n_steps: int = 64):
        """hair_l2_load_microbench over `pairs` (int64 device tensor [n][2]); returns (loads, ms)."""
        ms, n = C.c_float(0), C.c_uint64(0)
        self._check(self.L.hair_l2_load_microbench(self.h, mode, C.c_void_p(pairs.data_ptr()), pairs.numel() // 2, pitch,
                                                   n_steps, C.byref(n), C.byref(ms)), "hair_l2_load_microbench")
        return n.value, ms.value


def scan_noalloc(counts, bases, totals, n: int | None = None, stream=None) -> None:
    """hair_scan_noalloc: the H2 scan for callers that may not allocate device memory (an engine whose own pool holds
    all of it, or a frame loop that bans the synchronising cudaMalloc / cudaFree). No context, no allocation here or in
    the library: `counts` [n][2] {N_LOD, C}, `bases` [n][2] and `totals` [2] are the caller's int32 CUDA tensors
    (uint32 bit patterns, contiguous); the library's scratch is a fixed array in its device code, so n is at most
    SCAN_NOALLOC_MAX and calls that could overlap on one GPU must be ordered by the caller. Enqueues on `stream`
    (default: torch's current stream of the tensors' device) and returns without waiting."""
    import torch
    dev = counts.device.index
    assert counts.is_contiguous() and bases.is_contiguous() and totals.is_contiguous()
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    L = load()
    rc = L.hair_scan_noalloc(dev, C.c_void_p(st.cuda_stream), C.c_void_p(counts.data_ptr()),
                             counts.shape[0] if n is None else int(n), C.c_void_p(bases.data_ptr()),
                             C.c_void_p(totals.data_ptr()))
    if rc != 0:
        raise HairError(f"hair_scan_noalloc failed ({rc}): {L.hair_scan_noalloc_error().decode()}")


def gbuffer_to_numpy(gb) -> np.ndarray:
    """int64 device tensor [H][W][2] -> uint64 numpy."""
    return gb.cpu().numpy().view(np.uint64)
