"""Seeded synthetic grooms shaped like the paper's workloads (BASELINE.json configs).

The paper measures on the authors' own grooms ("a hair scene with 127k strands";
PAPER.md:7 Fig. 1 "total of 483k strands, 4K"), which are not available; these inputs take their
shapes (strand counts, control-point counts, resolutions, camera distances, LOD strengths) and
stand in for them.

This module is INPUT DATA ONLY: numpy arrays and parameter dicts. It holds none of the method's
arithmetic (no hash, no spline, no projection, no packing) and imports neither the CUDA binding
nor the oracle, so both may be fed from it. Randomness: numpy PCG64 ``default_rng(seed)``.
"""
from __future__ import annotations

import math

import numpy as np

VFOV = math.radians(45.0)
NEAR, FAR = 0.1, 100.0


# --------------------------------------------------------------------------- scalp + cage
def scalp_patch(nu: int, nv: int, phi_range, radius=0.1):
    """Spherical patch of a hemisphere, y up; (nu x nv) cells, two triangles per cell."""
    th = np.linspace(0.15, math.pi / 2, nv + 1)
    ph = np.linspace(phi_range[0], phi_range[1], nu + 1)
    T, P = np.meshgrid(th, ph, indexing="ij")  # [nv+1][nu+1]
    n = np.stack([np.sin(T) * np.cos(P), np.cos(T), np.sin(T) * np.sin(P)], -1).reshape(-1, 3)
    pos = radius * n
    tris = []
    for a in range(nv):
        for b in range(nu):
            i00 = a * (nu + 1) + b
            i01 = i00 + 1
            i10 = i00 + (nu + 1)
            i11 = i10 + 1
            tris.append((i00, i10, i01))
            tris.append((i01, i10, i11))
    return pos.astype(np.float64), n.astype(np.float64), np.asarray(tris, np.uint32)


def _smooth_field(rng, x):
    """Seeded smooth direction field: sum of 3 low-frequency sinusoids of position."""
    out = np.zeros_like(x)
    for _ in range(3):
        k = rng.uniform(-12.0, 12.0, size=(3, 3))
        ph = rng.uniform(0, 2 * math.pi, size=3)
        out += np.sin(x @ k.T + ph)
    return out / 3.0


def build_cage(rng, scalp, normals, n_prisms, length, mode):
    """Cage vertex layers X_i = X_{i-1} + h * normalize(dir_i)."""
    lv = n_prisms + 1
    X = np.zeros((lv,) + scalp.shape)
    X[0] = scalp
    h = length / n_prisms
    g = np.array([0.0, -1.0, 0.0])
    if mode == "droop":  # config 1: along normals plus a quadratic gravity droop
        for i in range(1, lv):
            X[i] = scalp + normals * (h * i)
            X[i, :, 1] -= 0.02 * (i / (lv - 1)) ** 2
        return X
    frng = np.random.default_rng(rng.integers(1 << 31))
    for i in range(1, lv):
        s = i / (lv - 1)
        d = (1.0 - 0.7 * s) * normals + (0.25 + 0.9 * s) * g + 0.45 * _smooth_field(
            np.random.default_rng(frng.integers(1 << 31)), X[i - 1] * 1.0)
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        X[i] = X[i - 1] + h * d
    return X


def strands_per_tri(scalp, tris, total):
    """N_t proportional to triangle area, largest-remainder rounding to the exact total."""
    a = scalp[tris[:, 1]] - scalp[tris[:, 0]]
    b = scalp[tris[:, 2]] - scalp[tris[:, 0]]
    area = 0.5 * np.linalg.norm(np.cross(a, b), axis=1)
    share = area / area.sum() * total
    n = np.floor(share).astype(np.int64)
    rem = total - n.sum()
    order = np.argsort(-(share - n), kind="stable")
    n[order[:rem]] += 1
    assert n.sum() == total
    return n.astype(np.uint32)


def make_groom(seed, nu, nv, n_prisms, spi, strands, ops=(), length=0.25, mode="field",
               phi_range=(math.pi / 2 - 0.75 * math.pi, math.pi / 2 + 0.75 * math.pi),
               xform=None, **style):
    rng = np.random.default_rng(seed)
    scalp, normals, tris = scalp_patch(nu, nv, phi_range)
    X = build_cage(rng, scalp, normals, n_prisms, length, mode)
    lv = n_prisms + 1
    ao = 0.35 + 0.65 * (np.arange(lv)[:, None] / (lv - 1)) * np.ones((1, scalp.shape[0]))
    ao = np.clip(ao * (1.0 + rng.uniform(-0.1, 0.1, size=ao.shape)), 0.0, 1.0)
    st = dict(spi=spi, seed=int(seed), ops=tuple(ops))
    st.update(style)
    return dict(pos=X.astype(np.float32), ao=ao.astype(np.float32), idx=tris,
                strands_per_tri=strands_per_tri(scalp, tris, strands),
                xform=None if xform is None else np.asarray(xform, np.float32).reshape(-1, 12),
                style=st)


# --------------------------------------------------------------------------- camera / lights
def look_from_z(center, distance, width, height):
    """Camera on +z of `center`, looking down -z; right = +x, up = +y (orthonormal, exact)."""
    c = np.asarray(center, np.float64)
    return dict(eye=tuple(float(v) for v in (c + np.array([0, 0, distance]))),
                right=(1.0, 0.0, 0.0), up=(0.0, 1.0, 0.0), forward=(0.0, 0.0, -1.0),
                vfov_y=VFOV, near_z=NEAR, far_z=FAR, width=int(width), height=int(height))


def moving_camera(cam: dict, i: int, yaw_step=0.004, dolly_step=0.004):
    """Frame i of a slow orbit of `cam`: yaw about the up axis by i * yaw_step rad while the eye swings sideways and
    dollies in and out (up to ~10 px of image motion per frame at 4K) — a bench leg whose depth ranges and hi-Z are one frame stale."""
    a = yaw_step * 10.0 * math.sin(i * 0.1)
    ca, sa = math.cos(a), math.sin(a)
    r, u, f = (np.asarray(cam[k], np.float64) for k in ("right", "up", "forward"))
    r2, f2 = ca * r + sa * f, ca * f - sa * r
    eye = np.asarray(cam["eye"], np.float64) + dolly_step * 10.0 * (math.sin(i * 0.07) * r + (1.0 - math.cos(i * 0.05)) * f)
    out = dict(cam)
    out.update(eye=tuple(float(v) for v in eye), right=tuple(float(v) for v in r2), forward=tuple(float(v) for v in f2))
    return out


def lights_around(rng, center, scale=1.0):
    out = []
    for i in range(3):  # PAPER.md:200 "three point light sources"
        d = rng.normal(size=3)
        d[2] = abs(d[2]) + 0.3  # camera side
        d /= np.linalg.norm(d)
        r = rng.uniform(1.0, 2.0) * scale
        inten = (r * r) * rng.uniform(0.6, 1.2) * np.array([1.0, 0.95, 0.9])
        out.append((tuple(float(v) for v in (np.asarray(center) + r * d)), tuple(float(v) for v in inten)))
    return out


def light_cameras(sc: dict, res: int = 512):
    """One square perspective camera per point light of sc["params"], looking from the light at the centre of the
    scene's cages with the whole scene inside its frustum and depth range (the views deep opacity maps are built
    from). Geometry only."""
    lo, hi = np.full(3, np.inf), np.full(3, -np.inf)
    for g in sc["grooms"]:
        p = g["pos"].reshape(-1, 3).astype(np.float64)
        xf = g["xform"] if g["xform"] is not None else np.array([[1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]], np.float64)
        for M in np.asarray(xf, np.float64).reshape(-1, 3, 4):
            q = p @ M[:, :3].T + M[:, 3]
            lo, hi = np.minimum(lo, q.min(0)), np.maximum(hi, q.max(0))
    c, R = 0.5 * (lo + hi), 0.5 * float(np.linalg.norm(hi - lo)) * 1.05
    cams = []
    for pos, _ in sc["params"]["lights"]:
        e = np.asarray(pos, np.float64)
        d = float(np.linalg.norm(c - e))
        f = (c - e) / d
        up0 = np.array([0.0, 1.0, 0.0]) if abs(f[1]) < 0.9 else np.array([1.0, 0.0, 0.0])
        r = np.cross(up0, -f)
        r /= np.linalg.norm(r)
        u = np.cross(-f, r)
        cams.append(dict(eye=tuple(float(v) for v in e), right=tuple(float(v) for v in r), up=tuple(float(v) for v in u),
                         forward=tuple(float(v) for v in f), vfov_y=float(2.0 * math.asin(min(R / d, 0.95)) * 1.05),
                         near_z=float(max(d - R, 0.05 * d) * 0.98), far_z=float((d + R) * 1.02),
                         width=int(res), height=int(res)))
    return cams


def default_params(rng, center, scale=1.0, **over):
    p = dict(center_diameter_px=0.5, filter_radius=5, s_par=0.5, s_perp=0.15, sigma_c=0.9,
             tau_z=1.45e-3, tau_fly=5e-4, w_strip=0.5, lights=lights_around(rng, center, scale),
             ambient_rgb=(0.15, 0.15, 0.15), k_d=0.4, k_R=0.25, k_TRT=0.5,
             background_rgb=(0.0, 0.0, 0.0), filter_on=True)
    p.update(over)
    return p


def _center(g):
    p = g["pos"].reshape(-1, 3).astype(np.float64)
    c = 0.5 * (p.min(0) + p.max(0))
    if g["xform"] is not None and g["xform"].shape[0] == 1:
        M = g["xform"][0].reshape(3, 4).astype(np.float64)
        c = M[:, :3] @ c + M[:, 3]
    return c


def _translate(t):
    return np.array([[1, 0, 0, t[0], 0, 1, 0, t[1], 0, 0, 1, t[2]]], np.float32)


def _scaled(n, scale, lo=1):
    return max(lo, int(round(n * scale)))


# --------------------------------------------------------------------------- the five configs
def config(index: int, scale: float = 1.0, res_scale: float = 1.0, distance=None, lam=None):
    """BASELINE.json configs[index-1] as concrete inputs. `scale` multiplies strand counts and
    `res_scale` the resolution (for parity cases the oracle finishes in seconds); 1.0 = as named."""
    seed = 1000 + index
    rng = np.random.default_rng(seed)

    def res(w, h):
        return max(32, int(round(w * res_scale))), max(32, int(round(h * res_scale)))

    if index == 1:  # tiny groom
        g = make_groom(seed, 8, 4, 2, 8, _scaled(1024, scale), ops=(), length=0.10, mode="droop",
                       phi_range=(math.pi / 4, 3 * math.pi / 4))
        w, h = res(256, 256)
        d = 0.5 if distance is None else distance
        cam = look_from_z(_center(g), d, w, h)
        return dict(name="tiny", grooms=[g], camera=cam, params=default_params(rng, _center(g)),
                    lam=[0.0 if lam is None else lam])
    if index == 2:  # single groom, curl + frizz
        g = make_groom(seed, 32, 32, 8, 4, _scaled(50_000, scale), ops=("curl", "frizz"),
                       curl_radius=0.004, curl_turns=3.0, curl_ramp_w0=0.1,
                       frizz_sigma=0.001, frizz_ramp_w0=0.1, frizz_cells=8, width_world=8e-5)
        w, h = res(1920, 1080)
        d = 0.5 if distance is None else distance
        cam = look_from_z(_center(g), d, w, h)
        return dict(name="single", grooms=[g], camera=cam, params=default_params(rng, _center(g)),
                    lam=[0.0 if lam is None else lam])
    if index == 3:  # dense long groom, twist + clump, lambda x distance sweep
        g = make_groom(seed, 64, 32, 12, 4, _scaled(150_000, scale), ops=("twist", "clump"),
                       twist_turns=1.5, clump_strength=0.6, clump_exp=1, length=0.30)
        w, h = res(3840, 2160)
        d = 2.0 if distance is None else distance
        cam = look_from_z(_center(g), d, w, h)
        return dict(name="dense", grooms=[g], camera=cam, params=default_params(rng, _center(g)),
                    lam=[4.0 if lam is None else lam],
                    sweep=dict(lam=(0.0, 1.0, 2.0, 4.0, 8.0), distance=(0.5, 2.0, 8.0)))
    if index == 4:  # five grooms, 483k strands: THE TARGET FRAME (Fig. 1)
        w, h = res(3840, 2160)
        thfov = (w / h) * math.tan(VFOV / 2)
        spec = [  # strands, prisms, spi, ops, distance, lambda, (nu, nv), style
            (120_000, 12, 4, ("curl",), 0.6, 4.0, (64, 32), dict(curl_radius=0.004, curl_turns=3.0, curl_ramp_w0=0.1)),
            (110_000, 8, 4, (), 1.5, 5.5, (32, 32), dict()),
            (95_000, 6, 4, ("clump",), 3.0, 2.0, (32, 32), dict(clump_strength=0.6, clump_exp=1)),
            (88_000, 10, 4, ("curl", "frizz"), 6.0, 2.8, (64, 32),
             dict(curl_radius=0.003, curl_turns=4.0, curl_ramp_w0=0.1, frizz_sigma=0.001, frizz_ramp_w0=0.1)),
            (70_000, 12, 3, ("clump", "twist"), 12.0, 3.0, (64, 32),
             dict(clump_strength=0.5, clump_exp=2, twist_turns=1.0)),
        ]
        xs = (-0.75, 0.15, 0.5, 0.72, 0.88)  # screen-space slots (NDC x); nearest groom on the left
        grooms, lams = [], []
        for gi, (n, prisms, spi, ops, dist, lm, (nu, nv), sty) in enumerate(spec):
            g = make_groom(seed + gi, nu, nv, prisms, spi, _scaled(n, scale), ops=ops, **sty)
            g["xform"] = _translate((xs[gi] * dist * thfov, 0.0, -dist))
            grooms.append(g)
            lams.append(lm)
        cam = look_from_z((0.0, -0.05, 0.0), 0.0, w, h)
        prm = default_params(rng, (0.0, 0.0, -2.0), scale=3.0)
        return dict(name="five_groom", grooms=grooms, camera=cam, params=prm,
                    lam=lams if lam is None else [lam] * 5)
    if index == 5:  # far-field crowd: 64 instances at 10-40 m
        w, h = res(3840, 2160)
        n_inst = 64
        thfov = (w / h) * math.tan(VFOV / 2)
        tv = math.tan(VFOV / 2)
        xf = []
        for _ in range(n_inst):
            z = rng.uniform(10.0, 40.0)
            x = rng.uniform(-0.9, 0.9) * z * thfov
            y = rng.uniform(-0.9, 0.9) * z * tv
            a = rng.uniform(0, 2 * math.pi)
            ca, sa = math.cos(a), math.sin(a)
            xf.append([ca, 0, sa, x, 0, 1, 0, y, -sa, 0, ca, -z])
        g = make_groom(seed, 32, 16, 6, 4, _scaled(30_000, scale), ops=("frizz",),
                       frizz_sigma=0.0005, frizz_ramp_w0=0.1, xform=np.asarray(xf, np.float32))
        cam = look_from_z((0.0, 0.0, 0.0), 0.0, w, h)
        prm = default_params(rng, (0.0, 0.0, -20.0), scale=10.0)
        return dict(name="crowd", grooms=[g], camera=cam, params=prm, lam=[4.0 if lam is None else lam])
    raise ValueError(index)


def n_strands(scene) -> int:
    return int(sum(int(g["strands_per_tri"].sum()) * (1 if g["xform"] is None else g["xform"].shape[0])
                   for g in scene["grooms"]))


# --------------------------------------------------------------------------- special scenes (tests)
def straight_prism(n_layers=5, h=0.05, axis=1, strands=32, spi=4, ops=(), **style):
    """One axis-aligned straight prism with equal layer spacing (closed-form pin, north_star)."""
    base = np.array([[0.0, 0.0, 0.0], [0.02, 0.0, 0.0], [0.0, 0.0, 0.02]])
    if axis == 0:
        base = base[:, [1, 0, 2]]
    elif axis == 2:
        base = base[:, [0, 2, 1]]
    X = np.zeros((n_layers, 3, 3))
    for i in range(n_layers):
        X[i] = base
        X[i, :, axis] += h * i
    st = dict(spi=spi, seed=7, ops=tuple(ops))
    st.update(style)
    return dict(pos=X.astype(np.float32), ao=None, idx=np.array([[0, 1, 2]], np.uint32),
                strands_per_tri=np.array([strands], np.uint32), xform=None, style=st)


def flat_prism(a, b, h, n_layers, strands=64, spi=4):
    """A flat prism in the plane z = 0: root triangle (0,0,0), (a,0,0), (0,b,0), layers stacked by h along +y.
    Every cage vertex has the same view depth for a camera on +z, so the projected AABB has a closed form."""
    X = np.zeros((n_layers, 3, 3))
    for i in range(n_layers):
        X[i] = np.array([[0.0, 0.0, 0.0], [a, 0.0, 0.0], [0.0, b, 0.0]])
        X[i, :, 1] += h * i
    return dict(pos=X.astype(np.float32), ao=None, idx=np.array([[0, 1, 2]], np.uint32),
                strands_per_tri=np.array([strands], np.uint32), xform=None, style=dict(spi=spi, seed=9, ops=()))


def straddle_prism(n_layers=5, dz=0.5, dx=0.06, strands=24, spi=4):
    """A prism whose layers march TOWARDS a camera on +z (layer i at z = i dz, x = i dx): a camera placed inside its
    depth range has some cage vertices and some strand vertices behind the near plane (R12, R13)."""
    base = np.array([[0.0, 0.0, 0.0], [0.05, 0.0, 0.0], [0.0, 0.05, 0.0]])
    X = np.zeros((n_layers, 3, 3))
    for i in range(n_layers):
        X[i] = base + np.array([dx * i, 0.0, dz * i])
    return dict(pos=X.astype(np.float32), ao=None, idx=np.array([[0, 1, 2]], np.uint32),
                strands_per_tri=np.array([strands], np.uint32), xform=None, style=dict(spi=spi, seed=13, ops=()))
