"""Pins of the oracle's projection, coverage predicates, packed word and resolve (O4/O5).

Independent checks: closed forms (horizontal segment, supercover count, Bresenham), a
double-precision brute force written here with different formulas (Liang-Barsky clipping for
segment-vs-square, vector projection for the centre distance), order independence.
"""
import math

import numpy as np
import pytest

from paper_2607_04230_b200 import synth

EMPTY = np.uint64(0xFFFFFFFFFFFFFFFF)


# ------------------------------------------------------------------------------- independent maths
def clip_segment_to_box(a, b, x0, y0, x1, y1):
    """Liang-Barsky: does the closed segment a-b meet the closed box? (double precision)"""
    t0, t1 = 0.0, 1.0
    dx, dy = b[0] - a[0], b[1] - a[1]
    for p, q in ((-dx, a[0] - x0), (dx, x1 - a[0]), (-dy, a[1] - y0), (dy, y1 - a[1])):
        if p == 0:
            if q < 0:
                return False
        else:
            r = q / p
            if p < 0:
                if r > t1:
                    return False
                t0 = max(t0, r)
            else:
                if r < t0:
                    return False
                t1 = min(t1, r)
    return t0 <= t1


def point_segment(c, a, b):
    """closest-point parameter and distance (double)"""
    d = b - a
    dd = d @ d
    t = 0.0 if dd == 0 else min(max(((c - a) @ d) / dd, 0.0), 1.0)
    q = a + t * d
    return t, math.hypot(*(c - q))


def pinhole(cam, p):
    """textbook pinhole projection in double: returns sx, sy, zn, zv"""
    eye, r, u, f = (np.asarray(cam[k], np.float64) for k in ("eye", "right", "up", "forward"))
    q = np.asarray(p, np.float64) - eye
    xv, yv, zv = q @ r, q @ u, q @ f
    fpx = 0.5 * cam["height"] / math.tan(0.5 * cam["vfov_y"])
    n, fa = cam["near_z"], cam["far_z"]
    zn = fa / (fa - n) - fa * n / ((fa - n) * zv)  # standard [0,1] depth: 0 at near, 1 at far
    return 0.5 * cam["width"] + fpx * xv / zv, 0.5 * cam["height"] - fpx * yv / zv, zn, zv


# ------------------------------------------------------------------------------- projection
def test_projection_matches_pinhole(orc):
    cam = synth.look_from_z((0.1, 0.2, 0.0), 1.5, 640, 360)
    rng = np.random.default_rng(0)
    for _ in range(200):
        p = rng.uniform(-0.5, 0.5, size=3) + np.array([0.1, 0.2, 0.0])
        o, valid = orc.project(cam, p)
        want = pinhole(cam, np.float32(p))
        assert valid
        assert abs(o[0] - want[0]) < 2e-3 and abs(o[1] - want[1]) < 2e-3  # fp32 at |sx| < 1024
        assert abs(o[2] - want[2]) < 2e-7 and abs(o[3] - want[3]) < 1e-6
    # optical axis -> image centre; top edge of the frustum -> sy = 0; near -> zn 0; far -> zn 1
    o, _ = orc.project(cam, (0.1, 0.2, 0.0))
    assert o[0] == 320.0 and o[1] == 180.0
    top = 1.5 * math.tan(0.5 * cam["vfov_y"])
    o, _ = orc.project(cam, (0.1, 0.2 + top, 0.0))
    assert abs(o[1]) < 1e-3
    o, v = orc.project(cam, (0.1, 0.2, 1.5 - 0.1))
    assert v and abs(o[2]) < 1e-6
    o, v = orc.project(cam, (0.1, 0.2, 1.5 - 100.0))
    assert v and abs(o[2] - 1.0) < 1e-6
    o, v = orc.project(cam, (0.1, 0.2, 1.5 - 0.05))
    assert not v  # in front of the near plane (R12)


# ------------------------------------------------------------------------------- word
def test_pack_unpack_round_trip_and_order(orc):
    rng = np.random.default_rng(1)
    for _ in range(200):
        zn, t = float(np.float32(rng.uniform())), float(np.float32(rng.uniform()))
        sid, j = int(rng.integers(1 << 24)), int(rng.integers(127))
        w = orc.pack(zn, sid, j, t)
        dq, s, jj, t9 = orc.unpack(w)
        assert (s, jj) == (sid, j)
        # fp32: zn*16777215 + 0.5 itself rounds once the product passes 2^23, so half a step becomes one step
        assert abs(dq / 16777215.0 - zn) <= (0.5 if zn < 0.5 else 1.0) / 16777215.0 + 1e-9
        assert abs(t9 / 511.0 - t) <= 0.5 / 511.0 + 1e-7
        assert w != int(EMPTY)
    assert orc.unpack(orc.pack(1.0, 0, 0, 0.0))[0] == 0xFFFFFE  # R8: capped below the clear value
    assert orc.unpack(orc.pack(0.0, 0, 0, 1.0)) == (0, 0, 0, 511)
    # depth in the high bits: a nearer hit always compares smaller, whatever the payload
    assert orc.pack(0.25, (1 << 24) - 1, 126, 1.0) < orc.pack(0.2500002, 0, 0, 0.0)
    zs = np.linspace(0, 1, 4001, dtype=np.float32)
    dqs = [orc.unpack(orc.pack(float(z), 0, 0, 0.0))[0] for z in zs]
    assert all(a <= b for a, b in zip(dqs, dqs[1:]))  # monotone


def test_depth_quantisation_unprojects_within_half_step(orc):
    cam = synth.look_from_z((0, 0, 0), 1.0, 64, 64)
    n, fa = cam["near_z"], cam["far_z"]
    for zv in (0.2, 0.5, 1.0, 3.0, 12.0, 40.0):
        o, _ = orc.project(cam, (0.0, 0.0, 1.0 - zv))
        dq = orc.unpack(orc.pack(float(o[2]), 0, 0, 0.0))[0]
        z = dq / 16777215.0
        zv_back = (fa * n / (fa - n)) / (fa / (fa - n) - z)
        step = zv * zv * (fa - n) / (fa * n) / 16777215.0  # d(zv)/d(zn) per quantisation step
        assert abs(zv_back - zv) <= 1.0 * step + 4e-7 * zv * zv / n  # one step (see above) + fp32 rounding of zn


# ------------------------------------------------------------------------------- coverage closed forms
def test_horizontal_segment_closed_form(orc):
    cover, tq = orc.segment_cover((2.5, 3.5), (10.5, 3.5), 0.25, 16, 8)
    ys, xs = np.nonzero(cover)
    assert set(zip(xs, ys)) == {(x, 3) for x in range(2, 11)}
    assert (cover[3, 2:11] == 3).all()  # both layers: the line runs through the pixel centres
    assert np.allclose(tq[3, 2:11], np.arange(9) / 8.0)


@pytest.mark.parametrize("seed", range(6))
def test_supercover_count_general_position(orc, seed):
    # a segment in general position touches |dfloor x| + |dfloor y| + 1 pixels
    rng = np.random.default_rng(seed)
    a, b = rng.uniform(1, 31, size=2), rng.uniform(1, 31, size=2)
    cover, _ = orc.segment_cover(a, b, 0.25, 32, 32)
    a32, b32 = np.float32(a), np.float32(b)
    want = abs(math.floor(b32[0]) - math.floor(a32[0])) + abs(math.floor(b32[1]) - math.floor(a32[1])) + 1
    assert int((cover & 1).sum()) == want


def bresenham(x0, y0, x1, y1):
    pts, dx, dy = [], abs(x1 - x0), -abs(y1 - y0)
    sx, sy = (1 if x0 < x1 else -1), (1 if y0 < y1 else -1)
    err = dx + dy
    while True:
        pts.append((x0, y0))
        if (x0, y0) == (x1, y1):
            return pts
        e2 = 2 * err
        if e2 >= dy:
            err += dy
            x0 += sx
        if e2 <= dx:
            err += dx
            y0 += sy


@pytest.mark.parametrize("p", [(3, 4, 20, 9), (25, 3, 4, 28), (5, 5, 5, 20), (2, 17, 29, 17), (7, 2, 11, 30)])
def test_centre_layer_contains_bresenham_line(orc, p):
    # rho = 0.5, endpoints on pixel centres: the centre layer holds the classic 1-px DDA line
    # ("single-pixel-wide lines"), and equals it for axis-aligned segments
    x0, y0, x1, y1 = p
    cover, _ = orc.segment_cover((x0 + 0.5, y0 + 0.5), (x1 + 0.5, y1 + 0.5), 0.5, 32, 32)
    centre = {(x, y) for y, x in zip(*np.nonzero(cover & 2))}
    line = set(bresenham(x0, y0, x1, y1))
    assert line <= centre
    if x0 == x1 or y0 == y1:
        assert line == centre
    assert len(centre) <= 2 * len(line)


def test_zero_length_segment_hits_one_pixel(orc):
    cover, _ = orc.segment_cover((7.2, 9.7), (7.2, 9.7), 0.25, 16, 16)
    assert int((cover & 1).sum()) == 1 and cover[9, 7] == 1  # 0.36 px from the centre (7.5, 9.5) > rho
    cover, _ = orc.segment_cover((7.45, 9.55), (7.45, 9.55), 0.25, 16, 16)
    assert cover[9, 7] == 3 and int((cover != 0).sum()) == 1


@pytest.mark.parametrize("seed", range(8))
def test_coverage_vs_double_precision_brute_force(orc, seed):
    # north_star: brute-force per-pixel segment tests on 32x32. Disagreement is allowed only where
    # the geometry is within 1e-4 px of a boundary.
    rng = np.random.default_rng(100 + seed)
    eps = 1e-4
    n_checked = 0
    for _ in range(40):
        a = rng.uniform(-2, 34, size=2)
        b = a + rng.normal(size=2) * rng.choice([0.3, 2.0, 12.0])
        rho = float(rng.choice([0.125, 0.25, 0.5]))
        a32, b32 = np.float32(a).astype(np.float64), np.float32(b).astype(np.float64)
        cover, tq = orc.segment_cover(a, b, rho, 32, 32)
        for y in range(32):
            for x in range(32):
                c = np.array([x + 0.5, y + 0.5])
                hit_out = clip_segment_to_box(a32, b32, x - eps, y - eps, x + 1 + eps, y + 1 + eps)
                hit_in = clip_segment_to_box(a32, b32, x + eps, y + eps, x + 1 - eps, y + 1 - eps)
                t, dist = point_segment(c, a32, b32)
                if hit_out == hit_in:  # firm decision
                    assert bool(cover[y, x] & 1) == hit_in, (a, b, x, y)
                    n_checked += 1
                if hit_in and abs(dist - rho) > eps:
                    assert bool(cover[y, x] & 2) == (dist < rho), (a, b, x, y, dist)
                if cover[y, x]:
                    assert abs(tq[y, x] - t) < 1e-4
                assert (cover[y, x] & 3) != 2  # centre subset of conservative, exactly
    assert n_checked > 30000


# ------------------------------------------------------------------------------- full frame
def _tiny_frame(orc, res=32, strands=96):
    sc = synth.config(1, scale=strands / 1024, res_scale=res / 256)
    f = orc.Frame(sc["grooms"])
    f.lod(sc["camera"], 0.0)
    f.generate()
    return sc, f


def test_gbuffer_vs_brute_force_32x32(orc):
    sc, f = _tiny_frame(orc)
    cam, prm = sc["camera"], sc["params"]
    counts = f.raster(cam, prm)
    G = f.gbuffer()
    V = f.vertices_f32().astype(np.float64)
    C = 17
    n_str = V.shape[0] // C
    rho = 0.5 * prm["center_diameter_px"]
    W = H = 32
    best = np.full((H, W, 2), None, dtype=object)
    cand = [[([], []) for _ in range(W)] for _ in range(H)]
    for s in range(n_str):
        P = [pinhole(cam, V[s * C + j, :3]) for j in range(C)]
        for j in range(C - 1):
            a, b = np.array(P[j][:2]), np.array(P[j + 1][:2])
            x0, x1 = int(math.floor(min(a[0], b[0]))) - 1, int(math.floor(max(a[0], b[0]))) + 1
            y0, y1 = int(math.floor(min(a[1], b[1]))) - 1, int(math.floor(max(a[1], b[1]))) + 1
            for y in range(max(y0, 0), min(y1, H - 1) + 1):
                for x in range(max(x0, 0), min(x1, W - 1) + 1):
                    if not clip_segment_to_box(a, b, x, y, x + 1, y + 1):
                        continue
                    t, dist = point_segment(np.array([x + 0.5, y + 0.5]), a, b)
                    zn = P[j][2] + t * (P[j + 1][2] - P[j][2])
                    dq = min(int(zn * 16777215.0 + 0.5), 0xFFFFFE)
                    cand[y][x][1].append((dq, s, j, dist))
                    if dist <= rho:
                        cand[y][x][0].append((dq, s, j, dist))
    n_px = n_same = 0
    for y in range(H):
        for x in range(W):
            for layer in (0, 1):
                c = cand[y][x][layer]
                w = int(G[y, x, layer])
                firm = [k for k in c if layer == 1 or abs(k[3] - rho) > 1e-4]
                if w == int(EMPTY):
                    assert not firm, (x, y, layer)  # nothing firmly covers an empty pixel
                    continue
                dq, sid, j, t9 = orc.unpack(w)
                n_px += 1
                assert c, (x, y, layer)
                dmin = min(k[0] for k in c)
                # the oracle's winner is a brute-force candidate within a few depth steps of the nearest:
                # zn = A - B/zv and its interpolation take ~4 fp32 roundings of 6e-8 = 1 step each
                match = [k for k in c if k[1] == sid and k[2] == j]
                assert match and abs(match[0][0] - dq) <= 3 and match[0][0] <= dmin + 3, (x, y, layer)
                if (sid, j) == min(c)[1:3]:  # same winning segment as the double-precision resolve
                    n_same += 1
    assert n_px > 300 and n_same >= 0.97 * n_px
    assert counts["segments"] == n_str * (C - 1)
    # centre subset of conservative, per pixel: cons word <= centre word
    assert (G[..., 1] <= G[..., 0]).all()


def test_segment_with_an_endpoint_behind_the_near_plane_is_dropped(orc):
    """DESIGN.md R12 (the paper is silent): a segment is drawn only if BOTH endpoints have zv >= near; no clipping.
    A camera inside the groom's depth range: the strands march towards it and cross the near plane."""
    g = synth.straddle_prism(n_layers=5, dz=0.5, strands=24, spi=4)
    cam = synth.look_from_z((0.1, 0.0, 0.0), 1.3, 96, 64)  # eye at z = 1.3 looking down -z
    prm = dict(center_diameter_px=1.0, lights=[])
    f = orc.Frame([g])
    f.lod(cam, 0.0)
    f.generate()
    v = f.vertices_f32()
    f.set_vertices_f32(v)
    cnt = f.raster(cam, prm)
    C = 17
    zv = np.float32(cam["eye"][2]) - v[:, 2].reshape(24, C)  # textbook: depth along -z from the eye
    valid = zv >= np.float32(cam["near_z"])
    assert np.abs(zv - np.float32(cam["near_z"])).min() > 1e-4  # no vertex sits on the plane itself
    drawn = valid[:, :-1] & valid[:, 1:]
    cut = valid[:, :-1] != valid[:, 1:]  # exactly one endpoint behind the plane
    assert cut.sum() == 24 and 0 < drawn.sum() < 24 * (C - 1)
    assert cnt["segments"] == int(drawn.sum())
    G = f.gbuffer()
    hit = G[..., 1] != EMPTY
    sid = ((G[..., 1] >> np.uint64(16)) & np.uint64(0xFFFFFF)).astype(np.int64)[hit]
    j = ((G[..., 1] >> np.uint64(9)) & np.uint64(0x7F)).astype(np.int64)[hit]
    assert hit.sum() > 50 and drawn[sid, j].all()          # no pixel names a cut or hidden segment
    last = drawn.shape[1] - 1 - np.argmax(drawn[:, ::-1], axis=1)  # last drawn segment of each strand ...
    seen = set(zip(sid.tolist(), j.tolist()))
    assert sum((s, int(last[s])) in seen for s in range(24)) >= 12  # ... is drawn right up to the cut


def test_resolve_is_order_independent(orc):
    # north_star invariant: the depth-sorted resolve is order-independent (min is commutative)
    sc, f = _tiny_frame(orc, res=64, strands=200)
    f.raster(sc["camera"], sc["params"])
    G0 = f.gbuffer()
    rng = np.random.default_rng(5)
    for _ in range(3):
        f.raster(sc["camera"], sc["params"], order=rng.permutation(f.n_strands))
        assert np.array_equal(f.gbuffer(), G0)
    f.raster(sc["camera"], sc["params"], order=np.arange(f.n_strands)[::-1])
    assert np.array_equal(f.gbuffer(), G0)


def test_nearer_duplicate_wins(orc):
    # two copies of the same groom, the second 5 cm nearer to the camera: it owns every pixel it covers
    sc = synth.config(1, scale=0.05, res_scale=0.25)
    g = sc["grooms"][0]
    g2 = dict(g)
    g2["xform"] = np.array([[1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0.05]], np.float32)
    n = int(g["strands_per_tri"].sum())
    f1 = orc.Frame([g2])
    f1.lod(sc["camera"], 0.0)
    f1.generate()
    f1.raster(sc["camera"], sc["params"])
    near_only = f1.gbuffer()
    f = orc.Frame([g, g2])
    f.lod(sc["camera"], 0.0)
    f.generate()
    f.raster(sc["camera"], sc["params"])
    G = f.gbuffer()
    covered = near_only[..., 1] != EMPTY
    sid = (G[..., 1] >> np.uint64(16)) & np.uint64(0xFFFFFF)
    # the far copy lies 5 cm behind everywhere, but its hair overlaps the near copy's depth range:
    # where the near copy covers a pixel, the winner is at least as near as the near copy's own hit
    assert (G[..., 1][covered] <= (near_only[..., 1][covered] + (np.uint64(n) << np.uint64(16)))).all()
    assert (sid[covered] >= n).mean() > 0.9


def test_width_world_sets_centre_radius(orc):
    # R9: projected width clamped to [0.25, 1] px; a wider strand hits more centre pixels
    sc = synth.config(1, scale=0.1, res_scale=0.5)
    hits = []
    for w in (0.0, 1e-6, 1.5e-3, 1e-2):  # 0, 3e-4, 0.46 and 3.1 px at f_px = 154.5, z ~ 0.5
        g = dict(sc["grooms"][0])
        g["style"] = dict(g["style"], width_world=w)
        f = orc.Frame([g])
        f.lod(sc["camera"], 0.0)
        f.generate()
        c = f.raster(sc["camera"], dict(sc["params"], center_diameter_px=0.25))
        hits.append(c["center"])
    assert hits[0] == hits[1]  # tiny width clamps to 0.25 px == center_diameter 0.25
    assert hits[1] < hits[2] < hits[3]
    assert hits[3] <= f.raster(sc["camera"], sc["params"])["cons"]


def test_window_samples_equal_full_frame(orc):
    """Frame.set_window (used to sample full-size frames in the GPU tests): inside the window the G-buffer
    and the filtered image are the full-frame values, outside nothing is written."""
    from paper_2607_04230_b200 import synth
    sc = synth.config(1, scale=0.5)
    cam, prm = sc["camera"], sc["params"]
    f = orc.Frame(sc["grooms"])
    f.lod(cam, sc["lam"])
    f.generate()
    f.set_vertices_f32(f.vertices_f32())
    f.raster(cam, prm)
    g_full = f.gbuffer().copy()
    f.shade(cam, prm)
    o_full = f.filter(cam, prm).copy()
    x0, y0, x1, y1 = 70, 60, 170, 141
    f.set_window(x0, y0, x1, y1)
    cnt = f.raster(cam, prm)
    g_win = f.gbuffer()
    assert np.array_equal(g_win[y0:y1, x0:x1], g_full[y0:y1, x0:x1])
    mask = np.ones(g_win.shape[:2], bool)
    mask[y0:y1, x0:x1] = False
    assert (g_win[mask] == np.uint64(0xFFFFFFFFFFFFFFFF)).all()
    assert 0 < cnt["cons"] < int((g_full[..., 1] != np.uint64(0xFFFFFFFFFFFFFFFF)).sum()) * 64
    f.set_gbuffer(g_full)
    f.shade(cam, prm)
    o_win = f.filter(cam, prm)
    assert np.array_equal(o_win[y0:y1, x0:x1], o_full[y0:y1, x0:x1])
    assert (o_win[mask] == 0).all()
    f.set_window()  # reset: whole image again
    f.raster(cam, prm)
    assert np.array_equal(f.gbuffer(), g_full)
