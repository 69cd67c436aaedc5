"""Pins of the oracle's deep opacity maps (§3.4 "Volumetric shadows are computed using deep-opacity maps
..., which we query using the depth-correction described in Section 3.2"; DESIGN.md R-dom). The paper prints no
formula for them, so the pins are: the lookup against closed forms on hand-made maps (Beer-Lambert, Eq. 6-7), and the
build against a recount from the primitives pinned elsewhere (orc.project, orc.segment_cover, orc.pack)."""
import math

import numpy as np

from paper_2607_04230_b200 import synth

D4 = np.array([100, 300, 700, 1500], np.uint32)


def _axis_cam(res=8):
    return synth.look_from_z((0.0, 0.0, 0.0), 2.0, res, res)


def _dq_of(orc, cam, p):
    o, valid = orc.project(cam, p)
    assert valid
    return orc.unpack(orc.pack(float(min(max(o[2], 0.0), 1.0)), 0, 0, 0.0))[0], o


def _point_at_texel(orc, cam, tx, ty, zv=2.0):
    """World point on the ray through screen position (tx, ty) at view depth zv, for the camera of look_from_z."""
    res = cam["width"]
    fpx = 0.5 * res / math.tan(0.5 * cam["vfov_y"])
    e = np.asarray(cam["eye"])
    p = e + np.array([(tx - 0.5 * res) * zv / fpx, (0.5 * res - ty) * zv / fpx, -zv])
    o, valid = orc.project(cam, p)
    assert valid and abs(o[0] - tx) < 1e-3 and abs(o[1] - ty) < 1e-3
    return p.astype(np.float32)


def test_lookup_is_beer_lambert_on_a_uniform_medium(orc):
    """Eq. 6-7: a medium of uniform density (fragments per layer proportional to the layer's thickness) gives
    V(d) = exp(-alpha sigma d) inside the layers and V'(d) = exp(-alpha sigma beta d) after thinning to beta, for
    every d — the closed form the depth-comparison fix is derived from. d <= 0 is unshadowed."""
    cam = _axis_cam()
    p = _point_at_texel(orc, cam, 4.5, 4.5)  # a texel centre: the bilinear weights select one texel
    dqp, _ = _dq_of(orc, cam, p)
    sigma, alpha = 0.02, 0.3
    cnt = np.zeros((8, 8, 4), np.uint32)
    cnt[...] = (sigma * np.diff(np.concatenate([[0], D4.astype(np.float64)]))).astype(np.uint32)  # 2, 4, 8, 16
    assert np.array_equal(cnt[0, 0], [2, 4, 8, 16])
    for d in (1, 50, 100, 299, 650, 1499):
        z0 = np.full((8, 8), dqp - d, np.uint32)
        for beta in (1.0, 0.5, 0.125):
            t = orc.dom_transmittance(cam, z0, cnt, D4, alpha, beta, p)
            assert abs(t - math.exp(-alpha * sigma * beta * d)) < 1e-12, (d, beta)
    for d in (0, -1, -500):  # at or in front of the nearest hair
        z0 = np.full((8, 8), dqp - d, np.uint32)
        assert orc.dom_transmittance(cam, z0, cnt, D4, alpha, 1.0, p) == 1.0
    # beyond the last layer end nothing more is in front: the total count
    z0 = np.full((8, 8), dqp - 5000, np.uint32)
    assert abs(orc.dom_transmittance(cam, z0, cnt, D4, alpha, 1.0, p) - math.exp(-alpha * 30.0)) < 1e-12
    # a pixel no hair touches casts no shadow
    assert orc.dom_transmittance(cam, np.full((8, 8), 0xFFFFFFFF, np.uint32), cnt, D4, alpha, 1.0, p) == 1.0


def test_lookup_is_piecewise_linear_in_the_fragment_count(orc):
    """Arbitrary counts: the optical depth at d is numpy's piecewise-linear interpolation of the cumulative count
    through the layer ends; beta scales d before the lookup (Eq. 7), so (beta, d) and (1, beta d) agree."""
    cam = _axis_cam()
    p = _point_at_texel(orc, cam, 2.5, 5.5)
    dqp, _ = _dq_of(orc, cam, p)
    rng = np.random.default_rng(7)
    for _ in range(20):
        c = rng.integers(0, 40, size=4).astype(np.uint32)
        cnt = np.zeros((8, 8, 4), np.uint32)
        cnt[...] = c
        d = int(rng.integers(1, 2000))
        beta = float(rng.uniform(0.05, 1.0))
        z0 = np.full((8, 8), dqp - d, np.uint32)
        xs = np.concatenate([[0.0], D4.astype(np.float64)])
        ys = np.concatenate([[0.0], np.cumsum(c.astype(np.float64))])
        want = math.exp(-0.1 * float(np.interp(beta * d, xs, ys)))
        assert abs(orc.dom_transmittance(cam, z0, cnt, D4, 0.1, beta, p) - want) < 1e-12
    # Eq. 7 as an identity between two lookups: thinning to beta at depth d == the full groom at depth beta d
    cnt[...] = np.array([7, 3, 11, 5], np.uint32)
    z_a, z_b = np.full((8, 8), dqp - 800, np.uint32), np.full((8, 8), dqp - 200, np.uint32)
    assert abs(orc.dom_transmittance(cam, z_a, cnt, D4, 0.1, 0.25, p) - orc.dom_transmittance(cam, z_b, cnt, D4, 0.1, 1.0, p)) < 1e-12


def test_lookup_blends_the_four_texels_around_the_point(orc):
    """Texel centres sit at integer + 1/2: at a centre only that texel counts, half way between two centres their
    optical depths average, at a corner all four do; empty texels and texels outside the map contribute nothing."""
    cam = _axis_cam()
    cnt = np.zeros((8, 8, 4), np.uint32)
    cnt[3, 3, 0], cnt[3, 4, 0], cnt[4, 3, 0], cnt[4, 4, 0] = 10, 20, 40, 80
    d, alpha = 100, 0.05  # at the end of layer 0: optical depth = the texel's count
    for (tx, ty), omega in (((3.5, 3.5), 10.0), ((4.5, 3.5), 20.0), ((4.0, 3.5), 15.0), ((3.5, 4.0), 25.0),
                            ((4.0, 4.0), 37.5), ((3.75, 3.5), 12.5)):
        p = _point_at_texel(orc, cam, tx, ty)
        dqp, _ = _dq_of(orc, cam, p)
        z0 = np.full((8, 8), dqp - d, np.uint32)
        t = orc.dom_transmittance(cam, z0, cnt, D4, alpha, 1.0, p)
        assert abs(-math.log(t) / alpha - omega) < 2e-3 * omega, ((tx, ty), -math.log(t) / alpha)
    # an empty neighbour weighs in with zero
    p = _point_at_texel(orc, cam, 4.0, 3.5)
    dqp, _ = _dq_of(orc, cam, p)
    z0 = np.full((8, 8), dqp - d, np.uint32)
    z0[3, 4] = 0xFFFFFFFF
    assert abs(-math.log(orc.dom_transmittance(cam, z0, cnt, D4, alpha, 1.0, p)) / alpha - 5.0) < 0.02
    # the map's border: the texels that do not exist contribute nothing
    cnt[0, 0, 0] = 12
    p = _point_at_texel(orc, cam, 0.25, 0.25)
    dqp, _ = _dq_of(orc, cam, p)
    z0 = np.full((8, 8), dqp - d, np.uint32)
    assert abs(-math.log(orc.dom_transmittance(cam, z0, cnt, D4, alpha, 1.0, p)) / alpha - 12.0 * 0.75 * 0.75) < 0.05


def _recount(orc, f, cam, prm, D3, z0):
    """The fragment counts again, from the primitives pinned elsewhere: every segment of the frame's fp32 vertices
    projected with orc.project, its conservative coverage and closest-point parameter from orc.segment_cover (pinned
    by the double-precision brute force of test_oracle_raster.py), depth at the hit as R11 states, quantised by
    orc.pack."""
    w, h = cam["width"], cam["height"]
    table, _ = f.table()
    v = f.vertices_f32().reshape(-1, 4)
    cnt = np.zeros((h, w, 4), np.uint32)
    n_hits = 0
    for nlod, C, _, vbase in table:
        for k in range(int(nlod)):
            P = [orc.project(cam, v[int(vbase) + k * int(C) + j, :3]) for j in range(int(C))]
            for j in range(int(C) - 1):
                (a, va), (b, vb) = P[j], P[j + 1]
                if not (va and vb):
                    continue  # R12
                cover, tq = orc.segment_cover(a[:2], b[:2], 0.5 * prm["center_diameter_px"], w, h)
                ys, xs = np.nonzero(cover & 1)
                for y, x in zip(ys, xs):
                    zn = np.float32(a[2]) + np.float32(tq[y, x]) * (np.float32(b[2]) - np.float32(a[2]))
                    if zn < 0 or zn > 1:
                        continue
                    d = orc.unpack(orc.pack(float(zn), 0, 0, 0.0))[0] - int(z0[y, x])
                    assert d >= 0
                    cnt[y, x, int(d >= D3[0]) + int(d >= D3[1]) + int(d >= D3[2])] += 1
                    n_hits += 1
    return cnt, n_hits


def test_build_equals_a_recount_from_pinned_primitives(orc):
    """z0 is the conservative layer of the light's G-buffer; the layer counts equal a recount done here, hit by hit,
    from orc.project / orc.segment_cover / orc.pack; their sum is the raster's own hit count."""
    sc = synth.config(1, scale=0.04)
    cam = synth.light_cameras(sc, 40)[1]
    prm = sc["params"]
    f = orc.Frame(sc["grooms"])
    f.lod(cam, [0.0])  # the maps are built from the full groom
    f.generate()
    D3 = np.array([2000, 6000, 14000], np.uint32)
    z0, cnt = f.dom_build(cam, prm, D3)
    G = f.gbuffer()
    none = (G[..., 1] & np.uint64(0xFFFFFFFFFF)) == np.uint64(0xFFFFFFFFFF)
    assert np.array_equal(z0[~none], (G[..., 1][~none] >> np.uint64(40)).astype(np.uint32)) and np.all(z0[none] == 0xFFFFFFFF)
    assert (~none).sum() > 100
    want, n_hits = _recount(orc, f, cam, prm, D3, z0)
    assert np.array_equal(cnt, want)
    assert int(cnt.sum()) == n_hits == f.raster(cam, prm)["cons"]
    assert np.all(cnt[~none][:, 0] >= 1)  # the nearest hit itself lies in layer 0
    assert np.all(cnt[none] == 0)
    assert cnt[..., 1:].sum() > 0  # the groom is deeper than one layer from this light


def test_shading_is_scaled_by_the_transmittance_light_by_light(orc):
    """O6 with a map: colour = ambient part + T_l x (light l's unshadowed part). Checked pixel by pixel on one
    light with the position rebuilt from the word; alpha_s = 0 changes nothing; shadows only ever darken."""
    sc = synth.config(1, scale=0.1, res_scale=0.25)
    cam, prm = sc["camera"], dict(sc["params"])
    prm["lights"] = prm["lights"][:1]
    lcam = synth.light_cameras(dict(sc, params=prm), 64)[0]
    full = orc.Frame(sc["grooms"])
    full.lod(lcam, [0.0])
    full.generate()
    D3 = np.array([3000, 9000, 21000], np.uint32)
    z0, cnt = full.dom_build(lcam, prm, D3)
    D4_ = np.array([3000, 9000, 21000, 45000], np.uint32)
    f = orc.Frame(sc["grooms"])
    f.lod(cam, [0.0])
    f.generate()
    f.raster(cam, prm)
    G = f.gbuffer()
    unshadowed = f.shade(cam, prm)
    amb = f.shade(cam, dict(prm, lights=[]))
    f.set_dom(0, lcam, z0, cnt, D4_, 0.0)
    assert np.array_equal(f.shade(cam, prm), unshadowed)  # alpha_s = 0: transmittance 1
    alpha = 0.08
    f.set_dom(0, lcam, z0, cnt, D4_, alpha)
    shadowed = f.shade(cam, prm)
    hit = (G[..., 0] & np.uint64(0xFFFFFFFFFF)) != np.uint64(0xFFFFFFFFFF)
    assert np.all(shadowed[hit] <= unshadowed[hit] + 1e-15) and (shadowed[hit] < unshadowed[hit] - 1e-6).any()
    v = f.vertices_f32()[:, :3].astype(np.float64)  # O6 shades from the fp32 vertex buffer
    table, _ = f.table()
    ys, xs = np.nonzero(hit)
    checked, lit = 0, 0
    for y, x in list(zip(ys, xs))[::7]:
        dq, sid, j, t9 = orc.unpack(int(G[y, x, 0]))
        # config 1 is one groom without LOD: strand sid starts at vertex sid * C
        C = int(table[0, 1])
        t = t9 / 511.0
        pos = (1 - t) * v[sid * C + j] + t * v[sid * C + j + 1]
        T = orc.dom_transmittance(lcam, z0, cnt, D4_, alpha, 1.0, pos.astype(np.float32))
        want = amb[y, x] + T * (unshadowed[y, x] - amb[y, x])
        assert np.allclose(shadowed[y, x], want, rtol=0, atol=1e-12), (y, x)
        checked += 1
        lit += T == 1.0
    assert checked > 50 and 0 < lit < checked  # some hits face the light unoccluded, some lie inside the groom
    f.set_dom(0, None)
    assert np.array_equal(f.shade(cam, prm), unshadowed)
    # the depth-comparison fix: a thinned groom (beta < 1) is looked up nearer to the light, so it is lit more
    f.set_dom(0, lcam, z0, cnt, D4_, alpha)
    f.set_dom_beta([0.4])
    brighter = f.shade(cam, prm)
    assert np.all(brighter[hit] >= shadowed[hit] - 1e-15) and (brighter[hit] > shadowed[hit] + 1e-6).any()


def test_light_cameras_frame_the_whole_scene(orc):
    """synth.light_cameras (input generator): orthonormal bases, eye at the light, every cage vertex of every groom
    and instance inside the view frustum and the depth range when the light stands outside the scene (config 1), and
    nothing in front of a light beyond its far plane otherwise."""
    for idx in (1, 4, 5):
        sc = synth.config(idx, scale=0.01, res_scale=0.1)
        cams = synth.light_cameras(sc, 128)
        assert len(cams) == len(sc["params"]["lights"])
        for cam, (pos, _) in zip(cams, sc["params"]["lights"]):
            r, u, f = (np.asarray(cam[k]) for k in ("right", "up", "forward"))
            assert np.allclose(cam["eye"], pos)
            assert np.allclose([r @ r, u @ u, f @ f], 1.0, atol=1e-12) and np.allclose([r @ u, r @ f, u @ f], 0.0, atol=1e-12)
            assert np.allclose(np.cross(r, u), -f, atol=1e-12)  # the handedness of look_from_z
            seen = total = 0
            for g in sc["grooms"]:
                p = g["pos"].reshape(-1, 3).astype(np.float64)[::7]
                xf = g["xform"] if g["xform"] is not None else np.array([[1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0]], np.float64)
                for M in np.asarray(xf, np.float64).reshape(-1, 3, 4)[::9]:
                    for q in (p @ M[:, :3].T + M[:, 3])[::5]:
                        o, valid = orc.project(cam, q)
                        if idx == 1:  # the lights stand outside the groom: all of it is in every map
                            assert valid and 0.0 <= o[0] <= 128.0 and 0.0 <= o[1] <= 128.0 and 0.0 < o[2] < 1.0, (idx, o)
                        elif valid:  # a light among the grooms cannot see behind itself (one perspective map per
                            assert o[2] < 1.0, (idx, o)  # light); what it sees is never beyond the far plane
                            seen += 1
                        total += 1
            assert idx == 1 or seen > 0.3 * total
