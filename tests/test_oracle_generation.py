"""Pins of the oracle's hash, LOD (O1), generation (O2) and calcTangent (O3).

Each test checks the oracle against something other than itself: values Eq. 1-5 fix, closed
forms named by BASELINE.json north_star, a library routine (scipy CubicHermiteSpline),
invariants, or statistics. Citations are PAPER.md lines / DESIGN.md readings.
"""
import math

import numpy as np
import pytest
from scipy.interpolate import CubicHermiteSpline

from paper_2607_04230_b200 import synth


# ------------------------------------------------------------------------------- hash / roots
def test_pcg_is_injective_and_avalanches(orc):
    # the PCG RXS-M-XS output permutation is a bijection on 32-bit words: no collisions
    xs = np.arange(0, 1 << 16, dtype=np.uint64)
    ys = np.array([orc.pcg(int(x)) for x in xs], dtype=np.uint64)
    assert len(np.unique(ys)) == len(xs)
    # avalanche: flipping one input bit flips about half of the output bits
    flips = []
    for x in range(0, 4096, 7):
        for b in (0, 5, 13, 31):
            flips.append(bin(orc.pcg(x) ^ orc.pcg(x ^ (1 << b))).count("1"))
    assert 13.0 < np.mean(flips) < 19.0


def test_root_barycentrics_uniform(orc):
    g = synth.straight_prism(strands=40000)
    f = orc.Frame([g])
    B = np.array([f.root(0, i)[0] for i in range(40000)])
    assert (B >= 0).all() and (B <= 1).all()
    assert np.array_equal(B.sum(1), np.ones(len(B)))  # multiples of 2^-24: exact
    assert np.allclose(B.mean(0), 1 / 3, atol=0.005)  # uniform on the triangle => mean 1/3 each
    # chi-square over the 16 congruent sub-triangles of a 4x4 barycentric subdivision
    i = np.minimum((B[:, 1] * 4).astype(int), 3)
    j = np.minimum((B[:, 2] * 4).astype(int), 3)
    up = (B[:, 1] * 4 - i) + (B[:, 2] * 4 - j) > 1.0
    cell = {}
    for a, b, u in zip(i, j, up):
        cell[(a, b, bool(u))] = cell.get((a, b, bool(u)), 0) + 1
    counts = np.array(list(cell.values()), float)
    assert len(counts) == 16
    chi2 = ((counts - counts.mean()) ** 2 / counts.mean()).sum()
    assert chi2 < 37.7  # chi2(15 dof) 99.9th percentile


def test_root_lies_on_scalp_triangle(orc):
    # north_star invariant: root vertices lie on the scalp triangle
    sc = synth.config(1)
    g = sc["grooms"][0]
    f = orc.Frame([g])
    for i in range(0, 1024, 37):
        b, tri = f.root(0, i)
        v, _ = f.strand(0, i, 17)
        X0 = g["pos"][0][g["idx"][tri]].astype(np.float64)
        assert np.allclose(v[0, :3], b @ X0, atol=1e-15)
        n = np.cross(X0[1] - X0[0], X0[2] - X0[0])
        assert abs(np.dot(v[0, :3] - X0[0], n / np.linalg.norm(n))) < 1e-15


# ------------------------------------------------------------------------------- O1: Eq. 1-5
@pytest.mark.parametrize("L,N,delta,want", [
    (1.0, 37, 0.0, 37), (1.0, 37, 0.999, 37),    # L = 1 => N_LOD = N for any delta (clamp)
    (0.0, 37, 0.5, 1),                            # L = 0 => lower clamp
    (0.5, 37, 0.0, 19), (0.5, 37, 0.5, 19),       # ceil(18.5), ceil(18.75)
    (0.12, 469, 0.5, 57),                         # ceil(0.12 * 469.5 = 56.34)
    (0.25, 8, 0.0, 2), (0.3, 0, 0.2, 0),
])
def test_eq1_strand_count(orc, L, N, delta, want):
    # Eq. 1
    assert orc.lod_counts(L, N, delta, 9, 127)[0] == want


@pytest.mark.parametrize("L,Lv,craw,C", [
    (1.0, 9, 127, 65),     # floor(127) ; 2^floor(log2 126) + 1
    (0.5, 9, 89, 65),      # floor(0.7071 * 127 = 89.8)
    (0.25, 9, 63, 33),     # floor(63.5)
    (0.0625, 9, 31, 17),   # floor(31.75)
    (0.01, 9, 12, 9),      # floor(12.7)
    (0.0, 13, 13, 9),      # C_layers bounds C_raw only (R14)
    (0.0, 3, 3, 3),
])
def test_eq4_eq5_control_points(orc, L, Lv, craw, C):
    # Eq. 4-5
    _, got_raw, got_c = orc.lod_counts(L, 10, 0.0, Lv, 127)
    assert (got_raw, got_c) == (craw, C)


def test_control_points_capped_by_c_full(orc):
    assert orc.lod_counts(1.0, 10, 0.0, 9, 33)[2] == 33  # R14: C = min(C, C_full)


def test_lod_frame_invariants(orc):
    sc = synth.config(3, scale=0.02, res_scale=0.25)
    g = sc["grooms"][0]
    f = orc.Frame([g])
    n_full = int(g["strands_per_tri"].sum())
    # lambda <= 0: LOD and culling off (R14)
    f.lod(sc["camera"], 0.0)
    t, L = f.table()
    assert f.n_strands == n_full and (t[:, 1] == 49).all() and np.array_equal(t[:, 0], g["strands_per_tri"])
    prev = None
    for lam in (0.5, 1.0, 2.0, 4.0, 8.0, 1000.0):
        f.lod(sc["camera"], lam)
        t, L = f.table()
        assert t[:, 0].sum() == f.n_strands  # strands generated == sum of N_LOD
        assert (t[:, 0] <= g["strands_per_tri"]).all()
        vis = L >= 0
        # north_star: strand count = roots x LOD fraction (Eq. 1: within the ceil and delta < 1)
        want = L[vis].astype(np.float64) * g["strands_per_tri"][vis]
        got = t[vis, 0].astype(np.float64)
        ok = (got >= np.floor(want)) & (got <= np.ceil(want) + 1) | (got == 1)
        assert ok.all()
        # scans
        assert np.array_equal(t[:, 2], np.concatenate([[0], np.cumsum(t[:, 0])[:-1]]))
        assert np.array_equal(t[:, 3], np.concatenate([[0], np.cumsum(t[:, 0].astype(np.int64) * t[:, 1])[:-1]]))
        if prev is not None:
            assert (t[:, 0] >= prev).all()  # monotone in lambda
        prev = t[:, 0].copy()
    assert f.n_strands == n_full  # huge lambda => L = 1 everywhere visible
    # monotone in 1/distance
    last = None
    for d in (8.0, 2.0, 0.5):
        sc2 = synth.config(3, scale=0.02, res_scale=0.25, distance=d)
        f.lod(sc2["camera"], 2.0)
        if last is not None:
            assert f.n_strands >= last
        last = f.n_strands


def test_offscreen_bundle_is_culled(orc):
    # PAPER.md:120 "Bundles with AABBs laying entirely outside the viewport are frustum-culled"
    g = synth.straight_prism(strands=8)
    cam = synth.look_from_z((10.0, 0.0, 0.0), 1.0, 64, 64)  # groom is 10 m to the left
    f = orc.Frame([g])
    f.lod(cam, 3.0)
    assert f.n_strands == 0
    cam = synth.look_from_z((0.0, 0.1, -3.0), 1.0, 64, 64)  # eye at z = -2 looking down -z: groom behind
    f.lod(cam, 3.0)
    assert f.n_strands == 0
    cam = synth.look_from_z((0.0, 0.1, 0.0), 1.0, 64, 64)
    f.lod(cam, 3.0)
    assert f.n_strands > 0


@pytest.mark.parametrize("W,H", [(640, 360), (300, 500)])
@pytest.mark.parametrize("a,b,h,lv", [(0.02, 0.02, 0.05, 7),    # tall bundle: the extent comes from the layers
                                      (0.3, 0.02, 0.004, 3)])   # wide bundle: the extent comes from the root triangle
def test_eq2_eq3_closed_form_of_L(orc, W, H, a, b, h, lv):
    """Eq. 2-3: L = clamp(||AABB_max - AABB_min|| / R_y * lambda) with the AABB over ALL layers'
    projected vertices, the 2-D diagonal in pixels and R_y = the vertical resolution. A flat prism facing the camera
    has every cage vertex at the same depth d, so the box is (f_px a / d) x (f_px (b + (Lv-1) h) / d) pixels."""
    d, lam = 2.0, 0.8
    g = synth.flat_prism(a, b, h, lv)
    ext_y = b + (lv - 1) * h
    cam = synth.look_from_z((0.5 * a, 0.5 * ext_y, 0.0), d, W, H)
    f = orc.Frame([g])
    f.lod(cam, lam)
    t, L = f.table()
    fpx = 0.5 * H / math.tan(0.5 * synth.VFOV)
    want = math.hypot(fpx * a / d, fpx * ext_y / d) / H * lam
    assert 0.05 < want < 0.5
    assert abs(float(L[0]) - want) < 1e-6
    # the mistakes this must catch: /W instead of /R_y, one axis instead of the diagonal, the root layer only
    assert abs(math.hypot(fpx * a / d, fpx * ext_y / d) / W * lam - want) > 1e-3
    assert abs(max(fpx * a / d, fpx * ext_y / d) / H * lam - want) > 1e-5
    assert abs(math.hypot(fpx * a / d, fpx * b / d) / H * lam - want) > 1e-4
    # and Eq. 1 on that L (delta < 1): N_LOD within one strand of L N
    assert abs(int(t[0, 0]) - want * 64) <= 1.0 + 1e-6


def test_near_plane_straddle_full_detail_or_culled(orc):
    """DESIGN.md R13 (PAPER.md:114-120 is silent on vertices behind the camera): a bundle with SOME cage vertices
    behind the near plane gets L = 1 whatever lambda says; one with ALL of them behind is culled."""
    g = synth.straddle_prism(n_layers=5, dz=0.5)  # layers at z = 0, 0.5, 1, 1.5, 2
    N = int(g["strands_per_tri"][0])
    f = orc.Frame([g])
    lam = 0.05
    f.lod(synth.look_from_z((0.1, 0.0, 0.0), 6.0, 96, 64), lam)  # whole cage in front: small L, few strands
    t, L = f.table()
    assert 0.0 < L[0] < 0.2 and 0 < t[0, 0] < N // 4
    f.lod(synth.look_from_z((0.1, 0.0, 0.0), 1.3, 96, 64), lam)  # eye at z = 1.3: layers 3, 4 are behind it
    t, L = f.table()
    assert L[0] == 1.0 and t[0, 0] == N
    assert t[0, 1] == orc.lod_counts(1.0, N, 0.0, 5, 17)[2] == 17  # Eq. 4-5 at L = 1, capped by C_full (R14)
    f.lod(synth.look_from_z((0.1, 0.0, 0.0), 0.55, 96, 64), lam)  # eye at z = 0.55: only layer 0 (zv 0.55) is in front
    assert f.table()[1][0] == 1.0
    f.lod(synth.look_from_z((0.1, 0.0, 0.0), 0.05, 96, 64), lam)  # zv = 0.05 < near for layer 0, negative for the rest
    t, L = f.table()
    assert t[0, 0] == 0 and f.n_strands == 0


# ------------------------------------------------------------------------------- O2: base spline
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_straight_prism_is_the_interpolated_line(orc, axis):
    # north_star closed form: an unstyled straight strand through an axis-aligned prism lies
    # exactly on the interpolated line, uniformly in w
    lv, h = 5, 0.05
    g = synth.straight_prism(n_layers=lv, h=h, axis=axis, strands=16)
    f = orc.Frame([g])
    for sid in range(16):
        for C in (17, 9, 33, 12):
            v, tan = f.strand(0, sid, C)
            b, _ = f.root(0, sid)
            root = b @ g["pos"][0].astype(np.float64)
            w = np.arange(C) / (C - 1)
            want = root[None, :] + np.outer(w * (lv - 1) * h, np.eye(3)[axis])
            assert np.abs(v[:, :3] - want).max() < 1e-8  # cage stored in fp32: 0.05*i rounds at ~1e-9
            assert np.allclose(tan, np.eye(3)[axis][None, :], atol=1e-6)


def _random_cage(seed, lv=6):
    rng = np.random.default_rng(seed)
    X = np.zeros((lv, 3, 3))
    X[0] = rng.normal(size=(3, 3)) * 0.02
    for i in range(1, lv):
        X[i] = X[i - 1] + rng.normal(size=(3, 3)) * 0.01 + np.array([0.0, 0.05, 0.0])
    return dict(pos=X.astype(np.float32), ao=rng.uniform(0.2, 1.0, size=(lv, 3)).astype(np.float32),
                idx=np.array([[0, 1, 2]], np.uint32), strands_per_tri=np.array([8], np.uint32),
                xform=None, style=dict(spi=4, seed=3, ops=()))


def test_base_spline_matches_scipy_cubic_hermite(orc):
    # Hermite spline from positions + finite-difference tangents (R4 Catmull-Rom)
    g = _random_cage(11)
    lv = g["pos"].shape[0]
    f = orc.Frame([g])
    for sid in range(8):
        b, _ = f.root(0, sid)
        P = np.einsum("k,lkc->lc", b, g["pos"].astype(np.float64))
        m = np.zeros_like(P)
        m[0], m[-1] = P[1] - P[0], P[-1] - P[-2]
        m[1:-1] = 0.5 * (P[2:] - P[:-2])
        sp = CubicHermiteSpline(np.arange(lv), P, m, axis=0)
        for C in (21, 9, 33):
            v, tan = f.strand(0, sid, C)
            s = np.arange(C) / (C - 1) * (lv - 1)
            assert np.abs(v[:, :3] - sp(s)).max() < 1e-14
            d = sp(s, 1)
            d /= np.linalg.norm(d, axis=1, keepdims=True)
            assert np.abs(tan - d).max() < 1e-12
        # interpolates every layer point when C-1 is a multiple of Lv-1 (R5)
        v, _ = f.strand(0, sid, 4 * (lv - 1) + 1)
        assert np.abs(v[::4, :3] - P).max() < 1e-15
        # AO: barycentric in the layer, linear between layers (R25)
        ao_l = g["ao"].astype(np.float64) @ b
        assert np.abs(v[::4, 3] - ao_l).max() < 1e-15
        assert abs(v[2, 3] - 0.5 * (ao_l[0] + ao_l[1])) < 1e-15


def test_base_spline_is_linear_in_barycentrics(orc):
    # p(b) = sum_k b_k * (spline along cage edge k): Hermite and Catmull-Rom are linear in P
    g = _random_cage(5)
    lv = g["pos"].shape[0]
    f = orc.Frame([g])
    C = 21
    s = np.arange(C) / (C - 1) * (lv - 1)
    edge = []
    for k in range(3):
        P = g["pos"][:, k, :].astype(np.float64)
        m = np.zeros_like(P)
        m[0], m[-1] = P[1] - P[0], P[-1] - P[-2]
        m[1:-1] = 0.5 * (P[2:] - P[:-2])
        edge.append(CubicHermiteSpline(np.arange(lv), P, m, axis=0)(s))
    for sid in range(8):
        b, _ = f.root(0, sid)
        v, _ = f.strand(0, sid, C)
        assert np.abs(v[:, :3] - sum(b[k] * edge[k] for k in range(3))).max() < 1e-14


# ------------------------------------------------------------------------------- O2: styling
def _dist_to_axis_line(p, root, axis):
    d = p - root
    d[:, axis] = 0
    return np.linalg.norm(d, axis=1)


def test_curl_keeps_distance_r_from_base_curve(orc):
    # north_star closed form: a curl operator of radius r keeps its distance r from the base curve
    r, turns, C = 0.004, 3.0, 65
    g = synth.straight_prism(strands=8, ops=("curl",), curl_radius=r, curl_turns=turns, curl_ramp_w0=0.0)
    base = synth.straight_prism(strands=8)
    f, fb = orc.Frame([g]), orc.Frame([base])
    for sid in range(8):
        v, _ = f.strand(0, sid, C)
        vb, _ = fb.strand(0, sid, C)
        off = v[:, :3] - vb[:, :3]
        assert np.abs(np.linalg.norm(off, axis=1) - r).max() < 1e-9  # r is float(0.004)
        assert np.abs(off[:, 1]).max() < 1e-12  # perpendicular to the (y-axis) tangent
        ang = np.unwrap(np.arctan2(off[:, 2], off[:, 0]))
        assert abs(abs(ang[-1] - ang[0]) - 2 * math.pi * turns) < 1e-9  # advances 2*pi*turns
        assert np.allclose(np.diff(ang), np.diff(ang)[0], atol=1e-9)  # uniformly in w


def test_curl_ramp_anchors_the_root(orc):
    g = synth.straight_prism(strands=4, ops=("curl",), curl_radius=0.004, curl_turns=2.0, curl_ramp_w0=0.25)
    base = synth.straight_prism(strands=4)
    v, _ = orc.Frame([g]).strand(0, 1, 17)
    vb, _ = orc.Frame([base]).strand(0, 1, 17)
    d = np.linalg.norm(v[:, :3] - vb[:, :3], axis=1)
    assert d[0] == 0.0 and abs(d[2] - 0.002) < 1e-9 and np.allclose(d[4:], 0.004, atol=1e-9)


def test_twist_by_whole_turns_returns_tip(orc):
    base = synth.straight_prism(strands=4)
    vb, _ = orc.Frame([base]).strand(0, 2, 33)
    for turns in (1.0, 2.0):
        g = synth.straight_prism(strands=4, ops=("twist",), twist_turns=turns)
        v, _ = orc.Frame([g]).strand(0, 2, 33)
        assert np.abs(v[-1, :3] - vb[-1, :3]).max() < 1e-12
        assert np.abs(v[0, :3] - vb[0, :3]).max() == 0.0
        assert np.abs(v[8, :3] - vb[8, :3]).max() > 1e-4  # but it did rotate in between
        # rotation about the centre curve keeps the distance to it
        c = g["pos"].astype(np.float64).mean(1)  # centroid line of the straight prism
        dist = np.linalg.norm((v[:, :3] - vb[:, :3] * 0)[:, [0, 2]] - c[0][[0, 2]], axis=1)
        assert np.allclose(dist, dist[0], atol=1e-12)
    g = synth.straight_prism(strands=4, ops=("twist",), twist_turns=0.5)  # half turn: point reflection
    v, _ = orc.Frame([g]).strand(0, 2, 33)
    c = base["pos"].astype(np.float64)[0].mean(0)
    assert np.allclose(v[-1, [0, 2]] - c[[0, 2]], -(vb[-1, [0, 2]] - c[[0, 2]]), atol=1e-12)


def test_clump_full_strength_puts_tip_on_centre_curve(orc):
    g = synth.straight_prism(strands=4, ops=("clump",), clump_strength=1.0, clump_exp=1)
    v, _ = orc.Frame([g]).strand(0, 3, 17)
    c_tip = g["pos"].astype(np.float64)[-1].mean(0)
    assert np.abs(v[-1, :3] - c_tip).max() < 1e-9
    g2 = synth.straight_prism(strands=4, ops=("clump",), clump_strength=1.0, clump_exp=2)
    v2, _ = orc.Frame([g2]).strand(0, 3, 17)
    vb, _ = orc.Frame([synth.straight_prism(strands=4)]).strand(0, 3, 17)
    # w^2 pulls less than w in the interior: at w = 0.5 a quarter vs a half of the way
    c_mid = 0.5 * (g["pos"].astype(np.float64)[0].mean(0) + c_tip)
    assert np.allclose(v[8, [0, 2]], 0.5 * (vb[8, [0, 2]] + c_mid[[0, 2]]), atol=1e-9)
    assert np.allclose(v2[8, [0, 2]], 0.75 * vb[8, [0, 2]] + 0.25 * c_mid[[0, 2]], atol=1e-9)


def test_frizz_is_perpendicular_unit_variance_and_zero_at_root(orc):
    sigma, n = 0.001, 3000
    g = synth.straight_prism(strands=n, ops=("frizz",), frizz_sigma=sigma, frizz_ramp_w0=0.1, frizz_cells=8)
    base = synth.straight_prism(strands=n)
    f, fb = orc.Frame([g]), orc.Frame([base])
    offs = []
    for sid in range(n):
        v, _ = f.strand(0, sid, 17)  # 16 segments over 8 cells: even CPs are lattice points
        vb, _ = fb.strand(0, sid, 17)
        offs.append(v[:, :3] - vb[:, :3])
    offs = np.array(offs)
    assert np.abs(offs[:, :, 1]).max() < 1e-15  # perpendicular to T (the y axis)
    assert np.abs(offs[:, 0, :]).max() == 0.0  # zero at the root (ramp)
    lat = offs[:, 2::2, :][:, :, [0, 2]] / sigma  # lattice points beyond the ramp
    assert abs(lat.var() - 1.0) < 0.05 and abs(lat.mean()) < 0.03
    assert np.abs(lat).max() <= 510 / math.sqrt(21845) + 1e-9  # (sum of 4 hash bytes - 510) / sqrt(21845)


def test_all_ops_off_is_bit_identical_to_base(orc):
    g0 = synth.straight_prism(strands=4)
    g1 = synth.straight_prism(strands=4, ops=(), curl_radius=0.1, twist_turns=3.0, clump_strength=1.0, frizz_sigma=1.0)
    a, _ = orc.Frame([g0]).strand(0, 1, 17)
    b, _ = orc.Frame([g1]).strand(0, 1, 17)
    assert np.array_equal(a, b)


def test_instances_share_roots_and_transform_last(orc):
    sc = synth.config(5, scale=0.002, res_scale=0.1)
    g = sc["grooms"][0]
    f = orc.Frame([g])
    f.lod(sc["camera"], 0.0)
    f.generate()
    V = f.vertices_f64()
    n_inst = g["xform"].shape[0]
    per = V.shape[0] // n_inst
    base = dict(g)
    base["xform"] = None
    fb = orc.Frame([base])
    fb.lod(sc["camera"], 0.0)
    fb.generate()
    Vb = fb.vertices_f64()
    for q in (0, 7, 63):
        M = g["xform"][q].reshape(3, 4).astype(np.float64)
        want = Vb[:, :3] @ M[:, :3].T + M[:, 3]
        assert np.abs(V[q * per:(q + 1) * per, :3] - want).max() < 1e-12
        assert np.array_equal(V[q * per:(q + 1) * per, 3], Vb[:, 3])


# ------------------------------------------------------------------------------- O3
def test_calc_tangent_three_cases(orc):
    # PAPER.md:353-359 verbatim: root n(next-curr), tip n(curr-prev), else n(next-prev)
    p, c, n = np.array([0.0, 0, 0]), np.array([1.0, 2, 0]), np.array([4.0, 2, 0])
    assert np.allclose(orc.calc_tangent(0, 5, p, c, n), [1, 0, 0])
    assert np.allclose(orc.calc_tangent(4, 5, p, c, n), np.array([1, 2, 0]) / math.sqrt(5))
    assert np.allclose(orc.calc_tangent(2, 5, p, c, n), np.array([4, 2, 0]) / math.sqrt(20))
    assert abs(np.linalg.norm(orc.calc_tangent(2, 5, p, c, n)) - 1) < 1e-15
