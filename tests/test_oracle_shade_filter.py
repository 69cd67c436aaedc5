"""Pins of the oracle's deferred shading (O6) and reconstruction filter (O7).

The shading model is a stand-in (R23: the paper gives no formulas), so it is pinned by
its own closed forms only — "parity unpinned" against the paper. The filter is pinned by closed
forms that follow from Eq. 9-10 and §3.3.2-3.3.3.
"""
import math

import numpy as np
import pytest

from paper_2607_04230_b200 import synth

EMPTY = 0xFFFFFFFFFFFFFFFF
W, H = 48, 32


def hand_frame(orc, verts, ao=1.0, n_strands=1, **style):
    """A frame whose vertex buffer is written by hand: `n_strands` strands of 5 vertices each."""
    st = dict(albedo_root=(0.5, 0.4, 0.3), albedo_tip=(0.5, 0.4, 0.3), roughness=0.3, tilt=-0.05)
    st.update(style)
    g = synth.straight_prism(n_layers=2, strands=n_strands, spi=4, **st)
    f = orc.Frame([g])
    cam = synth.look_from_z((0.0, 0.0, 0.0), 1.0, W, H)
    f.lod(cam, 0.0)
    v = np.zeros((n_strands * 5, 4), np.float32)
    v[:, :3] = np.asarray(verts, np.float32).reshape(-1, 3)
    v[:, 3] = ao
    f.set_vertices_f32(v)
    return f, cam


def params(**over):
    p = dict(center_diameter_px=0.5, filter_radius=5, s_par=0.5, s_perp=0.15, sigma_c=0.9,
             tau_z=1.45e-3, tau_fly=5e-4, w_strip=0.5, lights=[], ambient_rgb=(0.2, 0.2, 0.2),
             k_d=0.4, k_R=0.25, k_TRT=0.5, background_rgb=(0.0, 0.0, 0.0), filter_on=True)
    p.update(over)
    return p


X_LINE = [(-0.2 + 0.1 * j, 0.0, 0.0) for j in range(5)]  # along +x through the origin, 1 m from the eye


def gbuf_with(words):
    g = np.full((H, W, 2), EMPTY, np.uint64)
    for (x, y, layer), w in words.items():
        g[y, x, layer] = w
    return g


# ------------------------------------------------------------------------------- O6 shading
def test_no_lights_gives_ambient_times_ao_times_albedo(orc):
    f, cam = hand_frame(orc, X_LINE, ao=0.6, albedo_root=(0.2, 0.4, 0.6), albedo_tip=(1.0, 0.8, 0.2))
    w_root = orc.pack(0.9, 0, 0, 0.0)
    w_tip = orc.pack(0.9, 0, 3, 1.0)
    w_mid = orc.pack(0.9, 0, 2, 0.0)
    f.set_gbuffer(gbuf_with({(5, 5, 0): w_root, (6, 5, 0): w_tip, (7, 5, 0): w_mid}))
    col = f.shade(cam, params())
    assert np.allclose(col[5, 5], 0.6 * 0.2 * np.float32([0.2, 0.4, 0.6]), atol=1e-12)  # w = 0: root albedo
    assert np.allclose(col[5, 6], 0.6 * 0.2 * np.float32([1.0, 0.8, 0.2]), atol=1e-12)  # w = 1: tip albedo
    mid = 0.5 * (np.float32([0.2, 0.4, 0.6]).astype(float) + np.float32([1.0, 0.8, 0.2]))
    assert np.allclose(col[5, 7], 0.6 * 0.2 * mid, atol=1e-12)
    assert (col[0, 0] == 0).all()
    f2, cam = hand_frame(orc, X_LINE, ao=0.0)
    f2.set_gbuffer(gbuf_with({(5, 5, 0): w_mid}))
    assert (f2.shade(cam, params())[5, 5] == 0).all()  # AO = 0 and no lights => black


def test_light_parallel_to_tangent_adds_nothing(orc):
    f, cam = hand_frame(orc, X_LINE)
    f.set_gbuffer(gbuf_with({(5, 5, 0): orc.pack(0.9, 0, 2, 0.0)}))  # hit at the origin, T = +x
    amb = f.shade(cam, params())[5, 5]
    lit = f.shade(cam, params(lights=[((3.0, 0.0, 0.0), (5.0, 5.0, 5.0))]))[5, 5]
    assert np.allclose(lit, amb, atol=1e-12)  # cos_i = 0


def test_perpendicular_light_and_view_closed_form(orc):
    beta, tilt = 0.3, -0.05
    f, cam = hand_frame(orc, X_LINE, roughness=beta, tilt=tilt)
    f.set_gbuffer(gbuf_with({(5, 5, 0): orc.pack(0.9, 0, 2, 0.0)}))  # p = origin, V = +z, T = +x
    prm = params(lights=[((0.0, 2.0, 0.0), (4.0, 2.0, 1.0))])
    got = f.shade(cam, prm)[5, 5]
    b, tl = float(np.float32(beta)), float(np.float32(tilt))
    MR = math.exp(-(tl ** 2) / (2 * b * b))
    MT = math.exp(-((1.5 * tl) ** 2) / (8 * b * b))
    alb = np.float32([0.5, 0.4, 0.3]).astype(float)
    E = np.array([4.0, 2.0, 1.0]) / 4.0  # inverse-square at 2 m
    kd, kR, kT = (float(np.float32(v)) for v in (0.4, 0.25, 0.5))
    want = float(np.float32(0.2)) * alb + E * (kd * alb + kR * MR + kT * MT * alb)  # cos_i = 1, theta_h = 0
    assert np.allclose(got, want, atol=1e-12)


def test_shading_uses_calc_tangent_of_styled_polyline(orc):
    # a bent polyline: the tangent at an interior vertex is n(next - prev), so a
    # light along that direction contributes nothing at t = 0 of that segment
    bent = [(-0.2, 0, 0), (-0.1, 0, 0), (0, 0, 0), (0.1, 0.1, 0), (0.2, 0.3, 0)]
    f, cam = hand_frame(orc, bent)
    f.set_gbuffer(gbuf_with({(5, 5, 0): orc.pack(0.9, 0, 2, 0.0)}))
    d = np.array([0.2, 0.1, 0.0]) / math.hypot(0.2, 0.1)  # v3 - v1
    amb = f.shade(cam, params())[5, 5]
    lit = f.shade(cam, params(lights=[(tuple(3 * d), (5.0, 5.0, 5.0))]))[5, 5]
    assert np.allclose(lit, amb, atol=1e-9)
    lit2 = f.shade(cam, params(lights=[((0.0, 0.0, 3.0), (5.0, 5.0, 5.0))]))[5, 5]
    assert (lit2 > amb + 1e-3).all()


def test_screen_tangent_of_winning_segment(orc):
    diag = [(-0.2 + 0.1 * j, 0.2 - 0.1 * j, 0.0) for j in range(5)]  # +x, -y in world => +x, +y on screen
    f, cam = hand_frame(orc, diag)
    f.set_gbuffer(gbuf_with({(5, 5, 0): orc.pack(0.9, 0, 1, 0.5), (5, 5, 1): orc.pack(0.9, 0, 1, 0.5),
                             (9, 9, 1): orc.pack(0.9, 0, 3, 0.2)}))
    f.shade(cam, params())
    t = f.tangents()
    s = math.sqrt(0.5)
    assert np.allclose(t[5, 5], [s, s, s, s], atol=1e-6)
    assert np.allclose(t[9, 9], [0, 0, s, s], atol=1e-6)  # conservative-only pixel has T_A only


# ------------------------------------------------------------------------------- O7 filter
def line_frame(orc, pattern, y=16, x0=6, n=36, **kw):
    """Horizontal strand on screen; pattern(i) -> 'c' centre+cons hit, 'a' cons-only, None empty."""
    f, cam = hand_frame(orc, X_LINE, **kw)
    words = {}
    w = orc.pack(0.9, 0, 2, 0.0)
    for i in range(n):
        k = pattern(i)
        if k == "c":
            words[(x0 + i, y, 0)] = w
        if k in ("c", "a"):
            words[(x0 + i, y, 1)] = w
    f.set_gbuffer(gbuf_with(words))
    return f, cam


def test_constant_colour_full_line_is_unchanged(orc):
    f, cam = line_frame(orc, lambda i: "c")
    col = f.shade(cam, params())
    out = f.filter(cam, params())
    assert np.allclose(out[16, 6:42, :3], col[16, 6:42], atol=1e-12)  # normalised sum of a constant
    assert np.allclose(out[16, 6:42, 3], 1.0)  # every strip pixel is centre-hit => alpha = 1
    assert (out[15] == 0).all() and (out[17] == 0).all()


def test_radius_zero_is_identity(orc):
    f, cam = line_frame(orc, lambda i: "c" if i % 2 == 0 else "a")
    col = f.shade(cam, params())
    out = f.filter(cam, params(filter_radius=0, background_rgb=(0.1, 0.2, 0.3)))
    assert np.allclose(out[16, 6:42:2, :3], col[16, 6:42:2], atol=1e-12) and (out[16, 6:42:2, 3] == 1).all()
    assert np.allclose(out[16, 7:42:2, :3], [0.1, 0.2, 0.3], atol=1e-7) and (out[16, 7:42:2, 3] == 0).all()
    assert np.allclose(out[3, 3], [0.1, 0.2, 0.3, 0.0], atol=1e-7)


@pytest.mark.parametrize("r", [3, 5, 7])
def test_alternating_line_alpha_closed_form(orc, r):
    # PAPER.md:176 alpha = H_center / H_cons over the tangent-aligned strip (R18): on a horizontal
    # line of alternating centre-hit / conservative-only pixels the strip is the row itself
    f, cam = line_frame(orc, lambda i: "c" if i % 2 == 0 else "a")
    col = f.shade(cam, params())
    out = f.filter(cam, params(filter_radius=r))
    a_centre = (2 * (r // 2) + 1) / (2 * r + 1)
    a_prom = 2 * ((r + 1) // 2) / (2 * r + 1)
    xs = np.arange(6 + 8, 42 - 8)
    for x in xs:
        want = a_centre if (x - 6) % 2 == 0 else a_prom
        assert abs(out[16, x, 3] - want) < 1e-12, (x, out[16, x, 3], want)
        # promoted pixels borrow the neighbours' colour; composited over black
        assert np.allclose(out[16, x, :3], want * col[16, 6], atol=1e-12)


def test_mirror_image_gives_mirrored_output(orc):
    pat = lambda i: "c" if i in (0, 1, 4, 9, 10, 11, 20) else ("a" if i in (2, 3, 12, 15, 30) else None)
    f, cam = line_frame(orc, pat, x0=6, n=36)
    f.shade(cam, params())
    out = f.filter(cam, params())
    f2, cam = line_frame(orc, lambda i: pat(35 - i), x0=6, n=36)
    f2.shade(cam, params())
    out2 = f2.filter(cam, params())
    assert np.allclose(out[:, 6:42], out2[:, 6:42][:, ::-1], atol=1e-12)


def test_bilateral_weights_closed_form(orc):
    # Eq. 10 on three centre pixels: P, Q1 two pixels along the tangent, Q2 one pixel across
    f, cam = hand_frame(orc, [X_LINE, [(x, 0.05, 0) for x, _, _ in X_LINE]], n_strands=2,
                        albedo_root=(0.2, 0.2, 0.2), albedo_tip=(1.0, 1.0, 1.0))
    wP = orc.pack(0.9, 0, 0, 0.0)   # root albedo
    wQ1 = orc.pack(0.9, 0, 3, 1.0)  # tip albedo
    wQ2 = orc.pack(0.9, 1, 1, 1.0)  # in between
    words = {(20, 16, 0): wP, (20, 16, 1): wP, (22, 16, 0): wQ1, (22, 16, 1): wQ1, (20, 17, 0): wQ2, (20, 17, 1): wQ2}
    f.set_gbuffer(gbuf_with(words))
    prm = params(s_par=0.5, s_perp=0.3, sigma_c=0.9)
    col = f.shade(cam, prm)
    out = f.filter(cam, prm)
    CP, C1, C2 = col[16, 20], col[16, 22], col[17, 20]
    sp, sq, sc = (5 * float(np.float32(0.5))), (5 * float(np.float32(0.3))), float(np.float32(0.9))
    w1 = math.exp(-4.0 / sp ** 2) * math.exp(-((CP - C1) ** 2).sum() / sc ** 2)
    w2 = math.exp(-1.0 / sq ** 2) * math.exp(-((CP - C2) ** 2).sum() / sc ** 2)
    want = (CP + w1 * C1 + w2 * C2) / (1 + w1 + w2)
    # strip (half-width 0.5 around the row): P and Q1 are in it, Q2 (d_perp = 1) is not => alpha = 2/2
    assert abs(out[16, 20, 3] - 1.0) < 1e-12
    assert np.allclose(out[16, 20, :3], want, atol=1e-12)


def test_depth_rejection(orc):
    # neighbours whose depth differs by more than 1.45e-3 are rejected before weighting
    f, cam = hand_frame(orc, X_LINE, albedo_root=(0.2, 0.2, 0.2), albedo_tip=(1.0, 1.0, 1.0))
    wP = orc.pack(0.9, 0, 0, 0.0)
    near_ok = orc.pack(0.9 + 1.40e-3, 0, 3, 1.0)
    too_far = orc.pack(0.9 + 1.50e-3, 0, 3, 1.0)
    for wQ, contributes in ((near_ok, True), (too_far, False)):
        f.set_gbuffer(gbuf_with({(20, 16, 0): wP, (20, 16, 1): wP, (22, 16, 0): wQ, (22, 16, 1): wQ}))
        col = f.shade(cam, params())
        out = f.filter(cam, params())
        same = np.allclose(out[16, 20, :3], col[16, 20], atol=1e-12)
        assert same != contributes


def test_flyaway_strand_in_front_gets_alpha_one(orc):
    # a closer strand in the conservative layer (depth mismatch >= 5e-4) is blended on
    # top of the centre-hit colour and the output opacity is 1
    f, cam = hand_frame(orc, [X_LINE, [(x, 0.0, 0.3) for x, _, _ in X_LINE]], n_strands=2,
                        albedo_root=(0.2, 0.2, 0.2), albedo_tip=(0.2, 0.2, 0.2))
    back = orc.pack(0.9, 0, 2, 0.0)
    front = orc.pack(0.9 - 6e-4, 1, 2, 0.0)
    nearly = orc.pack(0.9 - 4e-4, 1, 2, 0.0)
    words = {}
    for x in range(10, 40):
        words[(x, 16, 0)] = back
        words[(x, 16, 1)] = back
    words[(25, 16, 1)] = front
    f.set_gbuffer(gbuf_with(words))
    f.shade(cam, params())
    out = f.filter(cam, params())
    assert out[16, 25, 3] == 1.0
    words[(25, 16, 1)] = nearly  # below the fly-away threshold: ordinary centre pixel
    f.set_gbuffer(gbuf_with(words))
    f.shade(cam, params())
    out2 = f.filter(cam, params())
    assert abs(out2[16, 25, 3] - 1.0) < 1e-12  # all strip pixels are centre hits anyway
    # genuine fly-away over a sparse background: alpha would be < 1 without the rule
    words = {(x, 16, 0): back for x in range(10, 40, 2)}
    words.update({(x, 16, 1): back for x in range(10, 40)})
    words[(24, 16, 1)] = front
    f.set_gbuffer(gbuf_with(words))
    f.shade(cam, params())
    out3 = f.filter(cam, params())
    assert out3[16, 24, 3] == 1.0 and out3[16, 26, 3] < 0.6


def test_flyaway_blend_of_two_different_colours(orc):
    """PAPER.md:175-176 / DESIGN.md R21: C = alpha_f C_f + (1 - alpha_f) C_c, alpha = 1, where C_c is the centre
    accumulation and (C_f, alpha_f) the accumulation around the conservative sample. Two strands whose hits differ in
    colour (root albedo at w = 0 against tip albedo at w = 1) and lie farther apart in depth than tau_z, so each
    accumulation sees one constant colour and alpha_f is a plain count: the blend is fixed by hand."""
    root, tip = (0.2, 0.4, 0.6), (1.0, 0.8, 0.2)
    f, cam = hand_frame(orc, [X_LINE, [(x, 0.0, 0.3) for x, _, _ in X_LINE]], n_strands=2, ao=0.5,
                        albedo_root=root, albedo_tip=tip)
    back = orc.pack(0.9, 0, 0, 0.0)            # strand 0 at w = 0
    front = orc.pack(0.9 - 3e-3, 1, 3, 1.0)    # strand 1 at w = 1, 3e-3 nearer: > tau_fly and > tau_z
    words = {}
    for x in range(10, 41):
        words[(x, 16, 0)] = back
        words[(x, 16, 1)] = back
    for x in (23, 24, 27):                     # centre hits of the front strand
        words[(x, 16, 0)] = front
        words[(x, 16, 1)] = front
    for x in (21, 22, 25, 26, 28, 29, 30):     # pixels the front strand only touches
        words[(x, 16, 1)] = front
    f.set_gbuffer(gbuf_with(words))
    col = f.shade(cam, params())
    out = f.filter(cam, params())
    amb = float(np.float32(0.2))
    C_c = 0.5 * amb * np.float32(root).astype(float)
    C_f = 0.5 * amb * np.float32(tip).astype(float)
    assert np.allclose(col[16, 25], C_c, atol=1e-12) and np.allclose(col[16, 24], C_f, atol=1e-12)
    # strip around (25, 16) along the row, x = 20 .. 30, classes relative to the FRONT depth: 23, 24, 27 centre;
    # 21, 22, 25, 26, 28, 29, 30 conservative-only; 20 (back in both layers) rejected by depth => alpha_f = 3 / 10
    alpha_f = 3.0 / 10.0
    want = alpha_f * C_f + (1.0 - alpha_f) * C_c
    assert out[16, 25, 3] == 1.0
    assert np.allclose(out[16, 25, :3], want, atol=1e-12)
    assert np.abs((1.0 - alpha_f) * C_f + alpha_f * C_c - want).max() > 1e-2   # swapped alpha would show
    assert np.abs(want - C_c).max() > 1e-2 and np.abs(want - C_f).max() > 1e-2


def test_filter_off_passes_centre_colour(orc):
    f, cam = line_frame(orc, lambda i: "c" if i % 3 == 0 else "a")
    col = f.shade(cam, params())
    out = f.filter(cam, params(filter_on=False, background_rgb=(0.3, 0.3, 0.3)))
    assert np.allclose(out[16, 6:42:3, :3], col[16, 6:42:3]) and (out[16, 6:42:3, 3] == 1).all()
    assert np.allclose(out[16, 7, :3], 0.3, atol=1e-7) and out[16, 7, 3] == 0


def test_end_to_end_alpha_and_energy_bounds(orc):
    sc = synth.config(1, scale=0.25, res_scale=0.5)
    f = orc.Frame(sc["grooms"])
    out = f.render(sc["camera"], sc["params"], 0.0)
    G = f.gbuffer()
    col = f.shade(sc["camera"], sc["params"])
    assert (out[..., 3] >= 0).all() and (out[..., 3] <= 1).all()
    empty = (G[..., 0] == np.uint64(EMPTY)) & (G[..., 1] == np.uint64(EMPTY))
    assert (out[empty] == 0).all()
    # a normalised average never exceeds the brightest shaded pixel
    assert out[..., :3].max() <= col.max() + 1e-12
    assert (out[~empty][:, 3] > 0).mean() > 0.5
