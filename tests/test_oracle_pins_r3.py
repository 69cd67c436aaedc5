"""Pins added in round 3 for five oracle behaviours that survived mutation of oracle/hair_oracle.cpp:

  mutant                                                      -> test that fails on it
  promoted pixel accumulated WITH the colour term             -> test_promoted_pixel_is_the_plain_spatial_mean
  fly-away accumulation WITH the colour term                  -> test_flyaway_accumulation_is_the_plain_spatial_mean
  theta_h = (theta_i - theta_o) / 2 (or any wrong half-angle) -> test_lobes_sit_on_the_mirror_cone, test_half_angle_pi_over_8
  upper clamp of the projected width 1 px -> 2 px             -> test_width_clamp_upper_end_is_one_pixel
  styling frame from cage edge v0->v2 instead of v0->v1       -> test_styling_frame_is_built_from_edge_v0_v1
and a diagonal tangent in the strip test (all other filter pins are horizontal): test_strip_follows_a_diagonal_tangent.
"""
import math

import numpy as np

from paper_2607_04230_b200 import synth
from test_oracle_shade_filter import EMPTY, H, W, X_LINE, gbuf_with, hand_frame, params


# ------------------------------------------------------------------ O7: w_color = 1
ROOT, TIP = (0.2, 0.4, 0.6), (1.0, 0.8, 0.2)


def _two_colour_row(orc, extra=None):
    """Horizontal strand; centre hits alternate between the root colour (w = 0) and the tip colour (w = 1)."""
    f, cam = hand_frame(orc, [X_LINE, [(x, 0.0, 0.3) for x, _, _ in X_LINE]], n_strands=2, ao=0.5,
                        albedo_root=ROOT, albedo_tip=TIP)
    return f, cam


def test_promoted_pixel_is_the_plain_spatial_mean(orc):
    """PAPER.md:175 "For promoted pixels the color-similarity term is disabled (w_color = 1)". A conservative-only pixel
    P with centre hits of colour A at offsets -1, +2 and colour B at +1, -2 along a horizontal tangent: every pair of
    equal |offset| has equal spatial weight (Eq. 10 with d_perp = 0), so with w_color = 1 the result is exactly the
    plain mean (A + B) / 2 whatever sigma_par is. With the colour term left on (C_P of a promoted pixel is black, so A
    and B get different colour weights) it is not."""
    f, cam = _two_colour_row(orc)
    wA = orc.pack(0.9, 0, 0, 0.0)   # root colour
    wB = orc.pack(0.9, 0, 3, 1.0)   # tip colour
    cons = orc.pack(0.9, 0, 2, 0.0)
    words = {(25, 16, 1): cons}
    for dx, w in ((-1, wA), (2, wA), (1, wB), (-2, wB)):
        words[(25 + dx, 16, 0)] = w
        words[(25 + dx, 16, 1)] = w
    f.set_gbuffer(gbuf_with(words))
    col = f.shade(cam, params())
    A, B = col[16, 24], col[16, 26]
    assert np.abs(A - B).max() > 0.02
    for r in (3, 5):
        out = f.filter(cam, params(filter_radius=r, sigma_c=0.05))  # a sharp colour term, were it on
        alpha = 4.0 / 5.0  # strip = the row: four centre hits, one conservative-only (P itself)
        assert abs(out[16, 25, 3] - alpha) < 1e-12
        assert np.allclose(out[16, 25, :3], alpha * 0.5 * (A + B), atol=1e-12)
    # the same geometry seen from a CENTRE pixel of colour A does use the colour term: B is suppressed
    words[(25, 16, 0)] = wA
    words[(25, 16, 1)] = wA
    f.set_gbuffer(gbuf_with(words))
    f.shade(cam, params())
    out = f.filter(cam, params(sigma_c=0.05))
    assert np.abs(out[16, 25, :3] - A).max() < 0.05 * np.abs(0.5 * (A + B) - A).max()


def test_flyaway_accumulation_is_the_plain_spatial_mean(orc):
    """PAPER.md:175-176 / DESIGN.md R21: the accumulation around the conservative sample of a fly-away pixel has
    w_color = 1 too. Front strand (3e-3 nearer: beyond tau_fly and tau_z) with centre hits of colour A at -1, +2 and B
    at +1, -2 around P; P's own centre hit belongs to the back strand (colour K). C = alpha_f (A + B)/2 + (1 - alpha_f) K
    with alpha_f = 4/5; with the colour term on (C_P = K = A's colour, far from B) the mean would tilt towards A."""
    f, cam = _two_colour_row(orc)
    back = orc.pack(0.9, 0, 0, 0.0)             # K: the root colour (== A), back strand
    fA = orc.pack(0.9 - 3e-3, 1, 0, 0.0)
    fB = orc.pack(0.9 - 3e-3, 1, 3, 1.0)
    fcons = orc.pack(0.9 - 3e-3, 1, 2, 0.0)
    words = {(25, 16, 0): back, (25, 16, 1): fcons}
    for dx, w in ((-1, fA), (2, fA), (1, fB), (-2, fB)):
        words[(25 + dx, 16, 0)] = w
        words[(25 + dx, 16, 1)] = w
    f.set_gbuffer(gbuf_with(words))
    col = f.shade(cam, params())
    A, B, K = col[16, 24], col[16, 26], col[16, 25]
    out = f.filter(cam, params(sigma_c=0.05))
    alpha_f = 4.0 / 5.0
    assert out[16, 25, 3] == 1.0
    # the centre accumulation sees only P itself at the back depth (the front hits are rejected by tau_z): C_c = K
    assert np.allclose(out[16, 25, :3], alpha_f * 0.5 * (A + B) + (1 - alpha_f) * K, atol=1e-12)
    assert np.abs(np.linalg.norm(K - A) - np.linalg.norm(K - B)) > 1e-3  # K is not equidistant: a colour term would show


def test_strip_follows_a_diagonal_tangent(orc):
    """Eq. 9 with T = (1, 1)/sqrt 2: d_perp of offset (dx, dy) is |dx - dy| / sqrt 2, so the strip of
    half-width 0.5 holds exactly the diagonal dx == dy (neighbouring diagonals are 0.707 away). Centre hits on the
    diagonal at even steps, conservative-only at odd steps: alpha is the count ratio ON THE DIAGONAL; hits placed on the
    row and the column of P (which a horizontal or vertical strip would count) must not change it."""
    diag = [(-0.2 + 0.1 * j, 0.2 - 0.1 * j, 0.0) for j in range(5)]  # +x, +y on screen
    f, cam = hand_frame(orc, diag)
    w = orc.pack(0.9, 0, 1, 0.5)
    words = {}
    for i in range(-8, 9):
        if i % 2 == 0:
            words[(24 + i, 16 + i, 0)] = w
        words[(24 + i, 16 + i, 1)] = w
    f.set_gbuffer(gbuf_with(words))
    f.shade(cam, params())
    r = 5
    out = f.filter(cam, params(filter_radius=r))
    want = (2 * (r // 2) + 1) / (2 * r + 1)
    assert abs(out[16, 24, 3] - want) < 1e-12
    for dx in (-3, -2, 2, 3):  # centre hits on P's row and column: outside the diagonal strip
        words[(24 + dx, 16, 0)] = w
        words[(24 + dx, 16, 1)] = w
        words[(24, 16 + dx, 0)] = w
        words[(24, 16 + dx, 1)] = w
    f.set_gbuffer(gbuf_with(words))
    f.shade(cam, params())
    assert abs(f.filter(cam, params(filter_radius=r))[16, 24, 3] - want) < 1e-12


# ------------------------------------------------------------------ O6: the half angle (DESIGN R23)
def _lit(orc, word, light_pos, beta=0.3, tilt=-0.05):
    f, cam = hand_frame(orc, X_LINE, roughness=beta, tilt=tilt)
    f.set_gbuffer(gbuf_with({(5, 5, 0): word}))
    L = (8.0, 8.0, 8.0)
    return f.shade(cam, params(lights=[(tuple(light_pos), L)]))[5, 5], f.shade(cam, params())[5, 5]


def _model(amb_rgb, cos_i, th, d2, beta, tilt):
    b, tl = float(np.float32(beta)), float(np.float32(tilt))
    MR = math.exp(-((th + tl) ** 2) / (2 * b * b))
    MT = math.exp(-((th - 1.5 * tl) ** 2) / (8 * b * b))
    alb = np.float32([0.5, 0.4, 0.3]).astype(float)
    kd, kR, kT = (float(np.float32(v)) for v in (0.4, 0.25, 0.5))
    return amb_rgb + (8.0 / d2) * cos_i * (kd * alb + kR * MR + kT * MT * alb)


def test_lobes_sit_on_the_mirror_cone(orc):
    """theta_h = (theta_i + theta_o) / 2 with both inclinations measured from the plane normal to T: when the light's
    inclination MIRRORS the view's (theta_i = -theta_o) the half angle is 0 and the lobes take the values of the
    perpendicular configuration; when it EQUALS the view's, theta_h = theta_o. Hit at the strand's tip (0.2, 0, 0), eye
    at (0, 0, 1): the view is oblique, sin theta_o = -0.2 / sqrt(1.04). A sign error in theta_h swaps the two cases."""
    P = np.array([0.2, 0.0, 0.0])
    word = orc.pack(0.9, 0, 3, 1.0)  # segment 3, t = 1: the last vertex; T = +x
    sin_o = -0.2 / math.sqrt(1.04)
    th_o = math.asin(sin_o)
    cos_o = math.cos(th_o)
    mirror, amb = _lit(orc, word, P + 2.0 * np.array([-sin_o, cos_o, 0.0]))
    same, _ = _lit(orc, word, P + 2.0 * np.array([sin_o, cos_o, 0.0]))
    assert np.allclose(mirror, _model(amb, cos_o, 0.0, 4.0, 0.3, -0.05), atol=1e-9)
    assert np.allclose(same, _model(amb, cos_o, th_o, 4.0, 0.3, -0.05), atol=1e-9)
    assert np.abs(mirror - same).max() > 1e-2  # the two cases are told apart


def test_half_angle_pi_over_8(orc):
    """Light 45 degrees off the normal plane (towards +T), view perpendicular to T: theta_h = pi / 8, cos_i = cos 45."""
    word = orc.pack(0.9, 0, 2, 0.0)  # the origin
    s = math.sqrt(0.5)
    got, amb = _lit(orc, word, 2.0 * np.array([s, s, 0.0]))
    assert np.allclose(got, _model(amb, s, math.pi / 8, 4.0, 0.3, -0.05), atol=1e-9)
    got2, _ = _lit(orc, word, 2.0 * np.array([-s, s, 0.0]))  # towards -T: theta_h = -pi / 8, the tilt breaks the symmetry
    assert np.allclose(got2, _model(amb, s, -math.pi / 8, 4.0, 0.3, -0.05), atol=1e-9)
    assert np.abs(got - got2).max() > 1e-3


# ------------------------------------------------------------------ O4: R9's upper clamp (centre within conservative)
def test_width_clamp_upper_end_is_one_pixel(orc):
    """R9: the projected width is clamped to [0.25, 1] px. A strand 2 cm wide projects to ~6 px here; its centre layer
    must be EXACTLY the centre layer of center_diameter_px = 1.0 (word for word), hold more hits than the 0.46 px
    strand, and stay inside the conservative layer (a centre radius above 0.5 px could claim pixels the segment never
    touches: the pixel square reaches only 0.707 px from its centre)."""
    sc = synth.config(1, scale=0.1, res_scale=0.5)

    def centre_layer(width_world, diameter):
        g = dict(sc["grooms"][0])
        g["style"] = dict(g["style"], width_world=width_world)
        f = orc.Frame([g])
        f.lod(sc["camera"], 0.0)
        f.generate()
        c = f.raster(sc["camera"], dict(sc["params"], center_diameter_px=diameter))
        return f.gbuffer().copy(), c

    G_wide, c_wide = centre_layer(2e-2, 0.3)
    G_one, c_one = centre_layer(0.0, 1.0)
    G_mid, c_mid = centre_layer(1.5e-3, 0.3)
    assert np.array_equal(G_wide, G_one) and c_wide["center"] == c_one["center"]
    assert c_wide["center"] > c_mid["center"]
    hit0, hit1 = G_wide[..., 0] != np.uint64(EMPTY), G_wide[..., 1] != np.uint64(EMPTY)
    assert hit0.sum() > 100 and not (hit0 & ~hit1).any()
    assert c_wide["center"] <= c_wide["cons"]


# ------------------------------------------------------------------ O2: the styling frame
def test_styling_frame_is_built_from_edge_v0_v1(orc):
    """O2.5: N = cage edge v0->v1 orthogonalised against the base tangent, B = T x N. straight_prism has v0->v1 = +x,
    v0->v2 = +z and T = +y, so N = +x and B = y x x = -z: with ramp 0 the curl offset of the ROOT vertex (w = 0) is
    r (cos phi, 0, -sin phi), phi = 2 pi u, u = the strand's curl phase (top 24 bits of hash stream 3, itself pinned
    against the published PCG values in test_oracle_generation). A frame from v0->v2 would give r (sin phi, 0, cos phi)."""
    r = 0.004
    g = synth.straight_prism(strands=8, ops=("curl",), curl_radius=r, curl_turns=3.0, curl_ramp_w0=0.0)
    base = synth.straight_prism(strands=8)
    f, fb = orc.Frame([g]), orc.Frame([base])
    rr = float(np.float32(r))
    seen = []
    for sid in range(8):
        v, _ = f.strand(0, sid, 17)
        vb, _ = fb.strand(0, sid, 17)
        off = v[0, :3] - vb[0, :3]
        phi = 2 * math.pi * ((orc.hash3(g["style"]["seed"], sid, 3) >> 8) / 16777216.0)
        assert np.allclose(off, rr * np.array([math.cos(phi), 0.0, -math.sin(phi)]), atol=1e-9), (sid, off, phi)
        seen.append(phi)
    assert np.ptp(seen) > 1.0  # the phases differ: the check is not vacuous
