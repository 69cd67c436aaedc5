"""Pins of the oracle's paper payload (DESIGN.md R-payload; "G-buffer compression": 24-bit depth,
position reconstructed from the depth, uvw styling coordinates, octahedral tangent, "all float values except for
depth are quantized as either uint8 or uint6").

What fixes it without another implementation: the octahedral map is a bijection of the unit sphere onto the square
(known codes of the axes, round trip within the grid's angular resolution, decode always unit length); the depth
bits of the resolve do not depend on the payload, so they must equal those of the separately pinned strand-id
resolve (O4) pixel by pixel; and every quantised field must agree, within its quantisation step, with the value
the strand-id word of the same pixel leads to through the pinned O2 / O3 / O6 code (tangent, w, AO, root
coordinates, hit position).
"""
import numpy as np
import pytest

from paper_2607_04230_b200 import synth

NONE40 = np.uint64((1 << 40) - 1)


def _frame(orc, sc, payload):
    f = orc.Frame(sc["grooms"])
    f.set_payload_mode(payload)
    f.lod(sc["camera"], sc["lam"])
    f.generate()
    f.set_vertices_f32(f.vertices_f32())
    return f


# ------------------------------------------------------------------------------------------- octahedral code
def test_oct_codes_of_the_axes(orc):
    # p = T / (|x|+|y|+|z|); upper hemisphere maps to the inner diamond, code = round((p/2 + 1/2) 255)
    assert orc.oct_encode([0, 0, 1]) == (128, 128)
    assert orc.oct_encode([1, 0, 0]) == (255, 128)
    assert orc.oct_encode([-1, 0, 0]) == (0, 128)
    assert orc.oct_encode([0, 1, 0]) == (128, 255)
    assert orc.oct_encode([0, -1, 0]) == (128, 0)
    # -z folds to the four corners of the square; with px = py = +0 it is the (+, +) corner
    assert orc.oct_encode([0, 0, -1]) == (255, 255)
    # the diagonal of the upper octant: p = (1/3, 1/3) -> round((1/6 + 1/2) 255) = 170
    s = 1 / np.sqrt(3)
    assert orc.oct_encode([s, s, s]) == (170, 170)
    # and its mirror below the equator: folded to (1 - 1/3, 1 - 1/3) -> round((1/3 + 1/2) 255) = 213 (212.5 + .5)
    ox, oy = orc.oct_encode([s, s, -s])
    assert abs(ox - 213) <= 1 and ox == oy


def test_oct_round_trip_within_grid_resolution(orc):
    rng = np.random.default_rng(3)
    T = rng.standard_normal((4000, 3))
    T /= np.linalg.norm(T, axis=1, keepdims=True)
    worst = 0.0
    for t in T.astype(np.float32):
        d = orc.oct_decode(*orc.oct_encode(t)).astype(np.float64)
        assert abs(np.linalg.norm(d) - 1.0) < 1e-6
        worst = max(worst, float(np.degrees(np.arccos(np.clip(np.dot(d, t / np.linalg.norm(t)), -1, 1)))))
    # grid step 2/255 in the square: half a step per axis is < 0.5 degrees on the sphere near the poles of the
    # map and about twice that at the stretched diamond edges
    assert worst < 1.0, worst


def test_oct_decode_covers_the_sphere_and_is_sign_symmetric(orc):
    # decode(255 - ox, oy) mirrors x up to the 1/255 asymmetry of the unorm grid around 127.5
    for ox, oy in [(10, 200), (128, 128), (77, 31), (250, 250)]:
        a = orc.oct_decode(ox, oy)
        b = orc.oct_decode(255 - ox, oy)
        assert np.allclose(a * np.array([-1, 1, 1], np.float32), b, atol=2e-6), (a, b)
    # every code decodes to a unit vector; the four corners are -z
    for ox, oy in [(0, 0), (255, 0), (0, 255), (255, 255)]:
        assert np.allclose(orc.oct_decode(ox, oy), [0, 0, -1], atol=1e-6)
    zs = [orc.oct_decode(ox, oy)[2] for ox in range(0, 256, 15) for oy in range(0, 256, 15)]
    assert min(zs) < -0.9 and max(zs) > 0.9


# ------------------------------------------------------------------------------------------- word layout
def test_payload_fields_closed_form_on_a_straight_vertical_strand(orc):
    # one strand along +y, AO = 1 (no AO array): tangent = +y -> (128, 255); w6 = round(63 (j + t)/(C-1)); ao6 = 63
    C = 9
    v = np.zeros((C, 4), np.float32)
    v[:, 1] = np.linspace(0, 0.2, C)
    v[:, 3] = 1.0
    a1, a2 = 3 << 20, 5 << 20  # 3/16, 5/16 -> round(63 * 3/16) = 12 (11.81), round(63 * 5/16) = 20 (19.69)
    for j, t in [(0, 0.0), (3, 0.5), (7, 1.0), (4, 0.25)]:
        p = orc.payload40(v, j, t, a1, a2)
        f = {k: int(x) for k, x in orc.unpack_payload(np.uint64(p)).items()}
        assert (f["ox"], f["oy"]) == (128, 255)
        assert f["w6"] == int(np.floor(63.0 * (j + t) / (C - 1) + 0.5))
        assert f["ao6"] == 63 and f["u6"] == 12 and f["v6"] == 20
        assert f["dq"] == 0  # orc_payload40 returns the low 40 bits only
    # AO ramp 0 -> 1 along the strand is interpolated linearly inside a segment
    v[:, 3] = np.linspace(0, 1, C)
    f = orc.unpack_payload(np.uint64(orc.payload40(v, 4, 0.5, a1, a2)))
    assert int(f["ao6"]) == int(np.floor(63.0 * 4.5 / 8 + 0.5))


def test_payload_tangent_follows_calc_tangent_on_a_bent_polyline(orc):
    # right-angle polyline in the xy plane: calcTangent at the corner is n(next - prev) = the
    # diagonal; root and tip are one-sided
    v = np.array([[0, 0, 0, 1], [1, 0, 0, 1], [1, 1, 0, 1]], np.float32)
    dec = lambda p: orc.oct_decode(*[int(x) for x in (orc.unpack_payload(np.uint64(p))["ox"], orc.unpack_payload(np.uint64(p))["oy"])])
    t_root = dec(orc.payload40(v, 0, 0.0, 0, 0))
    t_corner = dec(orc.payload40(v, 0, 1.0, 0, 0))
    t_tip = dec(orc.payload40(v, 1, 1.0, 0, 0))
    assert np.allclose(t_root, [1, 0, 0], atol=0.02)
    assert np.allclose(t_corner, np.array([1, 1, 0]) / np.sqrt(2), atol=0.02)
    assert np.allclose(t_tip, [0, 1, 0], atol=0.02)
    # halfway along the first segment: normalised mean of (1,0,0) and the diagonal = 22.5 degrees
    t_mid = dec(orc.payload40(v, 0, 0.5, 0, 0))
    assert abs(np.degrees(np.arctan2(t_mid[1], t_mid[0])) - 22.5) < 1.0


def test_root_codes_never_look_like_no_hit(orc):
    # folded roots have r1 + r2 <= 1, so u6 and v6 cannot both be 63: the payload of a hit is never all ones
    sc = synth.config(1)
    f = orc.Frame(sc["grooms"])
    n = int(sc["grooms"][0]["strands_per_tri"].sum())
    for i in range(0, n, 7):
        b, _ = f.root(0, i)
        u6 = int(np.floor(b[1] * 63 + 0.5))
        v6 = int(np.floor(b[2] * 63 + 0.5))
        assert u6 + v6 <= 64 and not (u6 == 63 and v6 == 63)


# ------------------------------------------------------------------------------------------- against the pinned O4 / O6
@pytest.fixture(scope="module")
def both(orc):
    sc = synth.config(2, scale=0.02, res_scale=0.25)  # curl + frizz, AO varies along the strand
    fid = _frame(orc, sc, False)
    fid.raster(sc["camera"], sc["params"])
    gid = fid.gbuffer().copy()
    fpp = _frame(orc, sc, True)
    fpp.raster(sc["camera"], sc["params"])
    gpp = fpp.gbuffer().copy()
    return sc, fid, gid, fpp, gpp


def test_depth_bits_equal_the_strand_id_resolve(both):
    sc, fid, gid, fpp, gpp = both
    # the min is taken on depth-major words: whatever rides in the low 40 bits, the winning depth is the same
    assert np.array_equal(gid >> np.uint64(40), gpp >> np.uint64(40))
    assert np.array_equal((gid & NONE40) == NONE40, (gpp & NONE40) == NONE40)
    assert ((gpp[..., 1] & NONE40) != NONE40).sum() > 2000


def test_fields_agree_with_what_the_strand_id_word_leads_to(orc, both):
    sc, fid, gid, fpp, gpp = both
    cam = sc["camera"]
    v = fid.vertices_f32()
    table, _ = fid.table()
    g = sc["grooms"][0]
    off = np.concatenate([[0], np.cumsum(g["strands_per_tri"])])
    hit = (gid[..., 0] & NONE40) != NONE40
    ys, xs = np.nonzero(hit)
    sel = np.random.default_rng(5).choice(len(ys), size=min(1500, len(ys)), replace=False)
    n_ok = 0
    worst_ang, worst_pos = 0.0, 0.0
    for y, x in zip(ys[sel], xs[sel]):
        wid, wpp = int(gid[y, x, 0]), int(gpp[y, x, 0])
        sid, j, t = (wid >> 16) & 0xFFFFFF, (wid >> 9) & 0x7F, (wid & 0x1FF) / 511.0
        tri = int(np.searchsorted(off, sid, side="right") - 1)
        nlod, C, _, vbase = [int(a) for a in table[tri]]
        k = sid - int(off[tri])
        s = v[vbase + k * C: vbase + (k + 1) * C].astype(np.float64)
        f = {kk: int(a) for kk, a in orc.unpack_payload(np.uint64(wpp)).items()}
        # w, AO: within one code of the exact values at the id word's (j, t) (t itself is a 9-bit code)
        ok = abs(f["w6"] - 63.0 * (j + t) / (C - 1)) <= 1.0
        ok &= abs(f["ao6"] - 63.0 * np.clip((1 - t) * s[j, 3] + t * s[j + 1, 3], 0, 1)) <= 1.0
        # root coordinates: half a code
        b, _ = fid.root(0, sid)
        ok &= abs(f["u6"] - 63.0 * b[1]) <= 0.5 + 1e-9 and abs(f["v6"] - 63.0 * b[2]) <= 0.5 + 1e-9
        # tangent: calcTangent (pinned, O3) interpolated at t, against the decoded code
        def ct(i):
            out = np.zeros(3)
            P = lambda q: np.ascontiguousarray(s[min(max(q, 0), C - 1), :3])
            orc.lib().orc_calc_tangent(i, C, P(i - 1).ctypes.data, P(i).ctypes.data, P(i + 1).ctypes.data, out.ctypes.data)
            return out
        T = (1 - t) * ct(j) + t * ct(j + 1)
        T /= np.linalg.norm(T)
        d = orc.oct_decode(f["ox"], f["oy"]).astype(np.float64)
        ang = float(np.degrees(np.arccos(np.clip(np.dot(d, T), -1, 1))))
        ok &= ang < 1.5
        # hit position (pinned O2 vertices) against the position rebuilt from the depth at the pixel centre: the hit
        # is the closest point of the segment to the pixel centre, at most rho <= 0.5 px away on screen
        pos = (1 - t) * s[j, :3] + t * s[j + 1, :3]
        zn = (wpp >> 40) / 16777215.0
        far, near = cam["far_z"], cam["near_z"]
        zv = (far * near / (far - near)) / (far / (far - near) - zn)
        fpx = 0.5 * cam["height"] / np.tan(0.5 * cam["vfov_y"])
        cx, cy = (x + 0.5 - 0.5 * cam["width"]) / fpx, (0.5 * cam["height"] - (y + 0.5)) / fpx
        rec = np.asarray(cam["eye"], float) + zv * (cx * np.asarray(cam["right"], float) + cy * np.asarray(cam["up"], float)
                                                    + np.asarray(cam["forward"], float))
        err_px = np.linalg.norm(rec - pos) * fpx / zv
        ok &= err_px < 0.75
        if ok:
            n_ok += 1
            worst_ang, worst_pos = max(worst_ang, ang), max(worst_pos, err_px)
    # two segments at the same 24-bit depth in one pixel are resolved by the payload bits, which differ between the
    # two layouts: allow a small share of such ties
    assert n_ok >= 0.98 * len(sel), (n_ok, len(sel))
    assert worst_ang < 1.5 and worst_pos < 0.75


def test_payload_shading_and_screen_tangent_close_to_the_exact_ones(orc, both):
    sc, fid, gid, fpp, gpp = both

    def orc_decode(w):
        return orc.oct_decode((w >> 32) & 0xFF, (w >> 24) & 0xFF).astype(np.float64)

    def orc_project(cc, p, out):
        import ctypes as C
        orc.lib().orc_project(C.byref(cc), p.ctypes.data, out.ctypes.data)

    cid = fid.shade(sc["camera"], sc["params"])
    tid = fid.tangents()
    cpp = fpp.shade(sc["camera"], sc["params"])
    tpp = fpp.tangents()
    hit = (gid[..., 0] & NONE40) != NONE40
    # 6-bit w / AO and a sub-degree tangent error move the colour by a few percent at most
    d = np.abs(cid - cpp)[hit]
    assert np.median(d) < 0.01 and np.percentile(d, 99) < 0.08, (np.median(d), np.percentile(d, 99))
    # screen tangent = projected direction of the decoded tangent at the rebuilt position: finite difference of the
    # pinned pinhole projection (orc_project) along the tangent, in double
    cam = sc["camera"]
    from oracle import make_camera
    import ctypes as C
    cc = make_camera(cam)
    far, near = cam["far_z"], cam["near_z"]
    fpx = 0.5 * cam["height"] / np.tan(0.5 * cam["vfov_y"])
    ys, xs = np.nonzero(hit)
    for i in np.random.default_rng(9).choice(len(ys), size=300, replace=False):
        y, x = int(ys[i]), int(xs[i])
        w = int(gpp[y, x, 0])
        T = orc_decode(w)
        zv = (far * near / (far - near)) / (far / (far - near) - (w >> 40) / 16777215.0)
        cx, cy = (x + 0.5 - 0.5 * cam["width"]) / fpx, (0.5 * cam["height"] - (y + 0.5)) / fpx
        pos = np.asarray(cam["eye"], float) + zv * (cx * np.asarray(cam["right"], float) + cy * np.asarray(cam["up"], float)
                                                    + np.asarray(cam["forward"], float))
        eps = 1e-2 * zv
        pa, pb = np.zeros(4, np.float32), np.zeros(4, np.float32)
        a = (pos - eps * T).astype(np.float32)
        b = (pos + eps * T).astype(np.float32)
        orc_project(cc, a, pa)
        orc_project(cc, b, pb)
        d = (pb[:2] - pa[:2]).astype(np.float64)
        if np.linalg.norm(d) < 0.5:  # tangent along the view ray: direction undefined
            continue
        d /= np.linalg.norm(d)
        assert abs(float(np.dot(d, tpp[y, x, :2]))) > np.cos(np.radians(0.5)), (x, y, d, tpp[y, x])
    # against the strand-id mode's chord direction: same up to sign and up to the bend of the strand inside one
    # segment (a curl of 3 turns over 32 segments turns ~34 degrees per segment)
    dots = np.abs((tid[..., :2] * tpp[..., :2]).sum(-1))[hit]
    assert np.median(dots) > np.cos(np.radians(6.0)) and np.percentile(dots, 2) > np.cos(np.radians(30.0)), \
        (np.median(dots), np.percentile(dots, 2))
    # and the filter runs unchanged on the payload G-buffer
    out = fpp.filter(sc["camera"], sc["params"])
    oid = fid.filter(sc["camera"], sc["params"])
    # (the strip that estimates alpha follows the screen tangent, which differs by the bend inside a segment)
    assert ((out[..., 3] > 0) == (oid[..., 3] > 0)).mean() > 0.97
    assert np.abs(out[..., :3] - oid[..., :3]).mean() < 0.03


def test_payload_shade_needs_exactly_one_groom(orc):
    sc = synth.config(4, scale=0.002, res_scale=0.1)
    f = _frame(orc, sc, True)
    f.raster(sc["camera"], sc["params"])
    from oracle import make_camera, make_params
    import ctypes as C
    c, p = make_camera(sc["camera"]), make_params(sc["params"])
    assert orc.lib().orc_frame_shade(f.h, C.byref(c), C.byref(p)) == -4  # five grooms in the mask
    f.set_pass(1 << 2)
    f.lod(sc["camera"], sc["lam"])
    f.generate()
    f.set_vertices_f32(f.vertices_f32())
    f.raster(sc["camera"], sc["params"])
    assert orc.lib().orc_frame_shade(f.h, C.byref(c), C.byref(p)) == 0
