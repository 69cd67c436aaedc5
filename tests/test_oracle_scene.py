"""Pins of the oracle's scene input (DESIGN.md R-scene; "reads the existing depth buffer ...
blended into the main render target", 208-210 "keeping depth").

What the mathematics fixes: the resolve is an elementwise 64-bit min, and min is associative, so drawing the
hair into a seeded buffer must equal min(hair-only buffer, seed) word by word; a scene in front of all hair
leaves only the scene; a scene at the far end changes nothing but the composite's background.
"""
import numpy as np
import pytest

from paper_2607_04230_b200 import synth

PAYLOAD_NONE = np.uint64((1 << 40) - 1)
EMPTY = np.uint64(0xFFFFFFFFFFFFFFFF)


def _frame(orc, sc):
    f = orc.Frame(sc["grooms"])
    f.lod(sc["camera"], sc["lam"])
    f.generate()
    f.set_vertices_f32(f.vertices_f32())
    return f


def _seed(zn):
    """R8 quantisation of a depth in fp32, payload all ones."""
    z = np.clip(zn.astype(np.float32), np.float32(0), np.float32(1))
    q = (z * np.float32(16777215.0) + np.float32(0.5)).astype(np.float32)
    dq = np.minimum(q.astype(np.uint64), np.uint64(0xFFFFFE))
    return (dq << np.uint64(40)) | PAYLOAD_NONE


@pytest.fixture(scope="module")
def base(orc):
    sc = synth.config(1, scale=0.5)
    f = _frame(orc, sc)
    f.raster(sc["camera"], sc["params"])
    g = f.gbuffer().copy()
    f.shade(sc["camera"], sc["params"])
    out = f.filter(sc["camera"], sc["params"]).copy()
    return sc, g, out


def test_seeded_resolve_is_min_of_hair_and_seed(orc, base):
    sc, g0, _ = base
    H, W = g0.shape[:2]
    hit = g0[..., 1] != EMPTY
    zn_hair = ((g0[..., 1] >> np.uint64(40)).astype(np.float64) / 16777215.0)[hit]
    rng = np.random.default_rng(7)
    # a bumpy wall through the middle of the hair's depth range: some hits in front, some behind
    yy, xx = np.mgrid[0:H, 0:W]
    zn = (np.median(zn_hair) + 0.5 * (zn_hair.max() - zn_hair.min()) * np.sin(xx / 9.0) * np.cos(yy / 13.0)
          + 1e-4 * rng.standard_normal((H, W))).astype(np.float32)
    f = _frame(orc, sc)
    f.set_scene(zn=zn)
    f.raster(sc["camera"], sc["params"])
    g1 = f.gbuffer()
    seed = _seed(zn)
    want = np.minimum(g0, seed[..., None])
    assert np.array_equal(g1, want)
    behind = hit & (g1[..., 1] == seed)
    front = hit & (g1[..., 1] != seed)
    assert behind.sum() > 100 and front.sum() > 100  # the wall really cuts through the groom


def test_scene_in_front_hides_everything(orc, base):
    sc, g0, _ = base
    H, W = g0.shape[:2]
    rgb = np.random.default_rng(3).random((H, W, 3)).astype(np.float32)
    f = _frame(orc, sc)
    f.set_scene(zn=np.zeros((H, W), np.float32), rgb=rgb)
    cnt = f.raster(sc["camera"], sc["params"])
    g = f.gbuffer()
    assert ((g & PAYLOAD_NONE) == PAYLOAD_NONE).all() and ((g >> np.uint64(40)) == 0).all()
    assert cnt["cons"] > 0  # the hits were produced, they lost the min
    f.shade(sc["camera"], sc["params"])
    out = f.filter(sc["camera"], sc["params"])
    assert np.array_equal(out[..., :3], rgb.astype(np.float64)) and (out[..., 3] == 0).all()


def test_scene_at_far_end_only_changes_the_background(orc, base):
    sc, g0, out0 = base
    H, W = g0.shape[:2]
    rgb = np.random.default_rng(4).random((H, W, 3)).astype(np.float32)
    f = _frame(orc, sc)
    f.set_scene(zn=np.ones((H, W), np.float32), rgb=rgb)
    f.raster(sc["camera"], sc["params"])
    g = f.gbuffer()
    hit = g0 != EMPTY
    assert np.array_equal(g[hit], g0[hit])
    assert ((g[~hit] & PAYLOAD_NONE) == PAYLOAD_NONE).all()
    f.shade(sc["camera"], sc["params"])
    out = f.filter(sc["camera"], sc["params"])
    # same alpha and same hair colour C: out = alpha C + (1 - alpha) bg with bg the scene instead of the constant
    a = out0[..., 3:4]
    bg0 = np.asarray(sc["params"].get("background_rgb", (0, 0, 0)), dtype=np.float64)
    want = out0[..., :3] - (1 - a) * bg0 + (1 - a) * rgb.astype(np.float64)
    assert np.allclose(out[..., 3], out0[..., 3], atol=0) and np.abs(out[..., :3] - want).max() < 1e-12


def test_half_wall_leaves_the_other_half_alone(orc, base):
    sc, g0, out0 = base
    H, W = g0.shape[:2]
    zn = np.ones((H, W), np.float32)
    zn[:, : W // 2] = 0.0
    f = _frame(orc, sc)
    f.set_scene(zn=zn)
    f.raster(sc["camera"], sc["params"])
    g = f.gbuffer()
    assert ((g[:, : W // 2] & PAYLOAD_NONE) == PAYLOAD_NONE).all()
    hit = g0[:, W // 2:] != EMPTY
    assert np.array_equal(g[:, W // 2:][hit], g0[:, W // 2:][hit])
    f.shade(sc["camera"], sc["params"])
    out = f.filter(sc["camera"], sc["params"])
    r = sc["params"].get("filter_radius", 5)
    assert np.array_equal(out[:, W // 2 + r:], out0[:, W // 2 + r:])  # beyond the filter's reach of the wall
    assert (out[:, : W // 2, 3] == 0).all()


# ------------------------------------------------------------------ sequential per-groom passes (R-seq)
def _two_grooms(dz, dx=0.0):
    """config-1 groom twice: the copy shifted by (dx, 0, -dz) (farther from the camera on +z for dz > 0)."""
    sc = synth.config(1, scale=0.5)
    g0 = sc["grooms"][0]
    g1 = dict(g0)
    g1["pos"] = (g0["pos"] + np.array([dx, 0.0, -dz], np.float32)).astype(np.float32)
    g1["style"] = dict(g0["style"], seed=g0["style"]["seed"] + 17)
    sc["grooms"] = [g0, g1]
    sc["lam"] = [0.0, 0.0]
    return sc


def test_sequential_single_groom_equals_single_resolve(orc, base):
    sc, g0, out0 = base
    f = orc.Frame(sc["grooms"])
    out, g, dq = f.render_sequential(sc["camera"], sc["params"], sc["lam"])
    assert np.array_equal(g, g0) and np.array_equal(out, out0)
    assert np.array_equal(dq, (g0[..., 0] >> np.uint64(40)).astype(np.uint32))


def test_sequential_disjoint_grooms_equal_single_resolve(orc):
    """Two grooms far apart on screen do not interact: both orders of processing and the one-resolve frame
    give the same image."""
    sc = _two_grooms(dz=0.0, dx=0.6)
    sc["camera"] = synth.look_from_z((0.3, 0.05, 0.0), 1.0, 400, 160)
    f = orc.Frame(sc["grooms"])
    out_seq, _, _ = f.render_sequential(sc["camera"], sc["params"], sc["lam"])
    f2 = orc.Frame(sc["grooms"])
    out_one = f2.render(sc["camera"], sc["params"], sc["lam"])
    hit = out_one[..., 3] > 0
    cols = np.where(hit.any(0))[0]
    assert (np.diff(cols) > 2 * 7 + 2).any(), "the two grooms must be separated by more than the filter's reach"
    assert np.abs(out_seq - out_one).max() < 1e-6  # fp32 target between the passes
    f3 = orc.Frame(sc["grooms"][::-1])
    out_rev, _, _ = f3.render_sequential(sc["camera"], sc["params"], sc["lam"])
    assert np.abs(out_rev - out_one).max() < 1e-6


def test_sequential_groom_behind_an_opaque_one_is_rejected(orc):
    """Second groom = a copy 40 cm behind the first (more than the groom is deep): wherever the first pass left centre hits, every hit of the
    second pass is farther and loses against the kept depth in both layers, so those pixels keep pass 1's
    depth, colour and alpha."""
    sc = _two_grooms(dz=0.4)
    cam, prm = sc["camera"], sc["params"]
    f1 = orc.Frame(sc["grooms"][:1])
    out1 = f1.render(cam, prm, 0.0)
    g1 = f1.gbuffer()
    f = orc.Frame(sc["grooms"])
    out, g, dq = f.render_sequential(cam, prm, sc["lam"])
    c1 = (g1[..., 0] & PAYLOAD_NONE) != PAYLOAD_NONE
    # centre layer of pass 2 at pass-1 centre pixels: no hit, depth = pass 1's
    assert ((g[..., 0][c1] & PAYLOAD_NONE) == PAYLOAD_NONE).all()
    assert np.array_equal(dq[c1], (g1[..., 0][c1] >> np.uint64(40)).astype(np.uint32))
    # the second groom does show where the first left holes
    assert (((g[..., 0] & PAYLOAD_NONE) != PAYLOAD_NONE) & ~c1).sum() > 50
    # alpha only grows, and is the "over" of the two passes: 1 - (1 - a1)(1 - a2) >= a1
    assert (out[..., 3] >= out1[..., 3].astype(np.float32) - 1e-7).all() and out[..., 3].max() <= 1 + 1e-7
    # no word of pass 2 at those pixels (both layers were seeded with the kept depth), so pass 2 composites
    # nothing there: the pixel keeps pass 1's colour and alpha (through the fp32 target)
    assert ((g[..., 1][c1] & PAYLOAD_NONE) == PAYLOAD_NONE).all()
    assert np.array_equal(out[c1][:, :3], out1[c1][:, :3].astype(np.float32).astype(np.float64))
    assert np.array_equal(out[c1][:, 3], out1[c1][:, 3].astype(np.float32).astype(np.float64))


def test_groom_mask_only_changes_the_masked_bundles(orc):
    sc = _two_grooms(dz=0.05)
    f = orc.Frame(sc["grooms"])
    f.lod(sc["camera"], sc["lam"])
    t_all, _ = f.table()
    f.set_pass(0b10)
    f.lod(sc["camera"], sc["lam"])
    t_1, _ = f.table()
    n0 = len(t_all) // 2
    assert (t_1[:n0, :2] == 0).all() and np.array_equal(t_1[n0:, :2], t_all[n0:, :2])
    assert np.array_equal(t_1[n0:, 2], t_all[n0:, 2] - t_all[n0, 2])  # scans restart: only this pass's strands exist
    f.set_pass()
    f.lod(sc["camera"], sc["lam"])
    assert np.array_equal(f.table()[0], t_all)
