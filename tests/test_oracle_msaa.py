"""Pins of the oracle's MSAA-k reference mode (DESIGN.md R-msaa).

k = 1 must reproduce the pinned centre layer of O4 and the filter-off image; every sample layer is checked
against a double-precision brute force written with other formulas (Liang-Barsky clip, vector projection);
closed-form alpha of a horizontal line from the pattern's offsets.
"""
import numpy as np
import pytest

from paper_2607_04230_b200 import synth
from test_oracle_raster import clip_segment_to_box, point_segment

EMPTY = np.uint64(0xFFFFFFFFFFFFFFFF)


def _frame(orc, sc):
    f = orc.Frame(sc["grooms"])
    f.lod(sc["camera"], sc["lam"])
    f.generate()
    f.set_vertices_f32(f.vertices_f32())
    return f


def test_one_sample_is_the_centre_layer_and_the_unfiltered_image(orc):
    sc = synth.config(1, scale=0.5)
    cam, prm = sc["camera"], dict(sc["params"], filter_on=False)
    f = _frame(orc, sc)
    f.raster(cam, prm)
    g = f.gbuffer().copy()
    f.shade(cam, prm)
    out_off = f.filter(cam, prm).copy()  # filter off: centre colour with alpha 1 over the background
    ms = f.raster_msaa(cam, prm, 1)
    assert ms.shape[0] == 1 and np.array_equal(ms[0], g[..., 0])
    assert np.array_equal(f.resolve_msaa(cam, prm), out_off)


@pytest.mark.parametrize("k", [2, 4, 8])
def test_sample_coverage_vs_double_precision_brute_force(orc, k):
    rng = np.random.default_rng(300 + k)
    eps = 1e-4
    offs = orc.MSAA_OFFSETS[k]
    assert len(offs) == k and len(set(offs)) == k and all(abs(x) < 8 and abs(y) < 8 for x, y in offs)
    assert abs(sum(x for x, _ in offs)) <= 0 and abs(sum(y for _, y in offs)) <= 0  # centred patterns
    n_checked = n_hit = 0
    for _ in range(25):
        a = rng.uniform(-2, 26, size=2)
        b = a + rng.normal(size=2) * rng.choice([0.3, 2.0, 12.0])
        rho = float(rng.choice([0.125, 0.25, 0.5]))
        a32, b32 = np.float32(a).astype(np.float64), np.float32(b).astype(np.float64)
        cover, tq = orc.segment_cover_msaa(a, b, rho, 24, 24, k)
        for s, (ox, oy) in enumerate(offs):
            for y in range(24):
                for x in range(24):
                    hit_out = clip_segment_to_box(a32, b32, x - eps, y - eps, x + 1 + eps, y + 1 + eps)
                    hit_in = clip_segment_to_box(a32, b32, x + eps, y + eps, x + 1 - eps, y + 1 - eps)
                    c = np.array([x + 0.5 + ox / 16.0, y + 0.5 + oy / 16.0])
                    t, dist = point_segment(c, a32, b32)
                    if hit_out == hit_in and abs(dist - rho) > eps:
                        assert bool(cover[s, y, x]) == (hit_in and dist < rho), (a, b, rho, s, x, y)
                        n_checked += 1
                    if cover[s, y, x]:
                        assert abs(tq[s, y, x] - t) < 1e-4
                        n_hit += 1
    assert n_checked > 25 * k * 500 and n_hit > 30 * k


def test_horizontal_line_alpha_closed_form(orc):
    """A horizontal segment through the pixel centres of row 5: sample s is hit iff |oy_s| / 16 <= rho."""
    for rho, k in ((0.125, 8), (0.25, 8), (0.5, 8), (0.2, 4), (0.25, 2), (0.3, 2)):
        cover, _ = orc.segment_cover_msaa((-3.0, 5.5), (40.0, 5.5), rho, 16, 12, k)
        want = np.array([abs(oy) / 16.0 <= rho for _, oy in orc.MSAA_OFFSETS[k]])
        assert (cover[:, 5, :] == want[:, None]).all()
        assert cover[:, :5].sum() == 0 and cover[:, 6:].sum() == 0


def test_resolve_is_the_mean_of_the_shaded_samples(orc):
    sc = synth.config(1, scale=0.5)
    cam, prm = sc["camera"], dict(sc["params"], background_rgb=(0.2, 0.4, 0.6))
    f = _frame(orc, sc)
    k = 4
    ms = f.raster_msaa(cam, prm, k)
    out = f.resolve_msaa(cam, prm)
    hit = ms != EMPTY
    assert np.allclose(out[..., 3], hit.mean(0), atol=0)
    # shade each layer on its own through the pinned O6: put layer s in the centre layer of a G-buffer
    acc = np.zeros(out.shape[:2] + (3,))
    for s in range(k):
        g = np.stack([ms[s], ms[s]], -1)
        f.set_gbuffer(g)
        acc += f.shade(cam, prm)
    bg = np.array([0.2, 0.4, 0.6], np.float32).astype(np.float64)
    want = acc / k + (1 - out[..., 3:4]) * bg
    assert np.abs(out[..., :3] - want).max() < 1e-12
    assert 0.02 < hit.mean() < 0.9


def test_more_samples_converge_to_coverage(orc):
    """Alpha of the 8-sample resolve correlates with the conservative layer's footprint and is never set where the
    conservative layer is empty (a sample hit requires the segment to cross the pixel)."""
    sc = synth.config(1, scale=0.5)
    cam, prm = sc["camera"], sc["params"]
    f = _frame(orc, sc)
    f.raster(cam, prm)
    cons = f.gbuffer()[..., 1] != EMPTY
    ms = f.raster_msaa(cam, prm, 8)
    any_hit = (ms != EMPTY).any(0)
    assert not (any_hit & ~cons).any()
    assert any_hit.sum() > 0.7 * cons.sum()
