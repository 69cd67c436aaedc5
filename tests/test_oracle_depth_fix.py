"""Pins of the oracle's depth-comparison fix (§3.2.3, Eq. 6-8; DESIGN.md R-beta): beta =
N_remaining / N_total per groom from the LOD table, delta = -log(beta), and the depth a thinned groom is tested at."""
import math

import numpy as np

from paper_2607_04230_b200 import synth


def test_no_thinning_means_no_shift(orc):
    """'This shift is delta = 0 when no culling occurs (beta = 1)'. LOD off keeps every strand."""
    sc = synth.config(4, scale=0.01, res_scale=0.1)
    f = orc.Frame(sc["grooms"])
    f.lod(sc["camera"], [0.0])
    beta, delta, bmin = f.beta()
    assert np.all(beta == 1.0) and np.all(delta == 0.0) and bmin == 1.0
    for d in (0.0, 1e-3, 0.7, 12.0):
        assert orc.depth_fix(d, 0.0) == d


def test_beta_is_the_ratio_of_the_table_and_delta_its_log(orc):
    """beta per groom, re-derived here from the table the oracle returns and the input strand counts (Eq. 8's
    N_remaining / N_total over the drawn bundles), five grooms with different lambda; delta = -ln beta."""
    sc = synth.config(4, scale=0.05, res_scale=0.25)
    f = orc.Frame(sc["grooms"])
    f.lod(sc["camera"], sc["lam"])
    table, _ = f.table()
    beta, delta, bmin = f.beta()
    gid, worst = 0, 1.0
    for gi, g in enumerate(sc["grooms"]):
        npt = g["strands_per_tri"].astype(np.int64)
        nl = table[gid:gid + len(npt), 0].astype(np.int64)
        drawn = nl > 0
        assert drawn.any()
        want = nl[drawn].sum() / npt[drawn].sum()
        assert beta[gi] == want and 0.0 < beta[gi] <= 1.0
        assert delta[gi] == -math.log(want) and delta[gi] >= 0.0
        worst = min(worst, float((nl[drawn] / npt[drawn]).min()))
        gid += len(npt)
    assert bmin == worst
    assert (beta < 1.0).any()  # the far grooms are thinned
    # Eq. 1: N_LOD = clamp(ceil(L (N + delta)), 1, N) >= L N, so no drawn bundle keeps less than its L
    _, L = f.table()
    nl, N = table[:, 0].astype(np.float64), np.concatenate([g["strands_per_tri"] for g in sc["grooms"]]).astype(np.float64)
    d = nl > 0
    assert np.all(nl[d] / N[d] >= np.minimum(L[d], 1.0) - 1e-7)


def test_delta_grows_as_strands_are_removed(orc):
    """delta 'increases smoothly as more strands are removed (beta -> 0)': monotone in lambda and distance."""
    prev = None
    for lam in (8.0, 4.0, 2.0, 1.0, 0.5):
        sc = synth.config(3, scale=0.5, res_scale=0.1, distance=4.0, lam=lam)
        f = orc.Frame(sc["grooms"])
        f.lod(sc["camera"], sc["lam"])
        beta, delta, _ = f.beta()
        if prev is not None:
            assert beta[0] <= prev[0] and delta[0] >= prev[1]
        prev = (beta[0], delta[0])
    assert prev[0] < 0.5 and prev[1] > math.log(2.0)
    prev = None
    for dist in (1.0, 2.0, 4.0, 8.0):
        sc = synth.config(3, scale=0.5, res_scale=0.1, distance=dist, lam=2.0)
        f = orc.Frame(sc["grooms"])
        f.lod(sc["camera"], sc["lam"])
        beta, _, _ = f.beta()
        assert prev is None or beta[0] <= prev
        prev = beta[0]


def test_depth_fix_is_eq7(orc):
    """Eq. 6-7: visibility through the thinned groom at depth d equals visibility through the full groom at the
    corrected depth, V'(d) = exp(-sigma beta d) = V(d_eff) with d_eff = depth_fix(d, -ln beta); the shift is additive in
    log depth (Eq. 8) and composes: thinning by beta1 then beta2 = thinning by beta1 beta2."""
    rng = np.random.default_rng(5)
    for _ in range(200):
        sigma, beta, d = rng.uniform(0.1, 50.0), rng.uniform(0.02, 1.0), rng.uniform(1e-4, 3.0)
        delta = -math.log(beta)
        de = orc.depth_fix(d, delta)
        assert math.isclose(math.exp(-sigma * beta * d), math.exp(-sigma * de), rel_tol=1e-12)
        assert math.isclose(math.log(de), math.log(d) - delta, rel_tol=0, abs_tol=1e-12)
        assert de <= d
        b2 = rng.uniform(0.05, 1.0)
        assert math.isclose(orc.depth_fix(de, -math.log(b2)), orc.depth_fix(d, -math.log(beta * b2)), rel_tol=1e-12)


def test_culled_and_masked_bundles_do_not_count(orc):
    """A groom that is not drawn at all (masked: R-seq) reports beta = 1, delta = 0; bundles outside the frustum are
    not 'removed strands' (PAPER.md:120 vs 144)."""
    sc = synth.config(4, scale=0.02, res_scale=0.1)
    f = orc.Frame(sc["grooms"])
    f.set_pass(0b00101)
    f.lod(sc["camera"], sc["lam"])
    beta, delta, _ = f.beta()
    assert beta[1] == 1.0 and delta[1] == 0.0 and beta[3] == 1.0 and beta[4] == 1.0
    f.set_pass()
    # camera turned away from everything: all bundles frustum-culled
    cam = dict(sc["camera"], forward=(0.0, 0.0, 1.0), right=(-1.0, 0.0, 0.0))
    f.lod(cam, sc["lam"])
    beta, delta, bmin = f.beta()
    assert f.n_strands == 0 and np.all(beta == 1.0) and np.all(delta == 0.0) and bmin == 1.0
