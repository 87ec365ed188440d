"""The reporting helpers of paper_1308_5426_b200/pt_math.py (Eqs. 10-12 on the exact integer accumulators, and the blocked
jack-knife that replaces the ALPS error analysis).  CPU only; the records come from the oracle."""
import math

import numpy as np

from paper_1308_5426_b200 import pt_math


def _snapshots(oracle, n_blocks=12, block=300):
    o = oracle.Oracle(8, 3, 0.5, 1, 3, [1 / 0.8, 1 / 1.5, 1 / 2.5], 99)
    o.sweeps(300, 1)
    snaps = [o.observables()]
    for _ in range(n_blocks):
        o.sweeps(block, 1)
        snaps.append(o.observables())
    return snaps


def test_wide_estimates_agree_with_the_plain_formulas(oracle):
    snaps = _snapshots(oracle)
    tot = pt_math.wide_sub(pt_math.widen(snaps[-1]), pt_math.widen(snaps[0]))
    est = pt_math.wide_estimates(tot, 8, 3)
    diff = pt_math.obs_diff(snaps[-1], snaps[0])
    d, c = pt_math.derived(diff, 8, 3), pt_math.cumulants(diff, 8, 3)
    for k in ("E_per_spin", "M", "M2"):
        np.testing.assert_allclose(est[k], d[k], rtol=1e-13)
    for k in ("U_E", "V_M"):
        np.testing.assert_allclose(est[k], c[k], rtol=1e-12)
    # Eq. 10 retyped: M = (q <Nmax>/L - 1)/(q - 1)
    n = diff["n_samples"].astype(float)
    np.testing.assert_allclose(est["M"], (3 * diff["sum_Nmax"] / (n * 8) - 1) / 2, rtol=1e-13)


def test_jackknife_of_a_mean_is_the_standard_error_of_the_block_means(oracle):
    snaps = _snapshots(oracle)
    blocks = pt_math.blocks_from_snapshots(snaps)
    est, err = pt_math.jackknife(blocks, lambda w: pt_math.wide_estimates(w, 8, 3)["E_per_spin"])
    means = np.stack([pt_math.wide_estimates(b, 8, 3)["E_per_spin"] for b in blocks])   # equal block lengths
    np.testing.assert_allclose(est, means.mean(axis=0), rtol=1e-12)
    np.testing.assert_allclose(err, means.std(axis=0, ddof=1) / math.sqrt(len(blocks)), rtol=1e-9)


def test_jackknife_of_the_cumulants_gives_finite_positive_errors(oracle):
    blocks = pt_math.blocks_from_snapshots(_snapshots(oracle))
    for key in ("U_E", "V_M"):
        est, err = pt_math.jackknife(blocks, lambda w, key=key: pt_math.wide_estimates(w, 8, 3)[key])
        assert np.isfinite(est).all() and (err > 0).all() and (err < 0.1).all()
    # the all-blocks estimate is the estimate of the summed record, not the mean of the block estimates (bias)
    tot = blocks[0]
    for b in blocks[1:]:
        tot = pt_math.wide_add(tot, b)
    est, _ = pt_math.jackknife(blocks, lambda w: pt_math.wide_estimates(w, 8, 3)["U_E"])
    np.testing.assert_allclose(est, pt_math.wide_estimates(tot, 8, 3)["U_E"], rtol=0)
