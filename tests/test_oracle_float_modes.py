"""Pins of the oracle's floating-point comparison modes (the paper's own arithmetic,
PAPER.md:106-108, with the thread-split sum of Listing 2's caption, :118-122).  CPU only.

The modes run the SAME quantised model with couplings (T)(Jq 2^-24).  In fp64 every sum of 25-bit couplings is exact, so
the fp64 mode must reproduce the pinned integer trajectory bit for bit: that pins the whole code path (indices, signs,
summation tree, acceptance, swaps) of the template, of which fp32 is the other instantiation.  For fp32 the rounding of
dE is bounded by the standard summation bound and the chain still samples the L=8 Boltzmann law."""
import math

import numpy as np
import pytest

from paper_1308_5426_b200 import inputs


@pytest.mark.parametrize("cfg,n,threads", [(0, 300, 1), (1, 60, 8)])
def test_fp64_mode_reproduces_the_integer_trajectory(oracle, cfg, n, threads):
    w = inputs.config(cfg)
    b = inputs.betas(w)
    oi = oracle.Oracle(w.L, w.q, w.sigma, 1, w.n_rep, b, w.seed)
    od = oracle.Oracle(w.L, w.q, w.sigma, 1, w.n_rep, b, w.seed)
    for k in (1, n):
        oi.sweeps(k, 1)
        od.sweeps_arith(k, 1, "fp64", threads)
        np.testing.assert_array_equal(oi.get_spins(), od.get_spins())
        np.testing.assert_array_equal(oi.energy(), od.energy())
        a, c = oi.observables(), od.observables()
        for f in a:
            np.testing.assert_array_equal(a[f], c[f], err_msg=f)
    with pytest.raises(ValueError):
        od.sweeps_arith(1, 1, "fp32")        # a context stays in the mode it entered


def test_fp32_delta_e_within_the_summation_bound_of_the_exact_value(oracle):
    L, q = 1024, 5
    o = oracle.Oracle(L, q, 0.8, 1, 1, [1.0], 11)
    Jsum = float(o.get_couplings().astype(np.int64).sum()) * 2.0 ** -24
    spins = o.get_spins()[0, 0]
    eps = 2.0 ** -24
    worst = 0.0
    for i in range(0, L, 37):
        b = 1 + (int(spins[i]) % q)          # a colour different from the site's own
        exact = o.delta_e(0, 0, i, b) * 2.0 ** -24
        assert o.delta_e_arith(0, 0, i, b, "fp64") == exact
        f32 = o.delta_e_arith(0, 0, i, b, "fp32")
        # couplings rounded to float (relative eps/2 each) + at most 8 + 7 additions on any path of the 128-way split
        bound = (0.5 + 15) * eps * Jsum
        assert abs(f32 - exact) <= bound, (i, f32, exact, bound)
        worst = max(worst, abs(f32 - exact))
    assert worst > 0.0                        # single precision does round here: the mode is not fp64 in disguise


def test_fp32_chain_samples_the_exact_boltzmann_law_L8_q3(oracle):
    from test_oracle_sweeps import exact_means
    Ts = [0.8, 1.5, 2.5]
    o = oracle.Oracle(8, 3, 0.5, 1, 3, [1 / T for T in Ts], 4242)
    o.sweeps_arith(2000, 1, "fp32")
    prev = o.observables()
    series = []
    for _ in range(48):
        o.sweeps_arith(2000, 1, "fp32")
        cur = o.observables()
        series.append((cur["sum_E"][0] - prev["sum_E"][0]) / (2000 * 2.0 ** 24))
        prev = cur
    series = np.array(series)
    mean, err = series.mean(axis=0), series.std(axis=0, ddof=1) / math.sqrt(len(series))
    for t, T in enumerate(Ts):
        x = exact_means(T)
        assert abs(mean[t] - x["E"]) < 3.5 * err[t] + 1e-5, (T, mean[t], x["E"], err[t])
        assert err[t] < 0.01 * abs(x["E"])
