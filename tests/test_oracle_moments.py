"""Pins for the higher-moment accumulators (sum E^4 as 256 bits, sum Nmax^3, sum Nmax^4 as 128 bits) and the
cumulants of Eqs. 11-12: exact agreement with Python big-integer arithmetic on a recorded time
series, and the exact Boltzmann values of the full enumeration at L=8, q=3."""
import itertools
import math

import numpy as np
import pytest

from paper_1308_5426_b200 import inputs

SCALE = 2 ** 24


def _e4(ob, t):
    return sum(int(ob["sum_E4"][0, t, k]) << (64 * k) for k in range(4))


def _n4(ob, t):
    return (int(ob["sum_Nmax4_hi"][0, t]) << 64) + int(ob["sum_Nmax4_lo"][0, t])


@pytest.mark.parametrize("L,q,sigma", [(64, 3, 0.5), (1024, 8, 0.3)])
def test_accumulators_equal_big_integer_sums_of_the_time_series(oracle, L, q, sigma):
    """Without swaps the configuration of a slot after sweep s is the one that was sampled (A15): the accumulators must
    equal the sums of E^k and Nmax^k over the recorded series, in exact integer arithmetic (E^4 ~ 2^150 at L=1024:
    all four limbs and their carries are exercised)."""
    n_rep = 3
    o = oracle.Oracle(L, q, sigma, 1, n_rep, inputs.geometric_betas(0.7, 2.5, n_rep), 11)
    s1 = [0] * n_rep; s2 = [0] * n_rep; s4 = [0] * n_rep
    m1 = [0] * n_rep; m2 = [0] * n_rep; m3 = [0] * n_rep; m4 = [0] * n_rep
    n = 25 if L > 100 else 200
    for _ in range(n):
        o.sweeps(1, 0)
        E, sp = o.energy()[0], o.get_spins()[0]
        for t in range(n_rep):
            e = int(E[t])
            nm = max(int((sp[t] == k).sum()) for k in range(1, q + 1))
            s1[t] += e; s2[t] += e ** 2; s4[t] += e ** 4
            m1[t] += nm; m2[t] += nm ** 2; m3[t] += nm ** 3; m4[t] += nm ** 4
    ob = o.observables()
    for t in range(n_rep):
        assert int(ob["n_samples"][0, t]) == n
        assert int(ob["sum_E"][0, t]) == s1[t]
        assert (int(ob["sum_E2_hi"][0, t]) << 64) + int(ob["sum_E2_lo"][0, t]) == s2[t]
        assert _e4(ob, t) == s4[t]
        assert int(ob["sum_Nmax"][0, t]) == m1[t] and int(ob["sum_Nmax2"][0, t]) == m2[t]
        assert int(ob["sum_Nmax3"][0, t]) == m3[t] and _n4(ob, t) == m4[t]
    if L > 100:
        assert max(s4).bit_length() > 128


def test_cumulants_match_exact_enumeration_L8_q3(oracle):
    """U_E = <E^4>/<E^2>^2 and V_M = 1 - <M^4>/(3<M^2>^2) (Eqs. 11, 12) from the oracle's accumulators against the
    exact Boltzmann averages over all 3^8 states; uniform configuration => M = 1 exactly => V_M = 2/3."""
    from paper_1308_5426_b200 import pt_math
    L, q = 8, 3
    Jq = oracle.couplings(L, 0.5).astype(np.int64)
    i, j = np.triu_indices(L, k=1)
    states = np.array(list(itertools.product(range(q), repeat=L)), dtype=np.int64)
    E = -((states[:, i] == states[:, j]) * Jq[j - i]).sum(axis=1).astype(np.float64) / SCALE
    nmax = np.stack([(states == k).sum(axis=1) for k in range(q)]).max(axis=0)
    M = (q * nmax / L - 1) / (q - 1)
    Ts = [1.0, 1.8, 3.0]
    o = oracle.Oracle(L, q, 0.5, 1, 3, [1 / T for T in Ts], 77)
    o.sweeps(2000, 1)
    base = o.observables()
    blocks = []
    for _ in range(32):
        o.sweeps(4000, 1)
        cur = o.observables()
        blocks.append(pt_math.cumulants(pt_math.obs_diff(cur, base), L, q))
        base = cur
    U = np.array([b["U_E"][0] for b in blocks]); V = np.array([b["V_M"][0] for b in blocks])
    for t, T in enumerate(Ts):
        w = np.exp(-(E - E.min()) / T); w /= w.sum()
        U_exact = (w * E ** 4).sum() / (w * E ** 2).sum() ** 2
        V_exact = 1 - (w * M ** 4).sum() / (3 * (w * M ** 2).sum() ** 2)
        for series, exact in ((U[:, t], U_exact), (V[:, t], V_exact)):
            err = series.std(ddof=1) / math.sqrt(len(series))
            assert abs(series.mean() - exact) < 4 * err + 2e-3 * abs(exact), (T, series.mean(), exact, err)
    # all-equal configuration sampled once: M = 1 => V_M = 1 - 1/3
    one = {k: np.zeros((1, 1) + v.shape[2:], dtype=v.dtype) for k, v in base.items()}
    one["n_samples"][0, 0] = 1; one["sum_Nmax"][0, 0] = L; one["sum_Nmax2"][0, 0] = L ** 2
    one["sum_Nmax3"][0, 0] = L ** 3; one["sum_Nmax4_lo"][0, 0] = L ** 4
    assert pt_math.cumulants(one, L, q)["V_M"][0, 0] == pytest.approx(2.0 / 3.0, rel=1e-15)
