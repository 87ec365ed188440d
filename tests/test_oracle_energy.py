"""Pins T4/T5/T6/T10: the oracle's total energy (Eq. 2, reading A1), its dE
and N_max (Eq. 10) against definitions written out here with numpy on small
random states, closed forms, and the q=2 <-> long-range Ising identity."""
import numpy as np
import pytest

from paper_1308_5426_b200 import inputs

# L=8, sigma=0.5 couplings, from the 40-digit mpmath evaluation in test_oracle_couplings.py
JQ8 = np.array([0, 20701016, 10017126, 7631696, 7083178, 7631696, 10017126, 20701016], dtype=np.int64)


def brute_energy(Jq, c):
    """Eq. 2 with each unordered pair once: E = -sum_{i<j} Jq[j-i] [c_i == c_j]."""
    L = len(c)
    E = 0
    for i in range(L):
        for j in range(i + 1, L):
            if c[i] == c[j]:
                E -= int(Jq[j - i])
    return E


def make(oracle, L, q, sigma, n_rep=3, seed=7):
    return oracle.Oracle(L, q, sigma, 1, n_rep, np.linspace(0.3, 1.2, n_rep), seed)


@pytest.mark.parametrize("L,q,sigma", [(8, 3, 0.5), (16, 2, 0.3), (64, 5, 0.8), (128, 16, 0.1), (64, 37, 0.6), (48, 64, 0.4)])
def test_total_energy_matches_definition(oracle, L, q, sigma):
    o = make(oracle, L, q, sigma)
    Jq = o.get_couplings().astype(np.int64)
    if (L, sigma) == (8, 0.5):
        assert np.array_equal(Jq, JQ8)
    s = inputs.random_spins(1, 3, L, q, seed=L * q)
    o.set_spins(s)
    E = o.energy()
    for t in range(3):
        assert int(E[0, t]) == brute_energy(Jq, s[0, t])
    assert np.array_equal(o.energy(recompute=True), E)
    assert np.array_equal(o.get_spins(), s)


def test_hot_start_is_philox_uniform(oracle):
    """INIT: c = mulhi32(P(i,0,t,(e<<4)|0).w0, q), API colour c+1; energy is that state's."""
    L, q = 64, 5
    o = oracle.Oracle(L, q, 0.5, 2, 3, [0.5, 0.6, 0.7], 0xABCDEF0123456789)
    s = o.get_spins()
    key = [0x23456789, 0xABCDEF01]
    for e in range(2):
        for t in range(3):
            for i in (0, 1, 17, 63):
                w0 = int(oracle.philox([i, 0, t, (e << 4) | 0], key)[0])
                assert s[e, t, i] == ((w0 * q) >> 32) + 1
    Jq = o.get_couplings().astype(np.int64)
    assert int(o.energy()[1, 2]) == brute_energy(Jq, s[1, 2])
    assert not np.array_equal(s[0], s[1])          # T9: different ensembles, different streams
    # colour frequencies roughly uniform over 2*3*64 = 384 draws
    cnt = np.bincount(s.ravel(), minlength=q + 1)[1:]
    assert cnt.min() > 40 and cnt.max() < 120


@pytest.mark.parametrize("L,q,sigma", [(8, 3, 0.5), (32, 4, 0.4), (64, 8, 0.3), (40, 29, 0.7)])
def test_delta_e_is_energy_difference(oracle, L, q, sigma):
    """T4: dE(i, a->b) == E(after) - E(before), both by the O(L^2) definition above."""
    o = make(oracle, L, q, sigma, n_rep=1)
    Jq = o.get_couplings().astype(np.int64)
    rng = np.random.default_rng(L + q)
    s = inputs.random_spins(1, 1, L, q, seed=99)
    o.set_spins(s)
    c = s[0, 0].copy()
    E0 = brute_energy(Jq, c)
    for _ in range(40):
        i = int(rng.integers(L))
        b = int(rng.integers(1, q + 1))
        c2 = c.copy()
        c2[i] = b
        assert o.delta_e(0, 0, i, b) == brute_energy(Jq, c2) - E0
    assert o.delta_e(0, 0, 3, int(c[3])) == 0


@pytest.mark.parametrize("L,q,sigma", [(8, 3, 0.5), (64, 3, 0.5), (256, 7, 0.2)])
def test_ground_state_energy(oracle, L, q, sigma):
    """T5: all spins equal => E = -(L/2) sum_r Jq[r] (every one of the L(L-1)/2 pairs counts)."""
    o = make(oracle, L, q, sigma, n_rep=2)
    Jq = o.get_couplings().astype(np.int64)
    for colour in (1, q):
        o.set_spins(np.full((1, 2, L), colour, dtype=np.uint8))
        E = o.energy()
        assert int(E[0, 0]) == int(E[0, 1]) == -(L // 2) * int(Jq.sum())
    if (L, sigma) == (8, 0.5):
        assert int(E[0, 0]) == -335131416         # = -4 * 83782854, SURVEY 8(c) T5


def test_q2_maps_onto_long_range_ising(oracle):
    """T6: with sigma_i = +-1, delta = (1 + sigma_i sigma_j)/2, so
    2 E_Potts = E_Ising - sum_{i<j} Jq[j-i],  E_Ising = -sum_{i<j} Jq[j-i] sigma_i sigma_j."""
    L = 32
    o = make(oracle, L, 2, 0.6, n_rep=3)
    Jq = o.get_couplings().astype(np.int64)
    s = inputs.random_spins(1, 3, L, 2, seed=5)
    o.set_spins(s)
    E = o.energy()
    i, j = np.triu_indices(L, k=1)
    Jsum = int(Jq[j - i].sum())
    for t in range(3):
        sg = 2 * s[0, t].astype(np.int64) - 3        # colours 1,2 -> -1,+1
        E_ising = -int((Jq[j - i] * sg[i] * sg[j]).sum())
        assert 2 * int(E[0, t]) == E_ising - Jsum


def test_nmax_and_accumulators_after_one_sweep(oracle):
    """T10 + MEASURE: after each sweep n_samples++, sum_E += E, sum_E2 += E^2 (128 bit),
    sum_Nmax += max_k N_k, sum_Nmax2 += Nmax^2 -- recomputed here from get_spins()."""
    L, q, R = 64, 4, 3
    o = oracle.Oracle(L, q, 0.5, 1, R, [2.0, 0.5, 0.0], 11)
    acc = np.zeros((R, 4), dtype=object)
    for n in range(1, 6):
        o.sweeps(1, swap_every=0)
        s = o.get_spins()
        E = o.energy()
        assert np.array_equal(E, o.energy(recompute=True))
        for t in range(R):
            nmax = int(np.bincount(s[0, t], minlength=q + 1).max())
            assert -(-L // q) <= nmax <= L
            acc[t] += np.array([int(E[0, t]), int(E[0, t]) ** 2, nmax, nmax * nmax], dtype=object)
        ob = o.observables()
        for t in range(R):
            assert ob["n_samples"][0, t] == n
            assert int(ob["sum_E"][0, t]) == acc[t, 0]
            e2 = (int(ob["sum_E2_hi"][0, t]) << 64) | int(ob["sum_E2_lo"][0, t])
            assert e2 == acc[t, 1]
            assert int(ob["sum_Nmax"][0, t]) == acc[t, 2]
            assert int(ob["sum_Nmax2"][0, t]) == acc[t, 3]
            assert ob["flip_attempts"][0, t] == n * L
    # beta = 0 slot accepts every proposal (A7)
    assert ob["flip_accepts"][0, 2] == 5 * L
    assert ob["swap_attempts"].sum() == 0
