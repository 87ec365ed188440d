"""Pins of the oracle's random-site update order (reading A5' of DESIGN.md; "L Metropolis steps ...
an average of one Monte Carlo step per spin").  CPU only."""
import math

import numpy as np

from test_oracle_sweeps import exact_means


def test_random_order_samples_the_exact_boltzmann_law_L8_q3(oracle):
    Ts = [0.8, 1.5, 2.5]
    o = oracle.Oracle(8, 3, 0.5, 1, 3, [1 / T for T in Ts], 20130827)
    o.set_site_order("random")
    o.sweeps(2000, 1)
    prev = o.observables()
    rows = []
    for _ in range(64):
        o.sweeps(2500, 1)
        cur = o.observables()
        rows.append(np.stack([(cur["sum_E"][0] - prev["sum_E"][0]) / (2500 * 2.0 ** 24),
                              (cur["sum_Nmax"][0] - prev["sum_Nmax"][0]) / 2500.0]))
        prev = cur
    rows = np.array(rows)
    mean, err = rows.mean(axis=0), rows.std(axis=0, ddof=1) / math.sqrt(len(rows))
    for t, T in enumerate(Ts):
        x = exact_means(T)
        assert abs(mean[0, t] - x["E"]) < 3.5 * err[0, t], (T, mean[0, t], x["E"])
        assert abs(mean[1, t] - x["Nmax"]) < 3.5 * err[1, t]
        assert err[0, t] < 0.01 * abs(x["E"])


def test_random_order_differs_from_sequential_and_is_deterministic(oracle):
    args = (64, 4, 0.6, 1, 3, [1.2, 0.8, 0.4], 5)
    a, b, c = oracle.Oracle(*args), oracle.Oracle(*args), oracle.Oracle(*args)
    a.set_site_order("random")
    b.set_site_order("random")
    a.sweeps(7, 1)
    a.sweeps(13, 1)
    b.sweeps(20, 1, field=True, threads=2)     # call splitting, field mode and threads change nothing
    c.sweeps(20, 1)
    np.testing.assert_array_equal(a.get_spins(), b.get_spins())
    np.testing.assert_array_equal(a.energy(), b.energy())
    np.testing.assert_array_equal(a.energy(), a.energy(recompute=True))   # sites visited twice keep E += dE exact
    assert not np.array_equal(a.get_spins(), c.get_spins())
    oa = a.observables()
    assert (oa["flip_attempts"] == 20 * 64).all()


def test_random_sites_are_mulhi_of_the_fourth_philox_word(oracle):
    """One sweep at beta = 0 accepts every step: the sites whose colour differs from the hot start afterwards are a
    subset of the sites drawn, and every drawn site whose LAST proposal differs from its start colour has changed."""
    L, q, seed = 64, 5, 9
    o = oracle.Oracle(L, q, 0.5, 1, 1, [0.0], seed)
    before = o.get_spins()[0, 0].astype(int) - 1
    o.set_site_order("random")
    o.sweeps(1, 0)
    after = o.get_spins()[0, 0].astype(int) - 1
    key = [seed & 0xFFFFFFFF, seed >> 32]
    cur = before.copy()
    for n in range(L):
        w = oracle.philox([n, 1, 0, 1], key)
        i = (int(w[3]) * L) >> 32
        k = (int(w[0]) * (q - 1)) >> 32
        cur[i] = k + (1 if k >= cur[i] else 0)
    np.testing.assert_array_equal(cur, after)
