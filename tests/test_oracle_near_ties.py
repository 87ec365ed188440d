"""Pin of the oracle's near-tie counter (finding 1).

The CUDA path never evaluates u < exp(-beta dE) for a Metropolis step: it compares integers with the threshold of
reading A9.  The two forms can only disagree when |u - exp(-beta dE)| is of the order of 1e-15, and the
oracle counts every step (and every swap) with |u - p| < 1e-12 so that the parity tests can assert that no such step
occurred.  A counter that can never fire would void that argument, so here it is MADE to fire: the temperature is
chosen so that the first proposal of the first sweep (resp. the first swap) lands on p = u to within an ulp, and a
control run with beta moved by 1e-6 (relative) must count nothing.

Everything the construction needs is recomputed here from published pieces (the Philox stream through orc_philox,
which has its own known-answer pin; the 53-bit uniform; dE through orc_delta_e, pinned against O(L^2) recounts in
test_oracle_energy.py) -- not from the sweep code under test.
"""
import math

import numpy as np
import pytest

TAG_SWEEP, TAG_SWAP = 1, 2


def _u53(w):
    return float(((int(w[1]) >> 5) << 26) | (int(w[2]) >> 6)) * 2.0 ** -53


def _first_step(oracle, o, seed, q, slot=0, site=0, sweep=1):
    """(b_api, dE, u) of the proposal at `site` of `slot` in sweep `sweep` for the CURRENT configuration."""
    key = [seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF]
    w = oracle.philox([site, sweep, slot, TAG_SWEEP], key)
    a = int(o.get_spins()[0, slot, site]) - 1
    k = (int(w[0]) * (q - 1)) >> 32
    b = k + (1 if k >= a else 0)
    return b + 1, int(o.delta_e(0, slot, site, b + 1)), _u53(w)


def _find_seed_with_uphill_first_step(oracle, L, q, sigma):
    for seed in range(1, 200):
        o = oracle.Oracle(L, q, sigma, 1, 1, [1.0], seed)
        b, dE, u = _first_step(oracle, o, seed, q)
        o.close()
        if dE > 0 and 0.05 < u < 0.95:
            return seed, dE, u
    raise AssertionError("no seed with an uphill first proposal")


def test_flip_near_tie_is_counted_and_control_is_not(oracle):
    L, q, sigma = 8, 3, 0.5
    seed, dE, u = _find_seed_with_uphill_first_step(oracle, L, q, sigma)
    beta = -math.log(u) / (dE * 2.0 ** -24)          # exp(-beta dE 2^-24) == u up to rounding
    assert abs(u - math.exp(-(beta * (dE * 2.0 ** -24)))) < 1e-14
    o = oracle.Oracle(L, q, sigma, 1, 1, [beta], seed)
    o.sweeps(1, 0)
    ob = o.observables()
    assert int(ob["near_ties"][0, 0]) >= 1, "the near-tie counter did not fire on a constructed tie"
    assert int(ob["flip_attempts"][0, 0]) == L
    o.close()
    # control: the same stream, beta moved by 1e-6 relative => |u - p| ~ 1e-6 * |ln u| * u >> 1e-12 at site 0;
    # the other sites of the sweep are generic (probability ~1e-12 each of a tie)
    for factor in (1.0 + 1e-6, 1.0 - 1e-6):
        o = oracle.Oracle(L, q, sigma, 1, 1, [beta * factor], seed)
        o.sweeps(1, 0)
        assert int(o.observables()["near_ties"].sum()) == 0
        o.close()


def test_flip_near_tie_window_is_1e_minus_12(oracle):
    """The window is |u - p| < 1e-12 (north_star): a miss by 1e-10 must not count, a miss by 1e-13 must."""
    L, q, sigma = 8, 3, 0.5
    seed, dE, u = _find_seed_with_uphill_first_step(oracle, L, q, sigma)
    x = dE * 2.0 ** -24
    for target, expect in ((u + 1e-13, 1), (u - 1e-13, 1), (u + 1e-10, 0), (u - 1e-10, 0)):
        beta = -math.log(target) / x
        p = math.exp(-(beta * x))
        assert (abs(u - p) < 1e-12) == bool(expect)   # the construction itself lands where intended
        o = oracle.Oracle(L, q, sigma, 1, 1, [beta], seed)
        o.sweeps(1, 0)
        assert int(o.observables()["near_ties"][0, 0]) == expect, (target - u, expect)
        o.close()


def test_downhill_steps_never_count(oracle):
    """dE <= 0 accepts without evaluating exp: such a step is never a near-tie, whatever u is (A7)."""
    L, q = 8, 3
    o = oracle.Oracle(L, q, 0.5, 1, 1, [0.0], 5)     # beta = 0: p = 1 for every step, u < 1 always
    o.sweeps(50, 0)
    ob = o.observables()
    assert int(ob["near_ties"].sum()) == 0 and int(ob["flip_accepts"].sum()) == 50 * L
    o.close()


def test_swap_near_tie_is_counted_and_control_is_not(oracle):
    """Eq. 9: d = (beta_0 - beta_1)(E_0 - E_1) 2^-24; choose beta_0 - beta_1 so that exp(d) == u of the first swap.
    Sweeps at beta = 0-like temperatures would change E, so the swap is made the first thing that happens: sweep 1
    runs with the final betas, then the event of sweep 1 sees the energies AFTER that sweep -- which depend on the
    betas.  The construction therefore iterates: guess, run, read E, solve for beta_0, until it reproduces itself."""
    L, q, sigma, seed = 8, 3, 0.5, 11
    key = [seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF]
    u = _u53(oracle.philox([0, 1, 0, TAG_SWAP], key))
    assert 0.0 < u < 1.0
    beta1 = 0.0                                      # slot 1 at infinite temperature: its sweep accepts everything
    beta0 = 0.3
    found = None
    for _ in range(60):
        o = oracle.Oracle(L, q, sigma, 1, 2, [beta0, beta1], seed)
        o.sweeps(1, 0)                               # the sweep only; energies just before the event
        E = o.energy()[0]
        o.close()
        dEs = int(E[0]) - int(E[1])
        if dEs >= 0:
            beta0 *= 1.7                             # colder slot 0 -> lower E_0
            continue
        new_beta0 = beta1 + math.log(u) / (dEs * 2.0 ** -24)   # d = ln u < 0
        if new_beta0 == beta0:
            found = beta0
            break
        beta0 = new_beta0
    if found is None:
        pytest.skip("construction did not reach a fixed point for this seed")
    d = (found - beta1) * (dEs * 2.0 ** -24)
    assert d < 0 and abs(u - math.exp(d)) < 1e-14
    o = oracle.Oracle(L, q, sigma, 1, 2, [found, beta1], seed)
    o.sweeps(1, 1)
    ob = o.observables()
    assert int(ob["swap_attempts"][0, 0]) == 1
    assert int(ob["near_ties"][0, 0]) >= 1, "the swap near-tie counter did not fire on a constructed tie"
    o.close()
    o = oracle.Oracle(L, q, sigma, 1, 2, [found * (1 + 1e-6), beta1], seed)
    o.sweeps(1, 0)
    if tuple(o.energy()[0]) == (int(E[0]), int(E[1])):          # same sweep outcome: only the swap test moved
        o.close()
        o = oracle.Oracle(L, q, sigma, 1, 2, [found * (1 + 1e-6), beta1], seed)
        o.sweeps(1, 1)
        assert int(o.observables()["near_ties"].sum()) == 0
    o.close()
