"""Pins T7/T8/T9: the oracle's Metropolis cycle (Eq. 8) and replica exchange
(Eq. 9, two stages :126) against the exact Boltzmann distribution from full
enumeration at L=8, q=3 (6561 states), beta=0, and its own invariants."""
import itertools
import math

import numpy as np
import pytest

JQ8 = np.array([0, 20701016, 10017126, 7631696, 7083178, 7631696, 10017126, 20701016], dtype=np.int64)
SCALE = float(2 ** 24)


def enumerate_L8_q3():
    """All 3^8 states: integer energy (Eq. 2, pairs once) and N_max."""
    L, q = 8, 3
    i, j = np.triu_indices(L, k=1)
    states = np.array(list(itertools.product(range(q), repeat=L)), dtype=np.int64)
    E = -((states[:, i] == states[:, j]) * JQ8[j - i]).sum(axis=1)
    nmax = np.stack([(states == k).sum(axis=1) for k in range(q)]).max(axis=0)
    return E, nmax


def exact_means(T):
    E, nmax = enumerate_L8_q3()
    if math.isinf(T):
        w = np.ones(len(E))
    else:
        w = np.exp(-(E - E.min()) / (SCALE * T))
    w /= w.sum()
    M = (3 * nmax / 8.0 - 1) / 2.0
    return dict(E=(w * E).sum() / SCALE, E2=(w * E.astype(np.float64) ** 2).sum() / SCALE ** 2,
                M=(w * M).sum(), M2=(w * M * M).sum(), Nmax=(w * nmax).sum())


def test_enumeration_matches_survey_printed_values():
    """SURVEY.md 8(c) T7 prints these (surveyor's independent scratch run)."""
    ref = {0.8: (-19.7988313117416, 392.945766055565, 0.993059597069154, 0.987768005456466, 7.96298451770216),
           1.5: (-15.4000560042365, 258.517741349843, 0.780882584517211, 0.672284128265076, 6.83137378409179),
           2.5: (-9.81298308303958, 111.581678271047, 0.466989948580927, 0.282056341175059, 5.15727972576494)}
    for T, (e, e2, m, m2, nm) in ref.items():
        x = exact_means(T)
        assert x["E"] == pytest.approx(e, rel=1e-12)
        assert x["E2"] == pytest.approx(e2, rel=1e-12)
        assert x["M"] == pytest.approx(m, rel=1e-12)
        assert x["M2"] == pytest.approx(m2, rel=1e-12)
        assert x["Nmax"] == pytest.approx(nm, rel=1e-12)
    x = exact_means(math.inf)
    assert x["E"] == pytest.approx(-6.658463001251221, rel=1e-13)     # = -(1/3)(8/2) sum Jq / 2^24
    assert x["E"] == pytest.approx(-(1 / 3) * 4 * JQ8.sum() / SCALE, rel=1e-13)
    assert x["M"] == pytest.approx(0.26406035665294925, rel=1e-13)


def blocked_series(o, n_blocks, block, swap_every, field=False):
    """Per-block means of E/2^24, E^2/2^48, Nmax, Nmax^2 per slot from accumulator snapshots."""
    prev = o.observables()
    out = []
    for _ in range(n_blocks):
        o.sweeps(block, swap_every=swap_every, field=field)
        cur = o.observables()
        e2c = cur["sum_E2_hi"][0].astype(object) * 2 ** 64 + cur["sum_E2_lo"][0].astype(object)
        e2p = prev["sum_E2_hi"][0].astype(object) * 2 ** 64 + prev["sum_E2_lo"][0].astype(object)
        out.append(np.stack([(cur["sum_E"][0] - prev["sum_E"][0]) / (block * SCALE),
                             np.array([float(v) for v in (e2c - e2p)]) / (block * SCALE ** 2),
                             (cur["sum_Nmax"][0] - prev["sum_Nmax"][0]) / block,
                             (cur["sum_Nmax2"][0] - prev["sum_Nmax2"][0]) / block]))
        prev = cur
    return np.array(out)            # [block, observable, slot]


@pytest.mark.parametrize("swap_every,field", [(0, False), (1, False), (3, True)])
def test_chain_samples_exact_boltzmann_L8_q3(oracle, swap_every, field):
    """T7: sampled <E>, <E^2>, <M>, <M^2> of every slot within 3 sigma (blocked error) of the
    enumeration -- without swaps, with swaps every sweep (PT leaves each slot's marginal
    Boltzmann), and in field mode with swaps every 3rd sweep."""
    Ts = [0.8, 1.5, 2.5]
    o = oracle.Oracle(8, 3, 0.5, 1, 3, [1 / T for T in Ts], 20130826 + swap_every)
    assert np.array_equal(o.get_couplings(), JQ8)
    o.sweeps(2000, swap_every=swap_every, field=field)
    series = blocked_series(o, n_blocks=64, block=2500, swap_every=swap_every, field=field)
    mean = series.mean(axis=0)
    err = series.std(axis=0, ddof=1) / math.sqrt(series.shape[0])
    for t, T in enumerate(Ts):
        x = exact_means(T)
        m_s = (3 * mean[2, t] / 8 - 1) / 2
        m_err = 3 * err[2, t] / 16
        assert abs(mean[0, t] - x["E"]) < 3.5 * err[0, t], (T, mean[0, t], x["E"], err[0, t])
        assert abs(mean[1, t] - x["E2"]) < 3.5 * err[1, t]
        assert abs(m_s - x["M"]) < 3.5 * m_err
        # <Nmax^2> <-> <M^2>: M^2 = (9 Nmax^2/64 - 6 Nmax/8 + 1)/4
        m2_s = (9 * mean[3, t] / 64 - 6 * mean[2, t] / 8 + 1) / 4
        assert m2_s == pytest.approx(x["M2"], abs=0.01)
        # errors small enough that a wrong sign/term in dE or Eq. 8 fails (rel. precision < 1%)
        assert err[0, t] < 0.01 * abs(x["E"])
    ob = o.observables()
    if swap_every:
        assert ob["swap_attempts"][0, 0] > 0 and ob["swap_attempts"][0, 2] == 0
        assert 0 < ob["swap_accepts"][0, 0] < ob["swap_attempts"][0, 0]
    assert ob["near_ties"].sum() == 0


@pytest.mark.parametrize("q", [4, 20])
def test_beta_zero_delta_is_one_over_q(oracle, q):
    """beta=0: every proposal accepted, stationary law uniform, <delta>=1/q so
    <E> = -(1/q)(L/2) sum_r Jq[r] (north_star pin); q = 20: the same closed form beyond 16 colours."""
    L = 32
    o = oracle.Oracle(L, q, 0.5, 1, 2, [0.0, 0.0], 3)
    Jsum = int(o.get_couplings().astype(np.int64).sum())
    o.sweeps(100, swap_every=1)
    series = blocked_series(o, n_blocks=40, block=500, swap_every=1)
    mean, err = series[:, 0, :].mean(axis=0), series[:, 0, :].std(axis=0, ddof=1) / math.sqrt(40)
    exact = -(1 / q) * (L / 2) * Jsum / SCALE
    for t in range(2):
        assert abs(mean[t] - exact) < 3.5 * err[t]
        assert err[t] < 0.01 * abs(exact)
    ob = o.observables()
    assert ob["flip_accepts"][0, 0] == ob["flip_attempts"][0, 0]
    # T8: equal betas => d = 0 => every swap accepted
    assert ob["swap_accepts"][0, 0] == ob["swap_attempts"][0, 0] == 100 + 40 * 500


def replay_sweep(oracle, c, E, Jq, q, beta, key, sweep, slot, ens):
    """One sequential-order sweep written out in Python from SURVEY 8(c) SWEEP (A5-A8), using
    only the KAT-pinned Philox and the energy definition (dE by two full recounts)."""
    L = len(c)
    i_, j_ = np.triu_indices(L, k=1)

    def energy(cc):
        return -int(((cc[i_] == cc[j_]) * Jq[j_ - i_]).sum())
    for i in range(L):
        w = [int(x) for x in oracle.philox([i, sweep, slot, (ens << 4) | 1], key)]
        a = int(c[i])
        k = (w[0] * (q - 1)) >> 32
        b = k + (1 if k >= a else 0)
        c2 = c.copy()
        c2[i] = b
        dE = energy(c2) - energy(c)
        u = (((w[1] >> 5) << 26) | (w[2] >> 6)) * 2.0 ** -53
        if dE <= 0 or u < math.exp(-(beta * (dE / SCALE))):
            c, E = c2, E + dE
    return c, E


@pytest.mark.parametrize("q", [3, 23])
def test_sweep_and_swap_replay_in_python(oracle, q):
    """Site order, counter layout, proposal rule, strict u<p, swap stages and slot keying:
    three sweeps with swaps replayed here and compared bit for bit (q = 23: more than 16 colours)."""
    L, R, ens = 16, 4, 1
    seed = 0x0123456789ABCDEF
    key = [seed & 0xFFFFFFFF, seed >> 32]
    betas = np.array([1.1, 0.9, 0.6, 0.3])
    o = oracle.Oracle(L, q, 0.5, 2, R, betas, seed)
    Jq = o.get_couplings().astype(np.int64)
    cs = [o.get_spins()[ens, t].astype(np.int64) - 1 for t in range(R)]
    Es = [int(v) for v in o.energy()[ens]]
    n_acc = 0
    for sweep in range(1, 4):
        for t in range(R):
            cs[t], Es[t] = replay_sweep(oracle, cs[t], Es[t], Jq, q, betas[t], key, sweep, t, ens)
        if sweep % 1 == 0:
            for stage in (0, 1):
                for t in range(stage, R - 1, 2):
                    d = (betas[t] - betas[t + 1]) * ((Es[t] - Es[t + 1]) / SCALE)
                    w = [int(x) for x in oracle.philox([t, sweep, 0, (ens << 4) | 2], key)]
                    u = (((w[1] >> 5) << 26) | (w[2] >> 6)) * 2.0 ** -53
                    if d >= 0 or u < math.exp(d):
                        cs[t], cs[t + 1] = cs[t + 1], cs[t]
                        Es[t], Es[t + 1] = Es[t + 1], Es[t]
                        n_acc += 1
        o.sweeps(1, swap_every=1)
        got = o.get_spins()[ens].astype(np.int64) - 1
        for t in range(R):
            assert np.array_equal(got[t], cs[t]), (sweep, t)
        assert [int(v) for v in o.energy()[ens]] == Es
    assert o.observables()["swap_accepts"][ens].sum() == n_acc
    assert o.sweep_counter() == 3


@pytest.mark.parametrize("L,q,sigma,R", [(64, 3, 0.5, 8), (128, 8, 0.3, 5), (64, 33, 0.5, 4)])
def test_field_mode_equals_direct_mode_and_recount(oracle, L, q, sigma, R):
    """north_star pin: incremental local-field energy == O(L^2) recompute after every sweep,
    and the field trajectory is the direct-sum trajectory bit for bit."""
    betas = 1.0 / np.geomspace(0.8, 2.5, R)
    a = oracle.Oracle(L, q, sigma, 1, R, betas, 42)
    b = oracle.Oracle(L, q, sigma, 1, R, betas, 42)
    for _ in range(25):
        a.sweeps(1, swap_every=1, field=False)
        b.sweeps(1, swap_every=1, field=True)
        assert np.array_equal(a.get_spins(), b.get_spins())
        assert np.array_equal(a.energy(), b.energy())
        assert np.array_equal(b.energy(), b.energy(recompute=True))
    oa, ob = a.observables(), b.observables()
    for k in oa:
        assert np.array_equal(oa[k], ob[k]), k


def test_call_splitting_threads_and_seed_determinism(oracle):
    """T9: sweeps(a); sweeps(b) == sweeps(a+b) (swap phase keyed on the global counter);
    replica-threaded == single-threaded; same seed => same bits; other seed differs."""
    L, q, R = 64, 5, 6
    betas = 1.0 / np.geomspace(0.5, 2.0, R)

    def run(chunks, threads=1, seed=5, field=False):
        o = oracle.Oracle(L, q, 0.8, 2, R, betas, seed)
        for n in chunks:
            o.sweeps(n, swap_every=3, threads=threads, field=field)
        return o.get_spins(), o.energy(), o.observables()
    s0, E0, ob0 = run([30])
    for chunks, th, fld in [([7, 23], 1, False), ([1] * 30, 1, True), ([30], 4, False), ([11, 19], 3, True)]:
        s1, E1, ob1 = run(chunks, th, field=fld)
        assert np.array_equal(s0, s1) and np.array_equal(E0, E1)
        for k in ob0:
            assert np.array_equal(ob0[k], ob1[k]), k
    assert ob0["swap_attempts"][0, 0] == 10 and ob0["swap_attempts"][0, R - 1] == 0
    s2, _, _ = run([30], seed=6)
    assert not np.array_equal(s0, s2)


def test_swap_invariants(oracle):
    """T8: n_rep=1 => swaps are no-ops; a swap event permutes (configuration, E) pairs, so the
    multiset of energies is unchanged by it."""
    o1 = oracle.Oracle(32, 3, 0.5, 1, 1, [0.7], 9)
    o2 = oracle.Oracle(32, 3, 0.5, 1, 1, [0.7], 9)
    o1.sweeps(20, swap_every=1)
    o2.sweeps(20, swap_every=0)
    assert np.array_equal(o1.get_spins(), o2.get_spins())
    assert o1.observables()["swap_attempts"].sum() == 0
    # swaps only permute: compare a run with swaps against per-slot recount
    R = 7
    o = oracle.Oracle(32, 4, 0.5, 1, R, 1.0 / np.linspace(0.5, 3.0, R), 10)
    for _ in range(30):
        o.sweeps(1, swap_every=1)
        assert np.array_equal(o.energy(), o.energy(recompute=True))
    ob = o.observables()
    assert np.all(ob["swap_attempts"][0, : R - 1] == 30) and ob["swap_attempts"][0, R - 1] == 0
    assert np.all(ob["swap_accepts"] <= ob["swap_attempts"])


def test_create_rejects_invalid_arguments(oracle):
    bad = [dict(L=7), dict(L=0), dict(q=1), dict(q=65), dict(sigma=0.0), dict(sigma=float("nan")),
           dict(n_ens=0), dict(betas=[-1.0, 1.0]), dict(sigma=0.01, L=4096)]
    for kw in bad:
        args = dict(L=16, q=3, sigma=0.5, n_ens=1, n_rep=2, betas=[0.5, 1.0], seed=1)
        args.update(kw)
        with pytest.raises(ValueError):
            oracle.Oracle(**args)
