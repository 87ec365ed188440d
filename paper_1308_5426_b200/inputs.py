"""Seeded, synthetic workload recipes (BASELINE.json `configs`).

This module holds NO arithmetic of the method: only the parameter tuples, the
temperature ladders (A14: computed once here in fp64 and handed to both the
CUDA path and the oracle, so no libm `pow` can differ between them) and the
start configurations that are not drawn by the method's own Philox stream.
It is the only module that both the product's tests/bench and the oracle's
callers import.
"""
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

SEED_BASE = 0x1308542600000000


@dataclass(frozen=True)
class Workload:
    name: str
    L: int
    q: int
    sigma: float
    n_ens: int
    n_rep: int
    T_lo: float
    T_hi: float
    sweeps: int
    swap_every: int = 1
    burn_in: int = 0
    cold_half: bool = False      # cfg2: slots t < n_rep/2 (the colder half) start all-1
    seed: int = SEED_BASE
    ladder: str = "geometric"    # "uniform": T_t equally spaced (the paper's ladder)

    @property
    def attempts(self) -> int:
        return self.L * self.n_ens * self.n_rep * self.sweeps


def geometric_betas(T_lo: float, T_hi: float, n_rep: int) -> np.ndarray:
    """beta_t = 1/T_t, T_t = T_lo (T_hi/T_lo)^(t/(R-1)), slot 0 = coldest (A14)."""
    if n_rep == 1:
        return np.array([1.0 / T_lo], dtype=np.float64)
    t = np.arange(n_rep, dtype=np.float64) / float(n_rep - 1)
    T = T_lo * np.power(T_hi / T_lo, t)
    return np.ascontiguousarray(1.0 / T, dtype=np.float64)


def uniform_betas(T_lo: float, T_hi: float, n_rep: int) -> np.ndarray:
    """beta_t = 1/T_t, T_t equally spaced in [T_lo, T_hi], slot 0 = coldest ("a uniform distribution of the
    temperatures")."""
    return np.ascontiguousarray(1.0 / np.linspace(T_lo, T_hi, n_rep, dtype=np.float64), dtype=np.float64)


PAPER_BENCH_SIZES = (512, 1024, 2048, 3072, 4096, 6144, 8192, 10240)


def paper_benchmark(L: int, n_rep: int = 400) -> Workload:
    """The shape of the paper's own runs: q = 3, 400 replicas on a uniform temperature
    ladder, lattice sizes 512..10240, swap event every sweep.  sigma = 0.5 (mid-range
    of the paper's [0.2, 0.8]) and T in [0.5, 3.0] (brackets the Table 1 critical temperatures) are this build's
    choices: the paper does not print the ladder's end points.  Synthetic parameters only; no dataset is involved.
    n_rep other than 400 gives the points of the replica-count scan (Fig. 5) on the same ladder range."""
    if L < 8 or L > 10240:
        raise ValueError("paper_benchmark: L must be in 8..10240")
    if n_rep < 2 or n_rep > 4096:
        raise ValueError("paper_benchmark: n_rep must be in 2..4096")
    return Workload("paper[L=%d,R=%d]" % (L, n_rep), L, 3, 0.5, 1, n_rep, 0.5, 3.0, 1000, ladder="uniform",
                    seed=SEED_BASE + 0x500 + L)


def config(k: int) -> Workload:
    """BASELINE.json configs[k] for k = 0..3 (one (q, sigma) per handle)."""
    table = {
        0: Workload("cfg0", 64, 3, 0.5, 1, 8, 0.8, 2.5, 1000),
        1: Workload("cfg1", 256, 3, 0.4, 1, 32, 1.0, 3.0, 10000, burn_in=2000),
        2: Workload("cfg2", 1024, 5, 0.8, 1, 64, 0.5, 2.0, 10000, cold_half=True),
        3: Workload("cfg3", 4096, 8, 0.3, 1, 128, 0.6, 2.5, 2000),
    }
    w = table[k]
    return Workload(**{**w.__dict__, "seed": SEED_BASE + k})


def config4() -> List[Workload]:
    """configs[4]: the sigma-q scan = 40 independent handles of 32 replicas each."""
    out = []
    for q in (3, 5, 7, 9):
        for s10 in range(1, 11):
            idx = len(out)
            out.append(Workload("cfg4[q=%d,sigma=%.1f]" % (q, s10 / 10.0), 2048, q, s10 / 10.0,
                                1, 32, 0.4, 3.0, 5000, seed=SEED_BASE + 4 + (idx << 8)))
    return out


def betas(w: Workload) -> np.ndarray:
    if w.ladder == "uniform":
        return uniform_betas(w.T_lo, w.T_hi, w.n_rep)
    return geometric_betas(w.T_lo, w.T_hi, w.n_rep)


def cold_half_spins(w: Workload, hot_spins: np.ndarray) -> np.ndarray:
    """cfg2 start: the colder half of the slots set to colour 1, the rest keep
    the hot start `hot_spins` ([n_ens, n_rep, L], values 1..q) the method drew."""
    s = np.array(hot_spins, dtype=np.uint8, copy=True).reshape(w.n_ens, w.n_rep, w.L)
    s[:, : w.n_rep // 2, :] = 1
    return s


def random_spins(n_ens: int, n_rep: int, L: int, q: int, seed: int) -> np.ndarray:
    """Arbitrary test configurations (numpy PCG64; not the method's stream)."""
    rng = np.random.default_rng(seed)
    return rng.integers(1, q + 1, size=(n_ens, n_rep, L), dtype=np.uint8)
