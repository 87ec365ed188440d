"""Reporting helpers on the integer accumulators of pt_obs (no CUDA, no libpt.so needed): one fixed fp64 formula for
<E>/L, <M>, <M^2> and the cumulants of Eqs. 11-12, used on the results of both the library and the oracle."""
import numpy as np


def obs_diff(cur, prev):
    """Accumulators gathered between two snapshots (burn-in removal, blocking): field-wise difference; the multi-word
    integers (sum_E2, sum_E4, sum_Nmax4) are differenced as whole integers and split back into their words."""
    out = {}
    for k in cur:
        if k in ("sum_E2_lo", "sum_E2_hi", "sum_E4", "sum_Nmax4_lo", "sum_Nmax4_hi"):
            continue
        out[k] = cur[k] - prev[k]
    shape = cur["n_samples"].shape
    out["sum_E2_lo"] = np.zeros(shape, dtype=np.uint64); out["sum_E2_hi"] = np.zeros(shape, dtype=np.int64)
    out["sum_Nmax4_lo"] = np.zeros(shape, dtype=np.uint64); out["sum_Nmax4_hi"] = np.zeros(shape, dtype=np.int64)
    out["sum_E4"] = np.zeros(shape + (4,), dtype=np.uint64)
    m64 = (1 << 64) - 1
    for idx in np.ndindex(*shape):
        for lo, hi in (("sum_E2_lo", "sum_E2_hi"), ("sum_Nmax4_lo", "sum_Nmax4_hi")):
            d = ((int(cur[hi][idx]) << 64) + int(cur[lo][idx])) - ((int(prev[hi][idx]) << 64) + int(prev[lo][idx]))
            out[lo][idx] = d & m64
            out[hi][idx] = d >> 64
        d = sum(int(cur["sum_E4"][idx + (k,)]) << (64 * k) for k in range(4)) - \
            sum(int(prev["sum_E4"][idx + (k,)]) << (64 * k) for k in range(4))
        for k in range(4):
            out["sum_E4"][idx + (k,)] = (d >> (64 * k)) & m64
    return out


def derived(obs, L, q):
    """<E>/L, <M>, <M^2> from the integer accumulators (one fixed fp64 formula; Eq. 10)."""
    n = obs["n_samples"].astype(np.float64)
    e = obs["sum_E"].astype(np.float64) / (n * L * 16777216.0)
    m1 = obs["sum_Nmax"].astype(np.float64) / (n * L)
    m2 = obs["sum_Nmax2"].astype(np.float64) / (n * float(L) * float(L))
    M = (q * m1 - 1.0) / (q - 1.0)
    M2 = (q * q * m2 - 2.0 * q * m1 + 1.0) / ((q - 1.0) ** 2)
    return {"E_per_spin": e, "M": M, "M2": M2}


def cumulants(obs, L, q):
    """Energy cumulant U_E = <E^4>/<E^2>^2 (Eq. 11) and Binder cumulant
    V_M = 1 - <M^4>/(3 <M^2>^2) (Eq. 12) per (ensemble, slot), from the exact integer accumulators
    (Python integers and fractions; only the last division is floating point).  With x = Nmax/L, Eq. 10 gives
    M = (q x - 1)/(q - 1), so <M^k> is a polynomial in the moments of Nmax."""
    from fractions import Fraction
    shape = obs["n_samples"].shape
    U = np.full(shape, np.nan)
    V = np.full(shape, np.nan)
    for idx in np.ndindex(*shape):
        n = int(obs["n_samples"][idx])
        if n == 0:
            continue
        e2 = (int(obs["sum_E2_hi"][idx]) << 64) + int(obs["sum_E2_lo"][idx])
        e4 = sum(int(obs["sum_E4"][idx + (k,)]) << (64 * k) for k in range(4))
        if e2:
            U[idx] = float(Fraction(e4 * n, e2 * e2))
        s1, s2, s3 = int(obs["sum_Nmax"][idx]), int(obs["sum_Nmax2"][idx]), int(obs["sum_Nmax3"][idx])
        s4 = (int(obs["sum_Nmax4_hi"][idx]) << 64) + int(obs["sum_Nmax4_lo"][idx])
        # sums over samples of (q Nmax - L)^k, k = 2 and 4 (the common factor ((q-1) L)^-k cancels in V_M)
        a, b = q, -L
        m2 = a * a * s2 + 2 * a * b * s1 + b * b * n
        m4 = a ** 4 * s4 + 4 * a ** 3 * b * s3 + 6 * a * a * b * b * s2 + 4 * a * b ** 3 * s1 + b ** 4 * n
        if m2:
            V[idx] = 1.0 - float(Fraction(m4 * n, 3 * m2 * m2))
    return {"U_E": U, "V_M": V}
