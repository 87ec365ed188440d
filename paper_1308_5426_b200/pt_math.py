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


# ---------------------------------------------------------------------------------------------------------------------
# Blocked jack-knife errors (section 5.1: "Errors were evaluated using the standard jack-knife technique";
# a blocked jack-knife replaces the ALPS library).  Works on the exact integer accumulators: a "wide"
# record holds every accumulator of pt_obs as an array of Python integers (the multi-word sums joined), so that blocks
# can be added and subtracted exactly; estimates (also the non-linear cumulants of Eqs. 11-12) are functions of such a
# record.
# ---------------------------------------------------------------------------------------------------------------------
_WIDE_PLAIN = ("n_samples", "sum_E", "sum_Nmax", "sum_Nmax2", "sum_Nmax3", "flip_attempts", "flip_accepts",
               "swap_attempts", "swap_accepts")


def widen(obs):
    """pt_obs fields (dict of numpy arrays, as returned by PT.observables / Oracle.observables) -> wide record."""
    shape = obs["n_samples"].shape
    w = {k: np.array([int(v) for v in obs[k].ravel()], dtype=object).reshape(shape) for k in _WIDE_PLAIN}
    e2 = [(int(h) << 64) + int(l) for h, l in zip(obs["sum_E2_hi"].ravel(), obs["sum_E2_lo"].ravel())]
    n4 = [(int(h) << 64) + int(l) for h, l in zip(obs["sum_Nmax4_hi"].ravel(), obs["sum_Nmax4_lo"].ravel())]
    e4 = [sum(int(x) << (64 * k) for k, x in enumerate(limbs)) for limbs in obs["sum_E4"].reshape(-1, 4)]
    w["sum_E2"] = np.array(e2, dtype=object).reshape(shape)
    w["sum_Nmax4"] = np.array(n4, dtype=object).reshape(shape)
    w["sum_E4"] = np.array(e4, dtype=object).reshape(shape)
    return w


def wide_sub(a, b):
    return {k: a[k] - b[k] for k in a}


def wide_add(a, b):
    return {k: a[k] + b[k] for k in a}


def blocks_from_snapshots(snaps):
    """Cumulative snapshots [s_0, s_1, ..., s_n] (pt_obs dicts) -> n wide block records s_i - s_{i-1}."""
    w = [widen(s) for s in snaps]
    return [wide_sub(w[i + 1], w[i]) for i in range(len(w) - 1)]


def wide_estimates(w, L, q):
    """<E>/L, <M>, <M^2> (Eq. 10), U_E (Eq. 11) and V_M (Eq. 12) per (ensemble, slot) from a wide record; exact integer
    and rational arithmetic up to the last division."""
    from fractions import Fraction
    shape = w["n_samples"].shape
    out = {k: np.full(shape, np.nan) for k in ("E_per_spin", "M", "M2", "U_E", "V_M")}
    for idx in np.ndindex(*shape):
        n = w["n_samples"][idx]
        if n <= 0:
            continue
        s1, s2, s3, s4 = w["sum_Nmax"][idx], w["sum_Nmax2"][idx], w["sum_Nmax3"][idx], w["sum_Nmax4"][idx]
        a, b = q, -L                               # (q Nmax - L)^k, k = 1, 2, 4; M = (q Nmax - L) / ((q - 1) L)
        m1 = a * s1 + b * n
        m2 = a * a * s2 + 2 * a * b * s1 + b * b * n
        m4 = a ** 4 * s4 + 4 * a ** 3 * b * s3 + 6 * a * a * b * b * s2 + 4 * a * b ** 3 * s1 + b ** 4 * n
        d = (q - 1) * L
        out["E_per_spin"][idx] = float(Fraction(w["sum_E"][idx], n * L * (1 << 24)))
        out["M"][idx] = float(Fraction(m1, n * d))
        out["M2"][idx] = float(Fraction(m2, n * d * d))
        if w["sum_E2"][idx]:
            out["U_E"][idx] = float(Fraction(w["sum_E4"][idx] * n, w["sum_E2"][idx] ** 2))
        if m2:
            out["V_M"][idx] = 1.0 - float(Fraction(m4 * n, 3 * m2 * m2))
    return out


def jackknife(blocks, fn):
    """Delete-one-block jack-knife of the estimate fn(wide record) -> array.  Returns (estimate on all blocks,
    jack-knife standard error).  For a linear estimate (a mean) this is the standard error of the block means; for the
    cumulants of Eqs. 11-12 it propagates the non-linearity."""
    n = len(blocks)
    if n < 2:
        raise ValueError("jackknife needs at least two blocks")
    total = blocks[0]
    for b in blocks[1:]:
        total = wide_add(total, b)
    full = np.asarray(fn(total), dtype=np.float64)
    leave = np.stack([np.asarray(fn(wide_sub(total, b)), dtype=np.float64) for b in blocks])
    mean = leave.mean(axis=0)
    err = np.sqrt((n - 1) / n * ((leave - mean) ** 2).sum(axis=0))
    return full, err
