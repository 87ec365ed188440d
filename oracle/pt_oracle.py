"""ctypes binding of the CPU oracle (oracle/pt_oracle.cpp).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from paper_1308_5426_b200.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pt_oracle.cpp")
_LIB = os.path.join(_HERE, "libpt_oracle.so")
# No -ffast-math, no FMA contraction: A8 (one rounding in beta*dE) must hold.
CXXFLAGS = ["-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-ffp-contract=off"]


def build(force=False):
    """Compile the oracle with g++ (building the checker is not using it)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["g++"] + CXXFLAGS + ["-o", tmp, _SRC])
    os.replace(tmp, _LIB)
    return _LIB


class Obs(ctypes.Structure):
    _fields_ = [("n_samples", ctypes.c_int64), ("sum_E", ctypes.c_int64),
                ("sum_E2_lo", ctypes.c_uint64), ("sum_E2_hi", ctypes.c_int64),
                ("sum_Nmax", ctypes.c_int64), ("sum_Nmax2", ctypes.c_int64),
                ("flip_attempts", ctypes.c_int64), ("flip_accepts", ctypes.c_int64),
                ("swap_attempts", ctypes.c_int64), ("swap_accepts", ctypes.c_int64),
                ("near_ties", ctypes.c_int64),
                ("sum_E4", ctypes.c_uint64 * 4), ("sum_Nmax3", ctypes.c_int64),
                ("sum_Nmax4_lo", ctypes.c_uint64), ("sum_Nmax4_hi", ctypes.c_int64)]


OBS_FIELDS = [f[0] for f in Obs._fields_]
_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, i32, i64, u64, dbl = (ctypes.c_void_p, ctypes.c_int, ctypes.c_int64,
                                  ctypes.c_uint64, ctypes.c_double)
        L.orc_jstar.argtypes = [i32, dbl, vp]
        L.orc_couplings.argtypes = [i32, dbl, vp]
        L.orc_philox.argtypes = [vp, vp, vp]
        L.orc_uniform53.argtypes = [ctypes.c_uint32, ctypes.c_uint32]
        L.orc_uniform53.restype = dbl
        L.orc_create.argtypes = [i32, i32, dbl, i32, i32, vp, u64]
        L.orc_create.restype = vp
        L.orc_create_ex.argtypes = [i32, i32, dbl, i32, i32, vp, u64, i32]
        L.orc_create_ex.restype = vp
        L.orc_destroy.argtypes = [vp]
        L.orc_destroy.restype = None
        L.orc_sweeps.argtypes = [vp, i64, i32, i32, i32]
        L.orc_sweeps_arith.argtypes = [vp, i64, i32, i32, i32]
        L.orc_delta_e_arith.argtypes = [vp, i32, i32, i32, i32, i32]
        L.orc_delta_e_arith.restype = dbl
        L.orc_energy.argtypes = [vp, vp, i32]
        L.orc_observables.argtypes = [vp, vp]
        L.orc_get_spins.argtypes = [vp, vp]
        L.orc_set_spins.argtypes = [vp, vp]
        L.orc_get_couplings.argtypes = [vp, vp]
        L.orc_sweep_counter.argtypes = [vp]
        L.orc_set_site_order.argtypes = [vp, i32]
        L.orc_sweep_counter.restype = i64
        L.orc_delta_e.argtypes = [vp, i32, i32, i32, i32]
        L.orc_delta_e.restype = i64
        assert L.orc_obs_size() == ctypes.sizeof(Obs)
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def jstar(L, sigma):
    out = np.zeros(L, dtype=np.float64)
    lib().orc_jstar(L, float(sigma), _p(out))
    return out


def couplings(L, sigma):
    out = np.zeros(L, dtype=np.int32)
    lib().orc_couplings(L, float(sigma), _p(out))
    return out


def philox(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    o = np.zeros(4, dtype=np.uint32)
    lib().orc_philox(_p(c), _p(k), _p(o))
    return o


def uniform53(w1, w2):
    return lib().orc_uniform53(int(w1), int(w2))


class Oracle:
    """Same call names as the product binding, CPU only."""

    def __init__(self, L, q, sigma, n_ens, n_rep, betas, seed, ens_base=0):
        b = np.ascontiguousarray(betas, dtype=np.float64)
        if b.shape != (n_rep,):
            raise ValueError("betas must have n_rep entries")
        self.L, self.q, self.n_ens, self.n_rep = L, q, n_ens, n_rep
        self.betas = b
        self._h = lib().orc_create_ex(L, q, float(sigma), n_ens, n_rep, _p(b), int(seed), int(ens_base))
        if not self._h:
            raise ValueError("orc_create: invalid arguments")

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    __del__ = close

    def sweeps(self, n, swap_every=1, field=False, threads=1):
        rc = lib().orc_sweeps(self._h, int(n), int(swap_every), int(bool(field)), int(threads))
        if rc:
            raise ValueError("orc_sweeps: invalid arguments")

    def set_site_order(self, order):
        if lib().orc_set_site_order(self._h, {"sequential": 0, "random": 1}[order]):
            raise ValueError("orc_set_site_order: invalid order")

    def sweeps_arith(self, n, swap_every=1, arith="fp32", threads=1):
        """The paper's floating-point arithmetic as a comparison mode (fp32 or fp64 sums of dE)."""
        rc = lib().orc_sweeps_arith(self._h, int(n), int(swap_every), {"fp32": 1, "fp64": 2}[arith], int(threads))
        if rc:
            raise ValueError("orc_sweeps_arith: invalid arguments (or the context is in the other mode)")

    def delta_e_arith(self, ens, slot, i, b, arith):
        return lib().orc_delta_e_arith(self._h, ens, slot, i, b, {"fp32": 1, "fp64": 2}[arith])

    def energy(self, recompute=False):
        E = np.zeros((self.n_ens, self.n_rep), dtype=np.int64)
        lib().orc_energy(self._h, _p(E), int(bool(recompute)))
        return E

    def observables(self):
        arr = (Obs * (self.n_ens * self.n_rep))()
        lib().orc_observables(self._h, ctypes.byref(arr))
        out = {}
        for name in OBS_FIELDS:
            if name == "sum_E4":   # [n_ens, n_rep, 4] little-endian 64-bit limbs
                out[name] = np.array([list(o.sum_E4) for o in arr], dtype=np.uint64).reshape(self.n_ens, self.n_rep, 4)
                continue
            dt = np.uint64 if name in ("sum_E2_lo", "sum_Nmax4_lo") else np.int64
            out[name] = np.array([getattr(o, name) for o in arr], dtype=dt).reshape(self.n_ens, self.n_rep)
        return out

    def get_spins(self):
        s = np.zeros((self.n_ens, self.n_rep, self.L), dtype=np.uint8)
        lib().orc_get_spins(self._h, _p(s))
        return s

    def set_spins(self, spins):
        s = np.ascontiguousarray(spins, dtype=np.uint8)
        if s.size != self.n_ens * self.n_rep * self.L:
            raise ValueError("spins must have n_ens*n_rep*L entries")
        if lib().orc_set_spins(self._h, _p(s)):
            raise ValueError("orc_set_spins: colour outside 1..q")

    def get_couplings(self):
        J = np.zeros(self.L, dtype=np.int32)
        lib().orc_get_couplings(self._h, _p(J))
        return J

    def sweep_counter(self):
        return lib().orc_sweep_counter(self._h)

    def delta_e(self, ens, slot, i, b):
        return lib().orc_delta_e(self._h, ens, slot, i, b)
