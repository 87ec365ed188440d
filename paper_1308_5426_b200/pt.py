"""Thin ctypes binding of libpt.so (include/pt.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  There is no
CPU fallback: a missing libpt.so raises at import, a missing GPU raises PTError
(PT_ECUDA) from pt_create.  PyTorch, when importable, supplies the CUDA stream
(`PT.use_torch_stream`) and device buffers for the *_dev calls.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# PT_LIBPT=<path> loads another build of the same library (development builds: -DPT_PARANOID, -DPT_TIMING)
LIB_PATH = os.environ.get("PT_LIBPT") or os.path.join(_HERE, "libpt.so")

VARIANT_AUTO, VARIANT_FIELD, VARIANT_DIRECT, VARIANT_FP32, VARIANT_FP64 = 0, 1, 2, 3, 4
_VARIANTS = {"auto": VARIANT_AUTO, "field": VARIANT_FIELD, "direct": VARIANT_DIRECT, "fp32": VARIANT_FP32,
             "fp64": VARIANT_FP64}
STATUS = {0: "PT_OK", -1: "PT_EINVAL", -2: "PT_EOVERFLOW", -3: "PT_ENOMEM", -4: "PT_ECUDA", -5: "PT_ECAPACITY"}

# every symbol include/pt.h declares
SYMBOLS = ["pt_create", "pt_create_ex", "pt_destroy", "pt_sweeps", "pt_energy", "pt_energy_dev",
           "pt_observables", "pt_get_spins", "pt_get_spins_dev", "pt_set_spins", "pt_get_couplings",
           "pt_sweep_counter", "pt_set_variant", "pt_get_variant", "pt_set_stream", "pt_sweeps_async",
           "pt_sync", "pt_last_error", "pt_create_shard", "pt_energy_storage_dev", "pt_swap_external",
           "pt_get_perm", "pt_measure_peaks", "pt_get_state", "pt_set_state", "pt_set_site_order",
           "pt_energy_storage_dev_async", "pt_swap_external_async", "pt_energy_static", "pt_describe"]


class PTError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s (%d): %s" % (STATUS.get(code, "?"), code, msg))
        self.code = code


class Obs(ctypes.Structure):  # pt_obs
    _fields_ = [("n_samples", ctypes.c_int64), ("sum_E", ctypes.c_int64),
                ("sum_E2_lo", ctypes.c_uint64), ("sum_E2_hi", ctypes.c_int64),
                ("sum_Nmax", ctypes.c_int64), ("sum_Nmax2", ctypes.c_int64),
                ("flip_attempts", ctypes.c_int64), ("flip_accepts", ctypes.c_int64),
                ("swap_attempts", ctypes.c_int64), ("swap_accepts", ctypes.c_int64),
                ("near_ties", ctypes.c_int64),
                ("sum_E4", ctypes.c_uint64 * 4), ("sum_Nmax3", ctypes.c_int64),
                ("sum_Nmax4_lo", ctypes.c_uint64), ("sum_Nmax4_hi", ctypes.c_int64)]


OBS_FIELDS = [f[0] for f in Obs._fields_]
# the same 144-byte record as a numpy structured type (argument marshalling without a Python loop per record)
OBS_DTYPE = np.dtype([(n, (np.uint64, (4,)) if n == "sum_E4" else
                      (np.uint64 if n in ("sum_E2_lo", "sum_Nmax4_lo") else np.int64)) for n in OBS_FIELDS])
assert OBS_DTYPE.itemsize == ctypes.sizeof(Obs)

if not os.path.exists(LIB_PATH):
    raise ImportError("libpt.so is not built (run `python -m paper_1308_5426_b200.build`); "
                      "there is no CPU fallback")

_lib = ctypes.CDLL(LIB_PATH)
_vp, _i32, _i64, _u64, _dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_uint64, ctypes.c_double
_lib.pt_create.argtypes = [ctypes.POINTER(_vp), _i32, _i32, _dbl, _i32, _i32, _vp, _u64]
_lib.pt_create_ex.argtypes = [ctypes.POINTER(_vp), _i32, _i32, _dbl, _i32, _i32, _vp, _u64, _i32]
_lib.pt_create_shard.argtypes = [ctypes.POINTER(_vp), _i32, _i32, _dbl, _i32, _vp, _u64, _i32, _i32, _i32]
_lib.pt_energy_storage_dev.argtypes = [_vp, _vp]
_lib.pt_swap_external.argtypes = [_vp, _vp]
_lib.pt_get_perm.argtypes = [_vp, _vp]
_lib.pt_destroy.argtypes = [_vp]
_lib.pt_destroy.restype = None
_lib.pt_sweeps.argtypes = [_vp, _i64, _i32]
_lib.pt_sweeps_async.argtypes = [_vp, _i64, _i32, ctypes.POINTER(_i64)]
_lib.pt_sync.argtypes = [_vp]
_lib.pt_energy.argtypes = [_vp, _vp, _i32]
_lib.pt_energy_dev.argtypes = [_vp, _vp, _i32]
_lib.pt_observables.argtypes = [_vp, _vp]
_lib.pt_get_spins.argtypes = [_vp, _vp]
_lib.pt_get_spins_dev.argtypes = [_vp, _vp]
_lib.pt_set_spins.argtypes = [_vp, _vp]
_lib.pt_get_couplings.argtypes = [_vp, _vp]
_lib.pt_sweep_counter.argtypes = [_vp]
_lib.pt_sweep_counter.restype = _i64
_lib.pt_set_variant.argtypes = [_vp, _i32]
_lib.pt_get_variant.argtypes = [_vp]
_lib.pt_describe.argtypes = [_vp, ctypes.c_char_p, ctypes.c_int]
_lib.pt_set_stream.argtypes = [_vp, _vp]
_lib.pt_last_error.restype = ctypes.c_char_p
_lib.pt_measure_peaks.argtypes = [_vp, _i32]
_lib.pt_get_state.argtypes = [_vp, _vp, _vp, _vp, ctypes.POINTER(_i64)]
_lib.pt_set_state.argtypes = [_vp, _vp, _vp, _vp, _i64]
_lib.pt_set_site_order.argtypes = [_vp, _i32]
_lib.pt_energy_storage_dev_async.argtypes = [_vp, _vp]
_lib.pt_swap_external_async.argtypes = [_vp, _vp]
_lib.pt_energy_static.argtypes = [_i32, _i32, _dbl, _vp, _i32, _vp, _vp, _vp]
STATIC_MAX_L, STATIC_MAX_SITES = 16384, 1048576     # PT_STATIC_MAX_L, PT_STATIC_MAX_SITES of include/pt.h

PEAK_PATTERNS = ["idp2a", "idp4a", "imad", "prmt", "lop3", "prmt+2idp2a (idp2a counted)", "lop3+2idp2a (idp2a counted)",
                 "lds128 (bytes)", "prmt+4idp2a (idp2a counted)", "2prmt+add+2idp2a (idp2a counted)",
                 "bulk tile, near form (idp2a counted)", "bulk tile, far form (idp4a counted)"]


def measure_peaks():
    """pt_measure_peaks: {pattern: [rate with 1, 2, 3, 4 warps per sub-partition]} in lane-operations per clock and SM."""
    r = np.zeros(len(PEAK_PATTERNS) * 4, dtype=np.float64)
    _check(_lib.pt_measure_peaks(_p(r), int(r.size)))
    return {name: [float(x) for x in r[4 * i:4 * i + 4]] for i, name in enumerate(PEAK_PATTERNS)}


def energy_static(L, q, sigma, spins_dev, n_conf, E_out_dev, status_dev=None, cuda_stream_ptr=None):
    """pt_energy_static: energies of n_conf caller-supplied configurations, allocation-free (shared static scratch:
    overlapping calls race).  spins_dev / E_out_dev / status_dev: objects with .data_ptr() on the current device
    (uint8 [n_conf, L], int64 [n_conf], int32 [1] or None).  Enqueues on the stream and returns."""
    _check(_lib.pt_energy_static(int(L), int(q), float(sigma), ctypes.c_void_p(spins_dev.data_ptr()), int(n_conf),
                                 ctypes.c_void_p(E_out_dev.data_ptr()),
                                 ctypes.c_void_p(status_dev.data_ptr()) if status_dev is not None else None,
                                 ctypes.c_void_p(int(cuda_stream_ptr)) if cuda_stream_ptr else None))


def _check(rc):
    if rc != 0:
        raise PTError(rc, (_lib.pt_last_error() or b"").decode())


def _p(a):
    return a.ctypes.data_as(_vp)


class PT:
    """One libpt context: n_ens ensembles x n_rep replicas of the (L, q, sigma) model."""

    def __init__(self, L, q, sigma, n_ens, n_rep, betas, seed, ens_base=0, variant="auto", shard=None):
        """shard = (rep_base, n_local): slot-sharded context (pt_create_shard; one ensemble)."""
        b = np.ascontiguousarray(betas, dtype=np.float64)
        if b.ndim != 1 or b.shape[0] != n_rep:
            raise ValueError("betas must have n_rep entries")
        self.L, self.q, self.n_ens, self.n_rep = int(L), int(q), int(n_ens), int(n_rep)
        self.betas = b
        self.shard = None if shard is None else (int(shard[0]), int(shard[1]))
        self._h = _vp()
        if self.shard is None:
            _check(_lib.pt_create_ex(ctypes.byref(self._h), int(L), int(q), float(sigma), int(n_ens), int(n_rep),
                                     _p(b), int(seed) & 0xFFFFFFFFFFFFFFFF, int(ens_base)))
        else:
            if n_ens != 1:
                raise ValueError("a slot-sharded context holds one ensemble")
            _check(_lib.pt_create_shard(ctypes.byref(self._h), int(L), int(q), float(sigma), int(n_rep), _p(b),
                                        int(seed) & 0xFFFFFFFFFFFFFFFF, int(ens_base), self.shard[0], self.shard[1]))
        if variant != "auto":
            self.set_variant(variant)

    def close(self):
        if getattr(self, "_h", None):
            _lib.pt_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- the calls of include/pt.h ------------------------------------------------
    def sweeps(self, n, swap_every=1):
        _check(_lib.pt_sweeps(self._h, int(n), int(swap_every)))

    def sweeps_async(self, n, swap_every=1):
        k = _i64(0)
        _check(_lib.pt_sweeps_async(self._h, int(n), int(swap_every), ctypes.byref(k)))
        return k.value

    def sync(self):
        _check(_lib.pt_sync(self._h))

    def energy(self, recompute=False):
        E = np.zeros((self.n_ens, self.n_rep), dtype=np.int64)
        _check(_lib.pt_energy(self._h, _p(E), int(bool(recompute))))
        return E

    def energy_dev(self, out, recompute=False):
        """out: torch int64 CUDA tensor with n_ens*n_rep elements (device pointer passed through)."""
        assert out.is_cuda and out.numel() == self.n_ens * self.n_rep and out.element_size() == 8
        _check(_lib.pt_energy_dev(self._h, ctypes.c_void_p(out.data_ptr()), int(bool(recompute))))
        return out

    def energy_storage_dev(self, out):
        """Slot-sharded contexts: out = torch int64 CUDA tensor with n_local elements (storage order)."""
        assert out.is_cuda and out.element_size() == 8
        _check(_lib.pt_energy_storage_dev(self._h, ctypes.c_void_p(out.data_ptr())))
        return out

    def swap_external(self, E_all):
        """Slot-sharded contexts: E_all = torch int64 CUDA tensor, energies of all n_rep configurations, storage order."""
        assert E_all.is_cuda and E_all.numel() == self.n_rep and E_all.element_size() == 8 and E_all.is_contiguous()
        _check(_lib.pt_swap_external(self._h, ctypes.c_void_p(E_all.data_ptr())))

    def energy_storage_dev_async(self, out):
        assert out.is_cuda and out.element_size() == 8
        _check(_lib.pt_energy_storage_dev_async(self._h, ctypes.c_void_p(out.data_ptr())))
        return out

    def swap_external_async(self, E_all):
        assert E_all.is_cuda and E_all.numel() == self.n_rep and E_all.element_size() == 8 and E_all.is_contiguous()
        _check(_lib.pt_swap_external_async(self._h, ctypes.c_void_p(E_all.data_ptr())))

    def get_perm(self):
        perm = np.zeros((self.n_ens, self.n_rep), dtype=np.int32)
        _check(_lib.pt_get_perm(self._h, _p(perm)))
        return perm

    def observables(self):
        rec = np.zeros(self.n_ens * self.n_rep, dtype=OBS_DTYPE)
        _check(_lib.pt_observables(self._h, _p(rec)))
        out = {}
        for name in OBS_FIELDS:   # sum_E4: [n_ens, n_rep, 4] little-endian 64-bit limbs of a 256-bit integer
            shape = (self.n_ens, self.n_rep, 4) if name == "sum_E4" else (self.n_ens, self.n_rep)
            out[name] = np.ascontiguousarray(rec[name]).reshape(shape)
        return out

    def get_spins(self):
        s = np.zeros((self.n_ens, self.n_rep, self.L), dtype=np.uint8)
        _check(_lib.pt_get_spins(self._h, _p(s)))
        return s

    def get_spins_dev(self, out):
        assert out.is_cuda and out.numel() == self.n_ens * self.n_rep * self.L and out.element_size() == 1
        _check(_lib.pt_get_spins_dev(self._h, ctypes.c_void_p(out.data_ptr())))
        return out

    def set_spins(self, spins):
        s = np.ascontiguousarray(spins, dtype=np.uint8)
        if s.size != self.n_ens * self.n_rep * self.L:
            raise ValueError("spins must have n_ens*n_rep*L entries")
        _check(_lib.pt_set_spins(self._h, _p(s)))

    def get_state(self):
        """pt_get_state: (spins uint8 [n_ens, n_rep, L], E int64 [n_ens, n_rep], obs raw ctypes array, sweep)."""
        s = np.zeros((self.n_ens, self.n_rep, self.L), dtype=np.uint8)
        E = np.zeros((self.n_ens, self.n_rep), dtype=np.int64)
        obs = (Obs * (self.n_ens * self.n_rep))()
        sw = _i64(0)
        _check(_lib.pt_get_state(self._h, _p(s), _p(E), ctypes.byref(obs), ctypes.byref(sw)))
        return s, E, obs, sw.value

    def set_state(self, spins, E=None, obs=None, sweep=0):
        """pt_set_state: E None -> recount from the spins; obs None -> keep the accumulators."""
        s = np.ascontiguousarray(spins, dtype=np.uint8)
        if s.size != self.n_ens * self.n_rep * self.L:
            raise ValueError("spins must have n_ens*n_rep*L entries")
        Ea = None if E is None else np.ascontiguousarray(E, dtype=np.int64)
        _check(_lib.pt_set_state(self._h, _p(s), None if Ea is None else _p(Ea),
                                 None if obs is None else ctypes.byref(obs), int(sweep)))

    def get_couplings(self):
        J = np.zeros(self.L, dtype=np.int32)
        _check(_lib.pt_get_couplings(self._h, _p(J)))
        return J

    def sweep_counter(self):
        return int(_lib.pt_sweep_counter(self._h))

    def set_variant(self, variant):
        _check(_lib.pt_set_variant(self._h, _VARIANTS[variant] if isinstance(variant, str) else int(variant)))

    def set_site_order(self, order):
        """'sequential' (default) or 'random' (pt_set_site_order; random order selects the field variant)."""
        _check(_lib.pt_set_site_order(self._h, {"sequential": 0, "random": 1}[order]))

    def get_variant(self):
        v = _lib.pt_get_variant(self._h)
        return {VARIANT_FIELD: "field", VARIANT_DIRECT: "direct", VARIANT_FP32: "fp32", VARIANT_FP64: "fp64"}.get(v, str(v))

    def describe(self):
        """pt_describe: the launch plan of the context as one line of text."""
        buf = ctypes.create_string_buffer(256)
        _check(_lib.pt_describe(self._h, buf, 256))
        return buf.value.decode()

    def set_stream(self, cuda_stream_ptr):
        _check(_lib.pt_set_stream(self._h, ctypes.c_void_p(int(cuda_stream_ptr) if cuda_stream_ptr else None)))

    def use_torch_stream(self, stream=None):
        """Run this context's kernels on a torch.cuda stream (default: the current one)."""
        import torch
        s = stream if stream is not None else torch.cuda.current_stream()
        self.set_stream(s.cuda_stream)
        return s

