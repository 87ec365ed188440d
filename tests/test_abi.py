"""CPU-side checks of the boundary: libpt.so builds, loads, and exports every symbol
include/pt.h declares; without a GPU the product fails loudly (no CPU path)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1308_5426_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "pt.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pt_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib_path):
    lib = ctypes.CDLL(lib_path)
    names = declared_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), "libpt.so does not export " + n


def test_binding_lists_every_symbol(lib_path):
    from paper_1308_5426_b200 import pt
    assert sorted(pt.SYMBOLS) == declared_symbols()
    assert ctypes.sizeof(pt.Obs) == 144


def test_no_cpu_fallback(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("box has a GPU")
    from paper_1308_5426_b200 import pt
    with pytest.raises(pt.PTError) as ei:
        pt.PT(64, 3, 0.5, 1, 2, [1.0, 0.5], 1)
    assert ei.value.code == -4  # PT_ECUDA


def test_argument_validation_before_any_device_work(lib_path):
    from paper_1308_5426_b200 import pt
    for kw in [dict(L=12), dict(q=1), dict(q=65), dict(sigma=-0.5), dict(n_ens=0), dict(betas=[float("inf"), 1.0])]:
        args = dict(L=64, q=3, sigma=0.5, n_ens=1, n_rep=2, betas=[1.0, 0.5], seed=1)
        args.update(kw)
        with pytest.raises(pt.PTError) as ei:
            pt.PT(**args)
        assert ei.value.code == -1


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1308_5426_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|#include\s+[\"<].*oracle|pt_oracle|libpt_oracle",
                                     src, flags=re.M), f


def test_input_recipes():
    from paper_1308_5426_b200 import inputs
    w = inputs.config(3)
    assert (w.L, w.q, w.n_rep, w.sweeps) == (4096, 8, 128, 2000) and w.attempts == 1048576000
    b = inputs.betas(w)
    assert b.shape == (128,) and np.isclose(1 / b[0], 0.6) and np.isclose(1 / b[-1], 2.5)
    assert np.all(np.diff(b) < 0)
    assert len(inputs.config4()) == 40 and len({c.seed for c in inputs.config4()}) == 40


def test_paper_benchmark_recipe():
    """The paper's own run shape: q=3, 400 replicas, temperatures equally spaced."""
    from paper_1308_5426_b200 import inputs
    for L in inputs.PAPER_BENCH_SIZES:
        w = inputs.paper_benchmark(L)
        assert (w.L, w.q, w.n_rep, w.n_ens, w.swap_every, w.ladder) == (L, 3, 400, 1, 1, "uniform")
        T = 1.0 / inputs.betas(w)
        assert T.shape == (400,) and np.isclose(T[0], w.T_lo) and np.isclose(T[-1], w.T_hi)
        assert np.allclose(np.diff(T), (w.T_hi - w.T_lo) / 399, rtol=1e-9)
    assert len({inputs.paper_benchmark(L).seed for L in inputs.PAPER_BENCH_SIZES}) == len(inputs.PAPER_BENCH_SIZES)
    with pytest.raises(ValueError):
        inputs.paper_benchmark(20480)
