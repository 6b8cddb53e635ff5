"""The C-ABI boundary (no GPU needed): libbd.so builds/loads, exports every symbol include/bd.h
declares, the Python binding declares the same names, and the product path fails loudly (no CPU
fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "bd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(bd_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for must in ("bd_create", "bd_assemble_hi", "bd_cholesky", "bd_brownian", "bd_step", "bd_observables"):
        assert must in names


def test_library_exports_every_declared_symbol():
    from paper_2208_06559_b200 import build
    lib = C.CDLL(build.build_lib())
    for name in _declared():
        assert hasattr(lib, name), name


def test_binding_covers_every_declared_symbol():
    from paper_2208_06559_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()
    assert C.sizeof(binding.bd_params) == 4 + 4 + 8 * 5 + 8 * 9 + 8 + 8 + 4 + 4 + 8      # matches the C struct layout


def test_header_has_no_torch_or_cxx_types():
    text = open(os.path.join(ROOT, "include", "bd.h")).read()
    assert "torch" not in text.lower().replace("torch tensor", "") and "std::" not in text and 'extern "C"' in text


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback_without_a_gpu():
    from paper_2208_06559_b200 import binding
    with pytest.raises(RuntimeError):
        binding.BD(n_rods=5, n_chains=1, dt=1e-4)
    lib = binding.load_library()
    p = binding.bd_params()
    p.n_rods, p.n_chains, p.b, p.hstar, p.a, p.K, p.dt = 5, 1, 1.0, 0.25, -1.0, -1.0, 1e-4
    ctx = C.c_void_p()
    assert lib.bd_create(C.byref(p), None, C.byref(ctx)) == binding.ERR_CUDA
    assert ctx.value is None
    assert lib.bd_step(None, None, 0, 1) == -1
    # the context-free entry point validates its arguments before touching the device
    assert lib.bd_cholesky_noalloc(None, 10, 1, 10, 100, None, None) == -1
    buf = C.create_string_buffer(64)
    addr = (C.addressof(buf) + 15) // 16 * 16
    assert lib.bd_cholesky_noalloc(C.c_void_p(addr), 0, 1, 10, 100, None, None) == -2
    assert lib.bd_cholesky_noalloc(C.c_void_p(addr), 10, 0, 10, 100, None, None) == -3
    assert lib.bd_cholesky_noalloc(C.c_void_p(addr), 10, 1, 9, 100, None, None) == -4
    assert lib.bd_cholesky_noalloc(C.c_void_p(addr), 10, 1, 10, 99, None, None) == -5
    assert lib.bd_cholesky_noalloc(C.c_void_p(addr), 128, 33, 128, 128 * 128, None, None) == binding.ERR_TOO_LARGE
    assert b"32" in lib.bd_strerror(binding.ERR_TOO_LARGE)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2208_06559_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "bd_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "#include" not in src or "bd.h\"" not in src.replace("bd_oracle.h\"", ""), f
            assert "import paper_2208" not in src and "from paper_2208" not in src, f


def test_user_scripts_import_and_fail_loudly_without_a_gpu():
    """nsweep / run_config / relaxation / variant_sweep are thin drivers of the binding: importable on a CPU box, and they raise
    (no fallback) as soon as they need a context."""
    import importlib
    import torch
    for name in ("nsweep", "run_config", "relaxation", "variant_sweep"):
        mod = importlib.import_module(f"paper_2208_06559_b200.{name}")
        assert hasattr(mod, "main")
    if not torch.cuda.is_available():
        from paper_2208_06559_b200 import relaxation
        with pytest.raises(RuntimeError):
            relaxation.measure(5, 2, 0.25, 1e-3, 0.1, 2)


def test_relaxation_fit_stops_at_the_noise_floor():
    """host logic of relaxation.py: lambda from the last 70 % of the RESOLVED part of C(t).  A synthetic
    exp(-t / lambda) with ensemble noise 1 / sqrt(chains), recorded far beyond its decay, must return lambda -- a fit over
    the whole window returns the window length instead (what the first version did for the runs with HI)."""
    import math
    import numpy as np
    from paper_2208_06559_b200.relaxation import fit_tail
    rng = np.random.default_rng(5)
    t = np.linspace(0.0, 440.0, 201)
    for lam in (25.0, 90.0, 280.0):
        acf = np.exp(-t / lam) + rng.normal(0.0, 1.0 / math.sqrt(2048), t.size)
        acf[0] = 1.0
        fit, t_cut = fit_tail(t, acf, 2048)
        assert abs(fit - lam) <= 0.08 * lam
        assert t_cut <= min(440.0, 3.5 * lam)
