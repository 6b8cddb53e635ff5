"""Thin Python binding of libbd (include/bd.h): argument marshalling only.

Same names as the C ABI (bd_create -> BD(...), bd_assemble_hi -> BD.assemble_hi, ...).  Every step of
the path runs in the CUDA kernels of libbd.so; torch is used for device memory and streams only.
There is no CPU fallback: without the built library or without a CUDA device this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

NOBS = 13
OBS_NAMES = ("R2", "Rx2", "Ry2", "Rz2", "Rg2", "Sxx", "Syy", "Szz", "Sxy", "Sxz", "Syz",
             "rod_dev_ms", "rod_dev_max")
ERR_CUDA, ERR_WORKSPACE, ERR_ALLOC, ERR_INTERNAL, ERR_TOO_LARGE = -100, -101, -102, -103, -104


class bd_params(C.Structure):
    _fields_ = [("n_rods", C.c_int32), ("n_chains", C.c_int32), ("b", C.c_double), ("hstar", C.c_double),
                ("a", C.c_double), ("K", C.c_double), ("dt", C.c_double), ("kappa", C.c_double * 9),
                ("seed", C.c_uint64), ("chain_id0", C.c_uint64), ("noise_kind", C.c_int32), ("spring_kind", C.c_int32),
                ("nu", C.c_double)]


EXPORTS = ("bd_create", "bd_destroy", "bd_workspace_bytes", "bd_set_workspace", "bd_set_flow",
           "bd_init_random_walk", "bd_assemble_hi", "bd_cholesky", "bd_cholesky_noalloc", "bd_brownian", "bd_noise", "bd_drift",
           "bd_update", "bd_set_path", "bd_set_cholesky", "bd_step", "bd_observables", "bd_end_to_end", "bd_autocorr", "bd_last_info", "bd_step_host", "bd_profile",
           "bd_stage_ms", "bd_launch_count", "bd_strerror", "bd_last_error")

_lib = None


def load_library(path: str | None = None) -> C.CDLL:
    """dlopen libbd.so (building it in-tree first if sources are newer) and declare the signatures."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _build.build_lib()
    if not os.path.exists(p):
        raise RuntimeError(f"libbd.so not found at {p}: the CUDA extension is required (no CPU fallback)")
    lib = C.CDLL(p)
    vp, i32, i64, u64, dp = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_void_p
    lib.bd_create.argtypes = [C.POINTER(bd_params), vp, C.POINTER(vp)]
    lib.bd_destroy.argtypes = [vp]
    lib.bd_workspace_bytes.argtypes = [vp]
    lib.bd_workspace_bytes.restype = C.c_size_t
    lib.bd_set_workspace.argtypes = [vp, dp, C.c_size_t]
    lib.bd_set_flow.argtypes = [vp, C.POINTER(C.c_double)]
    lib.bd_init_random_walk.argtypes = [vp, dp, u64]
    lib.bd_assemble_hi.argtypes = [vp, dp, dp, i64, i64, i32]
    lib.bd_cholesky.argtypes = [vp, dp, i64, i64, dp]
    lib.bd_cholesky_noalloc.argtypes = [dp, i32, i32, i64, i64, dp, vp]
    lib.bd_brownian.argtypes = [vp, dp, i64, i64, u64, dp, dp]
    lib.bd_noise.argtypes = [vp, u64, dp]
    lib.bd_drift.argtypes = [vp, dp, dp, dp, dp]
    lib.bd_update.argtypes = [vp, dp, dp, dp, dp]
    lib.bd_set_path.argtypes = [vp, i32]
    lib.bd_set_cholesky.argtypes = [vp, i32]
    lib.bd_step.argtypes = [vp, dp, u64, i32]
    lib.bd_observables.argtypes = [vp, dp, dp, dp]
    lib.bd_end_to_end.argtypes = [vp, dp, dp]
    lib.bd_autocorr.argtypes = [vp, dp, dp, dp]
    lib.bd_last_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i32)]
    lib.bd_step_host.argtypes = [vp, dp, u64, i32, dp]
    lib.bd_profile.argtypes = [vp, i32]
    lib.bd_stage_ms.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i64)]
    lib.bd_launch_count.argtypes = [vp]
    lib.bd_launch_count.restype = i64
    lib.bd_strerror.argtypes = [C.c_int]
    lib.bd_strerror.restype = C.c_char_p
    lib.bd_last_error.argtypes = [vp]
    lib.bd_last_error.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("bd_workspace_bytes", "bd_launch_count", "bd_strerror", "bd_last_error"):
            getattr(lib, name).restype = C.c_int
    if path is None:
        _lib = lib
    return lib


class BDError(RuntimeError):
    def __init__(self, fn: str, code: int, text: str):
        super().__init__(f"{fn} failed with code {code}: {text}")
        self.code = code


def _dptr(t):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor")
    return C.c_void_p(t.data_ptr())


def cholesky_noalloc(DL: torch.Tensor, info: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None):
    """bd_cholesky_noalloc: in-place tile Cholesky of DL [C][M][ld] (lower triangle) with the library's fixed scratch array;
    no context, no allocation.  Limit C * ceil(M / 128) <= 32; calls that overlap on the GPU race (one shared array)."""
    lib = load_library()
    Cn, M, ld = int(DL.shape[0]), int(DL.shape[1]), int(DL.shape[2])
    st = stream if stream is not None else torch.cuda.current_stream(DL.device)
    rc = lib.bd_cholesky_noalloc(_dptr(DL), M, Cn, ld, ld * M, _dptr(info), C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise BDError("bd_cholesky_noalloc", rc, lib.bd_strerror(rc).decode())
    return DL


class BD:
    """One libbd context (one CUDA stream).  Parameters follow the paper's problem statement."""

    def __init__(self, n_rods: int, n_chains: int, dt: float, hstar: float = 0.25, b: float = 1.0,
                 a: float = -1.0, K: float = -1.0, kappa=None, seed: int = 0, chain_id0: int = 0,
                 noise_kind: int = 0, spring_kind: int = 0, nu: float = 0.0, stream: torch.cuda.Stream | None = None,
                 device: str = "cuda:0"):
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("libbd needs a CUDA device (B200): there is no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        p = bd_params()
        p.n_rods, p.n_chains = int(n_rods), int(n_chains)
        p.b, p.hstar, p.a, p.K, p.dt = float(b), float(hstar), float(a), float(K), float(dt)
        k = np.zeros(9) if kappa is None else np.asarray(kappa, dtype=np.float64).reshape(9)
        for i in range(9):
            p.kappa[i] = float(k[i])
        p.seed, p.chain_id0, p.noise_kind = int(seed), int(chain_id0), int(noise_kind)
        p.spring_kind, p.nu = int(spring_kind), float(nu)
        self.params = p
        self.N, self.C, self.M = int(n_rods), int(n_chains), 3 * (int(n_rods) + 1)
        self._ctx = C.c_void_p()
        self._check("bd_create", self.lib.bd_create(C.byref(p), C.c_void_p(self.stream.cuda_stream), C.byref(self._ctx)))
        self._ws = None

    # ------------------------------------------------------------------ helpers
    def _check(self, fn: str, rc: int):
        if rc != 0:
            text = self.lib.bd_strerror(rc).decode()
            if rc == ERR_CUDA and getattr(self, "_ctx", None) is not None and self._ctx.value:
                text = self.lib.bd_last_error(self._ctx).decode()
            raise BDError(fn, rc, text)

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.bd_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def empty(self, *shape, dtype=torch.float64):
        return torch.empty(*shape, dtype=dtype, device=self.device)

    @property
    def ld(self) -> int:
        return (self.M + 15) // 16 * 16

    def matrix_storage(self, ld: int | None = None):
        """caller-owned D/L storage [C][M][ld] (row-major, lower triangle used)."""
        return self.empty(self.C, self.M, ld or self.ld)

    # ------------------------------------------------------------------ C ABI, same names
    def workspace_bytes(self) -> int:
        return int(self.lib.bd_workspace_bytes(self._ctx))

    def set_workspace(self, ws: torch.Tensor | None = None):
        if ws is None:
            ws = torch.empty(self.workspace_bytes() // 8, dtype=torch.float64, device=self.device)
        self._check("bd_set_workspace", self.lib.bd_set_workspace(self._ctx, _dptr(ws), ws.numel() * ws.element_size()))
        self._ws = ws
        return ws

    def set_flow(self, kappa):
        k = (C.c_double * 9)(*[float(x) for x in np.asarray(kappa, dtype=np.float64).reshape(9)])
        self._check("bd_set_flow", self.lib.bd_set_flow(self._ctx, k))

    def init_random_walk(self, init_seed: int, r: torch.Tensor | None = None):
        r = self.empty(self.C, self.N + 1, 3) if r is None else r
        self._check("bd_init_random_walk", self.lib.bd_init_random_walk(self._ctx, _dptr(r), init_seed))
        return r

    def assemble_hi(self, r, D=None, full: bool = False, chain_stride: int | None = None):
        D = self.matrix_storage() if D is None else D
        ld = D.shape[-1]
        self._check("bd_assemble_hi", self.lib.bd_assemble_hi(self._ctx, _dptr(r), _dptr(D), ld, chain_stride or ld * self.M, int(full)))
        return D

    def cholesky(self, DL, info: torch.Tensor | None = None, chain_stride: int | None = None):
        ld = DL.shape[-1]
        self._check("bd_cholesky", self.lib.bd_cholesky(self._ctx, _dptr(DL), ld, chain_stride or ld * self.M, _dptr(info)))
        return DL

    def noise(self, step: int, dW=None):
        dW = self.empty(self.C, self.M) if dW is None else dW
        self._check("bd_noise", self.lib.bd_noise(self._ctx, step, _dptr(dW)))
        return dW

    def brownian(self, L, step: int = 0, dW=None, y=None, chain_stride: int | None = None):
        y = self.empty(self.C, self.M) if y is None else y
        ld = L.shape[-1]
        self._check("bd_brownian", self.lib.bd_brownian(self._ctx, _dptr(L), ld, chain_stride or ld * self.M, step, _dptr(dW), _dptr(y)))
        return y

    def drift(self, r):
        T, F, v = self.empty(self.C, self.N, 3), self.empty(self.C, self.N + 1, 3), self.empty(self.C, self.M)
        self._check("bd_drift", self.lib.bd_drift(self._ctx, _dptr(r), _dptr(T), _dptr(F), _dptr(v)))
        return T, F, v

    def update(self, r, v, y, r_out=None):
        r_out = torch.empty_like(r) if r_out is None else r_out
        self._check("bd_update", self.lib.bd_update(self._ctx, _dptr(r), _dptr(v), _dptr(y), _dptr(r_out)))
        return r_out

    def set_path(self, path: int):
        """0 auto, 1 staged kernels, 2 fused per-chain kernel."""
        self._check("bd_set_path", self.lib.bd_set_path(self._ctx, int(path)))

    def set_cholesky(self, algo: int):
        """0 auto, 1 multi-launch blocked factorisation, 2 persistent tile kernel."""
        self._check("bd_set_cholesky", self.lib.bd_set_cholesky(self._ctx, int(algo)))

    def step(self, r, first_step: int = 0, n_steps: int = 1):
        if self._ws is None:
            self.set_workspace()
        self._check("bd_step", self.lib.bd_step(self._ctx, _dptr(r), first_step, n_steps))
        return r

    def observables(self, r):
        per, ens = self.empty(self.C, NOBS), self.empty(2, NOBS)
        self._check("bd_observables", self.lib.bd_observables(self._ctx, _dptr(r), _dptr(per), _dptr(ens)))
        return per, ens

    def end_to_end(self, r, R=None):
        R = self.empty(self.C, 3) if R is None else R
        self._check("bd_end_to_end", self.lib.bd_end_to_end(self._ctx, _dptr(r), _dptr(R)))
        return R

    def autocorr(self, r, R0, out=None):
        """device tensor [3]: sum_c R.R0, sum_c (R.R0)^2, sum_c R0.R0."""
        out = self.empty(3) if out is None else out
        self._check("bd_autocorr", self.lib.bd_autocorr(self._ctx, _dptr(r), _dptr(R0), _dptr(out)))
        return out

    def last_info(self):
        n, first = C.c_int32(0), C.c_int32(-1)
        self._check("bd_last_info", self.lib.bd_last_info(self._ctx, C.byref(n), C.byref(first)))
        return int(n.value), int(first.value)

    def step_host(self, r_host: torch.Tensor, first_step: int = 0, n_steps: int = 1, ensemble_host: torch.Tensor | None = None):
        """HOST buffers (pinned recommended): H2D, n_steps, observables, D2H inside the call."""
        if self._ws is None:
            self.set_workspace()
        assert (not r_host.is_cuda) and r_host.is_contiguous() and r_host.dtype == torch.float64
        eh = C.c_void_p(ensemble_host.data_ptr()) if ensemble_host is not None else None
        self._check("bd_step_host", self.lib.bd_step_host(self._ctx, C.c_void_p(r_host.data_ptr()), first_step, n_steps, eh))
        return r_host

    STAGES = ("drift", "assemble", "cholesky", "noise", "brownian", "update", "fused")

    def profile(self, enable: bool = True):
        self._check("bd_profile", self.lib.bd_profile(self._ctx, int(enable)))

    def stage_ms(self):
        """(dict stage -> accumulated ms, steps covered); synchronises and resets."""
        ms = (C.c_double * 7)()
        n = C.c_int64(0)
        self._check("bd_stage_ms", self.lib.bd_stage_ms(self._ctx, ms, C.byref(n)))
        return dict(zip(self.STAGES, [float(x) for x in ms])), int(n.value)

    def launch_count(self) -> int:
        return int(self.lib.bd_launch_count(self._ctx))
