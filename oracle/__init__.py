"""CPU ORACLE -- test infrastructure, NOT the product path.

Thin ctypes/numpy wrapper around ``oracle/bd_oracle.c`` (plain C, FP64,
``gcc -O2 -ffp-contract=off``), the step-by-step restatement of the hot path of
/root/reference/PAPER.md.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  It imports nothing from ``paper_2208_06559_b200`` (the CUDA path) and
the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bd_oracle.c")
_HDR = os.path.join(_HERE, "bd_oracle.h")
_LIB = os.path.join(_HERE, "libbd_oracle.so")

NOBS = 13
OBS_NAMES = ("R2", "Rx2", "Ry2", "Rz2", "Rg2", "Sxx", "Syy", "Szz", "Sxy", "Sxz", "Syz",
             "rod_dev_ms", "rod_dev_max")


def build(force: bool = False) -> str:
    """Compile the oracle (gcc, no FMA contraction).  Building the checker is not using it."""
    # BD_ORACLE_SANITIZE=1: a second build with AddressSanitizer + UBSan for checking the checker itself
    # (run the CPU tests with LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0).
    san = bool(os.environ.get("BD_ORACLE_SANITIZE"))
    out = _LIB.replace(".so", "_san.so") if san else _LIB
    stale = (not os.path.exists(out)) or any(
        os.path.getmtime(s) > os.path.getmtime(out) for s in (_SRC, _HDR))
    if force or stale:
        extra = ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] if san else []
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c99", "-shared", "-fPIC", *extra,
               "-o", out, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return out


class _Params(C.Structure):
    _fields_ = [("n_rods", C.c_int32), ("b", C.c_double), ("hstar", C.c_double), ("a", C.c_double),
                ("K", C.c_double), ("dt", C.c_double), ("kappa", C.c_double * 9),
                ("seed", C.c_uint64), ("noise_kind", C.c_int32), ("spring_kind", C.c_int32), ("nu", C.c_double)]


class _Trace(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("T", "F", "D", "L", "dW", "v", "y", "u", "Y")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_u01.restype = C.c_double
        _lib.orc_u01.argtypes = [C.c_uint64]
        for name in ("orc_cholesky", "orc_finish_step", "orc_step", "orc_step_ensemble", "orc_num_threads"):
            getattr(_lib, name).restype = C.c_int32
        _lib.orc_spring_coeff.restype = C.c_double
        _lib.orc_implicit_length.restype = C.c_double
    return _lib


@dataclass
class Params:
    """Physical parameters in the paper's notation."""
    n_rods: int
    dt: float
    hstar: float = 0.25
    b: float = 1.0
    a: float = -1.0          # <= 0: a = hstar * b (reading A3)
    K: float = -1.0          # <= 0: K = 1/dt (reading A6)
    kappa: np.ndarray = field(default_factory=lambda: np.zeros((3, 3)))
    seed: int = 0
    noise_kind: int = 0
    spring_kind: int = 0     # 0 Fraenkel rod (Eq. 3), 1 Cohen-Pade spring (Eq. 4)
    nu: float = 0.0          # Kuhn steps per spring (kind 1)

    def c(self) -> _Params:
        p = _Params()
        p.n_rods = int(self.n_rods)
        p.b = float(self.b)
        p.hstar = float(self.hstar)
        p.a = float(self.a) if self.a > 0 else float(self.hstar) * float(self.b)
        p.K = float(self.K) if self.K > 0 else 1.0 / float(self.dt)
        p.dt = float(self.dt)
        k = np.asarray(self.kappa, dtype=np.float64).reshape(9)
        for i in range(9):
            p.kappa[i] = float(k[i])
        p.seed = int(self.seed)
        p.noise_kind = int(self.noise_kind)
        p.spring_kind = int(self.spring_kind)
        p.nu = float(self.nu)
        return p

    @property
    def M(self) -> int:
        return 3 * (self.n_rods + 1)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def u01(x: int) -> float:
    return float(lib().orc_u01(C.c_uint64(int(x))))


def normals(seed: int, chain: int, step: int, M: int) -> np.ndarray:
    g = np.empty(M, dtype=np.float64)
    lib().orc_normals(C.c_uint64(seed), C.c_uint64(chain), C.c_uint64(step), C.c_int32(M), _ptr(g))
    return g


def uniforms_pm1(seed: int, chain: int, step: int, M: int) -> np.ndarray:
    g = np.empty(M, dtype=np.float64)
    lib().orc_uniforms_pm1(C.c_uint64(seed), C.c_uint64(chain), C.c_uint64(step), C.c_int32(M), _ptr(g))
    return g


def noise_dW(p: Params, chain: int, step: int) -> np.ndarray:
    dW = np.empty(p.M, dtype=np.float64)
    cp = p.c()
    lib().orc_noise_dW(C.byref(cp), C.c_uint64(chain), C.c_uint64(step), _ptr(dW))
    return dW


def init_random_walk(n_rods: int, b: float, init_seed: int, chains) -> np.ndarray:
    """chains: iterable of global chain ids -> r[C][N_b][3]."""
    chains = list(chains)
    r = np.empty((len(chains), n_rods + 1, 3), dtype=np.float64)
    for i, c in enumerate(chains):
        lib().orc_init_random_walk(C.c_int32(n_rods), C.c_double(b), C.c_uint64(init_seed),
                                   C.c_uint64(c), _ptr(r[i]))
    return r


def spring_coeff(p: Params, q: float) -> float:
    """T = spring_coeff(|Q|) * Q (Eq. 3 or Eq. 4)."""
    cp = p.c()
    return float(lib().orc_spring_coeff(C.byref(cp), C.c_double(q)))


def implicit_length(p: Params, Yn: float) -> float:
    """|Q'| from |Y| (Eq. 17, or the Cohen-Pade cubic)."""
    cp = p.c()
    return float(lib().orc_implicit_length(C.byref(cp), C.c_double(Yn)))


def spring_tensions(p: Params, r) -> np.ndarray:
    r = _f64(r)
    T = np.empty((p.n_rods, 3), dtype=np.float64)
    cp = p.c()
    lib().orc_spring_tensions(C.byref(cp), _ptr(r), _ptr(T))
    return T


def bead_forces(n_rods: int, T) -> np.ndarray:
    T = _f64(T)
    F = np.empty((n_rods + 1, 3), dtype=np.float64)
    lib().orc_bead_forces(C.c_int32(n_rods), _ptr(T), _ptr(F))
    return F


def rpy_block(p: Params, ri, rj) -> np.ndarray:
    ri, rj = _f64(ri), _f64(rj)
    B = np.empty((3, 3), dtype=np.float64)
    cp = p.c()
    lib().orc_rpy_block(C.byref(cp), _ptr(ri), _ptr(rj), _ptr(B))
    return B


def assemble(p: Params, r) -> np.ndarray:
    r = _f64(r)
    D = np.empty((p.M, p.M), dtype=np.float64)
    cp = p.c()
    lib().orc_assemble(C.byref(cp), _ptr(r), _ptr(D))
    return D


def cholesky(A):
    """returns (L, info)."""
    A = _f64(A)
    M = A.shape[0]
    L = np.empty((M, M), dtype=np.float64)
    info = lib().orc_cholesky(C.c_int32(M), _ptr(A), _ptr(L))
    return L, int(info)


def symv(D, x) -> np.ndarray:
    D, x = _f64(D), _f64(x).reshape(-1)
    v = np.empty(D.shape[0], dtype=np.float64)
    lib().orc_symv(C.c_int32(D.shape[0]), _ptr(D), _ptr(x), _ptr(v))
    return v


def trmv_lower(L, x) -> np.ndarray:
    L, x = _f64(L), _f64(x).reshape(-1)
    y = np.empty(L.shape[0], dtype=np.float64)
    lib().orc_trmv_lower(C.c_int32(L.shape[0]), _ptr(L), _ptr(x), _ptr(y))
    return y


def drift_onthefly(p: Params, r, F) -> np.ndarray:
    r, F = _f64(r), _f64(F)
    v = np.empty(p.M, dtype=np.float64)
    cp = p.c()
    lib().orc_drift_onthefly(C.byref(cp), _ptr(r), _ptr(F), _ptr(v))
    return v


def finish_step(p: Params, r, T, v, y):
    """steps 7-10 from given v = D.F and y = L.dW -> (r_new, u, Y, info)."""
    r, T, v, y = _f64(r), _f64(T), _f64(v).reshape(-1), _f64(y).reshape(-1)
    r_out = np.empty_like(r)
    u = np.empty(p.M, dtype=np.float64)
    Y = np.empty((p.n_rods, 3), dtype=np.float64)
    cp = p.c()
    info = lib().orc_finish_step(C.byref(cp), _ptr(r), _ptr(T), _ptr(v), _ptr(y), _ptr(r_out), _ptr(u), _ptr(Y))
    return r_out, u, Y, int(info)


def step(p: Params, chain: int, step_index: int, r, trace: bool = False):
    """One chain, one step.  returns (r_new, info) or (r_new, info, dict of intermediates)."""
    r = _f64(r)
    N, M = p.n_rods, p.M
    r_out = np.empty_like(r)
    cp = p.c()
    if not trace:
        info = lib().orc_step(C.byref(cp), C.c_uint64(chain), C.c_uint64(step_index), _ptr(r), _ptr(r_out), None)
        return r_out, int(info)
    tr = dict(T=np.zeros((N, 3)), F=np.zeros((N + 1, 3)), D=np.zeros((M, M)), L=np.zeros((M, M)),
              dW=np.zeros(M), v=np.zeros(M), y=np.zeros(M), u=np.zeros(M), Y=np.zeros((N, 3)))
    ct = _Trace()
    for k, a in tr.items():
        setattr(ct, k, a.ctypes.data)
    info = lib().orc_step(C.byref(cp), C.c_uint64(chain), C.c_uint64(step_index), _ptr(r), _ptr(r_out), C.byref(ct))
    return r_out, int(info), tr


def step_ensemble(p: Params, r, first_step: int, n_steps: int, chain0: int = 0):
    """r[C][N_b][3] -> (r_new, info[C]); OpenMP over chains."""
    r = np.array(r, dtype=np.float64, order="C", copy=True)
    Cn = r.shape[0]
    info = np.zeros(Cn, dtype=np.int32)
    cp = p.c()
    lib().orc_step_ensemble(C.byref(cp), C.c_int32(Cn), C.c_uint64(chain0), C.c_uint64(first_step),
                            C.c_int32(n_steps), _ptr(r), _ptr(info))
    return r, info


def observables(p: Params, r):
    """r[C][N_b][3] -> (per_chain[C][NOBS], ensemble[2][NOBS])."""
    r = _f64(r)
    Cn = r.shape[0]
    per = np.empty((Cn, NOBS), dtype=np.float64)
    ens = np.empty((2, NOBS), dtype=np.float64)
    cp = p.c()
    lib().orc_observables(C.byref(cp), C.c_int32(Cn), _ptr(r), _ptr(per), _ptr(ens))
    return per, ens


def end_to_end(n_rods: int, r) -> np.ndarray:
    """r[C][N_b][3] -> R[C][3] = r_N - r_0."""
    r = _f64(r)
    R = np.empty((r.shape[0], 3), dtype=np.float64)
    lib().orc_end_to_end(C.c_int32(n_rods), C.c_int32(r.shape[0]), _ptr(r), _ptr(R))
    return R


def autocorr(n_rods: int, r, R0) -> np.ndarray:
    """(sum_c R.R0, sum_c (R.R0)^2, sum_c R0.R0) of the end-to-end vectors."""
    r, R0 = _f64(r), _f64(R0)
    out = np.empty(3, dtype=np.float64)
    lib().orc_autocorr(C.c_int32(n_rods), C.c_int32(r.shape[0]), _ptr(r), _ptr(R0), _ptr(out))
    return out


def num_threads() -> int:
    return int(lib().orc_num_threads())
