"""FP64 issue-rate microbenchmark (DFMA and DMMA m8n8k4): the FP64 roofline denominator, because
MEASURED_PEAKS.json records no FP64 number.  bench.py calls `measure()` inside its own process and run;
`python -m paper_2208_06559_b200.bench.fp64_peak` prints the table kept in profiles/."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "fp64_peak.cu")
LIB = os.path.join(_HERE, "libbd_peak.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(SRC) > os.path.getmtime(LIB):
        subprocess.run([os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"), "-gencode", "arch=compute_100a,code=sm_100a",
                        "-O3", "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "-o", LIB, SRC], check=True)
    return LIB


def measure(kind: str = "dmma", warps_per_sm: int = 16, iters: int = 20000, reps: int = 5, stream: int = 0):
    """(TFLOP/s, best ms) of the FP64 pipe on the current CUDA device."""
    lib = C.CDLL(build())
    lib.bdpeak_fp64.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    tf, ms = C.c_double(0.0), C.c_double(0.0)
    rc = lib.bdpeak_fp64(1 if kind == "dmma" else 0, warps_per_sm, iters, reps, C.c_void_p(stream), C.byref(tf), C.byref(ms))
    if rc != 0:
        raise RuntimeError(f"bdpeak_fp64 failed with code {rc} (needs a CUDA device)")
    return tf.value, ms.value


if __name__ == "__main__":
    for wps in (4, 8, 16, 32):
        for kind in ("dfma", "dmma"):
            tf, ms = measure(kind, wps)
            print(f"{kind.upper():5s} ilp8 warps/SM={wps:2d}: {ms:8.3f} ms  {tf:6.2f} TFLOP/s")
