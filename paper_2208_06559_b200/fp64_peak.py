"""FP64 issue-rate microbenchmark (DFMA vs DMMA m8n8k4 and the m16n8k* f64 shapes): the FP64 roofline
denominator, because MEASURED_PEAKS.json records no FP64 number.  `python -m paper_2208_06559_b200.fp64_peak`
compiles csrc/fp64_peak.cu for sm_100a and runs it on the current GPU."""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))


def build() -> str:
    src = os.path.join(_HERE, "csrc", "fp64_peak.cu")
    exe = os.path.join(_HERE, "csrc", "build", "fp64_peak")
    os.makedirs(os.path.dirname(exe), exist_ok=True)
    if not os.path.exists(exe) or os.path.getmtime(src) > os.path.getmtime(exe):
        subprocess.run([os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"), "-gencode", "arch=compute_100a,code=sm_100a",
                        "-O3", "-DBIGSHAPES", "-o", exe, src], check=True)
    return exe


if __name__ == "__main__":
    sys.exit(subprocess.run([build()]).returncode)
