"""Build and run the FP4 tensor-core peak probe (csrc/probe_fp4_peak.cu): a measurement utility, not part
of the library.  `python -m paper_2607_05711_b200.probe [iterations]` on a B200."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build():
    out = os.path.join(HERE, "build", "probe_fp4_peak")
    os.makedirs(os.path.dirname(out), exist_ok=True)
    subprocess.run([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "--expt-relaxed-constexpr",
                    "-o", out, os.path.join(HERE, "csrc", "probe_fp4_peak.cu"), "-lcuda"], check=True)
    return out


if __name__ == "__main__":
    subprocess.run([build()] + sys.argv[1:], check=True)
