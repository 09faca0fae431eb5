"""Build and run the microbenchmarks behind the kernel designs (csrc/ubench.cu).

    python -m paper_2106_15350_b200.ubench          # needs a B200; prints markdown tables

Stand-alone: it does not touch liblbcnn.so, the oracle or any data."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))


def build() -> str:
    exe = os.path.join(HERE, "ubench.bin")
    src = os.path.join(HERE, "csrc", "ubench.cu")
    if not os.path.exists(exe) or os.path.getmtime(exe) < os.path.getmtime(src):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-o", exe, src], check=True)
    return exe


if __name__ == "__main__":
    sys.exit(subprocess.run([build()]).returncode)
