"""Build step: compile csrc/*.cu into paper_2607_04516_b200/liblbm_b200.so for sm_100a (in tree).

    python -m paper_2607_04516_b200.build [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SO = os.path.join(HERE, "liblbm_b200.so")
# two translation units, compiled side by side (the template instantiations of the step kernels dominate the build time)
SOURCES = [os.path.join(HERE, "csrc", "lbm_api.cu"), os.path.join(HERE, "csrc", "lbm_inplace_launch.cu")]
DEPS = SOURCES + glob.glob(os.path.join(HERE, "csrc", "*.cuh")) + glob.glob(os.path.join(HERE, "csrc", "*.h")) + [os.path.join(ROOT, "include", "lbm.h")]
OBJDIR = os.path.join(HERE, "build")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo", "--expt-relaxed-constexpr",
    "-Xcompiler", "-fPIC",
    # no --use_fast_math: divisions and square roots stay IEEE (1e-5 parity budget)
]


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "nvcc")
        os.makedirs(OBJDIR, exist_ok=True)
        objs, jobs = [], []
        for src in SOURCES:
            obj = os.path.join(OBJDIR, os.path.splitext(os.path.basename(src))[0] + ".o")
            objs.append(obj)
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
            jobs.append((cmd, subprocess.Popen(cmd)))
        for cmd, job in jobs:
            if job.wait() != 0:
                raise subprocess.CalledProcessError(job.returncode, cmd)
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-o", SO] + objs, check=True)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
