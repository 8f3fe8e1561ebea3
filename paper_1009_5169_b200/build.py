"""Build libwd.so (the C-ABI library of include/wd.h) in-tree with nvcc for sm_100a.

    python -m paper_1009_5169_b200.build [--force]

WD_NVCC_DEFINES (environment) adds -D flags for measurement builds, e.g. the ablation switches of csrc/wd_hop_zm.cu:
    WD_NVCC_DEFINES="-DWD_ZM_ABLATE=1" python -m paper_1009_5169_b200.build --force     (and --force again without it afterwards)
Such a library computes wrong results on purpose; wd_version() then ends in "MEASUREMENT BUILD: <the defines>", the Python
binding refuses to load it unless WD_ALLOW_MEASUREMENT_BUILD=1 is set (bench.py --hop-only timing runs), and
tests/test_abi.py fails on it.

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libwd.so")
SOURCES = ["wd_ctx.cu", "wd_layout.cu", "wd_hop.cu", "wd_hop_tma.cu", "wd_hop_zm.cu", "wd_solve.cu", "wd_solve_h16.cu", "wd_solve_gl.cu", "wd_force.cu", "wd_md.cu", "wd_noalloc.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "--use_fast_math=false"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "wd.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    os.makedirs(os.path.join(HERE, "build"), exist_ok=True)
    for s in SOURCES:
        o = os.path.join(HERE, "build", s.replace(".cu", ".o"))
        objs.append(o)
        defines = os.environ.get("WD_NVCC_DEFINES", "").split()
        if defines:   # a measurement build says so in wd_version(); tests/test_abi.py and wd.lib() refuse to go on with one
            defines = defines + ['-DWD_BUILD_DEFINES="' + " ".join(defines).replace('"', "") + '"']
        cmd = [nvcc] + [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")] + defines + \
              (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, s), "-o", o]
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for s, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode:
            sys.stderr.write(out)
        failed = failed or p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs + ["-lcudart"], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
