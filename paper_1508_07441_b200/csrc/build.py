"""Builds libpm.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Two steps: (1) pm_codegen (host tool, g++) turns the channel sets below into gen/pm_spec_gen.cuh — the
channel-specialised ket code of the fill kernel (see pm_codegen.cpp); (2) nvcc compiles the library.
A lattice whose channel set is not listed here still works: pm_fill falls back to the table-driven kernel.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
PKG = os.path.dirname(HERE)
LIB = os.path.join(PKG, "libpm.so")
GEN_DIR = os.path.join(HERE, "gen")
GEN = os.path.join(GEN_DIR, "pm_spec_gen.cuh")
CODEGEN = os.path.join(GEN_DIR, "pm_codegen")
SOURCES = ["pm_api.cu", "pm_kernels.cu", "pm_fill.cu", "pm_stream.cu", "pm_tables.cpp"]
HEADERS = ["pm_device.cuh", "pm_kernels.cuh", "pm_fill.cuh", "pm_tables.hpp", "pm_ylm.h", "pm_codegen.cpp", "build.py",
           os.path.join("..", "inputs.py"), os.path.join("..", "..", "include", "pm.h")]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "--shared", "-cudart", "shared"]


def channel_sets():
    """(name, J2, parity, T2, statistics, channels) of the sets that get a specialised kernel: the channel sets of
    BASELINE.json configs[0..4] (inputs.py holds the enumeration; no arithmetic of the method lives there)."""
    if PKG not in sys.path:
        sys.path.insert(0, os.path.dirname(PKG))
    from paper_1508_07441_b200 import inputs as I
    return [
        ("boson_s", 0, 1, 0, I.PM_SPINLESS_BOSON, I.boson_channel(0, 0)),
        ("nnn_s2", 1, 1, 1, I.PM_FERMION_ISOSPIN, I.swave_3n_channels()),
        ("nnn_j2", 1, 1, 1, I.PM_FERMION_ISOSPIN, I.enumerate_3n_channels(1, +1, 1, 2)),
        ("nnn_j3", 1, 1, 1, I.PM_FERMION_ISOSPIN, I.enumerate_3n_channels(1, +1, 1, 3)),
    ]


def generate(verbose: bool = False) -> str:
    os.makedirs(GEN_DIR, exist_ok=True)
    cxx = os.environ.get("CXX", "g++")
    subprocess.check_call([cxx, "-std=c++17", "-O1", "-o", CODEGEN, os.path.join(HERE, "pm_codegen.cpp"),
                           os.path.join(HERE, "pm_tables.cpp")])
    sets = os.path.join(GEN_DIR, "sets.txt")
    with open(sets, "w") as f:
        for name, J2, par, T2, stat, ch in channel_sets():
            f.write(f"{name} {J2} {par} {T2} {stat} {len(ch)}\n")
            for c in ch:
                f.write(" ".join(str(int(c[k])) for k in ("l", "s", "j", "t", "lam", "I2")) + "\n")
    subprocess.run([CODEGEN, sets, GEN], check=True, stderr=None if verbose else subprocess.DEVNULL)
    return GEN


def stale() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(GEN):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        generate(verbose)
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + f".{os.getpid()}.tmp"                 # link beside the target, then rename: readers never see a partial file
        cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *[os.path.join(HERE, s) for s in SOURCES]]
        try:
            subprocess.check_call(cmd)
            os.replace(tmp, LIB)
        finally:
            if os.path.exists(tmp):
                os.remove(tmp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
