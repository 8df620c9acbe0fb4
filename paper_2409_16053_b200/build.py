"""Build libak.so (the C-ABI library of include/ak.h) in-tree with nvcc for sm_100a.

    python -m paper_2409_16053_b200.build [--force]

nvcc cross-compiles without a GPU.  ak_exact.cu (ghost fill, dt) and ak_stage.cu (stage kernels, flux correction, FOFC)
(and mhd/ak_mhd.cu; only mhd/ak_mhd_fast.cu, the MHD sweeps of the default arithmetic flavour, allows contraction)
are compiled with -fmad=false: no contraction behind the source's back, every fused multiply-add of the stage kernel is
written out, so the same face solved by two tiles gives the same bits.  -lineinfo maps ncu's source page to these files.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
SO = os.path.join(HERE, "libak.so")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", INCLUDE, "-I", CSRC]
UNITS = {                      # translation unit -> extra flags
    "ak_api.cu": [],
    "ak_exact.cu": ["-fmad=false"],
    "ak_stage.cu": ["-fmad=false", "-Xptxas", "-v"],
    "mhd/ak_mhd.cu": ["-fmad=false", "-Xptxas", "-v"],        # MHD + CT (include/ak_mhd.h)
    "mhd/ak_mhd_fast.cu": ["-I", os.path.join(CSRC, "mhd"), "-Xptxas", "-v"],   # its default-flavour sweeps, contraction allowed
}


def _sources():
    src = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if os.path.isfile(os.path.join(CSRC, f))]
    src += [os.path.join(CSRC, "mhd", f) for f in os.listdir(os.path.join(CSRC, "mhd"))]
    return src + [os.path.join(INCLUDE, "ak.h"), os.path.join(INCLUDE, "ak_mhd.h")]


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(s) for s in _sources()):
        return SO
    bdir = os.path.join(HERE, "build")
    os.makedirs(bdir, exist_ok=True)
    objs = []
    for unit, extra in UNITS.items():
        obj = os.path.join(bdir, os.path.basename(unit).replace(".cu", ".o"))
        cmd = [nvcc, *ARCH, *COMMON, *extra, "-c", os.path.join(CSRC, unit), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {unit}")
        with open(os.path.join(bdir, os.path.basename(unit) + ".log"), "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        objs.append(obj)
    subprocess.run([nvcc, *ARCH, "-shared", "-o", SO, *objs], check=True)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
