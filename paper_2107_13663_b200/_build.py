"""In-tree nvcc build of libm3dk for sm_100a (no JIT cache: the .so travels with the repository snapshot).

Two variants of the same sources:
  libm3dk.so         timing build, FMA contraction on (nvcc default)
  libm3dk_verify.so  verification build: -fmad=false -DM3DK_NO_FMA (no fused multiply-add anywhere), the build the
                     1e-12 / 1e-8 parity bars of BASELINE.json are stated for ("FMA contraction disabled").
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
SOURCES = ["m3dk_api.cu", "m3dk_push.cu", "m3dk_sort.cu", "m3dk_deposit.cu", "m3dk_gc.cu"]
HEADERS = ["m3dk_internal.h", "m3dk_device.cuh", os.path.join("..", "..", "include", "m3dk.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def lib_path(verify: bool = False) -> str:
    return os.path.join(_HERE, "libm3dk_verify.so" if verify else "libm3dk.so")


def _stale(out: str) -> bool:
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    deps = [os.path.join(_CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def nvcc_cmd(verify: bool, out: str, extra=()):
    cmd = ["nvcc", "-O3", "-std=c++17", *ARCH, "-lineinfo", "-shared", "-Xcompiler", "-fPIC,-ffp-contract=off",
           "-Xptxas", "-v", "-o", out]
    if verify:
        cmd += ["-fmad=false", "-DM3DK_NO_FMA"]
    cmd += list(extra)
    cmd += [os.path.join(_CSRC, s) for s in SOURCES]
    return cmd


def build(verify: bool = False, force: bool = False, verbose: bool = False) -> str:
    out = lib_path(verify)
    if force or _stale(out):
        r = subprocess.run(nvcc_cmd(verify, out), capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed building " + out)
        with open(out + ".ptxas.log", "w") as fh:
            fh.write(r.stdout + r.stderr)
    return out


def build_all(force: bool = False, verbose: bool = False):
    return build(False, force, verbose), build(True, force, verbose)


if __name__ == "__main__":
    print(build_all(force="--force" in sys.argv, verbose=True))
