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
SOURCES = ["m3dk_api.cu", "m3dk_push.cu", "m3dk_sort.cu", "m3dk_deposit.cu", "m3dk_gc.cu", "m3dk_noalloc.cu"]
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


def nvcc_flags(verify: bool, extra=()):
    flags = ["-O3", "-std=c++17", *ARCH, "-lineinfo", "-Xcompiler", "-fPIC,-ffp-contract=off", "-Xptxas", "-v"]
    if verify:
        flags += ["-fmad=false", "-DM3DK_NO_FMA"]
    return flags + list(extra)


def nvcc_cmd(verify: bool, out: str, extra=()):
    """The single-command form of the build (what the object-by-object build below is equivalent to)."""
    return ["nvcc", *nvcc_flags(verify, extra), "-shared", "-o", out] + [os.path.join(_CSRC, s) for s in SOURCES]


def build(verify: bool = False, force: bool = False, verbose: bool = False, extra=()) -> str:
    """Compile every source to an object (in parallel: ptxas on the push kernels takes a minute) and link the library."""
    from concurrent.futures import ThreadPoolExecutor

    out = lib_path(verify)
    if not (force or _stale(out)):
        return out
    objdir = os.path.join(_HERE, "build", "verify" if verify else "timing")
    os.makedirs(objdir, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        r = subprocess.run(["nvcc", *nvcc_flags(verify, extra), "-c", "-o", obj, os.path.join(_CSRC, src)],
                           capture_output=True, text=True)
        return obj, r

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as pool:
        results = list(pool.map(compile_one, SOURCES))
    log = "".join(r.stdout + r.stderr for _, r in results)
    if verbose or any(r.returncode != 0 for _, r in results):
        sys.stderr.write(log)
    if any(r.returncode != 0 for _, r in results):
        raise RuntimeError("nvcc failed building " + out)
    r = subprocess.run(["nvcc", *ARCH, "-shared", "-o", out] + [o for o, _ in results], capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed linking " + out)
    with open(out + ".ptxas.log", "w") as fh:
        fh.write(log)
    return out


def build_all(force: bool = False, verbose: bool = False):
    from concurrent.futures import ThreadPoolExecutor

    with ThreadPoolExecutor(max_workers=2) as pool:
        a, b = pool.submit(build, False, force, verbose), pool.submit(build, True, force, verbose)
        return a.result(), b.result()


if __name__ == "__main__":
    print(build_all(force="--force" in sys.argv, verbose=True))
