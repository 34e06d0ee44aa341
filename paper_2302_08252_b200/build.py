"""Builds libadept_b200.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo).

Flags are part of the arithmetic contract (DESIGN.md rule M7): --fmad=false (no contraction), and the
nvcc defaults --prec-div=true --prec-sqrt=true --ftz=false; never -use_fast_math.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libadept_b200.so")
LIB_TIMING = os.path.join(HERE, "libadept_b200_timing.so")   # same sources, -DADEPT_TIMING_SECTIONS (include/adept.h)
SOURCES = ["layout_aos.cu", "layout_soa.cu", "layout_aosoa32.cu", "layout_aosoa64.cu", "layout_soa16.cu", "layout_aosoa16.cu", "layout_aosoa128.cu", "layout_hc16.cu", "layout_aosoa8.cu",
           "adept_api.cu", "step_static.cu"]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--fmad=false", "--prec-div=true", "--prec-sqrt=true", "--ftz=false",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _deps():
    out = [os.path.join(HERE, "..", "include", "adept.h")]
    out += [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    return out


def is_stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in _deps())


def build_all(force: bool = False) -> None:
    """The library and its timing variant."""
    build(force=force)
    if force or is_stale(LIB_TIMING):
        build(extra_flags=("-DADEPT_TIMING_SECTIONS",), out=LIB_TIMING)


def build(force: bool = False, verbose: bool = False, extra_flags=(), out: str | None = None) -> str:
    """Compile the library.  `extra_flags` / `out` build a variant (e.g. -DADEPT_STEP_MIN_CTAS=3)
    under another name; binding.py loads $ADEPT_B200_LIB instead of the default when it is set."""
    lib = LIB if out is None else out
    obj_dir = OBJ if out is None else OBJ + "_" + os.path.basename(out).replace(".so", "")
    if out is None and not force and not is_stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(obj_dir, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(obj_dir, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, *extra_flags, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        with open(obj + ".log", "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s" % (src, r.stderr[-4000:]))
        if verbose:
            sys.stderr.write(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    tmp = lib + ".tmp%d" % os.getpid()
    r = subprocess.run([nvcc, "-shared", "-cudart", "static", "-o", tmp, *objs], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + r.stderr[-4000:])
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--no-variants" not in sys.argv:
        build_all()
