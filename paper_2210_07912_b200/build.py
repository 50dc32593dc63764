"""Build librift_ile.so in-tree with nvcc for sm_100a (no torch involved).

    python -m paper_2210_07912_b200.build [--force] [--ptxas]

Every object is keyed by a SHA-256 over its source, every header of csrc/ and include/, and the compiler flags (kept in
build/<name>.o.key), so a stale or foreign object or library is never reused: `build()` recompiles exactly what changed and
relinks when any object did or when the library's own key (over the object keys) does not match.
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(ROOT, "include")
LIB = os.path.join(HERE, "librift_ile.so")
OBJ_DIR = os.path.join(HERE, "build")
SOURCES = ["api.cu", "geometry.cu", "lnl_direct.cu", "lnl_direct_ext.cu", "lnl_tc.cu", "lnl_tcs.cu", "lnl_mma.cu", "lnl_sky.cu", "lnl_sky64.cu", "sky_sort.cu",
           "reduce.cu", "convert.cu", "precompute.cu", "ac.cu", "sky_frame.cu", "gmm.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-I", INCLUDE, "-I", CSRC]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    return "nvcc"


def _headers_digest() -> bytes:
    h = hashlib.sha256()
    for d in (CSRC, INCLUDE):
        for f in sorted(os.listdir(d)):
            if f.endswith((".h", ".cuh")):
                h.update(f.encode())
                h.update(open(os.path.join(d, f), "rb").read())
    return h.digest()


def _read(path: str) -> str:
    try:
        return open(path).read().strip()
    except OSError:
        return ""


def build(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    os.makedirs(OBJ_DIR, exist_ok=True)
    nvcc = _nvcc()
    hd = _headers_digest()
    flags = [*NVCC_FLAGS, *extra_flags]

    def key_of(src: str) -> str:
        h = hashlib.sha256(hd)
        h.update(open(os.path.join(CSRC, src), "rb").read())
        h.update(" ".join(flags).replace(ROOT, "").encode())
        return h.hexdigest()

    keys = {src: key_of(src) for src in SOURCES}

    def compile_one(src: str) -> bool:
        obj = os.path.join(OBJ_DIR, src.replace(".cu", ".o"))
        if not force and os.path.exists(obj) and _read(obj + ".key") == keys[src]:
            return False
        cmd = [nvcc, *flags, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            print(" ".join(cmd), flush=True)
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        if verbose and (r.stdout or r.stderr):
            print(r.stdout, r.stderr, flush=True)
        open(obj + ".key", "w").write(keys[src])
        return True

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        changed = list(ex.map(compile_one, SOURCES))
    lib_key = hashlib.sha256("".join(keys[s] for s in SOURCES).encode()).hexdigest()
    if any(changed) or not os.path.exists(LIB) or _read(os.path.join(OBJ_DIR, "lib.key")) != lib_key:
        objs = [os.path.join(OBJ_DIR, s.replace(".cu", ".o")) for s in SOURCES]
        cmd = [nvcc, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a"]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
        open(os.path.join(OBJ_DIR, "lib.key"), "w").write(lib_key)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True,
                extra_flags=("-Xptxas", "-v") if "--ptxas" in sys.argv else ()))
