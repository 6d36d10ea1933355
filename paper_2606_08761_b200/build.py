"""Builds libapex4.so (the C-ABI library of include/apex4.h) in-tree with nvcc for sm_100a.

`python -m paper_2606_08761_b200.build` or `build()` from Python.  nvcc cross-compiles without a
GPU.  The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libapex4.so")
SOURCES = ["apex4_api.cu", "apex4_quant.cu", "apex4_fused_quant.cu", "apex4_gemm_pair.cu", "apex4_gemm_pair_m0.cu", "apex4_gemm_pair_m1.cu", "apex4_gemm_pair_m2.cu", "apex4_gemm_pair_m3.cu", "apex4_gemv.cu", "apex4_rho.cu", "apex4_e4m3.cu",
           "apex4_static_ws.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
    "-Xcompiler", "-fPIC", "--shared",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found (needed to build libapex4.so for sm_100a)")


def _source_hash(extra=()) -> str:
    """SHA-256 over every file under csrc/, include/apex4.h, the nvcc version and the flags: a library built from other
    sources (a stale prebuilt .so that travelled with a snapshot) is rebuilt, whatever the file times say."""
    import hashlib
    h = hashlib.sha256()
    for f in sorted(os.listdir(CSRC)):
        h.update(f.encode())
        h.update(open(os.path.join(CSRC, f), "rb").read())
    h.update(open(os.path.join(os.path.dirname(PKG), "include", "apex4.h"), "rb").read())
    try:
        h.update(subprocess.run([_nvcc(), "--version"], capture_output=True, text=True).stdout.encode())
    except OSError:
        pass
    h.update(" ".join(NVCC_FLAGS + list(extra)).encode())
    return h.hexdigest()


def needs_build(lib: str = LIB, extra=()) -> bool:
    stamp = lib + ".sha256"
    if not os.path.exists(lib) or not os.path.exists(stamp):
        return True
    return open(stamp).read().strip() != _source_hash(extra)


def build(force: bool = False, verbose: bool = False, out: str = LIB, defines=()) -> str:
    """Compiles every source to an object file (in parallel) and links the library.  `defines` (e.g.
    ["-DAPEX4_TIMELINE"], the tuning switches named in profiles/) and `out` build a variant next to the product
    library (load it with APEX4_LIB=<out>); the default builds paper_2606_08761_b200/libapex4.so."""
    defines = list(defines)
    if not force and not needs_build(out, defines):
        return out
    from concurrent.futures import ThreadPoolExecutor
    tag = "" if out == LIB else "_" + os.path.splitext(os.path.basename(out))[0]
    objdir = os.path.join(PKG, "_obj" + tag)
    os.makedirs(objdir, exist_ok=True)
    base = [_nvcc()] + [f for f in NVCC_FLAGS if f != "--shared"] + defines + (["-Xptxas", "-v"] if verbose else [])

    def compile_one(src):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        res = subprocess.run(base + ["-c", os.path.join(CSRC, src), "-o", obj], capture_output=True, text=True)
        return src, obj, res

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    for src, obj, res in results:
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError(f"nvcc failed on {src}")
        if verbose:
            sys.stderr.write(res.stderr)
    link = [_nvcc(), "--shared", "-gencode", "arch=compute_100a,code=sm_100a"] + [o for _, o, _ in results] + ["-o", out]
    res = subprocess.run(link, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking " + out)
    with open(out + ".sha256", "w") as f:
        f.write(_source_hash(defines) + "\n")
    return out


if __name__ == "__main__":
    # python -m paper_2606_08761_b200.build [--force] [-v] [--out PATH] [-DNAME[=VALUE] ...]
    args = sys.argv[1:]
    out = LIB
    if "--out" in args:
        out = os.path.abspath(args[args.index("--out") + 1])
    print(build(force="--force" in args, verbose="-v" in args, out=out, defines=[a for a in args if a.startswith("-D")]))
