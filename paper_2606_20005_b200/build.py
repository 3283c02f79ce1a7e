"""In-tree build of libstreamkl.so (sm_100a only) with nvcc.  No JIT cache, no torch extension machinery:
the product is a plain C-ABI shared library (include/streamkl.h) that travels with the source tree.

    python -m paper_2606_20005_b200.build [--force] [--debug-timeout]
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG_DIR, "csrc")
INCLUDE = os.path.join(os.path.dirname(PKG_DIR), "include")
LIB_PATH = os.path.join(PKG_DIR, "libstreamkl.so")
STAMP_PATH = os.path.join(PKG_DIR, "libstreamkl.so.stamp")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "--expt-relaxed-constexpr",
    "-cudart", "static",
]


def _sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cu"))


def _all_inputs():
    files = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh", ".h", ".inc"))]
    files += [os.path.join(INCLUDE, f) for f in sorted(os.listdir(INCLUDE)) if f.endswith(".h")]
    return files


def _digest(extra_flags) -> str:
    h = hashlib.sha256()
    h.update(" ".join(NVCC_FLAGS + list(extra_flags)).encode())
    for f in _all_inputs():
        with open(f, "rb") as fh:
            h.update(os.path.relpath(f, os.path.dirname(PKG_DIR)).encode())   # (relative: the stamp survives another checkout location)
            h.update(fh.read())
    return h.hexdigest()


def find_nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libstreamkl.so cannot be built (there is no CPU fallback)")


def build_library(force: bool = False, debug_timeout: bool = False, verbose: bool = False) -> str:
    """Compile every .cu under csrc/ into paper_2606_20005_b200/libstreamkl.so; returns its path."""
    extra = ["-DSTREAMKL_DEBUG_TIMEOUT"] if debug_timeout else []
    extra += os.environ.get("STREAMKL_NVCC_EXTRA", "").split()   # tuning macros, e.g. -DSTREAMKL_FWD_POLY_EVERY=3
    want = _digest(extra)
    if not force and os.path.exists(LIB_PATH) and os.path.exists(STAMP_PATH):
        with open(STAMP_PATH) as fh:
            if fh.read().strip() == want:
                return LIB_PATH
    nvcc = find_nvcc()
    objs = []
    procs = []
    build_dir = os.path.join(PKG_DIR, "build")
    os.makedirs(build_dir, exist_ok=True)
    for src in _sources():
        obj = os.path.join(build_dir, os.path.basename(src) + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *extra, "-I", INCLUDE, "-I", CSRC, "-c", src, "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{out}")
        if verbose and out:
            print(out)
    link = [nvcc, "-shared", "-cudart", "static", "-o", LIB_PATH, *objs]
    r = subprocess.run(link, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}")
    with open(STAMP_PATH, "w") as fh:
        fh.write(want + "\n")
    return LIB_PATH


if __name__ == "__main__":
    path = build_library(force="--force" in sys.argv, debug_timeout="--debug-timeout" in sys.argv,
                         verbose="--verbose" in sys.argv)
    print(path)
