"""Builds libbsa.so (the C-ABI CUDA library, include/bsa.h) in-tree with nvcc for sm_100a.

    python -m paper_2607_07724_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the
repository snapshot.
"""
from __future__ import annotations

import hashlib
import os
import shlex
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libbsa.so")
STAMP = LIB + ".srchash"
SOURCES = ["api.cu", "pool.cu", "select.cu", "score_tc_quest.cu", "score_tc_mean.cu", "attn.cu", "attn_t.cu", "diag.cu", "rowsel.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]
NVCC_FLAGS += shlex.split(os.environ.get("BSA_NVCC_FLAGS", ""))   # developer knob, e.g. -DBSA_TC_OCC2=0
if os.environ.get("BSA_DEBUG_TRAP", "0") not in ("", "0"):
    # debug builds only: a protocol bug traps after ~4 s of spinning on an mbarrier instead of hanging
    NVCC_FLAGS.append("-DBSA_MBAR_TRAP=1")


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found; libbsa cannot be built")


def _src_hash() -> str:
    """Hash of everything libbsa.so is built from: csrc/*, include/bsa.h and the nvcc flags.  mtimes
    are not used -- a repository snapshot copied to another box need not keep them."""
    h = hashlib.sha256()
    files = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC))
    files.append(os.path.join(_HERE, "..", "include", "bsa.h"))
    for f in files:
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def _stale() -> bool:
    """True when libbsa.so is missing or was not built from the sources as they are now."""
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as f:
        return f.read().strip() != _src_hash()


def build_lib(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu -> libbsa.so (one object per source, then a shared link)."""
    if not force and not _stale():
        return LIB
    nvcc = _nvcc()
    objdir = os.path.join(_HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    procs, objs = [], []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        objs.append(obj)
        cmd = [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)))
    failed = False
    for src, p in procs:
        out = p.communicate()[0].decode()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- nvcc {src} ---\n{out}\n")
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed while building libbsa.so")
    subprocess.check_call([nvcc, "-shared", "-o", LIB, *objs, "-gencode",
                           "arch=compute_100a,code=sm_100a"])
    with open(STAMP, "w") as f:
        f.write(_src_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
