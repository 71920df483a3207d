"""Builds the C-ABI library liber_b200.so from csrc/*.cu for sm_100a, in-tree (nvcc cross-compiles
without a GPU).  `python -m paper_2606_18967_b200.build` or `build_library()`.

`--dev` / `build_library(dev=True)` builds liber_b200_dev.so instead: the same sources with -DER_DEV, which adds the
partition / launch-mode knobs of csrc/er_dev.h (tests only; the shipped library does not contain them)."""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG_DIR, "csrc")
INCLUDE = os.path.join(os.path.dirname(PKG_DIR), "include")
LIB_PATH = os.path.join(PKG_DIR, "liber_b200.so")
DEV_LIB_PATH = os.path.join(PKG_DIR, "liber_b200_dev.so")
SOURCES = ["er_api.cu", "er_host.cu", "quantize_pack.cu", "spec_verify.cu", "w4a16_gemm_simt.cu", "w4a16_gemm.cu",
           "w4a16_gemm_small.cu", "w4a16_gemm_wide.cu", "w4a16_gemm_large.cu", "bf16_gemm.cu", "sd_policy.cu", "quantize_pack8.cu"]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-I", INCLUDE, "-I", CSRC]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: cannot build liber_b200.so (there is no CPU fallback)")


def _stale(lib_path: str) -> bool:
    if not os.path.exists(lib_path):
        return True
    t = os.path.getmtime(lib_path)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, "er.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force: bool = False, verbose: bool = False, dev: bool = False) -> str:
    lib_path = DEV_LIB_PATH if dev else LIB_PATH
    if not force and not _stale(lib_path):
        return lib_path
    nvcc = _nvcc()
    objdir = os.path.join(PKG_DIR, "build_dev" if dev else "build")
    flags = NVCC_FLAGS + (["-DER_DEV"] if dev else [])
    os.makedirs(objdir, exist_ok=True)
    procs = []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        cmd = [nvcc, *flags, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            print(" ".join(cmd))
        procs.append((src, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    objs = []
    for src, obj, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{out}")
        objs.append(obj)
    cmd = [nvcc, "-shared", "-o", lib_path, *objs, "-gencode", "arch=compute_100a,code=sm_100a"]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}")
    return lib_path


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose=True, dev="--dev" in sys.argv))
