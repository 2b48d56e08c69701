"""Build librfi.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  The translation units are compiled in parallel and linked into one
shared object.  The .so is git-ignored but travels to the GPU box with the repo snapshot.
Usage: `python -m paper_2412_14775_b200.build [--force]`.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(CSRC, "librfi.so")
OBJ_DIR = os.path.join(CSRC, "build")
SOURCES = [os.path.join(CSRC, f) for f in
           ("rfi_api.cu", "rfi_launch_direct.cu", "rfi_launch_split.cu", "rfi_launch_tma.cu", "rfi_launch_batched.cu", "rfi_launch_batched_tma.cu", "rfi_launch_batched_mask_f32.cu", "rfi_launch_batched_mask_f16.cu", "rfi_launch_tables.cu", "rfi_launch_tables_ps0.cu", "rfi_launch_tables_ps1.cu", "rfi_launch_tables_ps2.cu", "rfi_launch_tables_ps3.cu", "rfi_confusion.cu", "rfi_probe.cu", "rfi_sim42.cu", "rfi_rl.cu", "rfi_adapt.cu")]
DEPS = SOURCES + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + sorted(glob.glob(os.path.join(CSRC, "*.inc"))) + [
    os.path.join(CSRC, "rfi_internal.h"), os.path.join(ROOT, "include", "rfi.h")]

# per-file additions: the RL-environment evaluator carries a double-precision ground-truth chain that must not be
# contracted into fused multiply-adds (its CPU restatement is compiled with -ffp-contract=off)
EXTRA_FLAGS = {"rfi_rl.cu": ["-fmad=false"]}

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-Xptxas=-v",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found; librfi.so cannot be built")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def _deps_of(src: str) -> list[str]:
    """Transitive `#include "..."` closure of one translation unit (files under csrc/ and include/)."""
    import re
    seen, todo = set(), [src]
    while todo:
        f = todo.pop()
        if f in seen or not os.path.exists(f):
            continue
        seen.add(f)
        with open(f) as fh:
            for inc in re.findall(r'^\s*#\s*include\s+"([^"]+)"', fh.read(), flags=re.M):
                todo.append(os.path.normpath(os.path.join(os.path.dirname(f), inc)))
    return sorted(seen)


def build_library(force: bool = False, verbose: bool = False) -> str:
    """Compile the translation units whose sources changed (objects are cached in csrc/build/) and link librfi.so."""
    if not force and not is_stale():
        return LIB
    nvcc = nvcc_path()
    os.makedirs(OBJ_DIR, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(OBJ_DIR, os.path.basename(src)[:-3] + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *EXTRA_FLAGS.get(os.path.basename(src), []), "-c", "-o", obj, src]
        log = obj[:-2] + ".log"
        fresh = (not force and os.path.exists(obj) and os.path.exists(log)
                 and all(os.path.getmtime(d) <= os.path.getmtime(obj) for d in _deps_of(src) + [os.path.abspath(__file__)]))
        if fresh:
            with open(log) as f:
                return obj, cmd, 0, f.read()
        tmp = obj + f".tmp{os.getpid()}"
        res = subprocess.run(cmd[:-3] + ["-o", tmp, src], capture_output=True, text=True)
        if res.returncode == 0:
            os.replace(tmp, obj)
            with open(log, "w") as f:
                f.write(res.stderr)
        return obj, cmd, res.returncode, res.stdout + res.stderr

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        results = list(ex.map(compile_one, SOURCES))
    log = []
    for obj, cmd, rc, out in results:
        log.append(" ".join(cmd) + "\n" + out)
        if verbose or rc != 0:
            sys.stderr.write(out)
        if rc != 0:
            raise RuntimeError(f"nvcc failed compiling {cmd[-1]}")
    tmp = LIB + f".tmp{os.getpid()}"
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-o", tmp,
            *[obj for obj, _, _, _ in results]]
    res = subprocess.run(link, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking librfi.so")
    os.replace(tmp, LIB)
    with open(os.path.join(CSRC, "ptxas_info.txt"), "w") as f:
        f.write("\n".join(log) + "\n" + " ".join(link) + "\n")
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
