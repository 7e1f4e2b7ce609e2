"""Build libwl.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2407_16032_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library lands in paper_2407_16032_b200/lib/libwl.so
(git-ignored, but it travels to the GPU box with the gpurun snapshot).
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIBDIR = PKG / "lib"
LIB = LIBDIR / "libwl.so"
SOURCES = ["wl_api.cu", "wl_flow.cu", "wl_convdiff.cu", "wl_poisson.cu", "wl_pcgfast.cu", "wl_pcgfused.cu", "wl_small.cu", "wl_generic.cu", "wl_noalloc.cu"]
HEADERS = ["wl_common.cuh", "wl_body.cuh", "wl_vec.cuh", "wl_tma.cuh", "wl_internal.h", "wl_dual.cuh"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libwl cannot be built (there is no CPU fallback)")


def _stamp() -> str:
    h = hashlib.sha1()
    for name in SOURCES + HEADERS:
        h.update((CSRC / name).read_bytes())
    h.update((PKG.parent / "include" / "wl.h").read_bytes())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> Path:
    LIBDIR.mkdir(exist_ok=True)
    stamp_file = LIBDIR / "libwl.stamp"
    stamp = _stamp()
    if not force and LIB.exists() and stamp_file.exists() and stamp_file.read_text() == stamp:
        return LIB
    nvcc = _nvcc()
    objs = []
    logs = []
    procs = []
    for src in SOURCES:
        obj = LIBDIR / (src + ".o")
        cmd = [nvcc, *NVCC_FLAGS, "-c", str(CSRC / src), "-o", str(obj)]
        procs.append((src, cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(str(obj))
    for src, cmd, p in procs:
        out, _ = p.communicate()
        logs.append(f"$ {' '.join(cmd)}\n{out}")
        if p.returncode != 0:
            sys.stderr.write(logs[-1])
            raise RuntimeError(f"nvcc failed on {src}")
    cmd = [nvcc, "-shared", "-o", str(LIB), *objs, "-lcudart", "-ldl"]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    logs.append(f"$ {' '.join(cmd)}\n{r.stdout}")
    if r.returncode != 0:
        sys.stderr.write(logs[-1])
        raise RuntimeError("link failed")
    (LIBDIR / "build.log").write_text("\n".join(logs))
    stamp_file.write_text(stamp)
    if verbose:
        print("\n".join(logs))
    return LIB


if __name__ == "__main__":
    path = build(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
    print(path)
