"""Build step: compile the CUDA sources to an in-tree shared library for sm_100a.

    python -m paper_1101_0876_b200.build [--force]

nvcc cross-compiles without a GPU.  One translation unit per kernel family, compiled in parallel into
`paper_1101_0876_b200/build/*.o`, then linked.  The library links the CUDA runtime statically, so it needs
only the driver at run time and shares the primary context (memory, streams) with PyTorch.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libpotts_b200.so")
SOURCES = ["potts_api.cu", "k_stream.cu", "k_stream_s1c0.cu", "k_stream_s1c1.cu", "k_stream_s2c0.cu", "k_stream_s2c1.cu",
           "k_packed.cu", "k_packed_s1.cu", "k_packed_s2.cu", "k_resident.cu", "k_cluster.cu", "potts3d_api.cu", "potts8_api.cu",
           "potts_noalloc.cu"]
HEADERS = ["potts_core.cuh", "potts_kernels.cuh", "potts_resident.cuh", "potts_packed.cuh", "potts_cluster.cuh",
           "potts_launch.cuh", "potts3d.cuh", "potts8.cuh", "k_stream.inl", "k_packed.inl", os.path.join(INCLUDE, "potts.h")]

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ["-O3", "-std=c++17", *ARCH, "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]

last_action = "none"          # "compiled" or "reused": what the last build() call did


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _mtime(p: str) -> float:
    return os.path.getmtime(p) if os.path.exists(p) else 0.0


def _stale(target: str, deps) -> bool:
    t = _mtime(target)
    return t == 0.0 or any(_mtime(d) > t for d in deps)


def needs_build() -> bool:
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS]
    return _stale(LIB, deps)


def _compile(src: str, verbose: bool) -> str:
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    cmd = [_nvcc(), *NVCC_FLAGS, "-I", INCLUDE, "-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile what is out of date and link.  Sets `last_action` to "compiled" or "reused"."""
    global last_action
    hdrs = [h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS]
    os.makedirs(OBJ, exist_ok=True)
    todo = [s for s in SOURCES
            if force or _stale(os.path.join(OBJ, os.path.splitext(s)[0] + ".o"), [os.path.join(CSRC, s)] + hdrs)]
    if not todo and not _stale(LIB, [os.path.join(OBJ, os.path.splitext(s)[0] + ".o") for s in SOURCES]):
        last_action = "reused"
        return LIB
    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as pool:
        list(pool.map(lambda s: _compile(s, verbose), todo))
    tmp = LIB + f".tmp{os.getpid()}"
    objs = [os.path.join(OBJ, os.path.splitext(s)[0] + ".o") for s in SOURCES]
    cmd = [_nvcc(), *ARCH, "-shared", "-cudart", "static", "-o", tmp, *objs]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("link failed: " + " ".join(cmd))
    os.replace(tmp, LIB)
    last_action = "compiled"
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv), last_action)
