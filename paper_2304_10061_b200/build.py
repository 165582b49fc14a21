"""Builds libb200allegro.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo).

Each source is compiled to an object under paper_2304_10061_b200/build/ (git-ignored) by its own nvcc
process, in parallel, and only when it is older than its dependencies; the objects are then linked."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libb200allegro.so")
# gen_tp_patterns.cpp is a build-time host tool, not part of the library
SOURCES = ["model.cu", "cg_tables.cpp", "neighbors.cu", "edge_kernels.cu", "tp_kernels.cu", "tp2_kernels.cu",
           "tp2_l3_fwd.cu", "tp2_l3_bwd.cu", "tpc_kernels.cu", "tpc_l3.cu", "gemm_simt.cu", "gemm_tc.cu", "compute.cu", "probe.cu", "halo.cu", "noalloc.cu"]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def lib_path() -> str:
    return LIB


def _headers():
    return [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh", ".inc"))] + \
           [os.path.join(ROOT, "include", "b200_allegro.h")]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f != "tp2_patterns.inc"] + \
           [os.path.join(ROOT, "include", "b200_allegro.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(src: str, force: bool, verbose: bool):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
    path = os.path.join(CSRC, src)
    if not force and os.path.exists(obj):
        t = os.path.getmtime(obj)
        if all(os.path.getmtime(d) <= t for d in [path] + _headers()):
            return obj, 0, ""
    cmd = [nvcc, *ARCH, "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"),
           "-I", CSRC, "-x", "cu", "-c", path, "-o", obj]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    return obj, r.returncode, r.stdout + r.stderr


def _generate_patterns():
    """tp2_patterns.inc: compile-time sparsity patterns of the fused CG tensors (see gen_tp_patterns.cpp)."""
    out = os.path.join(CSRC, "tp2_patterns.inc")
    srcs = [os.path.join(CSRC, f) for f in ("gen_tp_patterns.cpp", "cg_tables.cpp", "internal.h")]
    if os.path.exists(out) and all(os.path.getmtime(s) <= os.path.getmtime(out) for s in srcs):
        return
    exe = os.path.join(OBJ, "gen_tp_patterns")
    cuda_inc = os.path.join(os.path.dirname(os.path.dirname(os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"))), "include")
    r = subprocess.run(["g++", "-O1", "-std=c++17", "-I", cuda_inc, "-I", os.path.join(ROOT, "include"), "-I", CSRC,
                        srcs[0], srcs[1], "-o", exe], capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("g++ failed building gen_tp_patterns")
    text = subprocess.run([exe], capture_output=True, text=True, check=True).stdout
    if not os.path.exists(out) or open(out).read() != text:
        open(out, "w").write(text)
    else:
        os.utime(out)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    _generate_patterns()
    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as ex:
        results = list(ex.map(lambda s: _compile(s, force, verbose), SOURCES))
    for obj, rc, log in results:
        if rc != 0:
            sys.stderr.write(log)
            raise RuntimeError(f"nvcc failed compiling {os.path.basename(obj)}")
        if verbose and log:
            sys.stderr.write(log)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    r = subprocess.run([nvcc, *ARCH, "-shared", "-Xcompiler", "-fPIC", "-o", LIB] + [o for o, _, _ in results],
                       capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed linking libb200allegro.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
