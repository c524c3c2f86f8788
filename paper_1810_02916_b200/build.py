"""Build libnf.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1810_02916_b200.build [--force] [-v]

nvcc cross-compiles without a GPU.  The built library is git-ignored but travels to the GPU
box with the repo snapshot.  Every translation unit is compiled on its own (in parallel) and
the objects are linked into one shared library.
"""
from __future__ import annotations

import concurrent.futures
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libnf.so")
SOURCES = ["nf_api.cu", "nf_scan.cu", "nf_bin.cu", "nf_forces.cu", "nf_stream.cu", "nf_step.cu", "nf_regroup.cu", "nf_dense.cu", "nf_tree.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC",
]
# Per-file flags.  Only the interaction kernel flushes float32 denormals (its PTX spells .ftz
# itself; the flag covers the plain C arithmetic around it: sentinel sources underflow to zero).
# The bit-exact float32 contracts of nf_bin / nf_kick_drift (include/nf.h) are IEEE, denormals
# included, like the oracle's.
EXTRA = {"nf_forces.cu": ["--ftz=true"]}


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f != "probe_sweep.cu"] + [os.path.join(HERE, "..", "include", "nf.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def _compile(nvcc: str, src: str, verbose: bool):
    obj = os.path.join(OBJ, src.replace(".cu", ".o"))
    cmd = [nvcc] + NVCC_FLAGS + EXTRA.get(src, []) + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    return src, obj, res


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    objs = []
    with concurrent.futures.ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        for src, obj, res in ex.map(lambda s: _compile(nvcc, s, verbose), SOURCES):
            if res.returncode != 0:
                sys.stderr.write(res.stdout + res.stderr)
                raise RuntimeError(f"nvcc failed compiling {src}")
            if verbose:
                sys.stderr.write(res.stderr)
            objs.append(obj)
    res = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking libnf.so")
    return LIB


def build_probe() -> str:
    """csrc/probe_sweep.cu -> ./probe_sweep: the sweep loops of the interaction kernel in isolation (a measuring tool)."""
    out = os.path.join(HERE, "probe_sweep")
    cmd = [os.environ.get("NVCC", "nvcc")] + NVCC_FLAGS[:5] + ["--ftz=true", "-o", out, os.path.join(CSRC, "probe_sweep.cu")]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed compiling probe_sweep.cu")
    return out


if __name__ == "__main__":
    if "--probe" in sys.argv:
        print(build_probe())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
