"""In-tree build of libskel.so: nvcc, sm_100a only (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libskel.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
# (source, object stem, extra defines); overlap2d_inst.cu is compiled once per radius (SKEL_INST),
# the slowest ones first so that the parallel build ends early
SOURCES = ([("overlap2d_inst.cu", f"overlap2d_inst{k}", [f"-DSKEL_INST={k}"]) for k in (3, 9, 8, 2, 1, 7, 6, 5, 0, 4)] +
           [(f, os.path.splitext(f)[0], []) for f in
            ("separable.cu", "fused.cu", "f64.cu", "scan.cu", "overlap1d.cu", "api.cu", "overlap2d.cu", "reduce.cu", "map.cu", "probe.cu", "noalloc.cu", "plan.cpp")])
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _deps_mtime() -> float:
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, "skel.h"), __file__]
    return max(os.path.getmtime(f) for f in files)


def _compile(item) -> str:
    src, stem, defines = item
    obj = os.path.join(OBJ, stem + ".o")
    srcp = os.path.join(CSRC, src)
    headers = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".hpp", ".cuh"))]
    headers.append(os.path.join(INCLUDE, "skel.h"))
    newest = max(os.path.getmtime(f) for f in [srcp, __file__] + headers)
    if not os.path.exists(obj) or os.path.getmtime(obj) < newest:
        cmd = [_nvcc(), *NVCC_FLAGS, *defines, "-x", "cu", "-I", INCLUDE, "-c", srcp, "-o", obj]
        subprocess.run(cmd, check=True)
    return obj


def build(force: bool = False) -> str:
    """Compile every translation unit (in parallel) and link libskel.so. Returns its path."""
    os.makedirs(OBJ, exist_ok=True)
    if force:
        for f in os.listdir(OBJ):
            os.remove(os.path.join(OBJ, f))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _deps_mtime():
        return LIB
    with ThreadPoolExecutor(max_workers=min(os.cpu_count() or 4, len(SOURCES))) as ex:
        objs = list(ex.map(_compile, SOURCES))
    subprocess.run([_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB, *objs], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in os.sys.argv))
