"""Build libds.so (the CUDA C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_2503_13092_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the repo snapshot.
"""
import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libds.so")
SOURCES = ["ds_api.cu", "ds_layout.cu", "ds_track.cu", "ds_event.cu", "ds_clone.cu", "ds_mlp.cu", "ds_vertex.cu", "ds_lines.cu"]
HEADERS = [os.path.join(CSRC, "ds_common.cuh"), os.path.join(CSRC, "ds_sort.cuh"), os.path.join(CSRC, "ds_track.cuh"), os.path.join(HERE, "..", "include", "ds.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--shared",
              "-Xcompiler", "-fPIC,-Wall,-Wextra", "-Xptxas", "-v", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + HEADERS + [os.path.abspath(__file__)]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    # one nvcc per source file, side by side (the tracking kernels take about a minute each), then the link
    objdir = tempfile.mkdtemp(prefix="libds_obj_")
    extra = os.environ.get("DS_NVCC_EXTRA", "").split()
    compile_flags = [f for f in NVCC_FLAGS if f not in ("--shared", "-cudart", "static")]

    def compile_one(src):
        obj = os.path.join(objdir, os.path.basename(src) + ".o")
        r = subprocess.run([_nvcc()] + compile_flags + extra + ["-c", "-o", obj, src], capture_output=True, text=True)
        return obj, r

    try:
        with ThreadPoolExecutor(max_workers=min(len(srcs), os.cpu_count() or 1)) as pool:
            results = list(pool.map(compile_one, srcs))
        failed = False
        for _, r in results:
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            failed |= r.returncode != 0
        if failed:
            raise RuntimeError("nvcc failed building libds.so")
        r = subprocess.run([_nvcc()] + NVCC_FLAGS + ["-o", tmp] + [o for o, _ in results], capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed linking libds.so")
    finally:
        shutil.rmtree(objdir, ignore_errors=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
