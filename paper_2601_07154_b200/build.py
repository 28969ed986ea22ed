"""Builds libmf_b200.so (the C-ABI library of include/mf.h) in-tree with nvcc for sm_100a.

    python -m paper_2601_07154_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so lands next to this file so that it travels with the
repo snapshot and shows up as an in-tree native library at run time.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libmf_b200.so")
SOURCES = ["api.cu", "api_host.cu", "chain.cu", "focus.cu", "attention.cu", "linear.cu", "depth.cu", "attention_d128.cu", "attention_clc.cu", "attention_split.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]
# chain.cu / focus.cu hold the bit-exact fp64 path: never contract mul+add into FMA there.
# (The fp32 render deliberately uses explicit fmaf, which -fmad=false does not touch.)
PER_FILE = {"chain.cu": ["-fmad=false"], "focus.cu": ["-fmad=false"]}


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _stale():
    if not os.path.exists(OUT):
        return True
    t = os.path.getmtime(OUT)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [
        os.path.join(HERE, "..", "include", "mf.h"), os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, out=None, extra_flags=(), build_dir=None):
    """Compiles every source and links the library.  `out` / `extra_flags` / `build_dir` build a variant somewhere else
    (tests/test_gpu_watchdog.py builds one with an injected pipeline bug); the default is the in-tree product library."""
    variant = out is not None
    out = out or OUT
    if not variant and not force and not _stale():
        return out
    nvcc = _nvcc()
    objs = []
    build_dir = build_dir or os.path.join(HERE, "build")
    os.makedirs(build_dir, exist_ok=True)
    for src in SOURCES:
        obj = os.path.join(build_dir, src.replace(".cu", ".o"))
        cmd = [nvcc] + NVCC_FLAGS + PER_FILE.get(src, []) + os.environ.get("MF_NVCC_EXTRA", "").split() + list(extra_flags) + [
            "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)
        objs.append(obj)
    cmd = [nvcc, "-shared", "-o", out] + objs + ["-cudart", "static"]
    subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
