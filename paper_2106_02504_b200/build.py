"""Builds librlxpp.so (the CUDA kernels + C ABI) in-tree for sm_100a.

    python -m paper_2106_02504_b200.build [--force]

nvcc cross-compiles without a GPU.  The multiplier rows (include/rlxpp_rows.cuh) are
regenerated first by csrc/gen_rows.py.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librlxpp.so")
SOURCES = ["rlxpp.cu"]
DEPS = ["rlxpp.cu", "arith.cuh", "state.cuh", "emit.cuh", "stages.cuh", "kernels_imad.cuh", "kernels_umma.cuh", "kernels_misc.cuh",
        "umma_path.cuh", "host_bigint.h", os.path.join("..", "..", "include", "rlxpp_rows.cuh"), "gen_rows.py", "normal_coeffs.cuh",
        os.path.join("..", "..", "include", "rlxpp.h"), os.path.join("..", "..", "include", "rlxpp_device.cuh"),
        os.path.join("..", "..", "include", "rlxpp_tile.cuh")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    sys.path.insert(0, CSRC)
    try:
        import gen_rows
        gen_rows.main()
    finally:
        sys.path.pop(0)
    deps = [os.path.join(CSRC, d) for d in DEPS]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + ["-o", LIB + ".tmp"] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
    with open(os.path.join(HERE, "build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building librlxpp.so (see output above)")
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
