"""Build the CUDA C-ABI library in-tree:  python -m paper_1903_09043_b200.build

nvcc cross-compiles for sm_100a without a GPU.  The .so is git-ignored but travels to the GPU box.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libark_b200.so")
SOURCES = ["ark.cu"]
HEADERS = ["ark_device.cuh", "ark_step.cuh", "ark_step3d.cuh", os.path.join("..", "..", "include", "ark.h")]
# tile of the fused step kernel: (TX, TY) outputs per block and plane, region (TX+4) x (TY+4) threads
# 3D: 28 outputs per row (32 lanes), ARK_NW3 row pairs per block (tile height 2 * NW3 - 4) on NW3 + 2 warps;
# ARK_REG_RING / ARK_REG_TILE: setmaxnreg targets of the ring warpgroup and of the tile warpgroups (per scheduler:
# 1 ring warp + 2 tile warps, REG_RING + 2 * REG_TILE <= 504: with 512 the allocation never completes)
TILES = {"ARK_TX3": 28, "ARK_NW3": 10, "ARK_REG_RING": 72, "ARK_REG_TILE": 216, "ARK_TX2": 28, "ARK_TY2": 8}


def nvcc_cmd(out, extra=()):
    # the product build takes nothing from the environment: the library the tests and bench.py load is the one the
    # committed profiles/ describe (tuning builds belong in _work/ with their own command line)
    defs = ["-D%s=%d" % (k, v) for k, v in TILES.items()]
    return (["nvcc", "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
             "-Xcompiler", "-fPIC", "-shared", "-o", out] + defs + list(extra)
            + [os.path.join(CSRC, s) for s in SOURCES])


LIB_STRICT = os.path.join(HERE, "libark_b200_strict.so")


def build_strict(force: bool = False) -> str:
    """The same sources with -DARK_STRICT --fmad=false (IEEE division / square root, no FMA contraction): not the
    product, a measuring instrument for reading A20 (tests/test_parity_gpu.py::test_strict_build_*)."""
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    if not force and os.path.exists(LIB_STRICT) and all(os.path.getmtime(LIB_STRICT) >= os.path.getmtime(d) for d in deps):
        return LIB_STRICT
    subprocess.run(nvcc_cmd(LIB_STRICT, ["-DARK_STRICT=1", "--fmad=false"]), check=True)
    return LIB_STRICT


def build(force: bool = False, verbose: bool = False) -> str:
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = nvcc_cmd(LIB, ["-Xptxas", "-v"] if verbose else [])
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--strict" in sys.argv:
        print(build_strict(force="--force" in sys.argv))
