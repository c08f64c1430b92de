"""Build libcube.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1211_4896_b200.build [--force]
"""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libcube.so")
SOURCES = ["cube.cu"]
DEPS = ["cube.cu", "cube_ooc.inl", "cube_kernels.cuh", "cube_common.cuh", "cube_select.cuh", "cube_fused.cuh", "cube_hist_big.cuh", "cube_minimap.cuh", "cube_minimap_tma.cuh", "cube_fused_big.cuh", "cube_torben.cuh", "cube_select_multi.cuh", "cube_render.cuh", "cube_minimap_median.cuh", "cube_gather.cuh", "cube_small.cuh", os.path.join("..", "..", "include", "cube.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=true",            # contraction is confined to fp64 fma() calls we write ourselves;
                                        # the float32 bin formula uses __fsub_rn/__fmul_rn (never contracted)
              "-Xcompiler", "-fPIC", "-shared"]


LIB_CHECKED = os.path.join(_HERE, "libcube_checked.so")


def build(force=False, verbose=False, checked=False):
    """checked=True: libcube_checked.so, the same source with -DCUBE_CHECKED (bounds checks that trap; load it with
    CUBE_LIBPATH=.../libcube_checked.so)."""
    lib = LIB_CHECKED if checked else LIB
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= newest:
        return lib
    tmp = lib + ".tmp.%d" % os.getpid()
    cmd = ["nvcc"] + NVCC_FLAGS + (["-DCUBE_CHECKED"] if checked else []) + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
