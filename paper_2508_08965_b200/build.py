"""Builds paper_2508_08965_b200/libcgks.so (hand-written CUDA for sm_100a) in-tree with nvcc."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcgks.so")
SOURCES = ["cgks_api.cu", "cgks_static.cu"]
HEADERS = ["cgks_common.cuh", "kernels_setup.cuh", "kernels_stage.cuh", "kernels_fused.cuh", "gks_flux.cuh", "fastmath64.cuh", "recon_gen.cuh", "math_gen.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _newer(a, b):
    return os.path.getmtime(a) > os.path.getmtime(b)


def generate(force=False):
    gen = os.path.join(CSRC, "gen_recon.py"); out = os.path.join(CSRC, "recon_gen.cuh")
    if force or not os.path.exists(out) or _newer(gen, out):
        subprocess.check_call([sys.executable, gen])
    gen = os.path.join(CSRC, "gen_math.py"); out2 = os.path.join(CSRC, "math_gen.cuh")
    if force or not os.path.exists(out2) or _newer(gen, out2):
        subprocess.check_call([sys.executable, gen])
    return out


def build(force=False, verbose=False):
    generate(force)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(HERE, "..", "include", "cgks.h")]
    if not force and os.path.exists(LIB) and all(not _newer(d, LIB) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


LIB_AB = os.path.join(HERE, "libcgks_ab.so")


def build_ab(force=False):
    """TEST-ONLY A/B library: the same sources with -DCGKS_AB_SPLIT_PIPELINE, i.e. every stage runs the three-kernel pipeline of
    rounds 1-2 (flux -> face-flux buffer -> update) instead of the sweep kernels.  tests/test_gpu_parity.py loads it to compare
    the two pipelines; the product (binding.py, bench.py) never does."""
    generate(False)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(HERE, "..", "include", "cgks.h")]
    if not force and os.path.exists(LIB_AB) and all(not _newer(d, LIB_AB) for d in deps):
        return LIB_AB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.check_call([nvcc] + NVCC_FLAGS + ["-DCGKS_AB_SPLIT_PIPELINE", "-o", LIB_AB] + [os.path.join(CSRC, s) for s in SOURCES])
    return LIB_AB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
