"""Build libvpmc.so in-tree with nvcc for sm_100a (python -m paper_2307_01416_b200.build)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvpmc.so")
SOURCES = ["vpmc_api.cu"]
DEPS = ["vpmc_api.cu", "vpmc_run.inl", "vpmc_influence.inl", "vpmc_host.h", "vpmc_kernels.cuh", "vpmc_transport.cuh",
        "vpmc_device.cuh", "vpmc_setup.cuh", "vpmc_spmv.cuh", "vpmc_spmv.inl", "vpmc_gamma.cuh", "../../include/vpmc.h"]


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
           "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr", "-ftz=true",
           "-Xptxas", "-v" if verbose else "-O3", "-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
