"""Compile csrc/ into paper_1808_10365_b200/libsk_b200.so (the product: include/sk_b200.h) and
csrc/bench/ into libsk_b200_bench.so (measurement kernels for bench.py: csrc/bench/sk_bench.h) for
sm_100a with nvcc (in-tree, so the built libraries travel with the repository snapshot).
`python -m paper_1808_10365_b200.build`."""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsk_b200.so")
BENCH_LIB = os.path.join(HERE, "libsk_b200_bench.so")
_HDR = os.path.join("..", "..", "include", "sk_b200.h")
_COMMON = ["sk_kernels.cuh", "sk_device.cuh", "sk_tma.cuh", _HDR]
# target -> (source, files it depends on), all relative to csrc/
TARGETS = {
    LIB: ("sk_api.cu", ["sk_api.cu", "sk_sim.cuh"] + _COMMON),
    BENCH_LIB: (os.path.join("bench", "sk_bench.cu"),
                [os.path.join("bench", f) for f in ("sk_bench.cu", "sk_bench.h", "sk_ceiling.cuh")] + _COMMON),
}


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the SK library cannot be built")


def up_to_date(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return False
    t = os.path.getmtime(lib)
    return all(os.path.getmtime(os.path.join(CSRC, d)) <= t for d in TARGETS[lib][1])


def build_one(lib: str, force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date(lib):
        return lib
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "--shared", "-Xcompiler", "-fPIC", "-cudart", "static"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, TARGETS[lib][0]), "-o", lib + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(lib + ".tmp", lib)
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    """The product library (returned) and the bench library."""
    build_one(BENCH_LIB, force, verbose)
    return build_one(LIB, force, verbose)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
