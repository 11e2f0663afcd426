"""Compile csrc/ into paper_1508_06268_b200/librfimpt.so for sm_100a with nvcc (in-tree).

Usage: python -m paper_1508_06268_b200.build [--force] [--verbose]

Debug builds: RFIM_PT_NVCC_FLAGS adds nvcc flags (e.g. -DRFIM_RES_CHECK: range checks on every address the resident kernel
forms) and RFIM_PT_LIB_OUT names another output file; point RFIM_PT_LIB at it to run the tests against that build.
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librfimpt.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _newest_input():
    deps = glob.glob(os.path.join(CSRC, "*")) + [os.path.join(HERE, "..", "include", "rfim_pt.h")]
    return max(os.path.getmtime(p) for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    extra = os.environ.get("RFIM_PT_NVCC_FLAGS", "").split()
    out = os.environ.get("RFIM_PT_LIB_OUT") or LIB
    if not force and not extra and os.path.exists(out) and os.path.getmtime(out) >= _newest_input():
        return out
    cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "--shared", "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math", "--fmad=false"] + extra + ["-o", out] + sources()
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True, cwd=HERE)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
