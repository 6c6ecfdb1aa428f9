"""Build paper_2606_21381_b200/libosog.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_21381_b200.build [--force] [--verbose]
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libosog.so")
SOURCES = ["osog_api.cu", "binning.cu", "compose.cu", "optics.cu"]
HEADERS = [os.path.join(CSRC, "osog_internal.cuh"), os.path.join(os.path.dirname(HERE), "include", "osog.h")]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libosog.so cannot be built (there is no CPU fallback)")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC,-Wall,-Wno-unused-function", "-shared",
           "-Xlinker", "-rpath=/usr/local/cuda/lib64",
           "-o", LIB + ".tmp"] + [os.path.join(CSRC, s) for s in SOURCES] + ["-lcufft"]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


def build_issue_rates() -> str:
    """The instruction-rate microbenchmark behind the ALU roofline (csrc/issue_rates.cu), a standalone executable."""
    out = os.path.join(HERE, "issue_rates")
    subprocess.run([_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-w", "-o", out,
                    os.path.join(CSRC, "issue_rates.cu")], check=True)
    return out


if __name__ == "__main__":
    if "--issue-rates" in sys.argv:
        print(build_issue_rates())
    else:
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
