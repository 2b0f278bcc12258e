"""In-tree build of the CUDA library (sm_100a only).  `python -m paper_2502_17805_b200.build [--force] [--verbose]`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libchorus_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def sources():
    out = [os.path.join(ROOT, "include", "chorus.h")]
    for f in sorted(os.listdir(CSRC)):
        out.append(os.path.join(CSRC, f))
    return out


def build(force: bool = False, verbose: bool = False, only_order: int | None = None, out: str = LIB) -> str:
    """only_order = n instantiates the kernels of one order only (-DCHORUS_ONLY_ORDER=n: a 25 s build instead of 2 min, for
    kernel development; such a library refuses every other order).  The default serves orders 2..9."""
    deps = sources()
    if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(d) for d in deps):
        return out
    cmd = [NVCC, "-std=c++17", "-O3", "-lineinfo", *ARCH, "-shared", "-Xcompiler", "-fPIC",
           "-o", out, os.path.join(CSRC, "chorus.cu")]
    if only_order is not None:
        cmd.insert(1, f"-DCHORUS_ONLY_ORDER={int(only_order)}")
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
