"""Build libamrhydro.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "amrhydro.cu")
OUT = os.path.join(HERE, "libamrhydro.so")
DEPS = [os.path.join(HERE, "csrc", f) for f in os.listdir(os.path.join(HERE, "csrc"))] + [
    os.path.join(os.path.dirname(HERE), "include", "amrhydro.h")]


def nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def build(force=False, verbose=False, out=None, extra=()):
    """extra: additional nvcc flags (tuning macros, e.g. -DAMR_MINB64=2); out: alternative .so path."""
    global OUT
    if out:
        OUT, force = out, True
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in DEPS):
        return OUT
    cmd = [nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
           "--use_fast_math" if os.environ.get("AMRHYDRO_FAST_MATH") else "-DAMRHYDRO_PRECISE",
           "-Xcompiler", "-fPIC", "-shared", "-o", OUT, SRC] + list(extra)
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    a = [x for x in sys.argv[1:] if x != "-v"]
    o = a[a.index("-o") + 1] if "-o" in a else None
    ex = [x for x in a if x.startswith("-D")]
    build(force=True, verbose="-v" in sys.argv, out=o, extra=ex)
    print(OUT)
