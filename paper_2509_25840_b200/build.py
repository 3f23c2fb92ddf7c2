"""In-tree build of libchfpe.so (hand-written sm_100a CUDA kernels + C-ABI host code) with nvcc."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(_HERE, "libchfpe.so")
SOURCES = ["chfpe_api.cu", "chfpe_kernels.cu", "chfpe_brick.cu", "chfpe_tma.cu", "chfpe_compact.cu", "chfpe_spectra.cu", "chfpe_hermite.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--use_fast_math=false", "-Xcompiler", "-fPIC", "-shared"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _deps():
    src = [os.path.join(_HERE, "csrc", s) for s in SOURCES]
    return src, src + [os.path.join(_HERE, "csrc", "chfpe_internal.cuh"), os.path.join(_HERE, "csrc", "chfpe_poly.h"), os.path.join(_HERE, "csrc", "chfpe_hermite_tma.cuh"), os.path.join(_HERE, "..", "include", "chfpe.h")]


def stale():
    """True if libchfpe.so is missing or older than any of its sources."""
    _, deps = _deps()
    return not os.path.exists(SO) or os.path.getmtime(SO) < max(os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    src, deps = _deps()
    if not force and not stale():
        return SO
    tmp = SO + ".tmp%d" % os.getpid()
    flags = [f for f in NVCC_FLAGS if f != "--use_fast_math=false"]
    cmd = [_nvcc()] + flags + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + src
    subprocess.check_call(cmd)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
