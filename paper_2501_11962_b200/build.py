"""Builds libmop_b200.so (the C-ABI of include/mop.h) from csrc/ with nvcc for sm_100a, in-tree."""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libmop_b200.so")
CHECKED_LIB = os.path.join(_HERE, "libmop_b200_checked.so")   # -DMOP_CHECK build of tests/sanitizer_target.py --checked
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--use_fast_math=false",
         "-Xcompiler", "-fPIC,-O2", "-shared", "-cudart", "static"]


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC))


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    inc = os.path.join(os.path.dirname(_HERE), "include", "mop.h")
    return any(os.path.getmtime(f) > t for f in sources() + [inc, os.path.abspath(__file__)])


def build(force=False, verbose=False, extra=(), out=None):
    """Compile the CUDA library if it is missing or older than its sources.  Returns the .so path.
    out: build to that file instead (always; e.g. CHECKED_LIB with extra=["-DMOP_CHECK"]) and leave the product alone."""
    if out is None and not (force or needs_build()):
        return LIB
    lib = out or LIB
    flags = [f for f in FLAGS if not f.startswith("--use_fast_math")]
    # mop_noalloc.cu is a translation unit of its own: its file-scope device array and the host code that looks up the
    # array's address have to live in one file
    cmd = ([NVCC] + flags + list(extra) + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib]
           + [os.path.join(CSRC, src) for src in ("mop_api.cu", "mop_noalloc.cu")])
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building " + os.path.basename(lib))
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
