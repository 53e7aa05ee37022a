"""Opcode histogram of the SASS of the pair kernels and the list builder in libmop_b200.so.

    python -m paper_2501_11962_b200.sass_histogram > profiles/rNN_sass_histogram.md

Runs `cuobjdump -sass` on the built library (no GPU needed) and prints, per kernel, the static instruction count by
opcode: the evidence that the pair math is issued as packed FP32 (FFMA2 / FMUL2 / FADD2), which loads and reductions
the kernel uses (LDS, LDGSTS = cp.async, RED), and how much of the code is not floating point."""
import collections
import re
import subprocess
import sys

from . import build as _build

KERNELS = ["k_nonbonded_p", "k_pairlist"]
FP = ("FFMA2", "FMUL2", "FADD2", "FFMA", "FMUL", "FADD", "MUFU", "FSEL", "FSETP", "FMNMX")


def main():
    lib = _build.build()
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True, check=True).stdout
    fn, hist = None, {}
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn = m.group(1)
            continue
        m = re.match(r"\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_]*)", line)
        if m and fn and any(k in fn for k in KERNELS):
            hist.setdefault(fn, collections.Counter())[m.group(1)] += 1
    names = subprocess.run(["c++filt"] + list(hist), capture_output=True, text=True).stdout.split("\n")
    print("# Static SASS opcode histogram (cuobjdump -sass %s)\n" % lib.split("/")[-1])
    print("Command: `python -m paper_2501_11962_b200.sass_histogram` (sm_100a, nvcc 12.9).  k_nonbonded_p<MODE, COUNT, CTAS>:")
    print("MODE 0 force, 1 force + energy (bead 1), 2 H.eta; COUNT 1 = counting instance used by the tests.\n")
    for fn, nm in zip(hist, names):
        h = hist[fn]
        tot = sum(h.values())
        fp = sum(v for k, v in h.items() if k in FP)
        print("## %s\n" % nm)
        print("%d instructions, %d floating-point (%.0f %%): " % (tot, fp, 100.0 * fp / tot) +
              ", ".join("%s %d" % (k, h[k]) for k in FP if h[k]) + "\n")
        print("| opcode | count |\n|---|---|")
        for k, v in h.most_common(28):
            print("| %s | %d |" % (k, v))
        print()


if __name__ == "__main__":
    sys.exit(main())
