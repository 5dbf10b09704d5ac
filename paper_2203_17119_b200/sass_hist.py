"""SASS opcode histogram of the Dhop TMA kernel instantiations in the built library (evidence that the hot kernel is
Blackwell-native tile movement -- UTMALDG = cp.async.bulk.tensor, SYNCS = mbarrier, USETMAXREG = setmaxnreg, UBLKPF = bulk L2
prefetch, LDGSTS = cp.async -- on plain FP pipes: the contraction is 3 x 3 complex, K = 3, so there is no UTC*MMA / HMMA).

    python -m paper_2203_17119_b200.sass_hist > profiles/r02_sass_hist.md

Needs cuobjdump and c++filt; reads paper_2203_17119_b200/libdwf_b200.so (build it first)."""
from __future__ import annotations

import collections
import os
import re
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libdwf_b200.so")
OPS = ["UTMALDG", "SYNCS", "USETMAXREG", "UBLKPF", "LDGSTS", "DFMA", "DMUL", "DADD", "FFMA", "FMUL", "FADD", "LDS", "LDG",
       "STG", "SHFL", "FSEL", "STL", "LDL", "BAR", "UTC", "HMMA"]


def histogram():
    sass = subprocess.run(["cuobjdump", "-sass", LIB], capture_output=True, text=True, check=True).stdout
    rows = []
    for f in re.split(r"\n\s*Function : ", sass)[1:]:
        mangled = f.split("\n", 1)[0].strip()
        if "dhop_tma_kernel" not in mangled:
            continue
        dem = subprocess.run(["c++filt", mangled], capture_output=True, text=True).stdout.strip()
        m = re.search(r"dhop_tma_kernel<([^>]*)>", dem)
        cnt, total = collections.Counter(), 0
        for line in f.split("\n"):
            mm = re.match(r"\s+/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\w+\s+)?([A-Z0-9_.]+)", line)
            if mm:
                total += 1
                for w in OPS:
                    if mm.group(1).startswith(w):
                        cnt[w] += 1
        rows.append(((m.group(1) if m else dem).replace("(int)", ""), cnt, total))
    return sorted(rows)


def main():
    print("# r02 -- SASS opcode histogram of `dwf::dhop_tma_kernel<R, TPS, NG, NST, MINB, EPI>` (sm_100a)\n")
    print("Command: `python -m paper_2203_17119_b200.sass_hist > profiles/r02_sass_hist.md` (cuobjdump -sass of the in-tree "
          "`libdwf_b200.so`; static instruction counts of the whole kernel: producer, link rebuild and one unrolled s-slice "
          "of the consumer loop).\n")
    print("| instantiation | " + " | ".join(OPS) + " | all |")
    print("|" + "---|" * (len(OPS) + 2))
    for name, c, total in histogram():
        print("| " + name + " | " + " | ".join(str(c[w]) for w in OPS) + f" | {total} |")
    print("\nReading: every instantiation moves its tiles with UTMALDG (3-D and 4-D tensor boxes) and LDGSTS gathers completing on "
          "SYNCS mbarriers, shrinks / grows its register file with USETMAXREG, prefetches the next tile's links with UBLKPF.L2; "
          "no UTC*MMA / HMMA (K = 3 contraction, SURVEY 8d). STL / LDL: 4-28 bytes of spills, all in the producer warp or "
          "loop-invariant (DESIGN.md section 5.1). s-loop bodies (one slice, per consumer thread): fp64 plain 432 FP64 + 48 LDS.128 "
          "+ 24 SHFL + 48 FSEL + 6 STG of 612 instructions; fp32 plain 870 FP32 + 48 LDS.128 + 6 STG of 959 (1032 FP32 of 1144 "
          "before the rebuilt third link row was pinned in registers, DESIGN.md section 7).")


if __name__ == "__main__":
    main()
