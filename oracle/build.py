"""Build the C oracle (test infrastructure) with gcc: two shared objects, fp64 and fp32.

    python -m oracle.build

Building the checker is not using it: __graft_entry__.build() calls this too.
"""
from __future__ import annotations

import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dwf_oracle.c")


def lib_path(prec: str) -> str:
    return os.path.join(HERE, f"liboracle_dwf_{prec}.so")


def _cpu_signature() -> str:
    """-march=native ties the objects to the CPU they were built on: a library built in one container must not be
    loaded on a box with another CPU (illegal instruction), so the build is redone when this signature changes."""
    model, flags = "", ""
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name") and not model:
                model = ln.split(":", 1)[1].strip()
            elif ln.startswith("flags") and not flags:
                flags = ln.split(":", 1)[1].strip()
            if model and flags:
                break
    except OSError:
        pass
    return hashlib.sha1((model + "|" + flags).encode()).hexdigest()


def build(force: bool = False) -> None:
    sig, stamp = _cpu_signature(), os.path.join(HERE, "build_stamp.txt")
    if not (os.path.exists(stamp) and open(stamp).read().strip() == sig):
        force = True
    for prec, real in (("f64", "double"), ("f32", "float")):
        out = lib_path(prec)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(SRC):
            continue
        # -O3 -march=native as SURVEY 8(d) "Oracle timing" asks; IEEE arithmetic kept (-fno-fast-math, no contraction
        # across statements beyond what the ISA's FMA gives)
        cmd = ["gcc", "-O3", "-march=native", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
               f"-DORC_REAL={real}", f"-DORC_SUFFIX=_{prec}", SRC, "-o", out, "-lm"]
        subprocess.run(cmd, check=True)
    with open(stamp, "w") as f:
        f.write(sig)


if __name__ == "__main__":
    build(force=True)
    print("built", lib_path("f64"), lib_path("f32"))
