"""oracle/build.py -- TEST INFRASTRUCTURE: compiles oracle/direct_sums.c with gcc.

Two instances of the same source are built: `long double` (parity reference)
and `double` (the timed CPU baseline).  Nothing here is used by the product
path (paper_2402_01282_b200/); see oracle/__init__.py.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "direct_sums.c")
VARIANTS = {
    "f80": ["-DREAL=long double"],
    "f64": ["-DREAL=double", "-DORC_DOUBLE"],
}


def lib_path(variant):
    return os.path.join(HERE, "liboracle_%s.so" % variant)


def build(force=False):
    """Compile both instances (no -ffast-math: IEEE evaluation order is kept)."""
    for variant, defs in VARIANTS.items():
        out = lib_path(variant)
        if (not force and os.path.exists(out)
                and os.path.getmtime(out) >= os.path.getmtime(SRC)):
            continue
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99",
               "-fno-fast-math", "-o", out, SRC, "-lm"] + defs
        subprocess.check_call(cmd)


if __name__ == "__main__":
    build(force=True)
    print("built", [lib_path(v) for v in VARIANTS])
