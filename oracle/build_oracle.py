"""Build oracle/liblrux_oracle.so from oracle/lrux_oracle_c.c with gcc (-O2, OpenMP).
TEST INFRASTRUCTURE ONLY: the checker, not the product (``__graft_entry__.build()``
compiles it; building the checker is not using it)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "lrux_oracle_c.c"), os.path.join(HERE, "lrux_oracle_body.h"), os.path.abspath(__file__)]
LIB = os.path.join(HERE, "liblrux_oracle.so")
# /usr/bin/gcc first: the image's $CC (/opt/gcc/bin/gcc) ships without libgomp.spec
COMPILERS = ["/usr/bin/gcc", os.environ.get("CC", "gcc"), "gcc", "cc"]
# -O2 without -ffast-math: IEEE semantics, no reassociation.  -fcx-limited-range: complex
# products and quotients by their textbook formulas (no __muldc3 NaN-recovery calls)
FLAGS = ["-O2", "-fcx-limited-range", "-shared", "-fPIC", "-std=c11", "-Wall", "-Wextra"]


def build(force=False, verbose=False):
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(s) for s in SRC):
        return LIB
    errs = []
    for omp in (["-fopenmp"], []):          # without OpenMP the batch runs on one core (reported as such)
        for cc in COMPILERS:
            cmd = [cc, *FLAGS, *omp, "-o", LIB, SRC[0], "-lm"]
            if verbose:
                print(" ".join(cmd), flush=True)
            try:
                r = subprocess.run(cmd, capture_output=True, text=True)
            except OSError as e:
                errs.append("%s: %s" % (cc, e))
                continue
            if r.returncode == 0:
                return LIB
            errs.append("%s: %s" % (" ".join(cmd), r.stderr.strip()[-400:]))
    raise RuntimeError("no C compiler built the C oracle:\n" + "\n".join(errs))


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
