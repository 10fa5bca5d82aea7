"""Build the CPU oracle (TEST INFRASTRUCTURE, not the product) with gcc.

Three shared objects from the one source dg_oracle.c:
  libdg_oracle.so      fp64, single-threaded, -ffp-contract=off   (the parity oracle)
  libdg_oracle_ld.so   x87 long double arbiter build, same source (-DORACLE_REAL="long double")
  libdg_oracle_omp.so  fp64 with `#pragma omp parallel for` over elements (timing baseline;
                       bit-identical to the single-threaded build, tests check that)
  libdg_oracle_ld_omp.so  the long double arbiter with the same OpenMP loops (bit-identical to
                       the single-threaded arbiter; used where the arbiter runs 100 steps)

Usage:  python oracle/build.py [--force]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dg_oracle.c")
HDR = os.path.join(HERE, "dg_oracle.h")

VARIANTS = {
    "libdg_oracle.so": [],
    "libdg_oracle_ld.so": ['-DORACLE_REAL=long double'],
    "libdg_oracle_omp.so": ["-fopenmp"],
    "libdg_oracle_ld_omp.so": ['-DORACLE_REAL=long double', "-fopenmp"],
}
CFLAGS = ["-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
          "-Wall", "-Wextra"]


def build(force=False, verbose=False):
    """Compile every variant that is missing or older than its source. Returns the paths."""
    out = {}
    newest_src = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
    for name, extra in VARIANTS.items():
        path = os.path.join(HERE, name)
        out[name] = path
        if not force and os.path.exists(path) and os.path.getmtime(path) >= newest_src:
            continue
        cmd = ["gcc"] + CFLAGS + extra + ["-o", path, SRC, "-lm"]
        if verbose:
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
