"""Build the float64 CPU oracle (test infrastructure only) with gcc.

Two shared objects from the same source: ``libnsm_oracle.so`` (single thread, deterministic
summation order; what the parity tests use) and ``libnsm_oracle_omp.so`` (``-fopenmp``; what
bench.py's cpu_baseline / --impl reference legs time).  ``-ffp-contract=off`` keeps the fp32 index path to exactly
the operations written in nsm_oracle.c.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nsm_oracle.c")
HDR = os.path.join(HERE, "nsm_oracle.h")
BASE = ["gcc", "-std=c11", "-O2", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
        "-Wall", "-Wextra", "-Wno-unknown-pragmas"]


def _stale(out):
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return t < os.path.getmtime(SRC) or t < os.path.getmtime(HDR)


def build(force=False):
    outs = {}
    for name, extra in (("libnsm_oracle.so", []), ("libnsm_oracle_omp.so", ["-fopenmp"])):
        out = os.path.join(HERE, name)
        if force or _stale(out):
            cmd = BASE + extra + [SRC, "-o", out + ".tmp", "-lm"]
            subprocess.run(cmd, check=True, cwd=HERE)
            os.replace(out + ".tmp", out)
        outs[name] = out
    return outs


if __name__ == "__main__":
    print(build(force=True))
