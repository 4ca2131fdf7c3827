"""Build the C oracle (test infrastructure) into oracle/libqarray_oracle.so and, if OpenMP is available,
oracle/libqarray_oracle_omp.so (the same source under an OpenMP parallel-for over pixels; bench.py's all-cores baseline).

    python oracle/build.py
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "qarray_oracle.c")
FLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra"]


def _stale(out):
    return (not os.path.exists(out)) or os.path.getmtime(out) < os.path.getmtime(SRC)


def build(force: bool = False, verbose: bool = False):
    outs = []
    for name, extra in (("libqarray_oracle.so", []), ("libqarray_oracle_omp.so", ["-fopenmp"])):
        out = os.path.join(HERE, name)
        if force or _stale(out):
            cmd = ["gcc", *FLAGS, *extra, "-o", out, SRC, "-lm"]
            if verbose:
                print(" ".join(cmd))
            r = subprocess.run(cmd, capture_output=True, text=True)
            if r.returncode != 0:
                if extra:            # OpenMP is optional
                    continue
                raise RuntimeError("oracle build failed:\n" + r.stderr)
        outs.append(out)
    return outs


if __name__ == "__main__":
    print("\n".join(build(force="--force" in sys.argv, verbose=True)))
