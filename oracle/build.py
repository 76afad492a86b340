"""Build the oracle shared library (test infrastructure; see ts_oracle.h).

    python -m oracle.build

gcc, C99, -O2, no FMA contraction, no fast-math (-fopenmp only serves orc_set_threads): fp32 results are those of the written
sequence of single operations (reading R21)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ts_oracle.c")
LIB = os.path.join(HERE, "libts_oracle.so")
FLAGS = ["-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra",
         "-fPIC", "-shared", "-fopenmp"]


def build(force=False):
    deps = [SRC, os.path.join(HERE, "ts_oracle.h")]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    subprocess.run(["gcc", *FLAGS, SRC, "-o", LIB, "-lm"], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
