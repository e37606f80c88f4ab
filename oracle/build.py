"""Build the CPU oracle (test infrastructure; see lisa_oracle.c header).

    python -m oracle.build

writes oracle/liblisa_oracle_ld.so (REAL = long double, the parity truth) and
oracle/liblisa_oracle_d.so (REAL = double, the timed CPU baseline).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lisa_oracle.c")
TARGETS = {
    "ld": (os.path.join(HERE, "liblisa_oracle_ld.so"), ["-DORC_REAL_LD"]),
    "d": (os.path.join(HERE, "liblisa_oracle_d.so"), []),
}


def build(force: bool = False) -> dict:
    out = {}
    for key, (lib, defs) in TARGETS.items():
        stale = (not os.path.exists(lib)) or os.path.getmtime(lib) < os.path.getmtime(SRC)
        if force or stale:
            cmd = ["gcc", "-std=c11", "-O2", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math",
                   "-ffp-contract=off", "-Wall", "-Wextra", "-Wno-unused-parameter",
                   *defs, SRC, "-o", lib, "-lm"]
            subprocess.run(cmd, check=True)
        out[key] = lib
    return out


if __name__ == "__main__":
    for k, v in build(force="--force" in sys.argv).items():
        print(k, v)
