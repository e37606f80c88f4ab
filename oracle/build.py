"""Build the CPU oracle (test infrastructure; see lisa_oracle.c header).

    python -m oracle.build

writes oracle/liblisa_oracle_ld.so (REAL = long double, the parity truth) and
oracle/liblisa_oracle_d.so (REAL = double, the timed CPU baseline).

With ORACLE_SANITIZE=1 in the environment the two libraries are built (under other names) with
-fsanitize=address,undefined, and oracle.binding loads those; run the CPU suite under them with

    LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 ORACLE_SANITIZE=1 \
        python -m pytest tests -q -m "not gpu"

(profiles/r2_sanitizers.md records the outcome).
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
    sanitize = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
    for key, (lib, defs) in TARGETS.items():
        opt = ["-O2"]
        if sanitize:
            lib = lib.replace(".so", "_asan.so")
            opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"]
        stale = (not os.path.exists(lib)) or os.path.getmtime(lib) < os.path.getmtime(SRC)
        if force or stale:
            cmd = ["gcc", "-std=c11", *opt, "-fPIC", "-shared", "-fopenmp", "-fno-fast-math",
                   "-ffp-contract=off", "-Wall", "-Wextra", "-Wno-unused-parameter",
                   *defs, SRC, "-o", lib, "-lm"]
            subprocess.run(cmd, check=True)
        out[key] = lib
    return out


if __name__ == "__main__":
    for k, v in build(force="--force" in sys.argv).items():
        print(k, v)
