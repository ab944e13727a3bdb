"""Build the CPU oracle (test infrastructure) into oracle/librpim_oracle.so.

    python oracle/build.py

Flags: -O2 -ffp-contract=off (no implicit fused multiply-add; fma() calls are explicit),
-march=native when the compiler accepts it so std::fma maps to the hardware instruction.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "rpim_oracle.cpp")
OUT = os.path.join(HERE, "librpim_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= os.path.getmtime(SRC):
        return OUT
    base = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", OUT, SRC]
    for extra in (["-march=native"], []):
        r = subprocess.run(base + extra, capture_output=True, text=True)
        if r.returncode == 0:
            return OUT
    sys.stderr.write(r.stderr)
    raise RuntimeError("oracle build failed")


if __name__ == "__main__":
    print(build(force=True))
