"""Build the CPU oracle shared libraries (TEST INFRASTRUCTURE, not the product).

    python oracle/build.py            # builds oracle/libdse_oracle.so and oracle/libdse_oracle_ld.so

-O2, no -ffast-math, -ffp-contract=off so that the arithmetic is exactly what the source states.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dse_oracle.c")
TARGETS = {
    "libdse_oracle.so": [],
    "libdse_oracle_ld.so": ["-DORACLE_LONG_DOUBLE"],
}


def build(force: bool = False) -> dict:
    out = {}
    for name, defs in TARGETS.items():
        so = os.path.join(HERE, name)
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(SRC):
            cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
                   "-Wall", "-Wextra", *defs, "-o", so, SRC, "-lm"]
            subprocess.run(cmd, check=True)
        out[name] = so
    return out


if __name__ == "__main__":
    for k, v in build(force="--force" in sys.argv).items():
        print(k, "->", v)
