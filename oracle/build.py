"""Build the CPU oracle shared libraries (test infrastructure, not the product).

    python oracle/build.py

produces, next to this file,
    libvoila_oracle_f32.so   real = float   (the oracle proper: north_star fixes fp32)
    libvoila_oracle_f64.so   real = double  (used only to derive tolerances / closed-form pins)

Only gcc and libm/libgomp are needed.  Nothing here touches the CUDA path.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "voila_oracle.c")
# -ffp-contract=off: no fused multiply-add unless the source says fmaf(); keeps the straight
# loops' rounding exactly as written on every host.
COMMON = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
          "-fno-fast-math", "-Wall", "-Wextra"]
TARGETS = {
    "libvoila_oracle_f32.so": [],
    "libvoila_oracle_f64.so": ["-DVO_REAL=double", "-DVO_REAL_IS_DOUBLE=1"],
}


def build(force: bool = False) -> dict:
    out = {}
    for name, defs in TARGETS.items():
        dst = os.path.join(HERE, name)
        out[name] = dst
        if (not force and os.path.exists(dst)
                and os.path.getmtime(dst) >= os.path.getmtime(SRC)):
            continue
        cmd = COMMON + defs + [SRC, "-o", dst, "-lm"]
        subprocess.check_call(cmd)
    return out


if __name__ == "__main__":
    for k, v in build(force="--force" in sys.argv).items():
        print(k, "->", v)
