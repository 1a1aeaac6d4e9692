"""Build the CPU oracle (TEST INFRASTRUCTURE) into oracle/liborc.so with gcc.

Three translation units from the same plain-C source, one per precision mode
(see the header of su2_oracle.c). -O2, no fast-math, no FMA contraction, so the
arithmetic is exactly what the source says.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "su2_oracle.c")
LIB = os.path.join(HERE, "liborc.so")

MODES = [
    # suffix, storage, arithmetic, uniform rule, extra
    ("f64", "double", "double", 64, ["-DORC_EMIT_COMMON"]),
    ("f32", "float", "float", 32, ["-DORC_AREAL_IS_FLOAT"]),
    ("f32x", "float", "double", 32, []),
]
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(__file__))):
        return LIB
    objs = []
    for sfx, real, areal, ubits, extra in MODES:
        obj = os.path.join(HERE, f"su2_oracle_{sfx}.o")
        cmd = ["gcc", *CFLAGS, f"-DORC_SFX={sfx}", f"-DORC_REAL={real}", f"-DORC_AREAL={areal}",
               f"-DORC_UNIFORM_BITS={ubits}", *extra, "-c", SRC, "-o", obj]
        subprocess.run(cmd, check=True)
        objs.append(obj)
    subprocess.run(["gcc", "-shared", "-o", LIB, *objs, "-lm"], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
