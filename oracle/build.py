"""Compile the oracle (TEST INFRASTRUCTURE ONLY) with gcc.  Building the checker is not using it.

  python -m oracle.build        -> oracle/liboracle_f64.so  (the oracle)
                                   oracle/liboracle_f32.so  (FP32 yardstick, DESIGN.md protocol P4)
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dm_oracle.c")


def lib_path(real: str = "f64") -> str:
    return os.path.join(HERE, f"liboracle_{real}.so")


def build(force: bool = False) -> None:
    for real, ctype in (("f64", "double"), ("f32", "float")):
        out = lib_path(real)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(SRC):
            continue
        # -O2 without -ffast-math: the summation orders written in the source are kept.
        cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra",
               f"-DORACLE_REAL={ctype}", SRC, "-o", out + ".tmp", "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)


if __name__ == "__main__":
    build(force=True)
    print("built", lib_path("f64"), lib_path("f32"))
