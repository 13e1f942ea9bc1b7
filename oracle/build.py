"""Compile the CPU oracle (test infrastructure) into oracle/libcdz_oracle.so with gcc."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "cdz_oracle.c")]
OUT = os.path.join(HERE, "libcdz_oracle.so")


def build(force: bool = False) -> str:
    srcs = [s for s in SRC if os.path.exists(s)]
    deps = srcs + [os.path.join(HERE, "cdz_oracle.h")]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wno-unused-function",
           "-o", OUT] + srcs + ["-lm"]
    subprocess.run(cmd, check=True)
    return OUT


if __name__ == "__main__":
    print(build(force=True))
