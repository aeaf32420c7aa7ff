"""Build the fp64 CPU oracle (oracle/gl_oracle.c) into oracle/libgl_oracle.so with gcc.

TEST INFRASTRUCTURE ONLY (see the header of gl_oracle.c).  `python -m oracle.build` or
`oracle.build.build()`; __graft_entry__.build() calls it too (building the checker is not using it).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gl_oracle.c")
LIB = os.path.join(HERE, "libgl_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # -ffp-contract=off: no FMA contraction, plain IEEE double round-to-nearest (reading S20).
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=gnu11",
           "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
