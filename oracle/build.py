"""Build the fp64 CPU oracle (oracle/birkhoff4_oracle.c -> oracle/libbirkhoff4_oracle.so) with gcc.

TEST INFRASTRUCTURE: the product (paper_2606_07574_b200) never imports or links this.
Run as `python -m oracle.build`; `__graft_entry__.build()` and the test fixtures call `build()`.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "birkhoff4_oracle.c")
LIB = os.path.join(HERE, "libbirkhoff4_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # no -ffast-math: the oracle must keep IEEE semantics (NaN/Inf propagation, exact rounding order)
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra",
           "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


SRC_OT = os.path.join(HERE, "ot_oracle.c")
LIB_OT = os.path.join(HERE, "libot_oracle.so")


def build_ot(force: bool = False) -> str:
    """the general small entropic-OT / n x n Birkhoff oracle (oracle/ot_oracle.c)"""
    if not force and os.path.exists(LIB_OT) and os.path.getmtime(LIB_OT) >= os.path.getmtime(SRC_OT):
        return LIB_OT
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra",
           "-o", LIB_OT + ".tmp", SRC_OT, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB_OT + ".tmp", LIB_OT)
    return LIB_OT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
    print(build_ot(force="--force" in sys.argv))
