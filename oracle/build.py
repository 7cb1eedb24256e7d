"""Build step of the CPU oracle (TEST INFRASTRUCTURE ONLY, see lbmimb_oracle.c).

`python oracle/build.py` (or `oracle.build.build()`) compiles
oracle/lbmimb_oracle.c with gcc into oracle/liblbmimb_oracle.so.
-ffp-contract=off: no FMA contraction (R4); -fopenmp: the outer node
loop only.  Nothing of paper_1011_2613_b200/ is read or linked here.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lbmimb_oracle.c")
LIB = os.path.join(HERE, "liblbmimb_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-std=gnu99", "-Wall", "-o", LIB + ".tmp%d" % os.getpid(), SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(cmd[cmd.index("-o") + 1], LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
