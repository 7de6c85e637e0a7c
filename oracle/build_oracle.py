"""Build oracle/liboracle.so (TEST INFRASTRUCTURE ONLY -- see hydro_oracle.cpp header).

g++ -O2 -ffp-contract=off: no FMA contraction, no fast-math, so the oracle's rounding is the
plain IEEE evaluation of the formulas as written.  Building the checker is not using it.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hydro_oracle.cpp")
SRCS = [SRC, os.path.join(HERE, "amr_oracle.cpp"),  # the fluid update; the flux fix-up / restriction that consume its fluxes
        os.path.join(HERE, "rtvd_oracle.cpp"),       # the directionally split relaxing-TVD update (the paper's contrast scheme)
        os.path.join(HERE, "waf_oracle.cpp")]        # the directionally split weighted-average-flux update
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in SRCS):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wextra", "-o", LIB + ".tmp"] + SRCS
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
