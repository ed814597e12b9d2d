"""Build the CPU oracle (oracle/pa_oracle.cpp) into oracle/libpa_oracle.so with g++.

Test infrastructure only: called by tests/, __graft_entry__.build() and bench.py's CPU legs.
-ffp-contract=off: no fused multiply-add may be formed (O6: tau_hat is one multiply
then one divide).  -O2 and OpenMP over replicas as stated in DESIGN.md section 7.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pa_oracle.cpp")
LIB = os.path.join(HERE, "libpa_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
