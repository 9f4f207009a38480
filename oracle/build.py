"""Build the CPU oracle (test infrastructure) with g++.  -ffp-contract=off: the float32 indexing
twin must execute exactly the operations written (explicit std::fmaf only)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))


def main() -> None:
    src = os.path.join(HERE, "gabsplat_oracle.cpp")
    out = os.path.join(HERE, "liboracle_gabsplat.so")
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-o", out, src]
    subprocess.check_call(cmd)
    print("built", out, file=sys.stderr)


if __name__ == "__main__":
    main()
