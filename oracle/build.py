"""Build the CPU oracle (test infrastructure) into oracle/libocnref.so.

    python oracle/build.py

Plain g++ -O2 -fopenmp; no fast-math (the long-double instantiation is the parity reference).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ocnref.cpp")
LIB = os.path.join(HERE, "libocnref.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(os.path.join(HERE, f)) for f in os.listdir(HERE)
                                             if f.endswith((".cpp", ".inc")))):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra",
           SRC, "-o", LIB]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
