"""Compile the CPU oracle (plain g++; no CUDA).  Test infrastructure only."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "picsarqed_oracle.cpp")
_LIB = os.path.join(_HERE, "libpicsarqed_oracle.so")


def lib_path() -> str:
    return _LIB


def build(force: bool = False) -> str:
    """g++ -O2 -std=c++17 -fopenmp -fPIC -shared picsarqed_oracle.cpp -lquadmath"""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
           _SRC, "-o", tmp, "-lquadmath"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


if __name__ == "__main__":
    print(build(force=True))
