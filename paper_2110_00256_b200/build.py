"""Compile libpicsarqed.so for sm_100a with nvcc, in-tree (no JIT cache, no CPU fallback).

nvcc cross-compiles without a GPU, so this also runs on the CPU-only build box.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_LIB = os.path.join(_HERE, "libpicsarqed.so")
_SOURCES = ["picsarqed.cu"]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def lib_path() -> str:
    return _LIB


def _stale() -> bool:
    if not os.path.exists(_LIB):
        return True
    t = os.path.getmtime(_LIB)
    # every file under csrc/ is a dependency (picsarqed.cu includes all the .cuh headers)
    deps = [os.path.join(_CSRC, f) for f in os.listdir(_CSRC) if f.endswith((".cu", ".cuh", ".h"))]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "picsarqed.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo ... -o libpicsarqed.so"""
    if not force and not _stale():
        return _LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + ["-o", tmp] + [os.path.join(_CSRC, s) for s in _SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stderr)
    os.replace(tmp, _LIB)
    return _LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
