"""Builds libnolsm.so (the C-ABI library of include/nolsm.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import glob
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
UNITS = ["abi.cpp", "assemble.cpp", "grouping.cpp", "engine.cu"]          # translation units (csrc/ctx.h says what each holds)
LIB = os.path.join(HERE, "libnolsm.so")
OBJ = os.path.join(HERE, "build")
STAMP = os.path.join(OBJ, "sources.sha256")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "-Xcompiler", "-pthread"]


def nvcc_path() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if p and (os.path.isabs(p) and os.path.exists(p) or not os.path.isabs(p)):
            return p
    return "nvcc"


def sources() -> list[str]:
    """Every file the library is built from: all of csrc/ and the public header."""
    return sorted(glob.glob(os.path.join(CSRC, "*"))) + [os.path.join(os.path.dirname(HERE), "include", "nolsm.h")]


def digest() -> str:
    h = hashlib.sha256()
    for f in sources():
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def needs_build() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as f:
        return f.read().strip() != digest()


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = nvcc_path()

    def compile_unit(u: str):
        obj = os.path.join(OBJ, os.path.splitext(u)[0] + ".o")
        cmd = [nvcc] + FLAGS + (["-Xptxas", "-v"] if verbose and u.endswith(".cu") else []) + ["-c", os.path.join(CSRC, u), "-o", obj]
        return obj, subprocess.run(cmd, capture_output=True, text=True)

    with ThreadPoolExecutor(len(UNITS)) as ex:
        results = list(ex.map(compile_unit, UNITS))
    for obj, res in results:
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
        if verbose:
            print(res.stderr)
    res = subprocess.run([nvcc, "-shared", "-o", LIB] + [o for o, _ in results] + ["-Xcompiler", "-pthread"],
                         capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + res.stdout + res.stderr)
    with open(STAMP, "w") as f:
        f.write(digest())
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
