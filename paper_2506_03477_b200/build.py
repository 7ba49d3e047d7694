"""In-tree build of libqsgw.so (hand-written CUDA for sm_100a + the C-ABI layer).

`python -m paper_2506_03477_b200.build` or `build()`; nvcc cross-compiles without a GPU.
Every csrc/*.cu is compiled to an object file under csrc/build/ (in parallel, only when stale) and the
objects are linked into the shared library.  The library links the CUDA runtime statically and resolves
the one driver entry point it needs (cuTensorMapEncodeTiled) at run time, so it loads on a machine
without a GPU driver (where every compute call then fails loudly).
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG_DIR, "csrc")
OBJ_DIR = os.path.join(CSRC, "build")
LIB_PATH = os.path.join(PKG_DIR, "libqsgw.so")
INCLUDE = os.path.join(os.path.dirname(PKG_DIR), "include")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static",
              "-Xcompiler", "-fPIC"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) \
        + glob.glob(os.path.join(INCLUDE, "*.h")) + [os.path.abspath(__file__)]


def _obj(src: str) -> str:
    return os.path.join(OBJ_DIR, os.path.splitext(os.path.basename(src))[0] + ".o")


def _run(cmd):
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout)
    return res.stdout


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ_DIR, exist_ok=True)
    hdr_t = max(os.path.getmtime(h) for h in _headers())
    todo = []
    for src in sources():
        o = _obj(src)
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(src), hdr_t):
            todo.append(src)
    for o in glob.glob(os.path.join(OBJ_DIR, "*.o")):          # objects of deleted sources
        if o not in [_obj(s) for s in sources()]:
            os.remove(o)
            force = True
    if not todo and not force and os.path.exists(LIB_PATH) and \
            os.path.getmtime(LIB_PATH) >= max(os.path.getmtime(_obj(s)) for s in sources()):
        return LIB_PATH
    extra = ["-Xptxas", "-v"] if verbose else []
    with ThreadPoolExecutor(max_workers=min(8, max(1, len(todo)))) as ex:
        outs = list(ex.map(lambda s: _run([nvcc] + NVCC_FLAGS + extra + ["-I", INCLUDE, "-c", s, "-o", _obj(s)]),
                           todo))
    if verbose:
        print("\n".join(outs))
    _run([nvcc] + LINK_FLAGS + ["-o", LIB_PATH] + [_obj(s) for s in sources()])
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
