"""nvcc build of the engine: csrc/*.cu -> paper_2607_07816_b200/libsparse_sv.so (sm_100a).

The library is built in-tree so that it travels to the GPU box with the repo snapshot.
Every translation unit is compiled on its own (in parallel, and only when it or a header
changed), then linked.
"""
import glob
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsparse_sv.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CFLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
          "--expt-extended-lambda", "-Xcompiler", "-fPIC"]
LFLAGS = ["-shared", "-cudart", "shared", "-gencode", "arch=compute_100a,code=sm_100a"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(os.path.dirname(HERE), "include", "*.h"))


def _compile(src, force, verbose, extra):
    obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
    deps = [src] + _headers()
    if (not force) and os.path.exists(obj) and all(os.path.getmtime(obj) >= os.path.getmtime(f) for f in deps):
        return obj
    cmd = [NVCC] + CFLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
    subprocess.run(cmd, check=True)
    return obj


def build(force: bool = False, verbose: bool = False, extra=(), checked: bool = False) -> str:
    """checked=True: the bounds-checked build (-DSV_CHECKED, see csrc/sv_device.cuh) INTO THE SAME libsparse_sv.so, for one
    run of the GPU tests; build again without it afterwards."""
    global OBJ
    if checked:
        OBJ = os.path.join(HERE, "build", "checked")
        extra = list(extra) + ["-DSV_CHECKED"]
        force = True
    os.makedirs(OBJ, exist_ok=True)
    srcs = sources()
    with ThreadPoolExecutor(max_workers=min(len(srcs), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(lambda s: _compile(s, force, verbose, list(extra)), srcs))
    if (not force) and (not checked) and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(o) for o in objs):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.run([NVCC] + LFLAGS + ["-o", tmp] + objs, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="-f" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
