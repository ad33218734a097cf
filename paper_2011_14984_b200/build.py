"""Build libfrost_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Every csrc/*.cu is compiled to its own object (in parallel, only when stale) under
paper_2011_14984_b200/build/, then linked with the static CUDA runtime.  probe/frost_probe.cu (the
FP64 issue-rate probe bench.py times) becomes its own libfrost_probe.so: measurement code stays out
of the product library."""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libfrost_b200.so")
PROBE_SRC = os.path.join(HERE, "probe", "frost_probe.cu")
PROBE_LIB = os.path.join(HERE, "libfrost_probe.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
CFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
          "-Xcompiler", "-fPIC"]
LFLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC",
          "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(HERE, "..", "include", "*.h"))


def _obj(src):
    return os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")


def _newer(deps, target):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build_probe(force: bool = False) -> str:
    deps = [PROBE_SRC, os.path.join(HERE, "probe", "frost_probe.h")]
    if force or _newer(deps, PROBE_LIB):
        subprocess.check_call([NVCC] + CFLAGS + ["-shared", "-cudart", "static", "-o", PROBE_LIB, PROBE_SRC])
    return PROBE_LIB


def build(force: bool = False, verbose: bool = False) -> str:
    build_probe(force)
    hdr = _headers()
    if not force and not _newer(sources() + hdr, LIB):
        return LIB                      # (a box that received the built library never recompiles)
    os.makedirs(OBJ, exist_ok=True)
    todo = [s for s in sources() if force or _newer([s] + hdr, _obj(s))]

    def compile_one(src):
        cmd = [NVCC] + CFLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", _obj(src), src]
        subprocess.check_call(cmd)

    if todo:
        with ThreadPoolExecutor(max_workers=min(len(todo), os.cpu_count() or 1)) as ex:
            list(ex.map(compile_one, todo))
    objs = [_obj(s) for s in sources()]
    stale = [o for o in glob.glob(os.path.join(OBJ, "*.o")) if o not in objs]
    for o in stale:                     # the object of a source file that no longer exists
        os.remove(o)
    if todo or stale or _newer(objs, LIB):
        subprocess.check_call([NVCC] + LFLAGS + ["-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
