"""Build libexx_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libexx_b200.so")
# middle-axis transform lengths: the three pass files are compiled once per length (-DEXX_TB=..., csrc/exx_inst.cuh)
TB_LENGTHS = [16, 24, 32, 48, 64, 72, 96, 128, 144, 192, 256]
# development shortcut: EXX_DEV_LENGTHS=96,192 builds only the mixes of those (main) lengths -- seconds instead of minutes
# while a kernel is being tuned.  The mode is recorded next to the objects; a library built in another mode is stale.
DEV = [int(x) for x in os.environ.get("EXX_DEV_LENGTHS", "").replace(" ", "").split(",") if x]
DEV_FLAGS = []
if DEV:
    TB_LENGTHS = sorted(DEV)
    DEV_FLAGS = ["-DEXX_DEV_LENGTHS_LIST=" + " ".join(f"X({t})" for t in TB_LENGTHS)]
MODE = "dev:" + ",".join(map(str, TB_LENGTHS)) if DEV else "full"
# (source, extra defines, object name); the heaviest units first so that the parallel build ends sooner
UNITS = [(f"exx_pass_{p}.cu", [f"-DEXX_TB={tb}"], f"exx_pass_{p}_{tb}.o") for tb in reversed(TB_LENGTHS) for p in "bca"] + \
        [("exx_api.cu", [], "exx_api.o"), ("exx_dispatch.cu", [], "exx_dispatch.o"), ("exx_diag.cu", [], "exx_diag.o"),
         ("exx_noalloc.cu", [], "exx_noalloc.o")]
SOURCES = sorted({u[0] for u in UNITS})
HEADERS = ["exx_dft.cuh", "exx_async.cuh", "exx_passes.cuh", "exx_launch.h", "exx_inst.cuh", "exx_sched.hpp", "../../include/exx.h"]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-std=c++17", "-O3", "-lineinfo", "-Xcompiler", "-fPIC"] + os.environ.get("EXX_EXTRA_NVCC_FLAGS", "").split()


def _nvcc() -> str:
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        raise RuntimeError("nvcc not found: the CUDA extension cannot be built")
    return nvcc


def _newest_dep() -> float:
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return max(os.path.getmtime(d) for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every CUDA source for sm_100a and link the C-ABI shared library.  Returns its path."""
    mode_file = os.path.join(OBJ, "mode.txt")
    same_mode = os.path.exists(mode_file) and open(mode_file).read().strip() == MODE
    if not force and same_mode and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_dep():
        return LIB
    nvcc = _nvcc()
    os.makedirs(OBJ, exist_ok=True)

    hdr_time = max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS + [os.path.basename(__file__)] if os.path.exists(os.path.join(CSRC, h)))
    hdr_time = max(hdr_time, os.path.getmtime(os.path.abspath(__file__)))

    def compile_one(unit) -> str:
        src, defines, objname = unit
        obj = os.path.join(OBJ, objname)
        # incremental: an object newer than its source, every header and this script is kept (same build mode only)
        if not force and same_mode and os.path.exists(obj) and os.path.getmtime(obj) >= max(hdr_time, os.path.getmtime(os.path.join(CSRC, src))):
            return obj
        cmd = [nvcc] + ARCH + FLAGS + DEV_FLAGS + defines + (["-Xptxas", "-v"] if verbose else []) + ["-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose:
            with open(obj + ".log", "w") as fh:
                fh.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src} {' '.join(defines)}:\n{r.stdout}\n{r.stderr[-6000:]}")
        return obj

    with ThreadPoolExecutor(max_workers=max(1, min(len(UNITS), os.cpu_count() or 4))) as ex:
        objs = list(ex.map(compile_one, UNITS))
    r = subprocess.run([nvcc] + ARCH + ["-shared", "-o", LIB] + objs + ["-ldl"], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    with open(mode_file, "w") as fh:
        fh.write(MODE + "\n")
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
