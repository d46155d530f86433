"""In-tree build of libspgpe.so with nvcc for sm_100a (no JIT cache: the built library travels with the tree)."""
from __future__ import annotations

import os
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor

_PKG = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_PKG, "csrc")
_OBJ = os.path.join(_CSRC, "build")
LIB_PATH = os.path.join(_PKG, "libspgpe.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-O3", "-lineinfo",
    "-Xcompiler", "-fPIC",
]
# extra compiler flags for diagnostic builds, e.g. SPGPE_NVCC_EXTRA="-DSPGPE_TIMELINE" (common.cuh)
NVCC_FLAGS += os.environ.get("SPGPE_NVCC_EXTRA", "").split()


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libspgpe cannot be built (there is no CPU fallback)")


def sources():
    return sorted(f for f in os.listdir(_CSRC) if f.endswith(".cu"))


def _newest_input() -> float:
    paths = [os.path.join(_CSRC, f) for f in os.listdir(_CSRC) if f.endswith((".cu", ".cuh", ".h"))]
    paths.append(os.path.join(os.path.dirname(_PKG), "include", "spgpe.h"))
    paths.append(os.path.abspath(__file__))
    return max(os.path.getmtime(p) for p in paths)


def is_stale() -> bool:
    return not os.path.exists(LIB_PATH) or os.path.getmtime(LIB_PATH) < _newest_input()


def build(force: bool = False, verbose: bool = False, jobs: int | None = None) -> str:
    """Compile every .cu under csrc/ and link libspgpe.so next to this file.  Returns its path."""
    if not force and not is_stale():
        return LIB_PATH
    nvcc = _nvcc()
    os.makedirs(_OBJ, exist_ok=True)
    newest_hdr = max(os.path.getmtime(os.path.join(_CSRC, f)) for f in os.listdir(_CSRC)
                     if f.endswith((".cuh", ".h")))
    newest_hdr = max(newest_hdr, os.path.getmtime(os.path.join(os.path.dirname(_PKG), "include", "spgpe.h")),
                     os.path.getmtime(os.path.abspath(__file__)))

    def compile_one(src: str) -> str:
        obj = os.path.join(_OBJ, src[:-3] + ".o")
        s = os.path.join(_CSRC, src)
        if not force and os.path.exists(obj) and os.path.getmtime(obj) >= max(os.path.getmtime(s), newest_hdr):
            return obj
        cmd = [nvcc, *NVCC_FLAGS, "-c", s, "-o", obj]
        if verbose:
            cmd.insert(-4, "-Xptxas")
            cmd.insert(-4, "-v")
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            print(r.stderr)
        return obj

    with ThreadPoolExecutor(max_workers=jobs or min(8, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(compile_one, sources()))
    tmp = LIB_PATH + f".tmp{os.getpid()}"
    r = subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *objs],
                       capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    import sys

    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
