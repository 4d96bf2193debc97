"""Compile the CUDA path into paper_2104_01636_b200/libps_poisson.so (in-tree, sm_100a only).

    python -m paper_2104_01636_b200.build [--force]

nvcc cross-compiles without a GPU.  Flags that matter for parity:
`--fmad=false` (no FMA contraction: every product and sum of the SOR update rounds separately,
as in the oracle's `-ffp-contract=off`), never `-use_fast_math`; fp64 division and sqrt are
IEEE-correct regardless.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_INC = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libps_poisson.so")
LIB_CHECKED = os.path.join(_HERE, "libps_poisson_checked.so")   # -DPS_CHECKED, tests only
SOURCES = ["ps_api.cu"]
HEADERS = sorted(f for f in os.listdir(_CSRC) if f.endswith(".cuh"))

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-std=c++17", "-O3", "--fmad=false", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    # the shared CUDA runtime (libcudart.so.12), so the shipped library carries none of the
    # runtime's own code.  binding.load() imports torch first, so in a Python process the library
    # binds the libcudart torch has already loaded (one runtime per process); a C program finds the
    # toolkit's copy through the rpath _rpath_flags() adds.  Needs a CUDA 12 runtime (12.0 or later:
    # cudaLaunchKernelEx with the cluster-dimension and programmatic-stream-serialization launch
    # attributes, cudaGetDriverEntryPoint with its query-result argument); built and tested with
    # the 12.9 toolkit against torch's 12.8 runtime.
    "-cudart", "shared",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")


def _rpath_flags(nvcc: str) -> list[str]:
    """-rpath of the lib64 directory of the toolkit the resolved nvcc belongs to (not a fixed
    /usr/local/cuda), for processes that have no libcudart loaded yet."""
    home = os.environ.get("CUDA_HOME") or os.path.dirname(os.path.dirname(os.path.realpath(nvcc)))
    for sub in ("lib64", os.path.join("targets", "x86_64-linux", "lib")):
        d = os.path.join(home, sub)
        if os.path.isdir(d):
            return ["-Xlinker", f"-rpath={d}"]
    return []


def _deps():
    yield os.path.join(_INC, "ps_poisson.h")
    for f in SOURCES + HEADERS:
        yield os.path.join(_CSRC, f)


def up_to_date(lib: str = LIB) -> bool:
    return os.path.exists(lib) and os.path.getmtime(lib) >= max(os.path.getmtime(d) for d in _deps())


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """Build libps_poisson.so (checked: the self-checking libps_poisson_checked.so, compiled with
    -DPS_CHECKED) if missing or older than its sources; returns its path."""
    lib = LIB_CHECKED if checked else LIB
    if not force and up_to_date(lib):
        return lib
    tmp = f"{lib}.{os.getpid()}.tmp"
    nvcc = _nvcc()
    cmd = [nvcc, *NVCC_FLAGS, *_rpath_flags(nvcc), *(["-DPS_CHECKED"] if checked else []),
           *(["-Xptxas", "-v"] if verbose else []),
           "-o", tmp, *[os.path.join(_CSRC, s) for s in SOURCES]]
    res = subprocess.run(cmd, cwd=_CSRC, capture_output=True, text=True)
    if res.returncode != 0:
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + res.stdout + res.stderr)
    if verbose:
        sys.stderr.write(res.stdout + res.stderr)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--checked" in sys.argv:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked=True))
