"""Build libtropical.so (sm_100a only) in-tree with nvcc.  `python -m paper_2606_16264_b200.build`."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtropical.so")
STAMP = LIB + ".flags"  # the extra nvcc flags the library on disk was built with (git-ignored, travels with the .so)
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "--use_fast_math",  # only affects the CUDA path; expf/exp2f intrinsics in softmax
    "-Xptxas", "-v",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cpp")))


def _extra_flags() -> list:
    # e.g. -DTROPICAL_DEBUG_WAIT (names a timed-out mbarrier wait), -DTROPICAL_WHATIF_* / -DTROPICAL_TIMELINE (measurement builds)
    return os.environ.get("TROPICAL_NVCC_EXTRA", "").split()


def _built_flags():
    try:
        with open(STAMP) as f:
            return f.read().split()
    except OSError:
        return None  # a library without a stamp: built by something else, taken as a plain build


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    # A measurement build (attention results wrong by design under -DTROPICAL_WHATIF_*) overwrites the same file:
    # a change of the flag set forces a rebuild, so a later plain run never loads it by accident.
    if (_built_flags() or []) != _extra_flags():
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.inc")) + \
        glob.glob(os.path.join(INCLUDE, "*.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB + f".tmp{os.getpid()}"
    extra = _extra_flags()
    cmd = [nvcc] + NVCC_FLAGS + extra + ["-I", INCLUDE, "-o", tmp] + sources()
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(HERE, "build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if res.returncode != 0:
        sys.stderr.write(log)
        raise RuntimeError("nvcc failed building libtropical.so")
    if verbose:
        print(log)
    os.replace(tmp, LIB)
    with open(STAMP, "w") as f:
        f.write(" ".join(extra) + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
