"""Build libspense.so (hand-written sm_100a CUDA + C ABI) in-tree with nvcc."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libspense.so")
SOURCES = ["spense_api.cu", "spense_gemm.cu", "spense_pack.cu", "spense_select.cu", "spense_prune.cu", "spense_probe.cu"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "spense.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, debug_hooks: bool = False, out: str | None = None) -> str:
    """debug_hooks: also compile the per-CTA timeline hook (spense_debug_set_trace, not declared in spense.h) into a
    library written to `out`; the default build exports exactly what include/spense.h declares."""
    if debug_hooks and (out is None or os.path.abspath(out) == LIB):
        raise ValueError("a debug_hooks build must be written to an explicit `out` other than libspense.so: it reads "
                         "SPENSE_* environment knobs and exports a symbol spense.h does not declare")
    lib = os.path.abspath(out) if out else LIB
    if lib == LIB and not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           "-o", lib] + [os.path.join(CSRC, s) for s in SOURCES] + ["-lcudart"]
    if debug_hooks:
        cmd.insert(1, "-DSPENSE_DEBUG_HOOKS")
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed building libspense.so")
    if verbose:
        print(r.stdout + r.stderr)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
