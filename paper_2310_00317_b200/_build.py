"""In-tree build of the C-ABI library with nvcc for sm_100a (cross-compiles without a GPU).

Two shared objects come from the same sources:
  * ``libxt_b200.so``        production: default ``--fmad=true`` (a*b+c contracts to DFMA)
  * ``libxt_b200_nofma.so``  validation: ``--fmad=false``; bit-identical to the oracle on
    cavity-free lattices (BASELINE.json north_star; reading A10)
"""
from __future__ import annotations

import os
import shutil
import subprocess
from typing import Dict, List

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["xt_api.cu", "xt_lattice.cu", "xt_track.cu", "xt_compact.cu", "xt_peak.cu", "xt_twiss.cu", "xt_refine.cu", "xt_knobs.cu"]
HEADERS = [os.path.join(CSRC, "xt_internal.h"), os.path.join(CSRC, "xt_line.h"),
           os.path.join(os.path.dirname(HERE), "include", "xt.h")]

LIBS: Dict[str, Dict] = {
    "prod": {"path": os.path.join(HERE, "libxt_b200.so"), "flags": []},
    "nofma": {"path": os.path.join(HERE, "libxt_b200_nofma.so"),
              "flags": ["--fmad=false", "-DXT_FMAD_OFF"]},
    # optional, built on first use: production FMA fusion with IEEE sqrt and division in the drift
    # (separates the two differences between the production and the validation arithmetic)
    "ieee_drift": {"path": os.path.join(HERE, "libxt_b200_ieee_drift.so"), "flags": ["-DXT_CANONICAL_DRIFT"]},
}

COMMON = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC,-ffp-contract=off",
    "-shared",
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA toolkit is required (there is no CPU fallback)")
    return exe


def _stale(path: str) -> bool:
    if not os.path.exists(path):
        return True
    t = os.path.getmtime(path)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def command(kind: str, extra: List[str] = ()) -> List[str]:
    lib = LIBS[kind]
    return [nvcc(), *COMMON, *lib["flags"], *extra,
            *[os.path.join(CSRC, s) for s in SOURCES], "-o", lib["path"]]


def build(kinds=("prod", "nofma"), force: bool = False, verbose: bool = False) -> None:
    for kind in kinds:
        if not force and not _stale(LIBS[kind]["path"]):
            continue
        cmd = command(kind, ["-Xptxas", "-v"] if verbose else [])
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose:
            print(res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), res.stderr))


if __name__ == "__main__":
    import sys
    build(force=True, verbose="-v" in sys.argv)
