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
SOURCES = ["xt_api.cu", "xt_lattice.cu", "xt_track.cu", "xt_compact.cu", "xt_peak.cu", "xt_twiss.cu", "xt_twiss6d.cu", "xt_refine.cu", "xt_knobs.cu"]
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


def _objdir(kind: str) -> str:
    d = os.path.join(HERE, "build", kind)
    os.makedirs(d, exist_ok=True)
    return d


def _stale(target: str, deps: List[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def compile_command(kind: str, src: str, obj: str, extra: List[str] = ()) -> List[str]:
    flags = [f for f in COMMON if f != "-shared"]
    return [nvcc(), *flags, *LIBS[kind]["flags"], *extra, "-c", os.path.join(CSRC, src), "-o", obj]


def command(kind: str, extra: List[str] = ()) -> List[str]:
    """The one-line equivalent of the build (every source in one nvcc call), for the record."""
    lib = LIBS[kind]
    return [nvcc(), *COMMON, *lib["flags"], *extra,
            *[os.path.join(CSRC, s) for s in SOURCES], "-o", lib["path"]]


def build(kinds=("prod", "nofma"), force: bool = False, verbose: bool = False, extra: List[str] = ()) -> None:
    """Each translation unit is compiled to an object file (in parallel, only when stale) and the objects
    are linked into the shared library: no device code crosses translation units, so no device link."""
    from concurrent.futures import ThreadPoolExecutor
    jobs = []
    for kind in kinds:
        od = _objdir(kind)
        for src in SOURCES:
            obj = os.path.join(od, src.replace(".cu", ".o"))
            deps = [os.path.join(CSRC, src)] + HEADERS + [os.path.abspath(__file__)]
            if force or _stale(obj, deps):
                jobs.append((kind, src, obj))

    def run(job):
        kind, src, obj = job
        cmd = compile_command(kind, src, obj, list(extra) + (["-Xptxas", "-v"] if verbose else []))
        res = subprocess.run(cmd, capture_output=True, text=True)
        return job, cmd, res

    with ThreadPoolExecutor(max_workers=max(1, min(len(jobs), os.cpu_count() or 4))) as ex:
        for job, cmd, res in ex.map(run, jobs):
            if verbose:
                print(res.stderr)
            if res.returncode != 0:
                raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), res.stderr))
    for kind in kinds:
        od = _objdir(kind)
        objs = [os.path.join(od, s.replace(".cu", ".o")) for s in SOURCES]
        if force or _stale(LIBS[kind]["path"], objs):
            cmd = [nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", *objs, "-o", LIBS[kind]["path"]]
            res = subprocess.run(cmd, capture_output=True, text=True)
            if res.returncode != 0:
                raise RuntimeError("link failed:\n%s\n%s" % (" ".join(cmd), res.stderr))


if __name__ == "__main__":
    import sys
    build(force=True, verbose="-v" in sys.argv)
