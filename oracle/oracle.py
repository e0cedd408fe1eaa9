"""ctypes front end of the CPU oracle (``xt_oracle.cpp``).  TEST INFRASTRUCTURE.

``build()`` compiles two shared objects from the one source:
  * ``liboracle_xt.so``      g++ -O2 -ffp-contract=off          -- THE oracle
  * ``liboracle_xt_fma.so``  g++ -O2 -ffp-contract=fast -mfma   -- the same expressions
    with FMA contraction, used only to *select* numerically stable particles for the
    100-turn comparison (reading A9); never as a source of expected values.

The oracle itself is single-threaded C++.  ``track(..., threads=N)`` merely runs N
independent oracle calls on disjoint particle slices (particles are independent,
PAPER.md:184), to shorten test wall-clock.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "xt_oracle.cpp")
_LIBS = {
    "strict": (os.path.join(_HERE, "liboracle_xt.so"), ["-O2", "-ffp-contract=off"]),
    "fma": (os.path.join(_HERE, "liboracle_xt_fma.so"), ["-O2", "-ffp-contract=fast", "-mfma"]),
}

F64 = ("x", "px", "y", "py", "zeta", "delta", "ptau", "rpp", "rvv", "s")
I64 = ("at_turn", "state", "at_element")


class _XoParticles(ctypes.Structure):
    _fields_ = ([(k, ctypes.POINTER(ctypes.c_double)) for k in F64]
                + [(k, ctypes.POINTER(ctypes.c_int64)) for k in I64]
                + [("min_margin", ctypes.POINTER(ctypes.c_double))])


def build(force: bool = False) -> None:
    for _, (path, flags) in _LIBS.items():
        if (not force and os.path.exists(path)
                and os.path.getmtime(path) >= os.path.getmtime(_SRC)):
            continue
        cmd = ["g++", "-std=c++17", "-shared", "-fPIC", "-fno-fast-math", *flags, _SRC, "-o", path]
        subprocess.run(cmd, check=True)


_loaded: Dict[str, ctypes.CDLL] = {}


def _lib(kind: str = "strict") -> ctypes.CDLL:
    if kind not in _loaded:
        build()
        lib = ctypes.CDLL(_LIBS[kind][0])
        lib.xo_track.restype = ctypes.c_int
        lib.xo_track.argtypes = [ctypes.c_char_p, ctypes.c_size_t, ctypes.POINTER(_XoParticles),
                                 ctypes.c_int64, ctypes.c_int64]
        lib.xo_init_derived.restype = ctypes.c_int
        lib.xo_init_derived.argtypes = [ctypes.c_char_p, ctypes.c_size_t] + \
            [ctypes.POINTER(ctypes.c_double)] * 4 + [ctypes.c_int64]
        lib.xo_reference.restype = ctypes.c_int
        lib.xo_reference.argtypes = [ctypes.c_char_p, ctypes.c_size_t,
                                     ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        lib.xo_s_table.restype = ctypes.c_int64
        lib.xo_s_table.argtypes = [ctypes.c_char_p, ctypes.c_size_t,
                                   ctypes.POINTER(ctypes.c_double), ctypes.c_int64]
        _loaded[kind] = lib
    return _loaded[kind]


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))


def reference(packed: bytes):
    """(beta0, gamma0) as derived by the oracle from the buffer's p0c, mass0."""
    b, g = ctypes.c_double(), ctypes.c_double()
    rc = _lib().xo_reference(packed, len(packed), ctypes.byref(b), ctypes.byref(g))
    if rc:
        raise ValueError("oracle: bad lattice buffer (rc=%d)" % rc)
    return b.value, g.value


def s_table(packed: bytes) -> np.ndarray:
    n = _lib().xo_s_table(packed, len(packed), None, 0)
    if n < 0:
        raise ValueError("oracle: bad lattice buffer (rc=%d)" % n)
    out = np.zeros(n, dtype=np.float64)
    _lib().xo_s_table(packed, len(packed), _dp(out), n)
    return out


def new_particles(packed: bytes, coords: Dict[str, np.ndarray], kind: str = "strict") -> Dict[str, np.ndarray]:
    """Full particle SoA (host, numpy) from the six primary coordinates: derives
    ptau, rpp, rvv with the oracle's init helper; s=0, at_turn=0, state=1, at_element=0."""
    n = len(coords["x"])
    p = {k: np.ascontiguousarray(coords[k], dtype=np.float64).copy()
         for k in ("x", "px", "y", "py", "zeta", "delta")}
    for k in ("ptau", "rpp", "rvv", "s"):
        p[k] = np.zeros(n, dtype=np.float64)
    p["at_turn"] = np.zeros(n, dtype=np.int64)
    p["state"] = np.ones(n, dtype=np.int64)
    p["at_element"] = np.zeros(n, dtype=np.int64)
    rc = _lib(kind).xo_init_derived(packed, len(packed), _dp(p["delta"]), _dp(p["ptau"]),
                                    _dp(p["rpp"]), _dp(p["rvv"]), n)
    if rc:
        raise ValueError("oracle: bad lattice buffer (rc=%d)" % rc)
    return p


def _track_slice(lib, packed, p, lo, hi, n_turns, margin):
    st = _XoParticles()
    for k in F64:
        setattr(st, k, _dp(p[k][lo:hi]))
    for k in I64:
        setattr(st, k, _ip(p[k][lo:hi]))
    st.min_margin = _dp(margin[lo:hi]) if margin is not None else None
    return lib.xo_track(packed, len(packed), ctypes.byref(st), hi - lo, n_turns)


def track(packed: bytes, p: Dict[str, np.ndarray], n_turns: int, *, kind: str = "strict",
          threads: int = 1, min_margin: Optional[np.ndarray] = None) -> None:
    """Track the SoA ``p`` in place for ``n_turns`` turns.  ``min_margin`` (optional,
    float64[n], pre-filled by the caller e.g. with +inf) receives per particle the minimum
    over this call's aperture checks of the distance to the aperture edge; it is
    min-combined with what the array already holds."""
    lib = _lib(kind)
    n = len(p["x"])
    for k in F64:
        assert p[k].dtype == np.float64 and p[k].flags.c_contiguous and len(p[k]) == n, k
    for k in I64:
        assert p[k].dtype == np.int64 and p[k].flags.c_contiguous and len(p[k]) == n, k
    margin = None
    if min_margin is not None:
        margin = np.full(n, np.inf)
    threads = max(1, min(threads, n))
    if threads == 1:
        rcs = [_track_slice(lib, packed, p, 0, n, n_turns, margin)]
    else:
        bounds = np.linspace(0, n, threads + 1).astype(np.int64)
        with ThreadPoolExecutor(threads) as ex:
            rcs = list(ex.map(lambda i: _track_slice(lib, packed, p, int(bounds[i]), int(bounds[i + 1]),
                                                     n_turns, margin), range(threads)))
    if any(rcs):
        raise ValueError("oracle: xo_track failed (rc=%s)" % rcs)
    if min_margin is not None:
        np.minimum(min_margin, margin, out=min_margin)


def copy_particles(p: Dict[str, np.ndarray]) -> Dict[str, np.ndarray]:
    return {k: v.copy() for k, v in p.items()}


def host_threads() -> int:
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
