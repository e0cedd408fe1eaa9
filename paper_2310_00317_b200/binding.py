"""Thin ctypes binding of ``include/xt.h`` -- argument marshalling only.

Every step of the tracking path runs inside ``libxt_b200.so`` (hand-written CUDA for
sm_100a).  PyTorch is used for device memory and streams, nothing else.  There is no CPU
fallback: if the library is missing it is built with nvcc, and if that fails, or no CUDA
device is present when a compute entry point is called, an exception is raised.

The functions carry the names of the C entry points they wrap.
"""
from __future__ import annotations

import ctypes
import os
from typing import Dict, Optional

import numpy as np

from . import _build

F64_FIELDS = ("x", "px", "y", "py", "zeta", "delta", "ptau", "rpp", "rvv", "s")
I64_FIELDS = ("at_turn", "state", "particle_id", "at_element")
ALL_FIELDS = F64_FIELDS + I64_FIELDS

XT_OK, XT_ERR_INVALID_ARG, XT_ERR_BAD_LATTICE, XT_ERR_CUDA, XT_ERR_NOMEM = 0, -1, -2, -3, -4


class XtError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("xt error %d: %s" % (code, msg))
        self.code = code


class xt_particles(ctypes.Structure):
    _fields_ = ([(k, ctypes.c_void_p) for k in F64_FIELDS] + [(k, ctypes.c_void_p) for k in I64_FIELDS])


XT_STATS_MAX_PASSES = 128


class xt_track_stats(ctypes.Structure):
    _fields_ = [("n_track_launches", ctypes.c_int64), ("n_passes", ctypes.c_int64),
                ("track_ms", ctypes.c_double), ("compact_ms", ctypes.c_double), ("compact_bytes", ctypes.c_double),
                ("scatter_ms", ctypes.c_double), ("scatter_bytes", ctypes.c_double),
                ("pass_n_in", ctypes.c_int64 * XT_STATS_MAX_PASSES),
                ("pass_n_out", ctypes.c_int64 * XT_STATS_MAX_PASSES),
                ("pass_ms", ctypes.c_double * XT_STATS_MAX_PASSES)]


class xt_track_opts(ctypes.Structure):
    _fields_ = [("turns_per_launch", ctypes.c_int64), ("compact_every", ctypes.c_int64),
                ("block_size", ctypes.c_int32), ("particles_per_thread", ctypes.c_int32),
                ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_uint64),
                ("stats", ctypes.POINTER(xt_track_stats)),
                ("cold_in_registers", ctypes.c_int32), ("balance", ctypes.c_int32)]


class xt_lattice_opts(ctypes.Structure):
    _fields_ = [("chunk_bytes", ctypes.c_int64), ("fuse", ctypes.c_int32), ("reserved", ctypes.c_int32)]


class xt_knob_link(ctypes.Structure):
    _fields_ = [("element", ctypes.c_int64), ("order", ctypes.c_int32), ("skew", ctypes.c_int32),
                ("knob", ctypes.c_int32), ("reserved", ctypes.c_int32), ("gain", ctypes.c_double)]


class xt_twiss4d_result(ctypes.Structure):
    _fields_ = ([("co", ctypes.c_double * 4), ("m", ctypes.c_double * 16)] +
                [(k, ctypes.c_double) for k in ("betx", "alfx", "mux", "qx_frac", "bety", "alfy", "muy", "qy_frac")] +
                [("iterations", ctypes.c_int32), ("stable", ctypes.c_int32)])


class xt_twiss4d_chrom_result(ctypes.Structure):
    _fields_ = ([("on", xt_twiss4d_result)] +
                [(k, ctypes.c_double) for k in ("dx", "dpx", "dy", "dpy", "dqx", "dqy")])


class xt_twiss6d_result(ctypes.Structure):
    _fields_ = [("co", ctypes.c_double * 6), ("m", ctypes.c_double * 36), ("q1_frac", ctypes.c_double),
                ("q2_frac", ctypes.c_double), ("qs", ctypes.c_double), ("iterations", ctypes.c_int32),
                ("reserved", ctypes.c_int32)]


class xt_twiss6d_modes(ctypes.Structure):
    _fields_ = [("q_frac", ctypes.c_double * 3), ("bet", (ctypes.c_double * 3) * 3), ("alf", (ctypes.c_double * 3) * 3),
                ("disp", ctypes.c_double * 4), ("v", (ctypes.c_double * 12) * 3),
                ("stable", ctypes.c_int32), ("degenerate", ctypes.c_int32)]


class xt_twiss6d_row(ctypes.Structure):
    _fields_ = [("s", ctypes.c_double), ("co", ctypes.c_double * 6), ("bet", (ctypes.c_double * 3) * 3),
                ("alf", (ctypes.c_double * 3) * 3), ("mu", ctypes.c_double * 3), ("disp", ctypes.c_double * 4)]


class xt_twiss_row(ctypes.Structure):
    _fields_ = [(k, ctypes.c_double) for k in ("s", "x", "px", "y", "py", "betx", "alfx", "mux", "bety", "alfy",
                                                "muy", "dx", "dpx", "dy", "dpy", "betx1", "bety1", "betx2", "bety2",
                                                "mu1", "mu2")]


class xt_twiss4d_modes(ctypes.Structure):
    _fields_ = ([(k, ctypes.c_double) for k in ("q1_frac", "q2_frac", "betx1", "alfx1", "bety1", "alfy1", "betx2",
                                                 "alfx2", "bety2", "alfy2")] +
                [("v1", ctypes.c_double * 8), ("v2", ctypes.c_double * 8), ("stable", ctypes.c_int32),
                 ("degenerate", ctypes.c_int32)])


class xt_lattice_info(ctypes.Structure):
    _fields_ = [("n_elements", ctypes.c_int64), ("n_records", ctypes.c_int64),
                ("n_chunks", ctypes.c_int64), ("image_bytes", ctypes.c_int64),
                ("chunk_bytes", ctypes.c_int64), ("n_by_type", ctypes.c_int64 * 8),
                ("sum_order", ctypes.c_int64), ("n_curved", ctypes.c_int64),
                ("has_aperture", ctypes.c_int64), ("beta0", ctypes.c_double),
                ("gamma0", ctypes.c_double), ("circumference", ctypes.c_double),
                ("n_drift_evals", ctypes.c_int64), ("n_thick", ctypes.c_int64),
                ("n_drift_applies", ctypes.c_int64)]

    def as_dict(self) -> Dict:
        d = {k: getattr(self, k) for k, _ in self._fields_ if k != "n_by_type"}
        d["n_by_type"] = list(self.n_by_type)
        return d


# name -> (restype, argtypes): every symbol include/xt.h declares
_VP, _I64, _SZ = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t
SIGNATURES = {
    "xt_lattice_create": (ctypes.c_int, [ctypes.c_char_p, _SZ, ctypes.POINTER(_VP)]),
    "xt_lattice_create_ex": (ctypes.c_int, [ctypes.c_char_p, _SZ, ctypes.POINTER(xt_lattice_opts),
                                            ctypes.POINTER(_VP)]),
    "xt_lattice_destroy": (ctypes.c_int, [_VP]),
    "xt_lattice_get_info": (ctypes.c_int, [_VP, ctypes.POINTER(xt_lattice_info)]),
    "xt_lattice_s_table": (_I64, [_VP, _VP, _I64]),
    "xt_lattice_pack_host": (_I64, [ctypes.c_char_p, _SZ, ctypes.POINTER(xt_lattice_opts), _VP, _SZ,
                                    ctypes.POINTER(xt_lattice_info)]),
    "xt_track": (ctypes.c_int, [_VP, ctypes.POINTER(xt_particles), _I64, _I64, _VP]),
    "xt_track_ex": (ctypes.c_int, [_VP, ctypes.POINTER(xt_particles), _I64, _I64, _VP,
                                   ctypes.POINTER(xt_track_opts)]),
    "xt_track_static": (ctypes.c_int, [_VP, ctypes.POINTER(xt_particles), _I64, _I64, _VP,
                                       ctypes.POINTER(xt_track_opts)]),
    "xt_track_host": (ctypes.c_int, [_VP, ctypes.POINTER(xt_particles), _I64, _I64, _VP,
                                     ctypes.POINTER(xt_track_opts)]),
    "xt_particles_init_derived": (ctypes.c_int, [_VP, ctypes.POINTER(xt_particles), _I64, _VP]),
    "xt_survival_histogram": (ctypes.c_int, [_VP, _VP, _I64, _I64, _I64, _VP, _VP]),
    "xt_fp64_fma_peak": (ctypes.c_int, [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), _VP]),
    "xt_track_workspace_bytes": (ctypes.c_uint64, [_I64]),
    "xt_fp64_fma_peak_sweep_size": (ctypes.c_int, []),
    "xt_fp64_fma_peak_sweep": (ctypes.c_int, [ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                              ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int), _VP]),
    "xt_fp64_fma_probe": (ctypes.c_int, [ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                         ctypes.POINTER(ctypes.c_double), _VP]),
    "xt_twiss4d": (ctypes.c_int, [_VP, ctypes.c_double, ctypes.POINTER(ctypes.c_double),
                                  ctypes.POINTER(xt_twiss4d_result), _VP]),
    "xt_refine_loss_location": (ctypes.c_int, [_VP, ctypes.POINTER(xt_particles), _I64, ctypes.c_double,
                                               ctypes.c_int32, ctypes.POINTER(ctypes.c_int64), _VP]),
    "xt_twiss4d_chrom": (ctypes.c_int, [_VP, ctypes.c_double, ctypes.c_double, ctypes.POINTER(ctypes.c_double),
                                        ctypes.POINTER(xt_twiss4d_chrom_result), _VP]),
    "xt_twiss6d": (ctypes.c_int, [_VP, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(xt_twiss6d_result), _VP]),
    "xt_twiss6d_normal_form": (ctypes.c_int, [ctypes.POINTER(ctypes.c_double), ctypes.c_double,
                                              ctypes.POINTER(xt_twiss6d_modes)]),
    "xt_twiss6d_line": (ctypes.c_int, [_VP, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(xt_twiss6d_result),
                                       ctypes.POINTER(xt_twiss6d_modes), ctypes.POINTER(xt_twiss6d_row), _I64, _VP]),
    "xt_twiss4d_normal_form": (ctypes.c_int, [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(xt_twiss4d_modes)]),
    "xt_twiss4d_line": (ctypes.c_int, [_VP, ctypes.c_double, ctypes.c_double, ctypes.POINTER(ctypes.c_double),
                                       ctypes.POINTER(xt_twiss4d_chrom_result), ctypes.POINTER(xt_twiss_row), _I64,
                                       _VP]),
    "xt_lattice_set_knobs": (ctypes.c_int, [_VP, ctypes.POINTER(ctypes.c_double), ctypes.c_int32, _I64,
                                            ctypes.POINTER(xt_knob_link), _I64]),
    "xt_track_knobs": (ctypes.c_int, [_VP, ctypes.POINTER(xt_particles), _I64, _I64, _I64, _VP]),
    "xt_launch_count": (_I64, []),
    "xt_last_error": (ctypes.c_char_p, []),
    "xt_build_info": (ctypes.c_char_p, []),
}

_libs: Dict[str, ctypes.CDLL] = {}


def load_library(kind: str = "prod") -> ctypes.CDLL:
    """Load (building first if stale/missing) ``libxt_b200.so`` (kind='prod') or the
    ``--fmad=false`` validation build (kind='nofma').  Fails loudly; no fallback."""
    if kind not in _libs:
        _build.build(kinds=(kind,))
        path = _build.LIBS[kind]["path"]
        if not os.path.exists(path):
            raise RuntimeError("CUDA extension %s is missing and could not be built" % path)
        lib = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)        # AttributeError if the symbol is not exported
            fn.restype, fn.argtypes = res, args
        _libs[kind] = lib
    return _libs[kind]


def _check(lib, rc: int) -> None:
    if rc != XT_OK:
        raise XtError(rc, lib.xt_last_error().decode("utf-8", "replace"))


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(int(stream.cuda_stream))


# ------------------------------------------------------------------------------ lattice
class Lattice:
    """Owner of an ``xt_lattice*`` (device image of a beam line)."""

    def __init__(self, handle: int, lib: ctypes.CDLL, kind: str):
        self._h, self._lib, self.kind = handle, lib, kind
        info = xt_lattice_info()
        _check(lib, lib.xt_lattice_get_info(_VP(handle), ctypes.byref(info)))
        self.info = info.as_dict()

    @property
    def handle(self) -> ctypes.c_void_p:
        if not self._h:
            raise ValueError("lattice already destroyed")
        return _VP(self._h)

    def close(self) -> None:
        if self._h:
            self._lib.xt_lattice_destroy(_VP(self._h))
            self._h = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _lattice_opts(chunk_bytes: int = 0, fuse: Optional[bool] = None):
    if not chunk_bytes and fuse is None:
        return None
    return xt_lattice_opts(int(chunk_bytes), 0 if fuse is None else (1 if fuse else 2), 0)


def xt_lattice_create(packed: bytes, kind: str = "prod") -> Lattice:
    lib = load_library(kind)
    out = _VP()
    _check(lib, lib.xt_lattice_create(packed, len(packed), ctypes.byref(out)))
    return Lattice(out.value, lib, kind)


def xt_lattice_create_ex(packed: bytes, kind: str = "prod", *, chunk_bytes: int = 0,
                         fuse: Optional[bool] = None) -> Lattice:
    """As ``xt_lattice_create`` with a staging-buffer size and/or record fusion switched off
    (``fuse=False``); neither changes any result."""
    lib = load_library(kind)
    out = _VP()
    o = _lattice_opts(chunk_bytes, fuse)
    _check(lib, lib.xt_lattice_create_ex(packed, len(packed), ctypes.byref(o) if o else None, ctypes.byref(out)))
    return Lattice(out.value, lib, kind)


def xt_lattice_destroy(lat: Lattice) -> None:
    lat.close()


def xt_lattice_get_info(lat: Lattice) -> Dict:
    return dict(lat.info)


def xt_lattice_s_table(lat: Lattice) -> np.ndarray:
    n = lat._lib.xt_lattice_s_table(lat.handle, None, 0)
    if n < 0:
        _check(lat._lib, int(n))
    out = np.zeros(n, dtype=np.float64)
    lat._lib.xt_lattice_s_table(lat.handle, out.ctypes.data_as(_VP), n)
    return out


def xt_lattice_pack_host(packed: bytes, kind: str = "prod", *, chunk_bytes: int = 0,
                         fuse: Optional[bool] = None):
    """(image bytes, info dict) of the device image; makes no CUDA call."""
    lib = load_library(kind)
    info = xt_lattice_info()
    o = _lattice_opts(chunk_bytes, fuse)
    op = ctypes.byref(o) if o else None
    n = lib.xt_lattice_pack_host(packed, len(packed), op, None, 0, ctypes.byref(info))
    if n < 0:
        _check(lib, int(n))
    buf = ctypes.create_string_buffer(int(n))
    lib.xt_lattice_pack_host(packed, len(packed), op, buf, int(n), ctypes.byref(info))
    return buf.raw, info.as_dict()


# ---------------------------------------------------------------------------- particles
def _struct_from_tensors(p: Dict) -> xt_particles:
    st = xt_particles()
    n = None
    for k in ALL_FIELDS:
        t = p.get(k)
        if t is None:
            setattr(st, k, None)
            continue
        import torch
        want = torch.float64 if k in F64_FIELDS else torch.int64
        if not (t.is_cuda and t.dtype == want and t.is_contiguous() and t.dim() == 1):
            raise ValueError("particle array %r must be a contiguous 1-D CUDA %s tensor" % (k, want))
        if n is None:
            n = t.numel()
        elif t.numel() != n:
            raise ValueError("particle array %r has a different length" % k)
        setattr(st, k, t.data_ptr())
    return st


def _struct_from_numpy(p: Dict) -> xt_particles:
    st = xt_particles()
    for k in ALL_FIELDS:
        a = p.get(k)
        if a is None:
            setattr(st, k, None)
            continue
        if hasattr(a, "data_ptr"):          # pinned torch CPU tensor
            if a.is_cuda or not a.is_contiguous():
                raise ValueError("host array %r must be a contiguous CPU tensor" % k)
            setattr(st, k, a.data_ptr())
        else:
            want = np.float64 if k in F64_FIELDS else np.int64
            if not (a.dtype == want and a.flags.c_contiguous and a.ndim == 1):
                raise ValueError("host array %r must be a contiguous 1-D %s array" % (k, want))
            setattr(st, k, a.ctypes.data)
    return st


def new_particles(lat: Lattice, coords: Dict[str, np.ndarray], device="cuda", stream=None) -> Dict:
    """Device SoA (dict of torch tensors) from the six primary coordinates; the derived
    ptau, rpp, rvv come from the library's own kernel (``xt_particles_init_derived``)."""
    import torch
    n = len(coords["x"])
    p = {}
    for k in ("x", "px", "y", "py", "zeta", "delta"):
        p[k] = torch.from_numpy(np.ascontiguousarray(coords[k], dtype=np.float64)).to(device)
    for k in ("ptau", "rpp", "rvv", "s"):
        p[k] = torch.zeros(n, dtype=torch.float64, device=device)
    p["at_turn"] = torch.zeros(n, dtype=torch.int64, device=device)
    p["state"] = torch.ones(n, dtype=torch.int64, device=device)
    p["at_element"] = torch.zeros(n, dtype=torch.int64, device=device)
    xt_particles_init_derived(lat, p, stream=stream)
    return p


def particles_to_device(p_host: Dict[str, np.ndarray], device="cuda") -> Dict:
    import torch
    return {k: torch.from_numpy(np.ascontiguousarray(v)).to(device) for k, v in p_host.items()
            if k in ALL_FIELDS}


def particles_to_host(p: Dict) -> Dict[str, np.ndarray]:
    return {k: v.cpu().numpy() for k, v in p.items()}


def _n_part(p: Dict) -> int:
    return int(p["x"].shape[0])


def _opts(turns_per_launch=0, compact_every=0, block_size=0, particles_per_thread=0, workspace=None, stats=None,
          cold_in_registers=0, balance=0):
    if not (turns_per_launch or compact_every or block_size or particles_per_thread or cold_in_registers or balance) \
            and workspace is None and stats is None:
        return None
    o = xt_track_opts(int(turns_per_launch), int(compact_every), int(block_size), int(particles_per_thread))
    o.cold_in_registers = int(cold_in_registers)
    o.balance = int(balance)
    if workspace is not None:                      # a torch uint8 CUDA tensor, caller-owned
        o.workspace = workspace.data_ptr()
        o.workspace_bytes = workspace.numel() * workspace.element_size()
    if stats is not None:
        o.stats = ctypes.pointer(stats)
    return o


def xt_track_workspace_bytes(n_part: int, kind: str = "prod") -> int:
    return int(load_library(kind).xt_track_workspace_bytes(int(n_part)))


def _stats_dict(st: "xt_track_stats") -> Dict:
    n = min(int(st.n_passes), XT_STATS_MAX_PASSES)
    return {"n_track_launches": int(st.n_track_launches), "n_passes": int(st.n_passes),
            "track_ms": st.track_ms, "compact_ms": st.compact_ms, "compact_bytes": st.compact_bytes,
            "scatter_ms": st.scatter_ms, "scatter_bytes": st.scatter_bytes,
            "pass_n_in": [int(v) for v in st.pass_n_in[:n]], "pass_n_out": [int(v) for v in st.pass_n_out[:n]],
            "pass_ms": [float(v) for v in st.pass_ms[:n]]}


def xt_particles_init_derived(lat: Lattice, p: Dict, stream=None) -> None:
    st = _struct_from_tensors(p)
    _check(lat._lib, lat._lib.xt_particles_init_derived(lat.handle, ctypes.byref(st), _n_part(p),
                                                        _stream_ptr(stream)))


def xt_track(lat: Lattice, p: Dict, n_turns: int, stream=None) -> None:
    """Track the device SoA ``p`` in place for ``n_turns`` turns (asynchronous on ``stream``)."""
    st = _struct_from_tensors(p)
    _check(lat._lib, lat._lib.xt_track(lat.handle, ctypes.byref(st), _n_part(p), int(n_turns),
                                       _stream_ptr(stream)))


def xt_track_ex(lat: Lattice, p: Dict, n_turns: int, stream=None, *, turns_per_launch: int = 0,
                compact_every: int = 0, block_size: int = 0, particles_per_thread: int = 0,
                workspace=None, stats: bool = False, cold_in_registers: int = 0, balance: int = 0):
    """``workspace``: optional torch uint8 CUDA tensor of xt_track_workspace_bytes(n) bytes; ``stats=True``
    returns the call's xt_track_stats as a dict (and makes the call synchronous)."""
    st = _struct_from_tensors(p)
    rec = xt_track_stats() if stats else None
    o = _opts(turns_per_launch, compact_every, block_size, particles_per_thread, workspace, rec, cold_in_registers,
              balance)
    _check(lat._lib, lat._lib.xt_track_ex(lat.handle, ctypes.byref(st), _n_part(p), int(n_turns),
                                          _stream_ptr(stream), ctypes.byref(o) if o else None))
    return _stats_dict(rec) if stats else None


XT_TRACK_STATIC_MAX_PARTICLES = 32768


def xt_track_static(lat: Lattice, p: Dict, n_turns: int, stream=None, *, turns_per_launch: int = 0,
                    compact_every: int = 0, block_size: int = 0, particles_per_thread: int = 0,
                    cold_in_registers: int = 0, balance: int = 0) -> None:
    """xt_track_ex without any allocation: step C's scratch is the library's static device array
    (at most XT_TRACK_STATIC_MAX_PARTICLES particles; calls that overlap on the GPU race, include/xt.h)."""
    st = _struct_from_tensors(p)
    o = _opts(turns_per_launch, compact_every, block_size, particles_per_thread, None, None, cold_in_registers,
              balance)
    _check(lat._lib, lat._lib.xt_track_static(lat.handle, ctypes.byref(st), _n_part(p), int(n_turns),
                                              _stream_ptr(stream), ctypes.byref(o) if o else None))


def xt_track_host(lat: Lattice, p_host: Dict, n_turns: int, stream=None, *, turns_per_launch: int = 0,
                  compact_every: int = 0, block_size: int = 0, particles_per_thread: int = 0) -> None:
    """End to end with HOST arrays (numpy or pinned torch CPU tensors): H2D, track, D2H, sync."""
    st = _struct_from_numpy(p_host)
    o = _opts(turns_per_launch, compact_every, block_size, particles_per_thread)
    _check(lat._lib, lat._lib.xt_track_host(lat.handle, ctypes.byref(st), _n_part(p_host), int(n_turns),
                                            _stream_ptr(stream), ctypes.byref(o) if o else None))


def xt_survival_histogram(p: Dict, bin_width: int, n_bins: int, stream=None, kind: str = "prod"):
    """int64[n_bins+1] device tensor: lost-turn histogram, last entry = survivors."""
    import torch
    lib = load_library(kind)
    hist = torch.empty(n_bins + 1, dtype=torch.int64, device=p["state"].device)
    _check(lib, lib.xt_survival_histogram(p["at_turn"].data_ptr(), p["state"].data_ptr(), _n_part(p),
                                          int(bin_width), int(n_bins), hist.data_ptr(), _stream_ptr(stream)))
    return hist


def xt_fp64_fma_peak(stream=None, kind: str = "prod"):
    """(FLOP/s, kernel ms) of the library's FP64 FMA microbenchmark on the current device."""
    lib = load_library(kind)
    f, ms = ctypes.c_double(), ctypes.c_double()
    _check(lib, lib.xt_fp64_fma_peak(ctypes.byref(f), ctypes.byref(ms), _stream_ptr(stream)))
    return f.value, ms.value


def xt_fp64_fma_peak_sweep(stream=None, kind: str = "prod"):
    """Every row of the peak sweep: list of dicts {chains, form, block, ctas_per_sm, tflops, ms}."""
    lib = load_library(kind)
    rows = []
    for i in range(lib.xt_fp64_fma_peak_sweep_size()):
        f, ms, d = ctypes.c_double(), ctypes.c_double(), (ctypes.c_int * 4)()
        _check(lib, lib.xt_fp64_fma_peak_sweep(i, ctypes.byref(f), ctypes.byref(ms), d, _stream_ptr(stream)))
        rows.append({"chains": d[0], "form": d[1], "block": d[2], "ctas_per_sm": d[3],
                     "tflops": f.value / 1e12, "ms": ms.value})
    return rows


def xt_fp64_fma_probe(pattern: int, stream=None, kind: str = "prod"):
    """(FLOP/s, kernel ms) of the DFMA probe with operand pattern 0, 1, 2 or 3 (see include/xt.h)."""
    lib = load_library(kind)
    f, ms = ctypes.c_double(), ctypes.c_double()
    _check(lib, lib.xt_fp64_fma_probe(int(pattern), ctypes.byref(f), ctypes.byref(ms), _stream_ptr(stream)))
    return f.value, ms.value


def xt_twiss4d(lat: Lattice, delta0: float = 0.0, guess4=None, stream=None) -> Dict:
    """Closed orbit, one-turn matrix and uncoupled optics at the start of the line (see include/xt.h)."""
    res = xt_twiss4d_result()
    g = (ctypes.c_double * 4)(*[float(v) for v in guess4]) if guess4 is not None else None
    _check(lat._lib, lat._lib.xt_twiss4d(lat.handle, float(delta0), g, ctypes.byref(res), _stream_ptr(stream)))
    out = {k: getattr(res, k) for k in ("betx", "alfx", "mux", "qx_frac", "bety", "alfy", "muy", "qy_frac",
                                        "iterations", "stable")}
    out["co"] = np.array(list(res.co))
    out["m"] = np.array(list(res.m)).reshape(4, 4)
    return out


def xt_refine_loss_location(lat: Lattice, p: Dict, ds: float, n_poly: int = 64, stream=None) -> int:
    """Refine in place the loss records of the device SoA ``p`` (see include/xt.h); returns how many moved."""
    st = _struct_from_tensors(p)
    moved = ctypes.c_int64(0)
    _check(lat._lib, lat._lib.xt_refine_loss_location(lat.handle, ctypes.byref(st), _n_part(p), float(ds),
                                                      int(n_poly), ctypes.byref(moved), _stream_ptr(stream)))
    return int(moved.value)


def _twiss_dict(res) -> Dict:
    out = {k: getattr(res, k) for k in ("betx", "alfx", "mux", "qx_frac", "bety", "alfy", "muy", "qy_frac",
                                        "iterations", "stable")}
    out["co"] = np.array(list(res.co))
    out["m"] = np.array(list(res.m)).reshape(4, 4)
    return out


def xt_twiss4d_chrom(lat: Lattice, delta0: float = 0.0, ddelta: float = 1e-4, guess4=None, stream=None) -> Dict:
    """xt_twiss4d plus dispersion (dx, dpx, dy, dpy) and chromaticity (dqx, dqy); see include/xt.h."""
    res = xt_twiss4d_chrom_result()
    g = (ctypes.c_double * 4)(*[float(v) for v in guess4]) if guess4 is not None else None
    _check(lat._lib, lat._lib.xt_twiss4d_chrom(lat.handle, float(delta0), float(ddelta), g, ctypes.byref(res),
                                               _stream_ptr(stream)))
    out = _twiss_dict(res.on)
    for k in ("dx", "dpx", "dy", "dpy", "dqx", "dqy"):
        out[k] = getattr(res, k)
    return out


def xt_twiss6d(lat: Lattice, guess6=None, stream=None) -> Dict:
    """Six-dimensional closed orbit, 6x6 one-turn matrix and the three tunes (include/xt.h)."""
    res = xt_twiss6d_result()
    g = (ctypes.c_double * 6)(*[float(v) for v in guess6]) if guess6 is not None else None
    _check(lat._lib, lat._lib.xt_twiss6d(lat.handle, g, ctypes.byref(res), _stream_ptr(stream)))
    return dict(co=np.array(list(res.co)), m=np.array(list(res.m)).reshape(6, 6), q1_frac=res.q1_frac,
                q2_frac=res.q2_frac, qs=res.qs, iterations=res.iterations)


_PLANES = ("x", "y", "z")


def _modes6_dict(res: "xt_twiss6d_modes") -> Dict:
    out = {"stable": int(res.stable), "degenerate": int(res.degenerate)}
    for k in range(3):
        out["q%d_frac" % (k + 1)] = res.q_frac[k]
        raw = np.array(list(res.v[k]))
        out["v%d" % (k + 1)] = raw[0::2] + 1j * raw[1::2]
        for u, name in enumerate(_PLANES):
            out["bet%s%d" % (name, k + 1)] = res.bet[u][k]
            out["alf%s%d" % (name, k + 1)] = res.alf[u][k]
    out["dx"], out["dpx"], out["dy"], out["dpy"] = list(res.disp)
    return out


def xt_twiss6d_normal_form(m, rvv_co: float = 1.0, kind: str = "prod") -> Dict:
    """Normal modes of a 6x6 one-turn matrix in (x, px, y, py, zeta, delta) (host arithmetic only; include/xt.h)."""
    lib = load_library(kind)
    a = np.ascontiguousarray(m, dtype=np.float64).reshape(36)
    res = xt_twiss6d_modes()
    _check(lib, lib.xt_twiss6d_normal_form(a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), float(rvv_co),
                                           ctypes.byref(res)))
    return _modes6_dict(res)


def xt_twiss6d_line(lat: Lattice, guess6=None, stream=None):
    """(start dict, list of row dicts): the six-dimensional optics carried along the line (include/xt.h)."""
    n = lat.info["n_elements"] + 1
    rows = (xt_twiss6d_row * n)()
    res, modes = xt_twiss6d_result(), xt_twiss6d_modes()
    g = (ctypes.c_double * 6)(*[float(v) for v in guess6]) if guess6 is not None else None
    _check(lat._lib, lat._lib.xt_twiss6d_line(lat.handle, g, ctypes.byref(res), ctypes.byref(modes), rows, n,
                                              _stream_ptr(stream)))
    start = dict(co=np.array(list(res.co)), m=np.array(list(res.m)).reshape(6, 6), qs=res.qs,
                 iterations=res.iterations)
    start.update(_modes6_dict(modes))          # q1_frac .. q3_frac of the normal form (arg(lambda)/2 pi)
    out = []
    for r in rows:
        d = {"s": r.s, "co": np.array(list(r.co)), "dx": r.disp[0], "dpx": r.disp[1], "dy": r.disp[2], "dpy": r.disp[3]}
        for k in range(3):
            d["mu%d" % (k + 1)] = r.mu[k]
            for u, name in enumerate(_PLANES):
                d["bet%s%d" % (name, k + 1)] = r.bet[u][k]
                d["alf%s%d" % (name, k + 1)] = r.alf[u][k]
        out.append(d)
    return start, out


def xt_twiss4d_normal_form(m, kind: str = "prod") -> Dict:
    """Normal modes of a 4x4 one-turn matrix (host arithmetic only; include/xt.h)."""
    lib = load_library(kind)
    a = np.ascontiguousarray(m, dtype=np.float64).reshape(16)
    res = xt_twiss4d_modes()
    _check(lib, lib.xt_twiss4d_normal_form(a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), ctypes.byref(res)))
    out = {k: getattr(res, k) for k, _ in xt_twiss4d_modes._fields_ if k not in ("v1", "v2")}
    for k in ("v1", "v2"):
        raw = np.array(list(getattr(res, k)))
        out[k] = raw[0::2] + 1j * raw[1::2]
    return out


def xt_twiss4d_line(lat: Lattice, delta0: float = 0.0, ddelta: float = 1e-4, guess4=None, stream=None):
    """Optics along the line: (start dict as xt_twiss4d_chrom, rows dict of arrays of n_elements + 1); include/xt.h."""
    n = int(lat.info["n_elements"]) + 1
    rows = (xt_twiss_row * n)()
    res = xt_twiss4d_chrom_result()
    g = (ctypes.c_double * 4)(*[float(v) for v in guess4]) if guess4 is not None else None
    _check(lat._lib, lat._lib.xt_twiss4d_line(lat.handle, float(delta0), float(ddelta), g, ctypes.byref(res), rows, n,
                                              _stream_ptr(stream)))
    start = _twiss_dict(res.on)
    for k in ("dx", "dpx", "dy", "dpy", "dqx", "dqy"):
        start[k] = getattr(res, k)
    arr = np.frombuffer(rows, dtype=np.float64).reshape(n, len(xt_twiss_row._fields_)).copy()
    return start, {k: arr[:, i] for i, (k, _) in enumerate(xt_twiss_row._fields_)}


def xt_lattice_set_knobs(lat: Lattice, table, links) -> None:
    """``table``: [n_knobs][n_steps] knob values; ``links``: (element, order, skew, knob, gain) tuples (include/xt.h)."""
    t = np.ascontiguousarray(table, dtype=np.float64)
    if t.ndim != 2:
        raise ValueError("table must be 2-D [n_knobs][n_steps]")
    arr = (xt_knob_link * max(1, len(links)))()
    for i, (element, order, skew, knob, gain) in enumerate(links):
        arr[i] = xt_knob_link(int(element), int(order), int(skew), int(knob), 0, float(gain))
    _check(lat._lib, lat._lib.xt_lattice_set_knobs(lat.handle, t.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                                   t.shape[0], t.shape[1], arr, len(links)))


def xt_track_knobs(lat: Lattice, p: Dict, n_turns: int, step0: int = 0, stream=None) -> None:
    st = _struct_from_tensors(p)
    _check(lat._lib, lat._lib.xt_track_knobs(lat.handle, ctypes.byref(st), _n_part(p), int(n_turns), int(step0),
                                             _stream_ptr(stream)))


def xt_launch_count(kind: str = "prod") -> int:
    return int(load_library(kind).xt_launch_count())


def xt_build_info(kind: str = "prod") -> str:
    return load_library(kind).xt_build_info().decode()
