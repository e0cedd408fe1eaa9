"""Packed lattice buffer: the user-level, serialised form of a beam line.

PAPER.md:70 ("Lattice modelling and single particle tracking"): "The beam line is
represented as a sequence of Python objects ..., each corresponding to an
accelerator element".  Here that sequence is flattened into one little-endian,
8-byte-aligned byte buffer (layout documented in ``include/xt.h`` and DESIGN.md §3):

    header (48 B):  char magic[8] = "XTLAT001"; uint32 version = 1; uint32 n_elements;
                    double p0c [eV]; double mass0 [eV]; double q0 [e]; uint64 total_bytes
    n_elements records:  uint32 type; uint32 aux; double params[...]

    type 0 MARKER        aux=0  (no params)
    type 1 DRIFT         aux=0  length
    type 2 MULTIPOLE     aux=N  hxl, length, knl[0..N], ksl[0..N]     (raw, NOT divided by n!)
    type 3 CAVITY        aux=0  voltage [V], frequency [Hz], lag [deg]
    type 4 SROTATION     aux=0  cos_z, sin_z
    type 5 XYSHIFT       aux=0  dx, dy
    type 6 LIMITRECT     aux=0  min_x, max_x, min_y, max_y
    type 7 LIMITELLIPSE  aux=0  a, b
    type 8 QUADRUPOLE    aux=0  k1 [1/m^2], length [m]   (thick; k1 != 0, length > 0)
    type 9 BEND          aux=m  k0 [1/m], h [1/m], length [m]   (thick sector bend: m = 0 the
                                'expanded' map, m = 1 the 'full' map; k0*h > 0, length > 0; a pure sector
                                bend has k0 = h)
    type 10 LIMITPOLYGON aux=n  x[0..n), y[0..n)   (closed polygon, 3 <= n <= 256 vertices; PAPER.md:178
                                "polygonal interpolation")
    type 12 RADMULTIPOLE aux=N  hxl, length, knl[0..N], ksl[0..N]   (thin multipole with "mean" synchrotron
                                radiation; length > 0)        [type 11 is internal to the library]

This module is pure serialisation (struct packing).  It performs no tracking
arithmetic: the same bytes are handed to the oracle and to ``xt_lattice_create``;
each parses them with its own code.
"""
from __future__ import annotations

import math
import struct
from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

MAGIC = b"XTLAT001"
VERSION = 1
HEADER_BYTES = 48

ELEMENT_TYPE_IDS = {
    "Marker": 0, "Drift": 1, "Multipole": 2, "Cavity": 3,
    "SRotation": 4, "XYShift": 5, "LimitRect": 6, "LimitEllipse": 7, "Quadrupole": 8, "Bend": 9, "LimitPolygon": 10, "RadMultipole": 12,
}


@dataclass(frozen=True)
class Marker:
    pass


@dataclass(frozen=True)
class Drift:
    length: float


@dataclass(frozen=True)
class Multipole:
    knl: Tuple[float, ...]
    ksl: Tuple[float, ...] = ()
    hxl: float = 0.0
    length: float = 0.0

    @property
    def order(self) -> int:
        return max(len(self.knl), len(self.ksl), 1) - 1


@dataclass(frozen=True)
class Cavity:
    voltage: float
    frequency: float
    lag: float  # degrees


@dataclass(frozen=True)
class SRotation:
    cos_z: float
    sin_z: float

    @staticmethod
    def from_angle(theta_rad: float) -> "SRotation":
        # cos/sin are stored so that both consumers get identical FP64 values
        return SRotation(math.cos(theta_rad), math.sin(theta_rad))


@dataclass(frozen=True)
class XYShift:
    dx: float
    dy: float


@dataclass(frozen=True)
class LimitRect:
    min_x: float
    max_x: float
    min_y: float
    max_y: float


@dataclass(frozen=True)
class LimitEllipse:
    a: float
    b: float


@dataclass(frozen=True)
class Quadrupole:
    """Thick quadrupole: gradient k1 = (dBy/dx)/(P0/q0), magnetic length."""
    k1: float
    length: float


@dataclass(frozen=True)
class Bend:
    """Thick sector bend: dipole strength k0 = By/(P0/q0), curvature h of the reference
    orbit, arc length; model 0 = the 'expanded' map, 1 = the 'full' map."""
    k0: float
    h: float
    length: float
    model: int = 0


@dataclass(frozen=True)
class LimitPolygon:
    """Aperture given by a closed polygon (the "locally refined aperture model obtained by
    polygonal interpolation"); vertices in order, the last one joins the first."""
    x: Tuple[float, ...]
    y: Tuple[float, ...]


@dataclass(frozen=True)
class RadMultipole:
    """Thin multipole slice that radiates ("mean" model); same parameters as Multipole, length > 0."""
    knl: Tuple[float, ...]
    ksl: Tuple[float, ...] = ()
    hxl: float = 0.0
    length: float = 1.0

    @property
    def order(self) -> int:
        return max(len(self.knl), len(self.ksl), 1) - 1


def _record(el) -> bytes:
    if isinstance(el, Marker):
        return struct.pack("<II", 0, 0)
    if isinstance(el, Drift):
        return struct.pack("<IId", 1, 0, el.length)
    if isinstance(el, (Multipole, RadMultipole)):
        n = el.order
        knl = list(el.knl) + [0.0] * (n + 1 - len(el.knl))
        ksl = list(el.ksl) + [0.0] * (n + 1 - len(el.ksl))
        return struct.pack("<II%dd" % (2 + 2 * (n + 1)), 12 if isinstance(el, RadMultipole) else 2, n, el.hxl,
                           el.length, *knl, *ksl)
    if isinstance(el, Cavity):
        return struct.pack("<II3d", 3, 0, el.voltage, el.frequency, el.lag)
    if isinstance(el, SRotation):
        return struct.pack("<II2d", 4, 0, el.cos_z, el.sin_z)
    if isinstance(el, XYShift):
        return struct.pack("<II2d", 5, 0, el.dx, el.dy)
    if isinstance(el, LimitRect):
        return struct.pack("<II4d", 6, 0, el.min_x, el.max_x, el.min_y, el.max_y)
    if isinstance(el, LimitEllipse):
        return struct.pack("<II2d", 7, 0, el.a, el.b)
    if isinstance(el, Quadrupole):
        return struct.pack("<II2d", 8, 0, el.k1, el.length)
    if isinstance(el, Bend):
        return struct.pack("<II3d", 9, int(el.model), el.k0, el.h, el.length)
    if isinstance(el, LimitPolygon):
        assert len(el.x) == len(el.y)
        return struct.pack("<II%dd" % (2 * len(el.x)), 10, len(el.x), *el.x, *el.y)
    raise TypeError("unknown element %r" % (el,))


def pack_lattice(elements: Sequence, p0c: float, mass0: float, q0: float = 1.0) -> bytes:
    """Serialise ``elements`` (in beam order) into the packed lattice buffer."""
    body = b"".join(_record(e) for e in elements)
    total = HEADER_BYTES + len(body)
    head = struct.pack("<8sIIdddQ", MAGIC, VERSION, len(elements), p0c, mass0, q0, total)
    assert len(head) == HEADER_BYTES
    return head + body


def unpack_lattice(buf: bytes):
    """Inverse of :func:`pack_lattice` -> (elements, p0c, mass0, q0).  Test helper."""
    magic, version, n, p0c, mass0, q0, total = struct.unpack_from("<8sIIdddQ", buf, 0)
    if magic != MAGIC or version != VERSION or total != len(buf):
        raise ValueError("not a packed lattice buffer")
    off = HEADER_BYTES
    out: List = []
    for _ in range(n):
        t, aux = struct.unpack_from("<II", buf, off)
        off += 8
        if t == 0:
            out.append(Marker())
        elif t == 1:
            (length,) = struct.unpack_from("<d", buf, off); off += 8
            out.append(Drift(length))
        elif t == 2:
            m = aux + 1
            vals = struct.unpack_from("<%dd" % (2 + 2 * m), buf, off); off += 8 * (2 + 2 * m)
            out.append(Multipole(knl=tuple(vals[2:2 + m]), ksl=tuple(vals[2 + m:2 + 2 * m]),
                                 hxl=vals[0], length=vals[1]))
        elif t == 3:
            v, f, lag = struct.unpack_from("<3d", buf, off); off += 24
            out.append(Cavity(v, f, lag))
        elif t == 4:
            c, s = struct.unpack_from("<2d", buf, off); off += 16
            out.append(SRotation(c, s))
        elif t == 5:
            dx, dy = struct.unpack_from("<2d", buf, off); off += 16
            out.append(XYShift(dx, dy))
        elif t == 6:
            vals = struct.unpack_from("<4d", buf, off); off += 32
            out.append(LimitRect(*vals))
        elif t == 7:
            a, b = struct.unpack_from("<2d", buf, off); off += 16
            out.append(LimitEllipse(a, b))
        elif t == 8:
            k1, length = struct.unpack_from("<2d", buf, off); off += 16
            out.append(Quadrupole(k1, length))
        elif t == 9:
            k0, h, length = struct.unpack_from("<3d", buf, off); off += 24
            out.append(Bend(k0, h, length, aux))
        elif t == 12:
            m = aux + 1
            vals = struct.unpack_from("<%dd" % (2 + 2 * m), buf, off); off += 8 * (2 + 2 * m)
            out.append(RadMultipole(knl=tuple(vals[2:2 + m]), ksl=tuple(vals[2 + m:2 + 2 * m]),
                                    hxl=vals[0], length=vals[1]))
        elif t == 10:
            vals = struct.unpack_from("<%dd" % (2 * aux), buf, off); off += 16 * aux
            out.append(LimitPolygon(tuple(vals[:aux]), tuple(vals[aux:])))
        else:
            raise ValueError("unknown element type %d" % t)
    return out, p0c, mass0, q0
