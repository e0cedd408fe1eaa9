"""Shared test helpers (host-side only; no tracking arithmetic beyond variable changes
needed to express invariants in canonical variables)."""
from __future__ import annotations

import json
import os
from typing import Dict, List, Sequence

import numpy as np

from oracle import oracle as O
from xt_inputs import packed as PK

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
P0C, MASS0, Q0 = 450e9, 938272088.16, 1.0
COORDS = ("x", "px", "y", "py", "zeta", "delta")


def load_golden():
    with open(os.path.join(GOLDEN, "worked_examples.json")) as fh:
        return json.load(fh)


def unhex(v):
    return float.fromhex(v)


def element_from_json(d):
    kw = {}
    for k, v in d.items():
        if k == "type":
            continue
        kw[k] = tuple(unhex(t) for t in v) if isinstance(v, list) else unhex(v)
    return getattr(PK, d["type"])(**kw)


def coords_from_rows(rows: Sequence[Sequence[float]]) -> Dict[str, np.ndarray]:
    a = np.asarray(rows, dtype=np.float64).reshape(-1, 6)
    return {k: np.ascontiguousarray(a[:, i]) for i, k in enumerate(COORDS)}


def oracle_particles_from_ptau(packed: bytes, x, px, y, py, zeta, ptau) -> Dict[str, np.ndarray]:
    """Particle SoA with ptau as the independent energy variable (for Jacobians in the
    canonical variables (x,px,y,py,zeta,ptau/beta0), reading A13): delta from the energy
    identity (1+delta)^2 = ptau^2 + 2 ptau/beta0 + 1, evaluated without cancellation."""
    beta0, _ = O.reference(packed)
    ptau = np.asarray(ptau, dtype=np.float64)
    t = ptau * (ptau + 2.0 / beta0)
    delta = t / (np.sqrt(t + 1.0) + 1.0)
    p = O.new_particles(packed, dict(x=x, px=px, y=y, py=py, zeta=zeta, delta=delta))
    p["ptau"] = ptau.copy()
    p["rpp"] = 1.0 / (1.0 + delta)
    p["rvv"] = (1.0 + delta) / (1.0 + beta0 * ptau)
    return p


def jacobian6(track_fn, packed: bytes, z0: Sequence[float], n_turns: int = 1,
              h: Sequence[float] = (1e-6, 1e-7, 1e-6, 1e-7, 1e-4, 1e-7)) -> np.ndarray:
    """6x6 central-difference Jacobian of the n-turn map in (x,px,y,py,zeta,pzeta=ptau/beta0)
    around z0 (Twiss step 2).  ``track_fn(packed, particles, n_turns)`` tracks
    in place (oracle or GPU front end)."""
    beta0, _ = O.reference(packed)
    z0 = np.asarray(z0, dtype=np.float64)
    pts = []
    for i in range(6):
        for sgn in (+1.0, -1.0):
            z = z0.copy()
            z[i] += sgn * h[i]
            pts.append(z)
    pts = np.asarray(pts)
    p = oracle_particles_from_ptau(packed, pts[:, 0].copy(), pts[:, 1].copy(), pts[:, 2].copy(),
                                   pts[:, 3].copy(), pts[:, 4].copy(), pts[:, 5] * beta0)
    track_fn(packed, p, n_turns)
    assert np.all(p["state"] == 1)
    out = np.stack([p["x"], p["px"], p["y"], p["py"], p["zeta"], p["ptau"] / beta0], axis=1)
    J = np.zeros((6, 6))
    for i in range(6):
        J[:, i] = (out[2 * i] - out[2 * i + 1]) / (2.0 * h[i])
    return J


S6 = np.zeros((6, 6))
for _i in range(3):
    S6[2 * _i, 2 * _i + 1] = 1.0
    S6[2 * _i + 1, 2 * _i] = -1.0


def reversed_lattice(elements: List) -> List:
    """Reading A11: reverse the order; Cavity lag -> -lag; SRotation (c,s)->(c,-s);
    XYShift -> (-dx,-dy); drifts, multipoles, apertures unchanged."""
    out = []
    for el in reversed(elements):
        if isinstance(el, PK.Cavity):
            out.append(PK.Cavity(el.voltage, el.frequency, -el.lag))
        elif isinstance(el, PK.SRotation):
            out.append(PK.SRotation(el.cos_z, -el.sin_z))
        elif isinstance(el, PK.XYShift):
            out.append(PK.XYShift(-el.dx, -el.dy))
        else:
            out.append(el)
    return out


def flip_R(p: Dict[str, np.ndarray]) -> None:
    """R: (x,px,y,py,zeta,delta) -> (x,-px,y,-py,-zeta,delta)."""
    p["px"] *= -1.0
    p["py"] *= -1.0
    p["zeta"] *= -1.0


def rel_err(a: np.ndarray, ref: np.ndarray, floor: float = 0.0) -> np.ndarray:
    """|a-ref| / max(|ref|, floor/tol-free): returns |a-ref|/|ref| with 0/0 = 0."""
    d = np.abs(a - ref)
    den = np.abs(ref)
    out = np.zeros_like(d)
    nz = den > 0
    out[nz] = d[nz] / den[nz]
    out[~nz & (d > floor)] = np.inf
    return out


def within(a: np.ndarray, ref: np.ndarray, rtol: float, atol: float) -> np.ndarray:
    """Reading A8: pass iff |a - ref| <= max(rtol*|ref|, atol), elementwise (NaN == NaN passes)."""
    both_nan = np.isnan(a) & np.isnan(ref)
    return both_nan | (np.abs(a - ref) <= np.maximum(rtol * np.abs(ref), atol))
