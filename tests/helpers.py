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


# ------------------------------------------------------------------ parity tolerance (reading A8)
FLOOR = 1e-15          # BASELINE.json north_star: "1e-12 relative (1e-15 absolute floor) per coordinate"
PARITY_KEYS = ("x", "px", "y", "py", "zeta", "delta", "ptau", "rpp", "rvv")


def parity_atol(ref_k: np.ndarray, rtol: float) -> float:
    """Absolute floor of one coordinate (reading A8): the north_star's 1e-15, or, where
    that is larger, rtol x the rms of THAT coordinate over the compared ensemble -- what an
    oscillating coordinate of that amplitude is allowed at the moment it crosses zero.  After one
    turn (rtol 1e-12, every rms <= 1e-3) this is the 1e-15 of the north_star for every coordinate;
    after 100 turns (rtol 1e-10) x, y (rms ~1e-4..1e-3 m) and zeta (0.05 m) get 1e-10 x their own
    scale, px, py (rms ~1e-6..1e-5) and delta, ptau (1e-4) stay at 1e-15, i.e. <= 1e-10 relative to
    their own rms -- never the blanket 1e-13 of round 1."""
    r = np.asarray(ref_k, dtype=np.float64)
    r = r[np.isfinite(r)]
    rms = float(np.sqrt(np.mean(r * r))) if r.size else 0.0
    return max(FLOOR, rtol * rms)


def parity_margins(got, ref, rtol, sel=None, keys=PARITY_KEYS):
    """-> {key: (worst |got-ref| / max(rtol |ref|, atol_k), atol_k, worst |got-ref| / (rtol rms_k), n_bad, first_bad)}."""
    out = {}
    for k in keys:
        a, r = np.asarray(got[k]), np.asarray(ref[k])
        if sel is not None:
            a, r = a[sel], r[sel]
        if a.size == 0:
            out[k] = (0.0, FLOOR, 0.0, 0, -1)
            continue
        atol = parity_atol(r, rtol)
        both_nan = np.isnan(a) & np.isnan(r)
        d = np.where(both_nan, 0.0, np.abs(a - r))
        bar = np.maximum(rtol * np.abs(np.where(both_nan, 0.0, r)), atol)
        ratio = d / bar
        ratio = np.where(np.isnan(ratio), np.inf, ratio)
        fin = r[np.isfinite(r)]
        rms = float(np.sqrt(np.mean(fin * fin))) if fin.size else 0.0
        bad = ratio > 1.0
        out[k] = (float(ratio.max()), atol, float(d.max() / (rtol * rms)) if rms > 0 else 0.0,
                  int(bad.sum()), int(np.argmax(bad)) if bad.any() else -1)
    return out


def assert_parity(got, ref, rtol, sel=None, keys=PARITY_KEYS, label=None):
    """The one floating-point parity check of every GPU test and of smoke(): per coordinate
    |got - ref| <= max(rtol |ref|, parity_atol).  With a label the measured margins are printed
    (pytest -s) in the form DESIGN.md section 9 tabulates."""
    m = parity_margins(got, ref, rtol, sel, keys)
    if label:
        print("PARITY %s rtol=%g " % (label, rtol) +
              " ".join("%s=%.3f(atol %.1e; /rms %.3f)" % (k, v[0], v[1], v[2]) for k, v in m.items()))
    for k, v in m.items():
        if v[3]:
            a, r = np.asarray(got[k]), np.asarray(ref[k])
            if sel is not None:
                a, r = a[sel], r[sel]
            j = v[4]
            raise AssertionError("%s: %d/%d outside tolerance (worst %.3g x the bar, atol %.2e); first %d gpu=%r ref=%r"
                                 % (k, v[3], a.size, v[0], v[1], j, a[j], r[j]))
    return m

