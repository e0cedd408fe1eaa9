"""The five synthetic workloads of BASELINE.json ``configs`` (recipe: DESIGN.md §4).

The paper names no public data set for single-particle tracking (its studies use
CERN machine models); these seeded synthetic lattices and particle
ensembles have the shapes and sizes BASELINE.json prescribes and stand in for them.

Only input construction lives here (element lists, random draws, amplitude grids).
No tracking arithmetic: optics values needed for matched distributions are *read*
from ``optics.json`` (written by ``oracle/make_optics.py`` from the oracle's one-turn
Jacobian, Twiss steps 2-3 of PAPER.md:97-98).

All random numbers come from ``numpy.random.default_rng(seed)`` (PCG64); seeds:
particles 1000+i, multipole errors 2002 (configs 2-4 share one "LHC-sized" machine),
misalignments 3003.
"""
from __future__ import annotations

import json
import math
import os
from typing import Dict, List, Optional, Tuple

import numpy as np

from .packed import (Bend, Cavity, Drift, LimitEllipse, LimitRect, Multipole, Quadrupole, SRotation,
                     XYShift, pack_lattice)

P0C = 450e9                 # eV, BASELINE.json configs[0]
MASS0 = 938272088.16        # eV, proton (CODATA 2018); the paper gives none
Q0 = 1.0
BETA0_GAMMA0 = P0C / MASS0  # p/(m c)

COORDS = ("x", "px", "y", "py", "zeta", "delta")

_OPTICS_PATH = os.path.join(os.path.dirname(__file__), "optics.json")


def load_optics() -> Dict[str, Dict[str, float]]:
    """Optics at the start point of each lattice, written by oracle/make_optics.py."""
    with open(_OPTICS_PATH) as fh:
        return json.load(fh)


# ----------------------------------------------------------------------------- lattices
def fodo_elements(sextupoles: bool, aperture: bool) -> List:
    """configs[0] / configs[1]: 10 thin-lens FODO cells + one cavity (C = 40 m)."""
    qf = Multipole(knl=(0.0, +0.1))
    qd = Multipole(knl=(0.0, -0.1))
    sf = Multipole(knl=(0.0, 0.0, +0.5))
    sd = Multipole(knl=(0.0, 0.0, -0.5))
    els: List = []
    for _ in range(10):
        els.append(qf)
        if sextupoles:
            els.append(sf)
        els.append(Drift(2.0))
        els.append(qd)
        if sextupoles:
            els.append(sd)
        els.append(Drift(2.0))
        if aperture:
            els.append(LimitRect(-0.010, 0.010, -0.010, 0.010))
    els.append(Cavity(1e6, 200e6, 180.0))
    return els


def lattice_cfg0() -> List:
    return fodo_elements(sextupoles=False, aperture=False)           # 41 elements


def lattice_cfg1() -> List:
    return fodo_elements(sextupoles=True, aperture=True)             # 71 elements


LHC_CIRC = 26658.883
LHC_NHALF = 400
LHC_LHALF = 66.6472075
LHC_KF = 1.6566 / LHC_LHALF
LHC_KD = 1.6273 / LHC_LHALF
LHC_NBEND = 1232
LHC_BEND_LEN = 14.3
LHC_ERR_ORDER = 15
LHC_ERR_RMS = 1e-4
LHC_ERR_RADIUS = 0.017
LHC_CAVITY_HALFCELLS = (80, 82, 180, 182, 280, 282, 380, 382)


def _with_errors(main_order: int, main_strength: float, rng: np.random.Generator,
                 hxl: float = 0.0, length: float = 0.0) -> Multipole:
    """Main field + relative-1e-4 random normal/skew errors of orders 0..15 at R = 17 mm."""
    n_max = LHC_ERR_ORDER
    knl = [0.0] * (n_max + 1)
    ksl = [0.0] * (n_max + 1)
    knl[main_order] = main_strength
    g = rng.standard_normal(n_max + 1)
    gp = rng.standard_normal(n_max + 1)
    for n in range(n_max + 1):
        scale = (LHC_ERR_RMS * main_strength * math.factorial(n) / math.factorial(main_order)
                 * LHC_ERR_RADIUS ** (main_order - n))
        knl[n] += scale * g[n]
        ksl[n] += scale * gp[n]
    return Multipole(knl=tuple(knl), ksl=tuple(ksl), hxl=hxl, length=length)


def lhc_like_elements(k3l: float = 1.0, misalign: bool = False, errors: bool = True,
                      apertures: bool = True,
                      err_seed: int = 2002, mis_seed: int = 3003,
                      n_halfcells: int = LHC_NHALF, thick: bool = False) -> List:
    """configs[2] (k3l=1), configs[3] (misalign=True), configs[4] (k3l=5).

    400 half-cells; each magnet (and cavity) sits mid-slot as [Drift(l/2), magnet, Drift(l/2)];
    a LimitEllipse(20 mm, 15 mm) follows every 10th element.

    ``thick=True`` (the thick-map bench workload): every quadrupole becomes a thick
    Quadrupole (length min(3.1 m, 0.8 slot), k1 = k1l/length) and every bend a thick sector Bend ('expanded';
    length 0.8 slot, k0 = h = hxl/length), each taking its length out of the two drifts of its slot; thick
    elements carry no multipole errors; sextupoles and octupoles stay thin with their order-15 errors.
    """
    rng = np.random.default_rng(err_seed)
    rng_mis = np.random.default_rng(mis_seed)
    hxl_bend = 2.0 * math.pi / LHC_NBEND

    def magnet(order: int, strength: float, hxl: float = 0.0, length: float = 0.0):
        if errors:
            return _with_errors(order, strength, rng, hxl=hxl, length=length)
        knl = [0.0] * (order + 1)
        knl[order] = strength
        return Multipole(knl=tuple(knl), hxl=hxl, length=length)

    base: List = []
    for j in range(n_halfcells):
        focusing = (j % 2 == 0)
        jm = j % 100
        arc = jm < 77
        sign = +1.0 if focusing else -1.0
        slots: List[List] = []
        quad = magnet(1, +LHC_KF if focusing else -LHC_KD)
        if thick:
            quad = ("quad", +LHC_KF if focusing else -LHC_KD)
        if misalign:
            dx, dy = rng_mis.normal(0.0, 1e-4, size=2)
            th = rng_mis.normal(0.0, 1e-4)
            slots.append([XYShift(dx, dy), SRotation.from_angle(th), quad,
                          SRotation.from_angle(-th), XYShift(-dx, -dy)])
        else:
            slots.append([quad])
        k2l = +0.006 if focusing else -0.014
        slots.append([magnet(2, k2l)])                                   # S1
        if jm < 42:
            slots.append([magnet(3, sign * k3l)])                        # O
        if arc:
            for b in range(4):
                slots.append([("bend", hxl_bend)] if thick else
                             [magnet(0, hxl_bend, hxl=hxl_bend, length=LHC_BEND_LEN)])
                if b == 1:
                    slots.append([magnet(2, k2l)])                       # S2 between bend pairs
        else:
            slots.append([magnet(2, k2l)])                               # S2
            if j in LHC_CAVITY_HALFCELLS:
                slots.append([Cavity(1e6, 400e6, 180.0)])
        half = 0.5 * (LHC_LHALF / len(slots))
        for group in slots:
            taken = 0.0
            for k, el in enumerate(group):
                if isinstance(el, tuple):                      # thick stand-in: (kind, integrated strength)
                    kind, strength = el
                    if kind == "quad":
                        length = min(3.1, 1.6 * half)
                        group[k] = Quadrupole(strength / length, length)
                    else:
                        length = 1.6 * half
                        group[k] = Bend(strength / length, strength / length, length)
                    taken = length
            base.append(Drift(half - 0.5 * taken))
            base.extend(group)
            base.append(Drift(half - 0.5 * taken))
    if not apertures:
        return base
    out: List = []
    for i, el in enumerate(base, start=1):
        out.append(el)
        if i % 10 == 0:
            out.append(LimitEllipse(0.020, 0.015))
    return out


def lattice_cfg2() -> List:
    return lhc_like_elements(k3l=1.0)


def lattice_cfg3() -> List:
    return lhc_like_elements(k3l=1.0, misalign=True)


def lattice_cfg4() -> List:
    return lhc_like_elements(k3l=5.0)


def lattice_cfg2_thick() -> List:
    """configs[2] with thick quadrupoles and thick sector bends (bench.py --workload thick)."""
    return lhc_like_elements(k3l=1.0, thick=True)


def strip_cavities(elements: List) -> List:
    """Cavity-free copy for the bit-exact (--fmad=false) comparison (reading A10)."""
    return [e for e in elements if not isinstance(e, Cavity)]


def pack(elements: List) -> bytes:
    return pack_lattice(elements, P0C, MASS0, Q0)


# ---------------------------------------------------------------------------- particles
def _empty(n: int) -> Dict[str, np.ndarray]:
    return {k: np.zeros(n, dtype=np.float64) for k in COORDS}


def particles_cfg0(n: int = 1000, seed: int = 1000) -> Dict[str, np.ndarray]:
    rng = np.random.default_rng(seed)
    p = _empty(n)
    p["x"] = rng.normal(0.0, 1e-4, n)
    p["px"] = rng.normal(0.0, 1e-5, n)
    p["y"] = rng.normal(0.0, 1e-4, n)
    p["py"] = rng.normal(0.0, 1e-5, n)
    p["zeta"] = rng.normal(0.0, 0.05, n)
    p["delta"] = rng.normal(0.0, 1e-4, n)
    return p


def particles_cfg1(n_r: int = 10000, n_theta: int = 100, sigma: float = 1e-4,
                   r_max: float = 20.0) -> Dict[str, np.ndarray]:
    """Uniform polar amplitude grid, delta = 0.  sigma=1e-3 gives the supplementary
    'configs[1b]' that actually loses particles."""
    r = r_max * np.arange(n_r, dtype=np.float64) / max(n_r - 1, 1)
    th = (math.pi / 2.0) * (np.arange(n_theta, dtype=np.float64) + 0.5) / n_theta
    rr, tt = np.meshgrid(r, th, indexing="ij")
    p = _empty(n_r * n_theta)
    p["x"] = (rr * sigma * np.cos(tt)).ravel()
    p["y"] = (rr * sigma * np.sin(tt)).ravel()
    return p


EPS_N = 2.5e-6   # normalised emittance [m]


def _add_closed_orbit(p: Dict[str, np.ndarray], optics: Dict[str, float]) -> None:
    """Centre the ensemble on the 4-D closed orbit at the start point (Twiss step 1)."""
    for k in ("x", "px", "y", "py"):
        p[k] = p[k] + optics.get(k + "_co", 0.0)


def matched_gaussian(n: int, seed: int, optics: Dict[str, float], n_sigma: float = 1.0,
                     sigma_zeta: float = 0.05, sigma_delta: float = 1e-4) -> Dict[str, np.ndarray]:
    """configs[2]/[3]: 6-D Gaussian matched to (beta, alpha) at the start point."""
    rng = np.random.default_rng(seed)
    eps = EPS_N / BETA0_GAMMA0
    p = _empty(n)
    g = rng.standard_normal((6, n))
    for (u, pu, i0) in (("x", "px", 0), ("y", "py", 2)):
        beta = optics["bet" + u]
        alpha = optics["alf" + u]
        p[u] = n_sigma * math.sqrt(eps * beta) * g[i0]
        p[pu] = n_sigma * math.sqrt(eps / beta) * (g[i0 + 1] - alpha * g[i0])
    p["zeta"] = n_sigma * sigma_zeta * g[4]
    p["delta"] = n_sigma * sigma_delta * g[5]
    _add_closed_orbit(p, optics)
    return p


def particles_cfg2(n: int = 100_000, seed: int = 1002, optics: Optional[dict] = None):
    optics = optics or load_optics()["cfg2"]
    return matched_gaussian(n, seed, optics, n_sigma=1.0)


def particles_cfg3(n: int = 10_000_000, seed: int = 1003, optics: Optional[dict] = None):
    optics = optics or load_optics()["cfg3"]
    return matched_gaussian(n, seed, optics, n_sigma=2.0)


CFG4_DELTAS = (-3e-4, -1.8e-4, -0.6e-4, 0.6e-4, 1.8e-4, 3e-4)


def particles_cfg4(n_r: int = 1667, n_theta: int = 200, r_max: float = 30.0,
                   optics: Optional[dict] = None) -> Dict[str, np.ndarray]:
    """Polar grid x 6 momentum offsets: 1667 x 200 x 6 = 2 000 400 particles
    (2 000 000 is not divisible by 1 200)."""
    optics = optics or load_optics()["cfg4"]
    eps = EPS_N / BETA0_GAMMA0
    sx = math.sqrt(eps * optics["betx"])
    sy = math.sqrt(eps * optics["bety"])
    r = r_max * np.arange(n_r, dtype=np.float64) / max(n_r - 1, 1)
    th = (math.pi / 2.0) * (np.arange(n_theta, dtype=np.float64) + 0.5) / n_theta
    d = np.asarray(CFG4_DELTAS)
    rr, tt, dd = np.meshgrid(r, th, d, indexing="ij")
    n = rr.size
    p = _empty(n)
    p["x"] = (rr * sx * np.cos(tt)).ravel()
    p["y"] = (rr * sy * np.sin(tt)).ravel()
    p["px"] = -optics["alfx"] * p["x"] / optics["betx"]
    p["py"] = -optics["alfy"] * p["y"] / optics["bety"]
    p["delta"] = dd.ravel().copy()
    _add_closed_orbit(p, optics)
    return p


# ------------------------------------------------------------------------------ registry
def n_turns(cfg: int) -> int:
    return (100, 1000, 1000, 100, 100_000)[cfg]


def lattice(cfg: int) -> List:
    return (lattice_cfg0, lattice_cfg1, lattice_cfg2, lattice_cfg3, lattice_cfg4)[cfg]()


def particles(cfg: int, n: Optional[int] = None) -> Dict[str, np.ndarray]:
    """Full-size ensemble of config ``cfg``; ``n`` overrides the count for the Gaussian
    configs (0, 2, 3) only."""
    if cfg == 0:
        return particles_cfg0(n or 1000)
    if cfg == 1:
        return particles_cfg1()
    if cfg == 2:
        return particles_cfg2(n or 100_000)
    if cfg == 3:
        return particles_cfg3(n or 10_000_000)
    if cfg == 4:
        return particles_cfg4()
    raise ValueError(cfg)


def subsample(p: Dict[str, np.ndarray], idx) -> Dict[str, np.ndarray]:
    return {k: np.ascontiguousarray(v[idx]) for k, v in p.items()}
