#!/usr/bin/env python
"""Writes tests/golden/worked_examples.json: 60-digit evaluations of the TEXTBOOK maps.

This script is the pin for the oracle's arithmetic (P1, P5, P6 in DESIGN.md §6).  It does
not call the oracle or the CUDA path.  It evaluates, with mpmath at 60 significant digits,
the *textbook* (not the cancellation-free, not the Horner) forms of the thin-lens maps the
paper refers to (PAPER.md:72 thin-lattice integration, ref [13] PAPER.md:255):

  drift      pz = sqrt((1+d)^2 - px^2 - py^2);  x += L px/pz;  y += L py/pz;
             zeta += L (1 - (1 + beta0 ptau)/pz)
  multipole  dpx - i dpy = - sum_n (knl[n] + i ksl[n]) (x + i y)^n / n!     (direct powers)
             curvature h = hxl: px += hxl (1+d) - (knl[0] hxl/length) x;  zeta -= hxl x beta0/beta
  cavity     ptau += (q0 V/p0c) sin(lag pi/180 - 2 pi f zeta/(beta0 c));  d = sqrt(ptau^2 + 2 ptau/beta0 + 1) - 1
  srotation  (x, y) -> (c x + s y, c y - s x), same for (px, py)
  xyshift    x -= dx, y -= dy
  init       ptau = sqrt((1+d)^2 + (mass0/p0c)^2) - 1/beta0

Inputs are stored as C99 hex floats so the oracle sees the identical FP64 numbers; outputs as
40-digit decimal strings.  Run:  python tests/golden/make_worked_examples.py
"""
import json
import math
import os
import sys

import mpmath as mp
import numpy as np

sys.path.insert(0, os.path.join(os.path.dirname(__file__), "..", ".."))
from xt_inputs.packed import (Cavity, Drift, LimitEllipse, LimitRect, Marker,  # noqa: E402
                              Multipole, SRotation, XYShift)
from xt_inputs import configs  # noqa: E402

mp.mp.dps = 60
C_LIGHT = mp.mpf(299792458)


class Ref:
    def __init__(self, p0c, mass0, q0=1.0):
        self.p0c, self.mass0, self.q0 = mp.mpf(p0c), mp.mpf(mass0), mp.mpf(q0)
        e0 = mp.sqrt(self.p0c ** 2 + self.mass0 ** 2)
        self.beta0 = self.p0c / e0
        self.gamma0 = e0 / self.mass0


def init_particle(ref, x, px, y, py, zeta, delta):
    d = mp.mpf(delta)
    ptau = mp.sqrt((1 + d) ** 2 + (ref.mass0 / ref.p0c) ** 2) - 1 / ref.beta0
    return dict(x=mp.mpf(x), px=mp.mpf(px), y=mp.mpf(y), py=mp.mpf(py), zeta=mp.mpf(zeta),
                delta=d, ptau=ptau)


def derived(ref, p):
    rpp = 1 / (1 + p["delta"])
    rvv = (1 + p["delta"]) / (1 + ref.beta0 * p["ptau"])
    return rpp, rvv


def apply(ref, el, p):
    """Textbook map of one element, in place."""
    if isinstance(el, (Marker, LimitRect, LimitEllipse)):
        return
    if isinstance(el, Drift):
        L = mp.mpf(el.length)
        pz = mp.sqrt((1 + p["delta"]) ** 2 - p["px"] ** 2 - p["py"] ** 2)
        p["x"] += L * p["px"] / pz
        p["y"] += L * p["py"] / pz
        p["zeta"] += L * (1 - (1 + ref.beta0 * p["ptau"]) / pz)
    elif isinstance(el, Multipole):
        n_ord = el.order
        knl = [mp.mpf(v) for v in el.knl] + [mp.mpf(0)] * (n_ord + 1 - len(el.knl))
        ksl = [mp.mpf(v) for v in el.ksl] + [mp.mpf(0)] * (n_ord + 1 - len(el.ksl))
        z = mp.mpc(p["x"], p["y"])
        acc = mp.mpc(0)
        for n in range(n_ord + 1):
            acc += mp.mpc(knl[n], ksl[n]) * z ** n / mp.factorial(n)
        dpx = -acc.real
        dpy = +acc.imag
        x0 = p["x"]
        p["px"] += dpx
        p["py"] += dpy
        if el.hxl != 0.0:
            h = mp.mpf(el.hxl)
            p["px"] += h * (1 + p["delta"])
            if el.length != 0.0:
                p["px"] -= (knl[0] * h / mp.mpf(el.length)) * x0
            beta0_over_beta = (1 + ref.beta0 * p["ptau"]) / (1 + p["delta"])
            p["zeta"] -= h * x0 * beta0_over_beta
    elif isinstance(el, Cavity):
        phase = mp.mpf(el.lag) * mp.pi / 180 - 2 * mp.pi * mp.mpf(el.frequency) * p["zeta"] / (ref.beta0 * C_LIGHT)
        p["ptau"] += ref.q0 * mp.mpf(el.voltage) / ref.p0c * mp.sin(phase)
        p["delta"] = mp.sqrt(p["ptau"] ** 2 + 2 * p["ptau"] / ref.beta0 + 1) - 1
    elif isinstance(el, SRotation):
        c, s = mp.mpf(el.cos_z), mp.mpf(el.sin_z)
        x, y, px, py = p["x"], p["y"], p["px"], p["py"]
        p["x"], p["y"] = c * x + s * y, c * y - s * x
        p["px"], p["py"] = c * px + s * py, c * py - s * px
    elif isinstance(el, XYShift):
        p["x"] -= mp.mpf(el.dx)
        p["y"] -= mp.mpf(el.dy)
    else:
        raise TypeError(el)


def s40(v):
    return mp.nstr(v, 40, strip_zeros=False, min_fixed=0, max_fixed=0)


def snapshot(ref, p):
    rpp, rvv = derived(ref, p)
    out = {k: s40(p[k]) for k in ("x", "px", "y", "py", "zeta", "delta", "ptau")}
    out["rpp"], out["rvv"] = s40(rpp), s40(rvv)
    return out


def el_json(el):
    d = {"type": type(el).__name__}
    for k, v in el.__dict__.items():
        d[k] = [float(t).hex() for t in v] if isinstance(v, tuple) else float(v).hex()
    return d


def worked_line(name, ref_args, els, start, cite):
    ref = Ref(*ref_args)
    p = init_particle(ref, *start)
    stages = [{"after": "init", "values": snapshot(ref, p)}]
    for el in els:
        apply(ref, el, p)
        stages.append({"after": type(el).__name__, "values": snapshot(ref, p)})
    return {"name": name, "cite": cite,
            "p0c": float(ref_args[0]).hex(), "mass0": float(ref_args[1]).hex(), "q0": float(ref_args[2]).hex(),
            "beta0": s40(ref.beta0), "gamma0": s40(ref.gamma0),
            "start": [float(v).hex() for v in start],
            "elements": [el_json(e) for e in els], "stages": stages}


def main():
    ref_args = (450e9, 938272088.16, 1.0)
    start = (1e-3, 2e-4, -5e-4, 1e-4, 0.01, 3e-4)
    out = {"_about": "60-digit mpmath evaluation of the textbook thin-lens maps; written by "
                     "tests/golden/make_worked_examples.py; inputs are hex floats", "lines": []}

    # W1 (SURVEY.md §8(c) worked example W1; north_star "1-particle, 3-element line")
    w1 = [Drift(1.5), Multipole(knl=(0.0, 0.1, 0.5)), Drift(1.0)]
    out["lines"].append(worked_line("W1", ref_args, w1, start, "SURVEY.md §8(c) W1"))

    # W2: every element type
    th = 1e-3
    w2 = [Drift(1.5), XYShift(1e-4, -2e-4), SRotation.from_angle(th),
          Multipole(knl=(5e-3, 0.1, 0.5, 5.0), ksl=(0.0, 1e-3, -0.2, 1.0), hxl=5e-3, length=14.3),
          SRotation.from_angle(-th), XYShift(-1e-4, 2e-4), Cavity(1e6, 200e6, 180.0), Drift(1.0)]
    out["lines"].append(worked_line("W2", ref_args, w2, start, "SURVEY.md §8(c) W2"))

    # W3: one full turn of configs[0] (41 elements) for 3 seeded particles
    rng = np.random.default_rng(424242)
    cfg0 = configs.lattice_cfg0()
    for i in range(3):
        st = (rng.normal(0, 1e-4), rng.normal(0, 1e-5), rng.normal(0, 1e-4), rng.normal(0, 1e-5),
              rng.normal(0, 0.05), rng.normal(0, 1e-4))
        line = worked_line("W3_%d" % i, ref_args, cfg0, st, "BASELINE.json configs[0], one turn")
        line["stages"] = [line["stages"][0], line["stages"][-1]]   # keep only init and end of turn
        out["lines"].append(line)

    # P1: exact drift, 16 seeded particles incl. large angles and off-momentum
    ref = Ref(*ref_args)
    drift_cases = []
    for i in range(16):
        scale = 10.0 ** rng.uniform(-6, -1.5)
        st = (rng.normal(0, 1e-3), rng.normal(0, scale), rng.normal(0, 1e-3), rng.normal(0, scale),
              rng.normal(0, 0.1), rng.normal(0, 3e-3))
        L = float(rng.uniform(0.1, 100.0))
        p = init_particle(ref, *st)
        apply(ref, Drift(L), p)
        drift_cases.append({"start": [float(v).hex() for v in st], "length": L.hex(),
                            "values": snapshot(ref, p)})
    out["drift_cases"] = drift_cases

    # P6: multipole kicks by direct complex powers, orders 0..20, normal + skew
    mult_cases = []
    for order in range(21):
        knl = tuple(float(rng.normal(0, 1.0) * math.factorial(n) / 0.02 ** max(n - 1, 0) * 1e-3)
                    for n in range(order + 1))
        ksl = tuple(float(rng.normal(0, 1.0) * math.factorial(n) / 0.02 ** max(n - 1, 0) * 1e-3)
                    for n in range(order + 1))
        st = (rng.normal(0, 8e-3), rng.normal(0, 1e-4), rng.normal(0, 8e-3), rng.normal(0, 1e-4),
              rng.normal(0, 0.05), rng.normal(0, 1e-3))
        el = Multipole(knl=knl, ksl=ksl)
        p = init_particle(ref, *st)
        apply(ref, el, p)
        mult_cases.append({"start": [float(v).hex() for v in st], "element": el_json(el),
                           "values": snapshot(ref, p)})
    out["multipole_cases"] = mult_cases

    path = os.path.join(os.path.dirname(__file__), "worked_examples.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
