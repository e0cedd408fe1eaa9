#!/usr/bin/env python
"""Writes xt_inputs/optics.json: start-point optics of the LHC-sized synthetic lattices.

TEST/INPUT INFRASTRUCTURE; calls only ``oracle/`` (never the CUDA path).  Follows the paper's
Twiss procedure, PAPER.md:96-98 ("Twiss module"):
  1. closed orbit = fixed point of the one-turn map (Newton on the 4-D transverse map at
     zeta = delta = 0),
  2. one-turn Jacobian by central differences of tracked particles,
  3. (uncoupled approximation of the normal form) per plane
     cos mu = (M11+M22)/2, beta = M12/sin mu, alpha = (M11-M22)/(2 sin mu).
The values only shape the synthetic *inputs* (matched Gaussian / amplitude grids of
configs[2..4]); they are not expected values of any parity test.

Run:  python oracle/make_optics.py
"""
import json
import math
import os
import sys

import numpy as np

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), ".."))
from oracle import oracle as O  # noqa: E402
from xt_inputs import configs as C  # noqa: E402


def one_turn(buf, z4):
    co = dict(x=np.array([z4[0]]), px=np.array([z4[1]]), y=np.array([z4[2]]), py=np.array([z4[3]]),
              zeta=np.zeros(1), delta=np.zeros(1))
    p = O.new_particles(buf, co)
    O.track(buf, p, 1)
    assert p["state"][0] == 1
    return np.array([p["x"][0], p["px"][0], p["y"][0], p["py"][0]])


def jac4(buf, z4, h=(1e-6, 1e-8, 1e-6, 1e-8)):
    n = 8
    pts = np.tile(np.asarray(z4, dtype=np.float64), (n, 1))
    for i in range(4):
        pts[2 * i, i] += h[i]
        pts[2 * i + 1, i] -= h[i]
    co = dict(x=pts[:, 0].copy(), px=pts[:, 1].copy(), y=pts[:, 2].copy(), py=pts[:, 3].copy(),
              zeta=np.zeros(n), delta=np.zeros(n))
    p = O.new_particles(buf, co)
    O.track(buf, p, 1)
    assert np.all(p["state"] == 1)
    out = np.stack([p["x"], p["px"], p["y"], p["py"]], axis=1)
    J = np.zeros((4, 4))
    for i in range(4):
        J[:, i] = (out[2 * i] - out[2 * i + 1]) / (2 * h[i])
    return J


def optics_of(buf):
    z = np.zeros(4)
    for _ in range(12):                                   # Twiss step 1: closed orbit
        J = jac4(buf, z)
        r = one_turn(buf, z) - z
        dz = np.linalg.solve(J - np.eye(4), -r)
        z = z + dz
        if np.max(np.abs(dz)) < 1e-13:
            break
    J = jac4(buf, z)                                      # Twiss step 2
    out = {"x_co": z[0], "px_co": z[1], "y_co": z[2], "py_co": z[3]}
    for name, i in (("x", 0), ("y", 2)):                  # Twiss step 3 (uncoupled)
        m = J[i:i + 2, i:i + 2]
        cosmu = 0.5 * (m[0, 0] + m[1, 1])
        assert abs(cosmu) < 1.0, "unstable plane %s: cos mu = %g" % (name, cosmu)
        sinmu = math.copysign(math.sqrt(1.0 - cosmu * cosmu), m[0, 1])
        out["bet" + name] = m[0, 1] / sinmu
        out["alf" + name] = (m[0, 0] - m[1, 1]) / (2.0 * sinmu)
        mu = math.atan2(sinmu, cosmu)
        out["q" + name + "_frac"] = (mu / (2 * math.pi)) % 1.0
    return out


def main():
    res = {"_about": "written by oracle/make_optics.py (oracle one-turn Jacobian at the 4-D closed "
                     "orbit, PAPER.md:96-98); input shaping only"}
    for cfg in (2, 3, 4):
        buf = C.pack(C.lattice(cfg))
        res["cfg%d" % cfg] = optics_of(buf)
        print(cfg, res["cfg%d" % cfg])
    path = os.path.join(os.path.dirname(os.path.abspath(C.__file__)), "optics.json")
    with open(path, "w") as fh:
        json.dump(res, fh, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
