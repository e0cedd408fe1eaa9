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


def one_turn(buf, z4, delta=0.0):
    co = dict(x=np.array([z4[0]]), px=np.array([z4[1]]), y=np.array([z4[2]]), py=np.array([z4[3]]),
              zeta=np.zeros(1), delta=np.full(1, delta))
    p = O.new_particles(buf, co)
    O.track(buf, p, 1)
    assert p["state"][0] == 1
    return np.array([p["x"][0], p["px"][0], p["y"][0], p["py"][0]])


def jac4(buf, z4, h=(1e-6, 1e-8, 1e-6, 1e-8), delta=0.0):
    n = 8
    pts = np.tile(np.asarray(z4, dtype=np.float64), (n, 1))
    for i in range(4):
        pts[2 * i, i] += h[i]
        pts[2 * i + 1, i] -= h[i]
    co = dict(x=pts[:, 0].copy(), px=pts[:, 1].copy(), y=pts[:, 2].copy(), py=pts[:, 3].copy(),
              zeta=np.zeros(n), delta=np.full(n, delta))
    p = O.new_particles(buf, co)
    O.track(buf, p, 1)
    assert np.all(p["state"] == 1)
    out = np.stack([p["x"], p["px"], p["y"], p["py"]], axis=1)
    J = np.zeros((4, 4))
    for i in range(4):
        J[:, i] = (out[2 * i] - out[2 * i + 1]) / (2 * h[i])
    return J


def optics_of(buf, delta=0.0, guess=None):
    z = np.zeros(4) if guess is None else np.asarray(guess, dtype=np.float64).copy()
    for _ in range(12):                                   # Twiss step 1: closed orbit
        J = jac4(buf, z, delta=delta)
        r = one_turn(buf, z, delta) - z
        dz = np.linalg.solve(J - np.eye(4), -r)
        z = z + dz
        if np.max(np.abs(dz)) < 1e-13:
            break
    J = jac4(buf, z, delta=delta)                         # Twiss step 2
    out = {"x_co": z[0], "px_co": z[1], "y_co": z[2], "py_co": z[3], "m": J}
    for name, i in (("x", 0), ("y", 2)):                  # Twiss step 3 (uncoupled)
        m = J[i:i + 2, i:i + 2]
        cosmu = 0.5 * (m[0, 0] + m[1, 1])
        if not abs(cosmu) < 1.0:                          # no uncoupled reading of this plane (coupled or unstable)
            out["bet" + name] = out["alf" + name] = out["q" + name + "_frac"] = float("nan")
            continue
        sinmu = math.copysign(math.sqrt(1.0 - cosmu * cosmu), m[0, 1])
        out["bet" + name] = m[0, 1] / sinmu
        out["alf" + name] = (m[0, 0] - m[1, 1]) / (2.0 * sinmu)
        mu = math.atan2(sinmu, cosmu)
        out["q" + name + "_frac"] = (mu / (2 * math.pi)) % 1.0
    return out


H6 = (1e-6, 1e-8, 1e-6, 1e-8, 1e-5, 1e-8)


def track6(buf, pts):
    """One turn of the rows (x, px, y, py, zeta, delta) of ``pts``."""
    pts = np.atleast_2d(np.asarray(pts, dtype=np.float64))
    p = O.new_particles(buf, dict(x=pts[:, 0].copy(), px=pts[:, 1].copy(), y=pts[:, 2].copy(), py=pts[:, 3].copy(),
                                  zeta=pts[:, 4].copy(), delta=pts[:, 5].copy()))
    O.track(buf, p, 1)
    assert np.all(p["state"] == 1)
    return np.stack([p["x"], p["px"], p["y"], p["py"], p["zeta"], p["delta"]], axis=1)


def jac6(buf, z, h=H6):
    pts = np.tile(np.asarray(z, dtype=np.float64), (12, 1))
    for i in range(6):
        pts[2 * i, i] += h[i]
        pts[2 * i + 1, i] -= h[i]
    out = track6(buf, pts)
    J = np.zeros((6, 6))
    for i in range(6):
        J[:, i] = (out[2 * i] - out[2 * i + 1]) / (2 * h[i])
    return J


def optics6d_of(buf, guess=None):
    """The paper's steps 1-3 in all six dimensions (a ring with an RF cavity): closed orbit
    by Newton on (x, px, y, py, zeta, delta), the 6x6 Jacobian there by central differences, and the three
    tunes from its eigenvalues exp(+-i mu_k): the synchrotron tune qs is the smallest angle (reported in
    (0, 1/2)); of the other two, q1 is the one whose cos mu is closer to that of the horizontal 2x2 block;
    their side of the half integer is read from the sign of that block's M12, as in ``optics_of``."""
    z = np.zeros(6) if guess is None else np.asarray(guess, dtype=np.float64).copy()
    for _ in range(20):
        J = jac6(buf, z)
        r = track6(buf, z)[0] - z
        dz = np.linalg.solve(J - np.eye(6), -r)
        z = z + dz
        if np.max(np.abs(dz)) < 1e-12:
            break
    J = jac6(buf, z)
    lam = np.linalg.eigvals(J)
    assert np.all(np.abs(np.abs(lam) - 1.0) < 1e-5), "unstable"
    ang = sorted(set(round(abs(math.atan2(l.imag, l.real)), 9) for l in lam))
    assert len(ang) == 3
    out = {"co": z, "m": J, "qs": ang[0] / (2 * math.pi)}
    rest = ang[1:]
    cx = 0.5 * (J[0, 0] + J[1, 1])
    if abs(math.cos(rest[0]) - cx) > abs(math.cos(rest[1]) - cx):
        rest = rest[::-1]
    for name, a, i in (("q1_frac", rest[0], 0), ("q2_frac", rest[1], 2)):
        out[name] = (math.copysign(a, J[i, i + 1]) / (2 * math.pi)) % 1.0
    return out


S4 = np.array([[0.0, 1.0, 0.0, 0.0], [-1.0, 0.0, 0.0, 0.0], [0.0, 0.0, 0.0, 1.0], [0.0, 0.0, -1.0, 0.0]])


def normal_form4(J):
    """Twiss step 3 in full ("Linear Normal Form of the map from the eigenvalues and eigenvectors
    of the Jacobian matrix"; step 5 "Mais-Ripken"): the two normal modes of the 4x4 one-turn matrix.
    numpy.linalg.eig gives eigenvalues exp(+-i mu_k) and eigenvectors; of each conjugate pair the one with
    v^H S v = +2i after scaling (positive symplectic norm) is kept -- in one uncoupled plane that is
    v = (sqrt(beta), (i - alpha)/sqrt(beta)) with eigenvalue exp(+i mu); mode 1 is the one with the larger
    horizontal part.  Mais-Ripken functions of mode k in plane u: beta_uk = |v_u|^2,
    alpha_uk = -Re(conj(v_u) v_pu).  Returns None if an eigenvalue is off the unit circle."""
    lam, vec = np.linalg.eig(np.asarray(J, dtype=np.float64))
    modes = []
    for k in range(4):
        if abs(abs(lam[k]) - 1.0) > 1e-6 or abs(lam[k].imag) < 1e-12:
            return None
        v = vec[:, k]
        norm = (np.conj(v) @ S4 @ v).imag / 2.0
        if norm > 0.0:
            modes.append((lam[k], v / math.sqrt(norm)))
    if len(modes) != 2:
        return None
    modes.sort(key=lambda m: -abs(m[1][0]) ** 2)
    out = {}
    for k, (lmb, v) in enumerate(modes, start=1):
        ref = v[0] if k == 1 else v[2]                     # phase origin: the mode's own plane is real positive
        v = v * (abs(ref) / ref)
        out["q%d_frac" % k] = (math.atan2(lmb.imag, lmb.real) / (2 * math.pi)) % 1.0
        out["v%d" % k] = v
        for name, i in (("x", 0), ("y", 2)):
            out["bet%s%d" % (name, k)] = abs(v[i]) ** 2
            out["alf%s%d" % (name, k)] = -(np.conj(v[i]) * v[i + 1]).real
    return out


S6 = np.zeros((6, 6))
for _k in range(3):
    S6[2 * _k, 2 * _k + 1], S6[2 * _k + 1, 2 * _k] = 1.0, -1.0


def normal_form6(J, rvv_co=1.0):
    """Twiss steps 3 and 5 in six dimensions ("Linear Normal Form of the map from the
    eigenvalues and eigenvectors of the Jacobian matrix", "Mais-Ripken").  J is the one-turn matrix in
    (x, px, y, py, zeta, delta) as ``jac6`` gives it; rvv_co = beta/beta0 on the closed orbit turns it into
    the canonical variables (..., zeta, pzeta = ptau/beta0): d pzeta = rvv d delta (dE = beta c dP).
    numpy.linalg.eig; of each conjugate pair the eigenvector with v^H S v = +2i after scaling is kept; the
    longitudinal mode (3) is the one with the smallest tune angle, of the other two mode 1 is the one with
    the larger horizontal part; phase origin: the mode's own plane (x, y, zeta) real positive.
    Mais-Ripken functions of mode k in plane u (x, y, zeta): beta_uk = |v_u|^2, alpha_uk = -Re(conj(v_u) v_pu).
    Dispersion "from the eigenvectors" (step 5): the transverse part of the longitudinal mode per unit of its
    momentum part, D_u = Re(v_u / v_pzeta) per pzeta, x rvv_co per delta.  Returns None if an eigenvalue is off
    the unit circle or real."""
    t = np.diag([1.0, 1.0, 1.0, 1.0, 1.0, rvv_co])
    jc = t @ np.asarray(J, dtype=np.float64) @ np.linalg.inv(t)
    lam, vec = np.linalg.eig(jc)
    modes = []
    for k in range(6):
        if abs(abs(lam[k]) - 1.0) > 1e-5 or abs(lam[k].imag) < 1e-12:
            return None
        v = vec[:, k]
        norm = (np.conj(v) @ S6 @ v).imag / 2.0
        if norm > 0.0:
            modes.append((lam[k], v / math.sqrt(norm)))
    if len(modes) != 3:
        return None
    modes.sort(key=lambda m: abs(math.atan2(m[0].imag, m[0].real)))
    longitudinal, rest = modes[0], modes[1:]
    rest.sort(key=lambda m: -abs(m[1][0]) ** 2)
    out = {}
    for k, (lmb, v) in enumerate(rest + [longitudinal], start=1):
        ref = v[2 * (k - 1)]
        v = v * (abs(ref) / ref)
        out["q%d_frac" % k] = (math.atan2(lmb.imag, lmb.real) / (2 * math.pi)) % 1.0
        out["v%d" % k] = v
        for name, i in (("x", 0), ("y", 2), ("z", 4)):
            out["bet%s%d" % (name, k)] = abs(v[i]) ** 2
            out["alf%s%d" % (name, k)] = -(np.conj(v[i]) * v[i + 1]).real
    v3 = out["v3"]
    for name, i in (("dx", 0), ("dpx", 1), ("dy", 2), ("dpy", 3)):
        out[name] = (v3[i] / v3[5]).real * rvv_co
    return out


def optics6d_along(elements, p0c, mass0, q0, rows, guess=None):
    """The six-dimensional optics carried along the line (steps 4-5: the eigenvectors are
    propagated "to all other elements by tracking").  For every requested row i (the entrance of element i):
    the 6x6 Jacobian J_i of the map from the start to row i by central differences around the 6-D closed
    orbit (steps of ``jac6``), in canonical variables at both ends (rvv at the start and at the row), and the
    three eigenvectors v_k(i) = J_i v_k(0): beta_uk = |v_u|^2, alpha_uk, the mode phases
    mu_k = arg of the mode's own component (mod 2 pi), and the dispersion of the longitudinal mode.  Each row
    is tracked through its own prefix line."""
    from xt_inputs import packed as PK
    buf = PK.pack_lattice(elements, p0c, mass0, q0)
    on = optics6d_of(buf, guess)
    z0 = on["co"]
    beta0, _ = O.reference(buf)

    def rvv_of(delta, ptau):
        return (1.0 + delta) / (1.0 + beta0 * ptau)

    def ptau_of(delta):
        tt = delta * (delta + 2.0)
        return tt / (math.sqrt(tt + 1.0 / beta0 ** 2) + 1.0 / beta0)

    rvv0 = rvv_of(z0[5], ptau_of(z0[5]))
    nf = normal_form6(on["m"], rvv0)
    assert nf is not None
    on.update(nf)
    pts = np.tile(z0, (13, 1))
    for i in range(6):
        pts[1 + 2 * i, i] += H6[i]
        pts[2 + 2 * i, i] -= H6[i]
    out = []
    for row in rows:
        prefix = PK.pack_lattice(list(elements[:row]) or [PK.Marker()], p0c, mass0, q0)
        p = O.new_particles(prefix, dict(x=pts[:, 0].copy(), px=pts[:, 1].copy(), y=pts[:, 2].copy(),
                                         py=pts[:, 3].copy(), zeta=pts[:, 4].copy(), delta=pts[:, 5].copy()))
        O.track(prefix, p, 1)
        assert np.all(p["state"] == 1)
        z = np.stack([p["x"], p["px"], p["y"], p["py"], p["zeta"], p["delta"]], axis=1)
        J = np.zeros((6, 6))
        for i in range(6):
            J[:, i] = (z[1 + 2 * i] - z[2 + 2 * i]) / (2 * H6[i])
        rvv1 = rvv_of(p["delta"][0], p["ptau"][0])
        jc = np.diag([1, 1, 1, 1, 1, rvv1]) @ J @ np.diag([1, 1, 1, 1, 1, 1.0 / rvv0])
        r = {"co": z[0].copy()}
        for k in (1, 2, 3):
            v = jc @ nf["v%d" % k]
            for name, i in (("x", 0), ("y", 2), ("z", 4)):
                r["bet%s%d" % (name, k)] = abs(v[i]) ** 2
                r["alf%s%d" % (name, k)] = -(np.conj(v[i]) * v[i + 1]).real
            own = v[2 * (k - 1)]
            r["mu%d" % k] = math.atan2(own.imag, own.real) % (2 * math.pi)
            if k == 3:
                for name, i in (("dx", 0), ("dpx", 1), ("dy", 2), ("dpy", 3)):
                    r[name] = (v[i] / v[5]).real * rvv1
        out.append(r)
    return on, out


def chromatic_optics_of(buf, ddelta=1e-4, delta=0.0):
    """Dispersion and chromaticity at the start of the line (the optics "as a function of the
    momentum"): central differences in delta of the closed orbit and of the tunes, each from the three steps
    above at delta -+ ddelta."""
    on = optics_of(buf, delta)
    z0 = [on["x_co"], on["px_co"], on["y_co"], on["py_co"]]
    hi, lo = optics_of(buf, delta + ddelta, z0), optics_of(buf, delta - ddelta, z0)
    out = dict(on)
    for name, key in (("dx", "x_co"), ("dpx", "px_co"), ("dy", "y_co"), ("dpy", "py_co")):
        out[name] = (hi[key] - lo[key]) / (2.0 * ddelta)
    for name, key in (("dqx", "qx_frac"), ("dqy", "qy_frac")):
        d = hi[key] - lo[key]
        d -= round(d)                                      # fractional tunes: the difference is taken on the circle
        out[name] = d / (2.0 * ddelta)
    return out


def optics_along(elements, p0c, mass0, q0, rows, ddelta=1e-4, delta=0.0):
    """Twiss along the line (the optics is propagated from the start "to all other elements
    by tracking"; beta functions along the ring).  For every requested row i (the ENTRANCE of
    element i; i = len(elements) is the end of the line): the closed orbit, the 4x4 Jacobian J_i of the map
    from the start to row i by central differences around the closed orbit (same steps as ``jac4``), then per
    plane with m = the plane's 2x2 block of J_i and (beta0, alpha0, gamma0) at the start:
        beta_i  = m11^2 beta0 - 2 m11 m12 alpha0 + m12^2 gamma0
        alpha_i = -m11 m21 beta0 + (m11 m22 + m12 m21) alpha0 - m12 m22 gamma0
        mu_i    = atan2(m12, m11 beta0 - m12 alpha0)   (mod 2 pi; the caller unwraps)
    and the dispersion as the central difference of the closed orbits at delta -+ ddelta tracked to row i.
    Each row is tracked through its own prefix line elements[:i] -- slow and obviously element i's entrance."""
    from xt_inputs import packed as PK
    buf = PK.pack_lattice(elements, p0c, mass0, q0)
    on = optics_of(buf, delta)
    z0 = np.array([on["x_co"], on["px_co"], on["y_co"], on["py_co"]])
    hi, lo = optics_of(buf, delta + ddelta, z0), optics_of(buf, delta - ddelta, z0)
    zh = np.array([hi["x_co"], hi["px_co"], hi["y_co"], hi["py_co"]])
    zl = np.array([lo["x_co"], lo["px_co"], lo["y_co"], lo["py_co"]])
    h = (1e-6, 1e-8, 1e-6, 1e-8)
    pts = np.tile(z0, (11, 1))
    for i in range(4):
        pts[1 + 2 * i, i] += h[i]
        pts[2 + 2 * i, i] -= h[i]
    pts[9], pts[10] = zh, zl
    deltas = np.full(11, delta)
    deltas[9], deltas[10] = delta + ddelta, delta - ddelta
    nf = normal_form4(on["m"])
    if nf is not None:
        on.update({k: v for k, v in nf.items()})
    out = []
    for row in rows:
        prefix = PK.pack_lattice(list(elements[:row]) or [PK.Marker()], p0c, mass0, q0)
        p = O.new_particles(prefix, dict(x=pts[:, 0].copy(), px=pts[:, 1].copy(), y=pts[:, 2].copy(),
                                         py=pts[:, 3].copy(), zeta=np.zeros(11), delta=deltas.copy()))
        O.track(prefix, p, 1)
        assert np.all(p["state"] == 1)
        z = np.stack([p["x"], p["px"], p["y"], p["py"]], axis=1)
        J = np.zeros((4, 4))
        for i in range(4):
            J[:, i] = (z[1 + 2 * i] - z[2 + 2 * i]) / (2 * h[i])
        r = {"x": z[0, 0], "px": z[0, 1], "y": z[0, 2], "py": z[0, 3]}
        for name, i in (("x", 0), ("y", 2)):
            m = J[i:i + 2, i:i + 2]
            b0, a0 = on["bet" + name], on["alf" + name]
            g0 = (1.0 + a0 * a0) / b0
            r["bet" + name] = m[0, 0] ** 2 * b0 - 2.0 * m[0, 0] * m[0, 1] * a0 + m[0, 1] ** 2 * g0
            r["alf" + name] = -m[0, 0] * m[1, 0] * b0 + (m[0, 0] * m[1, 1] + m[0, 1] * m[1, 0]) * a0 - m[0, 1] * m[1, 1] * g0
            r["mu" + name] = math.atan2(m[0, 1], m[0, 0] * b0 - m[0, 1] * a0) % (2 * math.pi)
        d = (z[9] - z[10]) / (2.0 * ddelta)
        r["dx"], r["dpx"], r["dy"], r["dpy"] = d
        if nf is not None:                                 # steps 4-5: the eigenvectors carried by the tracked Jacobian
            for k in (1, 2):
                v = J @ nf["v%d" % k]
                r["betx%d" % k], r["bety%d" % k] = abs(v[0]) ** 2, abs(v[2]) ** 2
                own = v[0] if k == 1 else v[2]
                r["mu%d" % k] = math.atan2(own.imag, own.real) % (2 * math.pi)
        out.append(r)
    return on, out


def main():
    res = {"_about": "written by oracle/make_optics.py (oracle one-turn Jacobian at the 4-D closed "
                     "orbit, PAPER.md:96-98); input shaping only"}
    for cfg in (2, 3, 4):
        buf = C.pack(C.lattice(cfg))
        res["cfg%d" % cfg] = {k: float(v) for k, v in optics_of(buf).items() if k != "m"}
        print(cfg, res["cfg%d" % cfg])
    path = os.path.join(os.path.dirname(os.path.abspath(C.__file__)), "optics.json")
    with open(path, "w") as fh:
        json.dump(res, fh, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
