"""Pins of the oracle's 'full' thick sector bend ("the bend can be 'full' or 'expanded'"; DESIGN.md
reading A23).  Pin P23.  The oracle evaluates a cancellation-free rearrangement of the textbook exact
sector-bend map; the pins do not retype it:

  (a) geometry: in a uniform field a charge moves on a helix.  In Cartesian coordinates of the bending plane
      the horizontal projection is a circle of radius p_h/k0 about a centre that follows from the entrance
      position and direction; the exit plane is the half line through the centre of curvature of the
      REFERENCE orbit at angle h L.  The crossing angle is found with a root finder in 40-digit arithmetic and
      x', px', y', zeta' follow from positions and path lengths -- no map formula involved;
  (b) the reference particle of a matched bend (k0 = h) is mapped to itself exactly, whatever the angle; an
      off-momentum particle starting on the axis lands where the two circles (radii 1/h and (1+delta)/k0) say;
  (c) for small amplitudes and a small bending angle the 'full' map tends to the 'expanded' map (reading A19):
      the difference falls by the factor 8 when amplitudes and angle are halved (third order);
  (d) it is symplectic (6x6 Jacobian in canonical variables) and reversible (reading A11);
  (e) bad parameters are rejected like those of the 'expanded' bend; an unknown model id is rejected.
"""
import math

import mpmath as mp
import numpy as np
import pytest

from oracle import oracle as O
from xt_inputs.packed import Bend, Cavity, Drift, Multipole, Quadrupole, pack_lattice
import helpers as H

P0C, MASS0 = 450e9, 938272088.16
mp.mp.dps = 40


def track_one(els, z, p0c=P0C, mass0=MASS0, turns=1):
    buf = pack_lattice(els, p0c, mass0, 1.0)
    p = O.new_particles(buf, H.coords_from_rows([z]))
    O.track(buf, p, turns)
    assert p["state"][0] == 1
    return {k: float(p[k][0]) for k in ("x", "px", "y", "py", "zeta", "delta", "ptau")}, buf


def helix(k0, h, length, z, beta0):
    """(x', px', y', zeta') of one particle through a uniform field k0, seen from the frame of curvature h."""
    x, px, y, py, zeta, delta = [mp.mpf(v) for v in z]
    k0, h, length, beta0 = mp.mpf(k0), mp.mpf(h), mp.mpf(length), mp.mpf(beta0)
    opd = 1 + delta
    ph = mp.sqrt(opd * opd - py * py)                     # momentum in the bending plane
    pz = mp.sqrt(ph * ph - px * px)
    rho0, theta, big_r = 1 / h, h * length, ph / k0
    # lab frame (X, Z): entrance plane Z = 0, reference orbit starts at the origin heading +Z and turns
    # counter-clockwise about (-rho0, 0); the particle starts at (x, 0) with momentum (px, pz)
    centre = mp.matrix([-rho0, 0])
    n0 = mp.matrix([-pz / ph, px / ph])                    # from the particle to its centre of gyration
    g = mp.matrix([x, 0]) + big_r * n0

    def rot(v, a):
        return mp.matrix([mp.cos(a) * v[0] - mp.sin(a) * v[1], mp.sin(a) * v[0] + mp.cos(a) * v[1]])

    s_hat = mp.matrix([-mp.sin(theta), mp.cos(theta)])     # normal of the exit plane
    x_hat = mp.matrix([mp.cos(theta), mp.sin(theta)])

    def miss(a):
        r = g - big_r * rot(n0, a)
        d = r - centre
        return d[0] * s_hat[0] + d[1] * s_hat[1]

    alpha = mp.findroot(miss, theta)
    r = g - big_r * rot(n0, alpha)
    d = r - centre
    mom = rot(mp.matrix([px, pz]), alpha)
    x1 = d[0] * x_hat[0] + d[1] * x_hat[1] - rho0
    px1 = mom[0] * x_hat[0] + mom[1] * x_hat[1]
    arc = big_r * alpha                                    # path length of the horizontal projection
    y1 = y + py / ph * arc
    path = opd / ph * arc
    # zeta = s - beta0 c t: the particle needs path/(beta c) for what the reference does in L/(beta0 c)
    gamma0 = 1 / mp.sqrt(1 - beta0 * beta0)
    p0 = beta0 * gamma0
    p = opd * p0
    beta = p / mp.sqrt(1 + p * p)
    zeta1 = zeta + length - beta0 / beta * path
    return x1, px1, y1, zeta1


CASES = [
    # k0, h, length, (x, px, y, py, zeta, delta), p0c
    (0.2, 0.2, 2.5, (3e-3, 2e-3, -2e-3, 1e-3, 0.01, 3e-3), 1e9),               # small ring, matched, 0.5 rad
    (0.2004, 0.2, 2.5, (-4e-3, -1e-3, 1e-3, -2e-3, -0.02, -5e-3), 1e9),        # mispowered
    (0.11, 0.1, 1.0, (1e-2, 5e-3, 5e-3, 5e-3, 0.0, 1e-2), 2e9),                 # large amplitudes, 10 % field error
    (2 * math.pi / 1232 / 14.3, 2 * math.pi / 1232 / 14.3, 14.3, (1e-3, 2e-5, -5e-4, 1e-5, 0.03, 3e-4), P0C),  # LHC-like
    (1.0, 1.0, 1.2, (1e-3, -3e-3, 2e-3, 1e-3, 0.0, -2e-3), 1e8),                # rho = 1 m, 69 degrees
]


@pytest.mark.parametrize("k0,h,length,z,p0c", CASES)
def test_full_bend_is_the_helix_cut_by_the_exit_plane(k0, h, length, z, p0c):
    got, buf = track_one([Bend(k0, h, length, 1)], z, p0c=p0c)
    beta0, _ = O.reference(buf)
    x1, px1, y1, zeta1 = helix(k0, h, length, z, mp.mpf(p0c) / mp.sqrt(mp.mpf(p0c) ** 2 + mp.mpf(MASS0) ** 2))
    assert abs(got["x"] - x1) <= 4e-16 * max(abs(x1), 1e-3) + 2e-19
    assert abs(got["px"] - px1) <= 4e-16 * max(abs(px1), 1e-3)
    assert abs(got["y"] - y1) <= 4e-16 * max(abs(y1), 1e-3)
    assert got["py"] == z[3] and got["delta"] == z[5]
    assert abs(got["zeta"] - zeta1) <= 4e-16 * max(abs(zeta1), 1e-2) + 1e-17
    assert abs(float(beta0) - float(mp.mpf(p0c) / mp.sqrt(mp.mpf(p0c) ** 2 + mp.mpf(MASS0) ** 2))) < 1e-15


def test_reference_particle_and_off_momentum_circle():
    for theta in (1e-3, 0.3, 1.0, 2.5):
        h = 0.4
        got, _ = track_one([Bend(h, h, theta / h, 1)], (0.0, 0.0, 0.0, 0.0, 0.0, 0.0), p0c=1e9)
        assert got["x"] == 0.0 and got["px"] == 0.0 and got["y"] == 0.0 and got["zeta"] == 0.0
    # off momentum, starting on the axis: circle of radius R = (1+delta)/k0 through the origin, tangent to +Z;
    # its crossing with the exit plane in closed form (law of cosines in the triangle of the two centres)
    h, theta, delta = 0.25, 0.6, 2e-2
    got, _ = track_one([Bend(h, h, theta / h, 1)], (0.0, 0.0, 0.0, 0.0, 0.0, delta), p0c=1e9)
    rho0, big_r = mp.mpf(1) / mp.mpf(h), (1 + mp.mpf(delta)) / mp.mpf(h)
    dcc = big_r - rho0                                     # distance of the two centres, along -X
    # point at distance lam from the reference centre on the exit ray, at distance R from the other centre:
    # lam^2 + 2 lam dcc cos(theta) + dcc^2 = R^2
    ct = mp.cos(mp.mpf(theta))
    lam = -dcc * ct + mp.sqrt(dcc * dcc * ct * ct - dcc * dcc + big_r * big_r)
    assert abs(got["x"] - float(lam - rho0)) < 1e-15
    assert got["x"] > 0.0 and got["px"] > 0.0              # dispersion: the stiffer particle drifts outwards


def test_full_tends_to_expanded_at_third_order():
    def diff(scale):
        z = (2e-3 * scale, 1e-3 * scale, -1e-3 * scale, 2e-3 * scale, 0.0, 4e-3 * scale)
        h = 0.05 * scale
        a, _ = track_one([Bend(h * 1.001, h, 1.0, 1)], z, p0c=1e9)
        b, _ = track_one([Bend(h * 1.001, h, 1.0, 0)], z, p0c=1e9)
        return max(abs(a[k] - b[k]) for k in ("x", "px", "y")), abs(a["zeta"] - b["zeta"])
    d1, z1 = diff(1.0)
    d2, z2 = diff(0.5)
    assert 1e-12 < d2 < d1 < 1e-6
    assert 6.0 < d1 / d2 < 11.0                            # third order in (amplitude, angle)
    assert z2 < z1 < 1e-6


def ring():
    return [Bend(0.2, 0.2, 1.5, 1), Drift(0.7), Quadrupole(0.6, 0.4), Drift(0.5), Bend(0.2006, 0.2, 1.5, 1),
            Multipole(knl=(0.0, 0.0, 0.3)), Drift(0.9), Quadrupole(-0.55, 0.4), Cavity(2e4, 50e6, 10.0), Drift(0.3)]


def test_full_bend_line_is_symplectic_and_reversible():
    els = ring()
    buf = pack_lattice(els, 1e9, MASS0, 1.0)
    z0 = (1e-3, 5e-4, -8e-4, 3e-4, 0.01, 1e-3)
    J = H.jacobian6(lambda b, p, n: O.track(b, p, n), buf, z0)
    assert abs(np.linalg.det(J) - 1.0) < 2e-7
    assert np.max(np.abs(J.T @ H.S6 @ J - H.S6)) < 2e-7
    # reversibility (reading A11): forward, flip, backward through the reversed line, flip
    rng = np.random.default_rng(5)
    rows = rng.normal(0, 1, (50, 6)) * np.array([2e-3, 1e-3, 2e-3, 1e-3, 0.02, 2e-3])
    p = O.new_particles(buf, H.coords_from_rows(rows))
    start = {k: p[k].copy() for k in ("x", "px", "y", "py", "zeta", "delta")}
    O.track(buf, p, 1)
    H.flip_R(p)
    back = pack_lattice(H.reversed_lattice(els), 1e9, MASS0, 1.0)
    p["at_turn"][:] = 0
    O.track(back, p, 1)
    H.flip_R(p)
    for k in start:
        assert np.max(np.abs(p[k] - start[k])) <= 1e-13 * max(1e-3, np.max(np.abs(start[k]))), k


def test_bad_full_bends_are_rejected():
    for bad in (Bend(0.1, -0.1, 1.0, 1), Bend(0.0, 0.1, 1.0, 1), Bend(0.1, 0.1, 0.0, 1), Bend(0.1, 0.1, 1.0, 2)):
        buf = pack_lattice([bad], P0C, MASS0, 1.0)
        with pytest.raises(Exception):
            O.new_particles(buf, H.coords_from_rows([[0.0] * 6]))
