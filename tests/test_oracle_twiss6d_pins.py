"""Pin P24: the six-dimensional linear normal form of the oracle procedure (oracle/make_optics.py:
normal_form6, optics6d_along, Twiss steps 3-5: eigenvectors of the one-turn Jacobian,
their propagation by tracking, Mais-Ripken functions, dispersion from the eigenvectors).

  (a) a thin FODO ring with a cavity and no bends (pin P22's ring): the three modes are the three planes --
      beta_x1, alpha_x1 = the horizontal Courant-Snyder values of the 4-D procedure (pins P2 / P19),
      beta_y2, alpha_y2 the vertical ones, the cross terms vanish; the longitudinal mode of the kick-slip
      map [[1, A], [-B, 1 - A B]] has beta_z3 = A / sin mu_s, alpha_z3 = A B / (2 sin mu_s) in closed form;
  (b) the eigenvectors are symplectically normalised: v_k^H S v_k = 2i, v_j^H S v_k = 0, v_j^T S v_k = 0;
  (c) seen from a frame rotated by theta about s the transverse modes share the planes as cos^2 / sin^2
      (pin P20's closed form), the longitudinal mode does not change;
  (d) in the ring of thin quadrupoles and thin sector dipoles of pin P18 with a weak cavity the dispersion
      "from the eigenvectors" equals the periodic dispersion of the 3x3 matrices (closed form) up to the
      synchrotron-motion correction, at the start and along the line, and closes after one turn;
  (e) carried along the line (optics6d_along) the transverse modes of an uncoupled ring reproduce the 4-D
      beta functions row by row and the phases advance to 2 pi q_k.
"""
import math

import numpy as np

from oracle import make_optics as MO
from oracle import oracle as O
from xt_inputs.packed import Cavity, Drift, Multipole, SRotation, pack_lattice
import helpers as H

P0C_SMALL = 1.0e9


def pack(els, p0c=H.P0C):
    return pack_lattice(els, p0c, H.MASS0, H.Q0)


def fodo_with_cavity(volt=1e5, freq=200e6, lag=0.0):
    cell = [Multipole(knl=(0.0, 0.1)), Drift(2.0), Multipole(knl=(0.0, -0.095)), Drift(2.0)]
    return cell * 10 + [Cavity(volt, freq, lag)], cell * 10


def test_P24a_b_uncoupled_modes_are_the_planes_and_normalised():
    els, flat_els = fodo_with_cavity()
    buf = pack(els, P0C_SMALL)
    got = MO.optics6d_of(buf)
    nf = MO.normal_form6(got["m"])
    flat = MO.optics_of(pack(flat_els, P0C_SMALL))
    assert abs(nf["betx1"] / flat["betx"] - 1) < 1e-6 and abs(nf["bety2"] / flat["bety"] - 1) < 1e-6
    assert abs(nf["alfx1"] - flat["alfx"]) < 1e-6 and abs(nf["alfy2"] - flat["alfy"]) < 1e-6
    for k in ("bety1", "betz1", "betx2", "betz2", "betx3", "bety3"):
        assert nf[k] < 1e-9, (k, nf[k])
    assert abs(nf["q1_frac"] - flat["qx_frac"]) < 1e-8 and abs(nf["q2_frac"] - flat["qy_frac"]) < 1e-8
    # longitudinal mode of the slip-then-kick map (P11 / P22 notation): no bends, so the slip is A = C / gamma0^2
    beta0, gamma0 = O.reference(buf)
    kz = 2 * math.pi * 200e6 / (beta0 * 299792458.0)
    A, B = 40.0 / gamma0 ** 2, (1e5 / P0C_SMALL) * kz / beta0
    mu_s = math.acos(1.0 - A * B / 2.0)
    assert abs(nf["q3_frac"] - mu_s / (2 * math.pi)) < 1e-9 or abs(nf["q3_frac"] - (1 - mu_s / (2 * math.pi))) < 1e-9
    assert abs(nf["betz3"] / (A / math.sin(mu_s)) - 1.0) < 1e-6
    assert abs(abs(nf["alfz3"]) - A * B / (2 * math.sin(mu_s))) < 1e-6
    # (b) symplectic normalisation
    vs = [nf["v1"], nf["v2"], nf["v3"]]
    for j in range(3):
        for k in range(3):
            herm = np.conj(vs[j]) @ MO.S6 @ vs[k]
            plain = vs[j] @ MO.S6 @ vs[k]
            assert abs(herm - (2j if j == k else 0.0)) < 1e-6, (j, k, herm)
            assert abs(plain) < 1e-6, (j, k, plain)


def test_P24c_rotated_frame_shares():
    els, flat_els = fodo_with_cavity()
    flat = MO.optics_of(pack(flat_els, P0C_SMALL))
    base = MO.normal_form6(MO.optics6d_of(pack(els, P0C_SMALL))["m"])
    th = 0.3
    rot = [SRotation.from_angle(-th)] + els + [SRotation.from_angle(th)]
    nf = MO.normal_form6(MO.optics6d_of(pack(rot, P0C_SMALL))["m"])
    c2, s2 = math.cos(th) ** 2, math.sin(th) ** 2
    assert abs(nf["q1_frac"] - base["q1_frac"]) < 1e-8 and abs(nf["q2_frac"] - base["q2_frac"]) < 1e-8
    assert abs(nf["betx1"] - c2 * flat["betx"]) < 1e-5 and abs(nf["bety1"] - s2 * flat["betx"]) < 1e-5
    assert abs(nf["betx2"] - s2 * flat["bety"]) < 1e-5 and abs(nf["bety2"] - c2 * flat["bety"]) < 1e-5
    assert abs(nf["betz3"] / base["betz3"] - 1) < 1e-7 and abs(nf["q3_frac"] - base["q3_frac"]) < 1e-9


def dispersion_ring(n_cells=8, L=3.0, kq=0.25, ell=1.5):
    th = 2.0 * math.pi / (2 * n_cells)
    bend = Multipole(knl=(th,), hxl=th, length=ell)
    cell = [Multipole(knl=(0.0, kq)), Drift(L), bend, Drift(L), Multipole(knl=(0.0, -kq)), Drift(L), bend, Drift(L)]
    quad = lambda k: np.array([[1.0, 0.0, 0.0], [-k, 1.0, 0.0], [0.0, 0.0, 1.0]])
    drift = np.array([[1.0, L, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]])
    dip = np.array([[1.0, 0.0, 0.0], [-th * th / ell, 1.0, th], [0.0, 0.0, 1.0]])
    mats = [quad(kq), drift, dip, drift, quad(-kq), drift, dip, drift]
    return cell, mats, n_cells


def test_P24d_dispersion_from_the_longitudinal_eigenvector():
    cell, mats, n_cells = dispersion_ring()
    # above transition (alpha_c > 1/gamma0^2 at 450 GeV): the stable phase is 180 degrees; a weak cavity keeps the
    # synchrotron tune at ~1e-3, so the eigenvector dispersion differs from the static one at the 1e-5 level
    els = cell * n_cells + [Cavity(2e4, 50e6, 180.0)]
    on, rows = MO.optics6d_along(els, H.P0C, H.MASS0, H.Q0, list(range(9)) + [len(els)])
    assert 1e-5 < on["qs"] < 5e-3
    m = np.eye(3)
    for e in mats:
        m = e @ m
    d = np.append(np.linalg.solve(np.eye(2) - m[:2, :2], m[:2, 2]), 1.0)
    assert abs(on["dx"] / d[0] - 1.0) < 2e-4 and abs(on["dpx"] - d[1]) < 2e-4 * max(abs(d[1]), 0.1)
    assert abs(on["dy"]) < 1e-7 and abs(on["dpy"]) < 1e-7
    for i in range(9):
        assert abs(rows[i]["dx"] / d[0] - 1.0) < 3e-4 and abs(rows[i]["dpx"] - d[1]) < 3e-4 * max(abs(d[1]), 0.1), i
        if i < 8:
            d = mats[i] @ d
    assert abs(rows[-1]["dx"] - rows[0]["dx"]) < 1e-3 * abs(rows[0]["dx"])        # behind the cavity: one turn closed


def test_P24e_modes_carried_along_the_line():
    els, flat_els = fodo_with_cavity()
    rows_i = list(range(0, len(flat_els) + 1, 3))
    on4, rows4 = MO.optics_along(flat_els, P0C_SMALL, H.MASS0, H.Q0, rows_i)
    on6, rows6 = MO.optics6d_along(els, P0C_SMALL, H.MASS0, H.Q0, rows_i + [len(els)])
    for r4, r6 in zip(rows4, rows6):
        assert abs(r6["betx1"] / r4["betx"] - 1) < 2e-6 and abs(r6["bety2"] / r4["bety"] - 1) < 2e-6
        assert abs(r6["alfx1"] - r4["alfx"]) < 2e-6 and abs(r6["alfy2"] - r4["alfy"]) < 2e-6
        assert r6["bety1"] < 1e-9 and r6["betx2"] < 1e-9 and r6["betx3"] < 1e-9
        for a, b in ((r6["mu1"], r4["mux"]), (r6["mu2"], r4["muy"])):
            dd = (a - b) % (2 * math.pi)
            assert min(dd, 2 * math.pi - dd) < 2e-6
    end = rows6[-1]                                                                # one full turn: eigenvectors x exp(i mu)
    for k, key in ((1, "betx1"), (2, "bety2"), (3, "betz3")):
        assert abs(end[key] / on6[key] - 1) < 1e-6
        dd = (end["mu%d" % k] - 2 * math.pi * on6["q%d_frac" % k]) % (2 * math.pi)
        assert min(dd, 2 * math.pi - dd) < 1e-6
