"""Twiss from tracking on the GPU path against
(a) the thin-FODO closed form of pin P2 and (b) the same three steps run on the oracle
(``oracle/make_optics.py``: Newton closed orbit, central-difference Jacobian, uncoupled optics).

Both sides use the same finite-difference steps, so they differ only by the tracking
arithmetic (FMA fusion) amplified by 1/(2h): the closed orbit agrees to 1e-12 m, the matrix
to 1e-7, tunes to 1e-8 -- the accuracy central differences give, far above the 1e-12 parity
bar of the tracking itself.
"""
import math

import numpy as np
import pytest

from oracle import make_optics as MO
from xt_inputs import configs as C
from xt_inputs.packed import Drift, LimitEllipse, Multipole, pack_lattice

pytestmark = pytest.mark.gpu

P0C, MASS0 = 450e9, 938272088.16


@pytest.fixture(scope="module")
def X():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m gpu on the B200 box)")
    import paper_2310_00317_b200 as X
    return X


def test_twiss_fodo_closed_form(X):
    """config[0] without its cavity: ten thin FODO cells, textbook values (pin P2)."""
    cell = [Multipole(knl=(0.0, 0.1)), Drift(2.0), Multipole(knl=(0.0, -0.1)), Drift(2.0)]
    lat = X.xt_lattice_create(pack_lattice(cell * 10, P0C, MASS0, 1.0))
    tw = X.xt_twiss4d(lat)
    lat.close()
    assert tw["stable"] == 1 and tw["iterations"] <= 3
    assert np.max(np.abs(tw["co"])) < 1e-15                       # the origin is the closed orbit
    mu_cell = math.acos(1.0 - 2.0 ** 2 / (2.0 * 10.0 ** 2))       # cos mu = 1 - L^2/(2 f^2), reading A15
    tune = 10 * mu_cell / (2 * math.pi)
    assert abs(tune - 0.31884280429259924) < 1e-15
    assert abs(tw["qx_frac"] - tune) < 1e-8 and abs(tw["qy_frac"] - tune) < 1e-8
    assert abs(tw["betx"] - 22.110831935702666) < 1e-6 and abs(tw["alfx"] + 1.1055415967851333) < 1e-7
    assert abs(tw["bety"] - 18.090680674665817) < 1e-6 and abs(tw["alfy"] - 0.90453403373329087) < 1e-7
    np.testing.assert_allclose(tw["m"][0:2, 0:2], [[-1.4229092060125620, 20.074399908620036],
                                                   [-0.091247272311909253, 0.58453078484944159]], atol=1e-7)
    assert np.max(np.abs(tw["m"][0:2, 2:4])) < 1e-8               # upright quads: no coupling
    assert abs(np.linalg.det(tw["m"]) - 1.0) < 1e-7               # symplectic map


@pytest.mark.parametrize("cfg", [0, 2, 3])
def test_twiss_matches_the_oracle_procedure(X, cfg):
    buf = C.pack(C.lattice(cfg))
    want = MO.optics_of(buf)
    lat = X.xt_lattice_create(buf)
    tw = X.xt_twiss4d(lat)
    lat.close()
    assert tw["stable"] == 1 and tw["iterations"] <= 8
    np.testing.assert_allclose(tw["co"], [want["x_co"], want["px_co"], want["y_co"], want["py_co"]], atol=1e-12)
    for k in ("betx", "bety"):
        assert abs(tw[k] / want[k] - 1.0) < 1e-7, k
    for k in ("alfx", "alfy"):
        assert abs(tw[k] - want[k]) < 1e-6, k
    for k in ("qx_frac", "qy_frac"):
        assert abs(tw[k] - want[k]) < 1e-8, k
    if cfg >= 2:                                                   # what shaped the matched ensembles
        ref = C.load_optics()["cfg%d" % cfg]
        assert abs(tw["betx"] / ref["betx"] - 1.0) < 1e-6 and abs(tw["qy_frac"] - ref["qy_frac"]) < 1e-7


def test_twiss_off_momentum_and_errors(X):
    """Off-momentum closed orbit of the LHC-sized ring moves with dispersion; a guess far inside
    the aperture still converges; an orbit outside the aperture is reported, not returned."""
    buf = C.pack(C.lattice(2))
    lat = X.xt_lattice_create(buf)
    on = X.xt_twiss4d(lat, 0.0)
    off = X.xt_twiss4d(lat, 1e-4, guess4=on["co"])
    dx = (off["co"][0] - on["co"][0]) / 1e-4                       # dispersion at the start point [m]
    assert 0.1 < abs(dx) < 10.0 and off["stable"] == 1
    again = X.xt_twiss4d(lat, 0.0, guess4=[1e-3, 0.0, -1e-3, 0.0])
    np.testing.assert_allclose(again["co"], on["co"], atol=1e-11)
    with pytest.raises(X.XtError) as e:
        X.xt_twiss4d(lat, 0.0, guess4=[0.5, 0.0, 0.0, 0.0])       # 0.5 m: outside the 20 mm ellipse
    assert e.value.code == -5
    lat.close()
    # an unstable plane is flagged, not an error: two focusing quads in a row
    bad = [Multipole(knl=(0.0, 0.9)), Drift(2.0), Multipole(knl=(0.0, 0.9)), Drift(2.0)]
    lat = X.xt_lattice_create(pack_lattice(bad, P0C, MASS0, 1.0))
    tw = X.xt_twiss4d(lat)
    assert tw["stable"] == 0 and (math.isnan(tw["bety"]) or math.isnan(tw["betx"]))
    lat.close()


def test_dispersion_and_chromaticity(X):
    """xt_twiss4d_chrom against closed forms (pin P18: thin-FODO natural chromaticity; periodic dispersion of a
    ring of thin quadrupoles and thin sector dipoles from 3x3 matrices) and against the oracle procedure
    on the LHC-sized ring."""
    n_cells, L, kq = 10, 2.0, 0.1
    cell = [Multipole(knl=(0.0, kq)), Drift(L), Multipole(knl=(0.0, -kq)), Drift(L)]
    lat = X.xt_lattice_create(pack_lattice(cell * n_cells, P0C, MASS0, 1.0))
    tw = X.xt_twiss4d_chrom(lat)
    lat.close()
    mu = math.acos(1.0 - (L * kq) ** 2 / 2.0)
    want = -n_cells * math.tan(mu / 2.0) / math.pi
    assert abs(tw["dqx"] - want) < 1e-5 * abs(want) and abs(tw["dqy"] - want) < 1e-5 * abs(want)
    assert max(abs(tw[k]) for k in ("dx", "dpx", "dy", "dpy")) < 1e-9

    n_cells, L, kq, ell = 8, 3.0, 0.25, 1.5
    th = 2.0 * math.pi / (2 * n_cells)
    bend = Multipole(knl=(th,), hxl=th, length=ell)
    cell = [Multipole(knl=(0.0, kq)), Drift(L), bend, Drift(L), Multipole(knl=(0.0, -kq)), Drift(L), bend, Drift(L)]
    lat = X.xt_lattice_create(pack_lattice(cell * n_cells, P0C, MASS0, 1.0))
    tw = X.xt_twiss4d_chrom(lat, 0.0, 1e-4)
    lat.close()
    quad = lambda k: np.array([[1.0, 0.0, 0.0], [-k, 1.0, 0.0], [0.0, 0.0, 1.0]])
    drift = np.array([[1.0, L, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]])
    dip = np.array([[1.0, 0.0, 0.0], [-th * th / ell, 1.0, th], [0.0, 0.0, 1.0]])
    m = np.eye(3)
    for e in (quad(kq), drift, dip, drift, quad(-kq), drift, dip, drift):
        m = e @ m
    d = np.linalg.solve(np.eye(2) - m[:2, :2], m[:2, 2])
    assert abs(tw["dx"] - d[0]) < 1e-6 * abs(d[0]) and abs(tw["dpx"] - d[1]) < 1e-6 * max(abs(d[1]), 0.1)
    assert abs(tw["dy"]) < 1e-9

    buf = C.pack(C.lattice(2))
    want = MO.chromatic_optics_of(buf, 1e-4)
    lat = X.xt_lattice_create(buf)
    tw = X.xt_twiss4d_chrom(lat, 0.0, 1e-4)
    assert abs(tw["dx"] - want["dx"]) < 1e-6 * max(abs(want["dx"]), 1.0) and abs(tw["dpx"] - want["dpx"]) < 1e-7
    assert abs(tw["dy"] - want["dy"]) < 1e-6 and abs(tw["dqx"] - want["dqx"]) < 2e-4 * max(abs(want["dqx"]), 1.0)
    assert abs(tw["dqy"] - want["dqy"]) < 2e-4 * max(abs(want["dqy"]), 1.0) and abs(tw["betx"] / want["betx"] - 1) < 1e-7
    with pytest.raises(X.XtError) as e:
        X.xt_twiss4d_chrom(lat, 0.0, 0.0)
    assert e.value.code == -1
    lat.close()


def test_optics_along_the_line(X):
    """xt_twiss4d_line (one launch through internal monitor records) against the thin-FODO closed forms of pin
    P19, against the oracle's prefix-tracking procedure on every row of configs[0] and on sampled rows of the
    LHC-sized configs[2]; the last row closes on the first and carries the whole tune."""
    from xt_inputs.packed import Marker
    n_cells, L, kq = 10, 2.0, 0.1
    cell = [Multipole(knl=(0.0, kq)), Drift(L / 2), Marker(), Drift(L / 2), Multipole(knl=(0.0, -kq)), Drift(L)]
    lat = X.xt_lattice_create(pack_lattice(cell * n_cells, P0C, MASS0, 1.0))
    start, rows = X.xt_twiss4d_line(lat)
    lat.close()
    mu = math.acos(1.0 - (L * kq) ** 2 / 2.0)
    bmax, bmin = 2 * L * (1 + math.sin(mu / 2)) / math.sin(mu), 2 * L * (1 - math.sin(mu / 2)) / math.sin(mu)
    qf, qd = np.arange(n_cells) * 6, np.arange(n_cells) * 6 + 4
    np.testing.assert_allclose(rows["betx"][qf], bmax, rtol=1e-6)
    np.testing.assert_allclose(rows["bety"][qf], bmin, rtol=1e-6)
    np.testing.assert_allclose(rows["betx"][qd], bmin, rtol=1e-6)
    np.testing.assert_allclose(rows["alfx"][qf], -bmax * kq / 2, atol=1e-6)
    np.testing.assert_allclose(rows["alfy"][qd], -bmax * kq / 2, atol=1e-6)
    np.testing.assert_allclose(rows["mux"][qf], np.arange(n_cells) * mu, atol=1e-6)
    np.testing.assert_allclose(rows["muy"][-1], n_cells * mu, atol=1e-6)
    np.testing.assert_allclose(rows["s"][qd], np.arange(n_cells) * 2 * L + L, atol=1e-12)
    assert np.array_equal(rows["betx"][qf + 2], rows["betx"][qf + 3])           # a marker's row = the next element's
    assert abs(rows["mux"][-1] / (2 * math.pi) % 1.0 - start["qx_frac"]) < 1e-7

    for cfg, pick in ((0, None), (2, 24)):
        els = C.lattice(cfg)
        n = len(els)
        sel = list(range(n + 1)) if pick is None else sorted(set(np.random.default_rng(3).integers(0, n + 1, pick)) | {0, n})
        want_on, want = MO.optics_along(els, C.P0C, C.MASS0, 1.0, sel)
        lat = X.xt_lattice_create(C.pack(els))
        start, rows = X.xt_twiss4d_line(lat)
        lat.close()
        assert abs(start["betx"] / want_on["betx"] - 1) < 1e-7
        for i, w in zip(sel, want):
            for k in ("x", "y"):
                assert abs(rows[k][i] - w[k]) < 1e-11, (cfg, i, k)
            for k in ("betx", "bety"):
                assert abs(rows[k][i] / w[k] - 1.0) < 2e-6, (cfg, i, k)
            for k in ("alfx", "alfy"):
                assert abs(rows[k][i] - w[k]) < 2e-6 * max(1.0, abs(w[k])), (cfg, i, k)
            for k in ("mux", "muy"):
                d = (rows[k][i] - w[k]) % (2 * math.pi)
                assert min(d, 2 * math.pi - d) < 1e-6, (cfg, i, k)
            for k in ("dx", "dy"):
                assert abs(rows[k][i] - w[k]) < 2e-6 * max(1.0, abs(w[k])), (cfg, i, k)
            if cfg == 2:                                                         # normal modes (coupling from the tilted magnets?)
                for k in ("betx1", "bety1", "betx2", "bety2"):
                    assert abs(rows[k][i] - w[k]) < 3e-5 * max(w["betx1"], w["bety2"], 1.0), (cfg, i, k, rows[k][i], w[k])
                for k in ("mu1", "mu2"):
                    d = (rows[k][i] - w[k]) % (2 * math.pi)
                    assert min(d, 2 * math.pi - d) < 1e-5, (cfg, i, k)
            else:                                                                # symmetric FODO: equal tunes, no modes
                assert np.isnan(rows["betx1"][i]) and np.isnan(rows["mu2"][i])
        assert np.all(np.diff(rows["mux"]) > -1e-9) and np.all(np.diff(rows["s"]) >= 0)
        assert abs(rows["betx"][-1] / rows["betx"][0] - 1) < 1e-5 and abs(rows["dx"][-1] - rows["dx"][0]) < 1e-5
        assert abs((rows["mux"][-1] / (2 * math.pi)) % 1.0 - start["qx_frac"]) < 1e-6
        if cfg == 2:
            assert abs(rows["mu1"][-1] / (2 * math.pi) % 1.0 - want_on["q1_frac"]) < 1e-6
            assert rows["mux"][-1] / (2 * math.pi) > 10.0                       # integer part of the tune included
            print("configs[2] tunes with integer part:", rows["mux"][-1] / (2 * math.pi), rows["muy"][-1] / (2 * math.pi))


def test_coupled_optics_along_the_line(X):
    """A FODO ring with unequal tunes seen from a frame rotated about s (pin P20): the normal-mode functions from
    the GPU path carry the cos^2 / sin^2 shares at the start and are the ring's own planes inside; with a skew
    quadrupole they follow the oracle procedure at every element."""
    from xt_inputs.packed import SRotation
    kq, L, th = 0.1, 2.0, 0.3
    ring = [Multipole(knl=(0.0, kq)), Drift(L), Multipole(knl=(0.0, -0.95 * kq)), Drift(L)] * 10
    lat = X.xt_lattice_create(pack_lattice(ring, P0C, MASS0, 1.0))
    flat, _ = X.xt_twiss4d_line(lat)
    lat.close()
    rot = [SRotation.from_angle(-th)] + ring + [SRotation.from_angle(th)]
    lat = X.xt_lattice_create(pack_lattice(rot, P0C, MASS0, 1.0))
    start, rows = X.xt_twiss4d_line(lat)
    modes = X.xt_twiss4d_normal_form(start["m"])
    lat.close()
    c2, s2 = math.cos(th) ** 2, math.sin(th) ** 2
    assert abs(modes["q1_frac"] - flat["qx_frac"]) < 1e-8 and abs(modes["q2_frac"] - flat["qy_frac"]) < 1e-8
    for i in (0, len(rot)):
        assert abs(rows["betx1"][i] - c2 * flat["betx"]) < 1e-5 and abs(rows["bety1"][i] - s2 * flat["betx"]) < 1e-5
        assert abs(rows["bety2"][i] - c2 * flat["bety"]) < 1e-5 and abs(rows["betx2"][i] - s2 * flat["bety"]) < 1e-5
    assert np.max(rows["bety1"][1:-1]) < 1e-9 and np.max(rows["betx2"][1:-1]) < 1e-9
    assert abs(rows["mu1"][-1] / (2 * math.pi) % 1.0 - flat["qx_frac"]) < 1e-7
    skew = [Multipole(knl=(0.0, 0.0), ksl=(0.0, 0.004))] + ring
    want_on, want = MO.optics_along(skew, P0C, MASS0, 1.0, list(range(len(skew) + 1)))
    lat = X.xt_lattice_create(pack_lattice(skew, P0C, MASS0, 1.0))
    start, rows = X.xt_twiss4d_line(lat)
    lat.close()
    assert want_on["bety1"] > 1e-3                                               # really coupled
    for i, w in enumerate(want):
        for k in ("betx1", "bety1", "betx2", "bety2"):
            assert abs(rows[k][i] - w[k]) < 1e-6 * max(w["betx1"], w["bety2"]), (i, k)
        for k in ("mu1", "mu2"):
            d = (rows[k][i] - w[k]) % (2 * math.pi)
            assert min(d, 2 * math.pi - d) < 1e-6, (i, k)


def test_six_dimensional_twiss(X):
    """xt_twiss6d: the closed forms of pin P22 (synchrotron tune of a cavity in a ring without bends, fixed point at
    zeta = lag/kz, FODO tunes) and the oracle procedure (make_optics.optics6d_of) on the LHC-sized configs[2] and
    configs[3] with their eight cavities; a ring without a cavity is reported, not solved."""
    from xt_inputs.packed import Cavity
    from oracle import oracle as O
    p0c, volt, freq = 1.0e9, 1e5, 200e6
    cell = [Multipole(knl=(0.0, 0.1)), Drift(2.0), Multipole(knl=(0.0, -0.095)), Drift(2.0)]
    for lag in (0.0, 25.0):
        buf = pack_lattice(cell * 10 + [Cavity(volt, freq, lag)], p0c, MASS0, 1.0)
        beta0, gamma0 = O.reference(buf)
        kz = 2 * math.pi * freq / (beta0 * 299792458.0)
        A, B = 40.0 / gamma0 ** 2, (volt / p0c) * kz / beta0
        lat = X.xt_lattice_create(buf)
        tw = X.xt_twiss6d(lat)
        flat = X.xt_twiss4d(lat)
        lat.close()
        assert abs(tw["qs"] - math.acos(1.0 - A * B / 2.0) / (2 * math.pi)) < 1e-8
        assert abs(tw["co"][4] - math.radians(lag) / kz) < 1e-9 and np.max(np.abs(tw["co"][[0, 1, 2, 3, 5]])) < 1e-12
        assert abs(tw["q1_frac"] - flat["qx_frac"]) < 1e-7 and abs(tw["q2_frac"] - flat["qy_frac"]) < 1e-7
    for cfg in (2, 3):
        buf = C.pack(C.lattice(cfg))
        want = MO.optics6d_of(buf)
        lat = X.xt_lattice_create(buf)
        tw = X.xt_twiss6d(lat)
        lat.close()
        np.testing.assert_allclose(tw["co"][:4], want["co"][:4], atol=1e-10)
        assert abs(tw["co"][4] - want["co"][4]) < 1e-8 and abs(tw["co"][5] - want["co"][5]) < 1e-10
        for k in ("q1_frac", "q2_frac"):
            assert abs(tw[k] - want[k]) < 2e-6, (cfg, k, tw[k], want[k])
        assert abs(tw["qs"] - want["qs"]) < 1e-7 and 0 < tw["qs"] < 0.1, (cfg, tw["qs"], want["qs"])
        print("configs[%d]: q1 %.6f q2 %.6f qs %.6f, %d Newton steps" % (cfg, tw["q1_frac"], tw["q2_frac"], tw["qs"], tw["iterations"]))
    # no cavity: singular; configs[0] (no bends, cavity at lag 180 deg: below transition that is the unstable phase,
    # the longitudinal eigenvalues are real, 1 -+ 4e-5): reported
    for buf in (pack_lattice(cell * 10, p0c, MASS0, 1.0), C.pack(C.lattice(0))):
        lat = X.xt_lattice_create(buf)
        with pytest.raises(X.XtError) as e:
            X.xt_twiss6d(lat)
        assert e.value.code == -5
        lat.close()


def test_six_dimensional_normal_form_along_the_line(X):
    """xt_twiss6d_line (steps 3-5 in six dimensions): (a) the closed forms of pin P24 on the GPU
    path -- the modes of an uncoupled FODO ring with a cavity are its planes (4-D Courant-Snyder values row by row,
    kick-slip closed form of the longitudinal mode), the dispersion ring gives the periodic dispersion of the 3x3
    matrices from the longitudinal eigenvector; (b) the oracle procedure (make_optics.optics6d_along) on every row
    of a skew-coupled ring with bends and on sampled rows of the LHC-sized configs[2]."""
    from xt_inputs.packed import Cavity
    from oracle import oracle as O
    two_pi = 2 * math.pi

    def phase_close(a, b, tol):
        d = (a - b) % two_pi
        return min(d, two_pi - d) < tol

    # (a) uncoupled FODO + cavity
    p0c = 1.0e9
    cell = [Multipole(knl=(0.0, 0.1)), Drift(2.0), Multipole(knl=(0.0, -0.095)), Drift(2.0)]
    els = cell * 10 + [Cavity(1e5, 200e6, 0.0)]
    buf = pack_lattice(els, p0c, MASS0, 1.0)
    lat = X.xt_lattice_create(buf)
    start, rows = X.xt_twiss6d_line(lat)
    flat_lat = X.xt_lattice_create(pack_lattice(cell * 10, p0c, MASS0, 1.0))
    _, cols4 = X.xt_twiss4d_line(flat_lat)
    rows4 = [{k: v[i] for k, v in cols4.items()} for i in range(len(cols4["s"]))]
    flat_lat.close()
    lat.close()
    assert len(rows) == len(els) + 1 and start["stable"] == 1
    for r6, r4 in zip(rows[:len(cell) * 10 + 1], rows4):
        assert abs(r6["betx1"] / r4["betx"] - 1) < 5e-6 and abs(r6["bety2"] / r4["bety"] - 1) < 5e-6
        assert abs(r6["alfx1"] - r4["alfx"]) < 5e-6 and abs(r6["alfy2"] - r4["alfy"]) < 5e-6
        assert r6["bety1"] < 1e-8 and r6["betx2"] < 1e-8 and r6["betx3"] < 1e-8 and r6["betz1"] < 1e-8
        assert abs(r6["mu1"] - r4["mux"]) < 5e-6 and abs(r6["mu2"] - r4["muy"]) < 5e-6       # both unwrapped
    beta0, gamma0 = O.reference(buf)
    kz = two_pi * 200e6 / (beta0 * 299792458.0)
    A, B = 40.0 / gamma0 ** 2, (1e5 / p0c) * kz / beta0
    mu_s = math.acos(1.0 - A * B / 2.0)
    assert abs(start["betz3"] / (A / math.sin(mu_s)) - 1) < 1e-5
    assert abs(rows[-1]["mu3"] - mu_s) < 1e-6 and abs(rows[-1]["mu1"] / two_pi - round(rows[-1]["mu1"] / two_pi - start["q1_frac"]) - start["q1_frac"]) < 1e-6
    # (a) dispersion ring of pin P18 / P24 with a weak cavity
    th = two_pi / 16
    bend = Multipole(knl=(th,), hxl=th, length=1.5)
    dcell = [Multipole(knl=(0.0, 0.25)), Drift(3.0), bend, Drift(3.0), Multipole(knl=(0.0, -0.25)), Drift(3.0), bend, Drift(3.0)]
    quad = lambda k: np.array([[1.0, 0.0, 0.0], [-k, 1.0, 0.0], [0.0, 0.0, 1.0]])
    drift = np.array([[1.0, 3.0, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]])
    dip = np.array([[1.0, 0.0, 0.0], [-th * th / 1.5, 1.0, th], [0.0, 0.0, 1.0]])
    mats = [quad(0.25), drift, dip, drift, quad(-0.25), drift, dip, drift]
    m = np.eye(3)
    for e in mats:
        m = e @ m
    d = np.append(np.linalg.solve(np.eye(2) - m[:2, :2], m[:2, 2]), 1.0)
    lat = X.xt_lattice_create(pack_lattice(dcell * 8 + [Cavity(2e4, 50e6, 180.0)], P0C, MASS0, 1.0))
    start, rows = X.xt_twiss6d_line(lat)
    lat.close()
    for i in range(9):
        assert abs(rows[i]["dx"] / d[0] - 1.0) < 3e-4 and abs(rows[i]["dpx"] - d[1]) < 3e-4 * max(abs(d[1]), 0.1), i
        assert abs(rows[i]["dy"]) < 1e-6
        if i < 8:
            d = mats[i] @ d
    # (b) oracle procedure: a skew-coupled ring with curved dipoles, every row
    ks = [Multipole(knl=(0.0, 0.0), ksl=(0.0, 0.03))]
    coupled = (ks + dcell) * 8 + [Cavity(2e5, 100e6, 180.0)]
    want_on, want = MO.optics6d_along(coupled, P0C, MASS0, 1.0, list(range(len(coupled) + 1)))
    lat = X.xt_lattice_create(pack_lattice(coupled, P0C, MASS0, 1.0))
    start, rows = X.xt_twiss6d_line(lat)
    lat.close()
    assert want_on["bety1"] > 1e-3 * want_on["betx1"]                                      # really coupled
    scale = max(want_on["betx1"], want_on["bety2"])
    for k in ("q1_frac", "q2_frac", "q3_frac"):
        assert abs(start[k] - want_on[k]) < 1e-7, k
    for r, w in zip(rows, want):
        np.testing.assert_allclose(r["co"], w["co"], atol=1e-9)
        for mode in (1, 2, 3):
            for pl in ("x", "y"):
                assert abs(r["bet%s%d" % (pl, mode)] - w["bet%s%d" % (pl, mode)]) < 2e-5 * scale
                assert abs(r["alf%s%d" % (pl, mode)] - w["alf%s%d" % (pl, mode)]) < 2e-5 * max(1.0, scale / 10)
            sense = -1.0 if (mode == 3 and start["q3_frac"] > 0.5) else 1.0
            assert phase_close(sense * r["mu%d" % mode], w["mu%d" % mode], 2e-5), (mode, r["mu%d" % mode], w["mu%d" % mode])
        assert abs(r["betz3"] / w["betz3"] - 1) < 1e-4
        for k in ("dx", "dpx", "dy", "dpy"):
            assert abs(r[k] - w[k]) < 1e-4 * max(1.0, abs(w[k])), (k, r[k], w[k])
    # (b) configs[2], sampled rows
    els2 = C.lattice(2)
    sample = [0, 1, 7, 200, 1234, 4321, len(els2) - 3, len(els2)]
    want_on, want = MO.optics6d_along(els2, P0C, MASS0, 1.0, sample)
    lat = X.xt_lattice_create(C.pack(els2))
    start, rows = X.xt_twiss6d_line(lat)
    lat.close()
    scale = max(want_on["betx1"], want_on["bety2"])
    for i, w in zip(sample, want):
        r = rows[i]
        np.testing.assert_allclose(r["co"][:4], w["co"][:4], atol=1e-9)
        for key in ("betx1", "bety1", "betx2", "bety2"):
            assert abs(r[key] - w[key]) < 1e-4 * scale, (i, key, r[key], w[key])
        for key in ("dx", "dy"):
            assert abs(r[key] - w[key]) < 2e-3 * max(1.0, abs(w[key])), (i, key, r[key], w[key])
    print("configs[2] 6-D: q = %.6f %.6f %.6f, betx1 %.2f bety2 %.2f betz3 %.1f, dx %.4f at the start"
          % (start["q1_frac"], start["q2_frac"], start["q3_frac"], start["betx1"], start["bety2"], start["betz3"], start["dx"]))
