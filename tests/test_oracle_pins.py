"""Pins of the CPU oracle against things other than itself (P1-P11).

None of these needs a GPU.  A pin either compares with the 60-digit *textbook*
evaluation stored in tests/golden/ (written by make_worked_examples.py, which never
calls the oracle), with a closed form, or checks an invariant of the mathematics.
"""
import math

import mpmath as mp
import numpy as np
import pytest

from oracle import oracle as O
from xt_inputs import configs as C
from xt_inputs.packed import (Cavity, Drift, LimitEllipse, LimitRect, Marker, Multipole,
                              SRotation, XYShift, pack_lattice)
import helpers as H

mp.mp.dps = 50
ULP = 2.0 ** -52


def pack(els, p0c=H.P0C, mass0=H.MASS0, q0=H.Q0):
    return pack_lattice(els, p0c, mass0, q0)


def track_one(els, start, n_turns=1, **kw):
    buf = pack(els, **kw)
    p = O.new_particles(buf, H.coords_from_rows([start]))
    O.track(buf, p, n_turns)
    return p


def assert_matches_golden(p, values, rtol, keys=("x", "px", "y", "py", "zeta", "delta", "ptau", "rpp", "rvv")):
    for k in keys:
        ref = mp.mpf(values[k])
        got = mp.mpf(float(p[k][0]))
        err = abs(got - ref)
        assert err <= rtol * abs(ref) or err == 0, (k, float(err / abs(ref)) if ref != 0 else float(err))


# ----------------------------------------------------------------------------- reference
def test_reference_particle_constants():
    g = H.load_golden()["lines"][0]
    beta0, gamma0 = O.reference(pack([Marker()]))
    assert abs(mp.mpf(beta0) - mp.mpf(g["beta0"])) <= 1 * ULP
    assert abs(mp.mpf(gamma0) - mp.mpf(g["gamma0"])) <= 2 * ULP * gamma0
    # SURVEY.md §8(c) worked-example constants (60-digit session check)
    assert abs(beta0 - 0.99999782629224451599) < 2e-16
    assert abs(gamma0 - 479.60605867866257519) < 2e-13


def test_init_helper_matches_textbook():
    g = H.load_golden()
    for case in g["drift_cases"]:
        st = [H.unhex(v) for v in case["start"]]
        buf = pack([Marker()])
        p = O.new_particles(buf, H.coords_from_rows([st]))
        ref = H.load_golden()  # noqa: F841
        # ptau, rpp, rvv are unchanged by a drift: compare to the stored post-drift values
        assert_matches_golden(p, case["values"], 4 * ULP, keys=("ptau", "rpp", "rvv", "delta"))


# ------------------------------------------------------------------------ P1 exact drift
def test_P1_exact_drift_closed_form():
    """x, y, zeta within 2 ulp of the 60-digit textbook exact drift."""
    g = H.load_golden()
    for case in g["drift_cases"]:
        st = [H.unhex(v) for v in case["start"]]
        p = track_one([Drift(H.unhex(case["length"]))], st)
        assert_matches_golden(p, case["values"], 2 * ULP, keys=("x", "y", "zeta"))
        assert p["px"][0] == st[1] and p["py"][0] == st[3] and p["delta"][0] == st[5]


# --------------------------------------------------------------- P5 worked examples W1..W3
@pytest.mark.parametrize("name", ["W1", "W2"])
def test_P5_worked_examples_stage_by_stage(name):
    g = H.load_golden()
    line = next(l for l in g["lines"] if l["name"] == name)
    els = [H.element_from_json(d) for d in line["elements"]]
    start = [H.unhex(v) for v in line["start"]]
    for k in range(len(els) + 1):
        p = track_one(els[:k] if k else [Marker()], start)
        assert_matches_golden(p, line["stages"][k]["values"], 1e-15)


def test_P5_survey_printed_values():
    """Digits printed in SURVEY.md §8(c) tables W1/W2 (final rows)."""
    g = H.load_golden()
    for name, exp in (("W1", dict(x=1.369506343806425560212e-3, px=6.961718789953393473442e-5,
                                  y=-2.852964188025315194125e-4, py=6.476798823145405988275e-5,
                                  zeta=9.999961263568563893139e-3)),
                      ("W2", dict(x=1.380951326487813852667e-3, px=8.106561136853177356806e-5,
                                  y=-2.643470141317643943199e-4, py=8.572368539549421031333e-5,
                                  zeta=9.993960029127754365771e-3, delta=3.000930656374122780101e-4,
                                  ptau=3.000924135184838653674e-4))):
        line = next(l for l in g["lines"] if l["name"] == name)
        els = [H.element_from_json(d) for d in line["elements"]]
        p = track_one(els, [H.unhex(v) for v in line["start"]])
        for k, v in exp.items():
            assert abs(p[k][0] - v) <= 2e-15 * abs(v), (name, k)


def test_P5_W3_full_turn_of_config0():
    g = H.load_golden()
    for line in (l for l in g["lines"] if l["name"].startswith("W3")):
        els = [H.element_from_json(d) for d in line["elements"]]
        assert len(els) == 41
        p = track_one(els, [H.unhex(v) for v in line["start"]])
        assert_matches_golden(p, line["stages"][-1]["values"], 2e-14)
        assert p["at_turn"][0] == 1 and p["state"][0] == 1 and p["s"][0] == 0.0


# ---------------------------------------------------------------- P6 Horner vs definition
def test_P6_horner_vs_direct_power_sum_orders_0_to_20():
    g = H.load_golden()
    assert len(g["multipole_cases"]) == 21
    for case in g["multipole_cases"]:
        el = H.element_from_json(case["element"])
        st = [H.unhex(v) for v in case["start"]]
        p = track_one([el], st)
        # kick magnitudes: compare the *kick* to 1e-14 relative (absolute floor from the sum's size)
        for k, i0 in (("px", 1), ("py", 3)):
            ref_after = mp.mpf(case["values"][k])
            kick_ref = ref_after - mp.mpf(st[i0])
            kick = mp.mpf(float(p[k][0])) - mp.mpf(st[i0])
            scale = max(abs(kick_ref), mp.mpf(1e-6))
            assert abs(kick - kick_ref) <= 1e-14 * scale + 2 * ULP * abs(ref_after), (el.order, k)
        assert p["x"][0] == st[0] and p["y"][0] == st[2] and p["zeta"][0] == st[4]


# -------------------------------------------------------------- P2 thin FODO closed form
def _cell_matrix_closed_form():
    """One FODO cell [QF, D(2), QD, D(2)] with thin quads f = 1/k1l = 10 m (textbook 2x2 algebra)."""
    def drift(L):
        return np.array([[1.0, L], [0.0, 1.0]])

    def quad(k):
        return np.array([[1.0, 0.0], [-k, 1.0]])
    mx = drift(2.0) @ quad(-0.1) @ drift(2.0) @ quad(+0.1)
    my = drift(2.0) @ quad(+0.1) @ drift(2.0) @ quad(-0.1)
    return mx, my


def test_P2_fodo_cell_matrix_tune_and_twiss():
    cell = [Multipole(knl=(0.0, 0.1)), Drift(2.0), Multipole(knl=(0.0, -0.1)), Drift(2.0)]
    buf = pack(cell)
    J = H.jacobian6(O.track, buf, np.zeros(6))
    mx, my = _cell_matrix_closed_form()
    np.testing.assert_allclose(mx, [[0.76, 4.4], [-0.02, 1.2]], atol=1e-15)
    np.testing.assert_allclose(my, [[1.16, 3.6], [-0.02, 0.8]], atol=1e-15)
    np.testing.assert_allclose(J[0:2, 0:2], mx, atol=1e-8)
    np.testing.assert_allclose(J[2:4, 2:4], my, atol=1e-8)
    # no x-y coupling for upright quads
    assert np.max(np.abs(J[0:2, 2:4])) < 1e-8 and np.max(np.abs(J[2:4, 0:2])) < 1e-8
    # cos(mu) = 1 - L^2/(2 f^2) with L = 2 m, f = 10 m  (north_star; reading A15)
    cosmu = 0.5 * (J[0, 0] + J[1, 1])
    assert abs(cosmu - (1.0 - 2.0 ** 2 / (2.0 * 10.0 ** 2))) < 1e-8
    assert abs(cosmu - 0.98) < 1e-8
    mu = math.acos(0.98)
    assert abs(mu - 0.20033484232311959) < 1e-15

    # Ten cells (config[0] without its cavity): ring tune 10 mu / 2 pi and M^10
    ring = cell * 10
    J10 = H.jacobian6(O.track, pack(ring), np.zeros(6))
    m10 = np.linalg.matrix_power(mx, 10)
    np.testing.assert_allclose(J10[0:2, 0:2], m10, atol=1e-7)
    np.testing.assert_allclose(m10, [[-1.4229092060125620, 20.074399908620036],
                                     [-0.091247272311909253, 0.58453078484944159]], rtol=1e-13)
    tune = math.acos(0.5 * (J10[0, 0] + J10[1, 1])) / (2 * math.pi)
    assert abs(tune - 0.31884280429259924) < 1e-8
    # Twiss at the QF entrance from the one-turn matrix (Twiss step 3)
    sinmu = math.sin(10 * mu)
    betx = J10[0, 1] / sinmu
    alfx = (J10[0, 0] - J10[1, 1]) / (2 * sinmu)
    bety = J10[2, 3] / sinmu
    alfy = (J10[2, 2] - J10[3, 3]) / (2 * sinmu)
    assert abs(betx - 22.110831935702666) < 1e-6 and abs(alfx + 1.1055415967851333) < 1e-7
    assert abs(bety - 18.090680674665817) < 1e-6 and abs(alfy - 0.90453403373329087) < 1e-7


# ------------------------------------------------------------------- P3 symplecticity
ALL_TYPES_LINE = [
    Drift(1.5), XYShift(1e-4, -2e-4), SRotation.from_angle(1e-3),
    Multipole(knl=(5e-3, 0.1, 0.5, 5.0), ksl=(0.0, 1e-3, -0.2, 1.0), hxl=5e-3, length=14.3),
    SRotation.from_angle(-1e-3), XYShift(-1e-4, 2e-4), LimitRect(-0.05, 0.05, -0.05, 0.05),
    Cavity(1e6, 200e6, 180.0), Drift(1.0), LimitEllipse(0.04, 0.03), Marker(),
]


def _check_symplectic(buf, z0, tol=1e-7):
    J = H.jacobian6(O.track, buf, z0)
    err = np.max(np.abs(J.T @ H.S6 @ J - H.S6))
    det = np.linalg.det(J)
    assert err < tol, err
    assert abs(det - 1.0) < tol, det


@pytest.mark.parametrize("z0", [np.zeros(6),
                                np.array([1e-3, 2e-4, -5e-4, 1e-4, 0.01, 3e-4]),
                                np.array([-2e-3, -1e-4, 1e-3, 3e-4, -0.02, -5e-4])])
def test_P3_symplectic_all_element_types(z0):
    _check_symplectic(pack(ALL_TYPES_LINE), z0)


@pytest.mark.parametrize("cfg", [0, 1])
def test_P3_symplectic_one_turn_small_configs(cfg):
    buf = C.pack(C.lattice(cfg))
    for z0 in (np.zeros(6), np.array([2e-4, 1e-5, -1e-4, 2e-5, 0.03, 1e-4])):
        _check_symplectic(buf, z0)


def test_P3_symplectic_one_turn_lhc_like():
    buf = C.pack(C.lattice(2))
    # amplification of finite-difference noise by the 8 606-element turn: loosen to 5e-6
    _check_symplectic(buf, np.array([3e-4, 1e-6, 1e-4, -2e-6, 0.01, 1e-4]), tol=5e-6)


def test_A13_determinant_in_zeta_delta_variables_is_not_one_with_cavity():
    """Reading A13: (zeta, delta) is not a canonical pair; with a cavity det != 1 there."""
    buf = pack(ALL_TYPES_LINE)
    J = H.jacobian6(O.track, buf, np.array([1e-3, 2e-4, -5e-4, 1e-4, 0.01, 3e-4]))
    assert abs(np.linalg.det(J) - 1.0) < 1e-7


# ------------------------------------------------------------------- P4 reversibility
@pytest.mark.parametrize("n_turns", [1, 3])
def test_P4_reversibility(n_turns):
    els = [e for e in ALL_TYPES_LINE]
    rng = np.random.default_rng(5)
    n = 64
    co = dict(x=rng.normal(0, 1e-3, n), px=rng.normal(0, 1e-4, n), y=rng.normal(0, 1e-3, n),
              py=rng.normal(0, 1e-4, n), zeta=rng.normal(0, 0.02, n), delta=rng.normal(0, 3e-4, n))
    fwd, bwd = pack(els), pack(H.reversed_lattice(els))
    p = O.new_particles(fwd, co)
    p0 = O.copy_particles(p)
    O.track(fwd, p, n_turns)
    ok = p["state"] == 1            # the line is not a stable ring: some leave the apertures
    assert ok.sum() > n // 2
    moved = max(np.max(np.abs(p[k] - p0[k])) for k in ("x", "y", "zeta"))
    assert moved > 1e-5                      # the forward pass did something
    H.flip_R(p)
    O.track(bwd, p, n_turns)
    H.flip_R(p)
    assert np.all(p["state"][ok] == 1)
    for k in ("x", "px", "y", "py", "zeta", "delta", "ptau"):
        # relative to the ensemble scale of the coordinate (a single |p0| may be ~0)
        scale = np.maximum(np.abs(p0[k]), {"x": 1e-3, "y": 1e-3, "px": 1e-4, "py": 1e-4,
                                           "zeta": 0.02, "delta": 3e-4, "ptau": 3e-4}[k])
        assert np.max((np.abs(p[k] - p0[k]) / scale)[ok]) < 1e-13, k


def test_P4_reversibility_config0_100_turns():
    els = C.lattice(0)
    fwd, bwd = C.pack(els), C.pack(H.reversed_lattice(els))
    p = O.new_particles(fwd, C.particles_cfg0(100))
    p0 = O.copy_particles(p)
    O.track(fwd, p, 100)
    H.flip_R(p)
    O.track(bwd, p, 100)
    H.flip_R(p)
    for k in ("x", "px", "y", "py", "zeta", "delta"):
        scale = {"x": 1e-4, "y": 1e-4, "px": 1e-5, "py": 1e-5, "zeta": 0.05, "delta": 1e-4}[k]
        assert np.max(np.abs(p[k] - p0[k])) < 1e-12 * scale, k


# -------------------------------------------------------------- P7 invariants
def test_P7_courant_snyder_invariant_and_frozen_energy():
    ring = [Multipole(knl=(0.0, 0.1)), Drift(2.0), Multipole(knl=(0.0, -0.1)), Drift(2.0)] * 10
    buf = pack(ring)
    betx, alfx = 22.110831935702666, -1.1055415967851333     # P2 values (closed form)
    bety, alfy = 18.090680674665817, +0.90453403373329087
    gamx, gamy = (1 + alfx ** 2) / betx, (1 + alfy ** 2) / bety
    rng = np.random.default_rng(11)
    n = 32
    # amplitude small enough that the exact drift's nonlinearity, (px^2+py^2)/2 per drift and
    # systematic over 2 000 drifts, stays below 1e-13
    co = dict(x=rng.normal(0, 1e-8, n), px=rng.normal(0, 1e-9, n), y=rng.normal(0, 1e-8, n),
              py=rng.normal(0, 1e-9, n), zeta=np.zeros(n), delta=np.zeros(n))
    p = O.new_particles(buf, co)
    d0, pt0 = p["delta"].copy(), p["ptau"].copy()

    def inv(p):
        jx = gamx * p["x"] ** 2 + 2 * alfx * p["x"] * p["px"] + betx * p["px"] ** 2
        jy = gamy * p["y"] ** 2 + 2 * alfy * p["y"] * p["py"] + bety * p["py"] ** 2
        return jx, jy
    jx0, jy0 = inv(p)
    # conditioning of the quadratic form: its error scales with the sum of |terms|, which can
    # exceed J itself (alpha != 0); normalise with that sum at the start point
    sx = gamx * p["x"] ** 2 + 2 * abs(alfx * p["x"] * p["px"]) + betx * p["px"] ** 2
    sy = gamy * p["y"] ** 2 + 2 * abs(alfy * p["y"] * p["py"]) + bety * p["py"] ** 2
    for _ in range(100):
        O.track(buf, p, 1)
        jx, jy = inv(p)
        assert np.max(np.abs(jx - jx0) / sx) < 1e-12 and np.max(np.abs(jy - jy0) / sy) < 1e-12
    assert np.array_equal(p["delta"], d0) and np.array_equal(p["ptau"], pt0)   # bit-unchanged


# ------------------------------------------------------------------ P8 aperture edges
def test_P8_rect_edges_inclusive_nan_lost_and_loss_record():
    els = [Drift(3.0), Marker(), LimitRect(-0.01, 0.02, -0.03, 0.04), Drift(1.0)]
    buf = pack(els)
    inf = math.inf
    rows = [
        [0.02, 0, 0, 0, 0, 0], [math.nextafter(0.02, inf), 0, 0, 0, 0, 0],
        [-0.01, 0, 0, 0, 0, 0], [math.nextafter(-0.01, -inf), 0, 0, 0, 0, 0],
        [0, 0, 0.04, 0, 0, 0], [0, 0, math.nextafter(0.04, inf), 0, 0, 0],
        [0, 0, -0.03, 0, 0, 0], [0, 0, math.nextafter(-0.03, -inf), 0, 0, 0],
        [math.nan, 0, 0, 0, 0, 0], [0, 0, math.nan, 0, 0, 0], [0, 0, 0, 0, 0, 0],
    ]
    p = O.new_particles(buf, H.coords_from_rows(rows))
    p["at_turn"][:] = 5
    margin = np.full(len(rows), np.inf)
    O.track(buf, p, 3, min_margin=margin)
    np.testing.assert_array_equal(p["state"], [1, 0, 1, 0, 1, 0, 1, 0, 0, 0, 1])
    lost = p["state"] == 0
    np.testing.assert_array_equal(p["at_turn"][lost], 5)          # completed turns only
    np.testing.assert_array_equal(p["at_turn"][~lost], 8)
    np.testing.assert_array_equal(p["at_element"][lost], 2)
    np.testing.assert_array_equal(p["s"][lost], 3.0)
    np.testing.assert_array_equal(p["s"][~lost], 0.0)
    assert p["x"][1] == rows[1][0]                                  # frozen at the aperture
    assert margin[0] == 0.0 and margin[1] < 1e-17 and margin[10] == 0.01


def test_P8_ellipse_edges():
    a, b = 0.02, 0.015
    els = [LimitEllipse(a, b)]
    buf = pack(els)
    inf = math.inf
    rows = [[a, 0, 0, 0, 0, 0], [math.nextafter(a, inf), 0, 0, 0, 0, 0],
            [0, 0, b, 0, 0, 0], [0, 0, -math.nextafter(b, inf), 0, 0, 0],
            [0.012, 0, 0.012, 0, 0, 0],   # (0.6)^2 + (0.8)^2 = 1 up to rounding
            [0.0121, 0, 0.012, 0, 0, 0], [math.inf, 0, 0, 0, 0, 0], [math.nan, 0, 0, 0, 0, 0],
            [0.001, 0, 0.001, 0, 0, 0]]
    p = O.new_particles(buf, H.coords_from_rows(rows))
    O.track(buf, p, 2)
    a2, b2 = a * a, b * b
    exp = [1 if (r[0] * r[0]) * b2 + (r[2] * r[2]) * a2 <= a2 * b2 else 0 for r in rows]
    assert exp[0] == 1 and exp[1] == 0 and exp[2] == 1 and exp[3] == 0 and exp[5:8] == [0, 0, 0] and exp[8] == 1
    np.testing.assert_array_equal(p["state"], exp)
    np.testing.assert_array_equal(p["at_turn"], [2 if e else 0 for e in exp])


# ------------------------------------------------------------------ P9 structural
def test_P9_continuation_order_and_freeze():
    els = C.lattice(1)
    buf = C.pack(els)
    co = C.subsample(C.particles_cfg1(sigma=1e-3), slice(None, None, 997))   # loses particles
    pa = O.new_particles(buf, co)
    pb = O.copy_particles(pa)
    O.track(buf, pa, 60)
    O.track(buf, pb, 25)
    snap = O.copy_particles(pb)
    O.track(buf, pb, 35)
    n_lost = int(np.sum(pa["state"] == 0))
    assert 0 < n_lost < len(pa["x"])
    for k in pa:
        np.testing.assert_array_equal(pa[k], pb[k], err_msg=k)            # track(60) == track(25)+track(35)
    dead = snap["state"] == 0
    for k in pa:
        np.testing.assert_array_equal(snap[k][dead], pb[k][dead], err_msg=k)   # lost never change again
    perm = np.random.default_rng(3).permutation(len(co["x"]))
    pc = O.new_particles(buf, {k: v[perm] for k, v in co.items()})
    O.track(buf, pc, 60)
    for k in pa:
        np.testing.assert_array_equal(pa[k][perm], pc[k], err_msg=k)      # independent of order
    pd = O.new_particles(buf, co)
    O.track(buf, pd, 60, threads=4)
    for k in pa:
        np.testing.assert_array_equal(pa[k], pd[k], err_msg=k)


def test_bad_buffers_rejected():
    good = pack([Drift(1.0)])
    for bad in (good[:-1], b"XXXX" + good[4:], good + b"\0" * 8,
                pack([Multipole(knl=(0.0,) * 22)]), pack([Drift(math.nan)]),
                pack_lattice([Drift(1.0)], -1.0, H.MASS0, 1.0)):
        with pytest.raises(ValueError):
            O.reference(bad)


# -------------------------------------------------------------- P10 energy identities
def test_P10_energy_identities_after_cavities():
    buf = C.pack(C.lattice(0))
    beta0, gamma0 = O.reference(buf)
    p = O.new_particles(buf, C.particles_cfg0(200))
    O.track(buf, p, 50)
    for i in range(200):
        d, pt = mp.mpf(float(p["delta"][i])), mp.mpf(float(p["ptau"][i]))
        lhs = (1 + d) ** 2
        rhs = pt ** 2 + 2 * pt / mp.mpf(beta0) + 1
        assert abs(lhs - rhs) <= 4 * ULP
        assert abs(mp.mpf(float(p["rvv"][i])) * (1 + mp.mpf(beta0) * pt) - (1 + d)) <= 4 * ULP
        assert abs(mp.mpf(float(p["rpp"][i])) * (1 + d) - 1) <= 2 * ULP


# --------------------------------------------- P11 cavity: linear synchrotron map, closed form
def test_P11_cavity_linear_synchrotron_trace():
    """Ring of drifts (C = 40 m) + one cavity at lag 0 (stable below transition: no bends, so
    the slip is purely kinematic).  Linearised one-turn longitudinal map in (zeta, ptau/beta0):
    [[1, A],[0, 1]] . [[1, 0],[-B, 1]],  A = C/gamma0^2,  B = (q0 V/p0c)(2 pi f/(beta0 c))/beta0,
    so trace = 2 - A B (closed form; pins kz, vn, lag units, sign conventions of reading A2)."""
    p0c = 1.0e9
    volt, freq, circ = 1e5, 200e6, 40.0
    els = [Drift(circ / 4)] * 4 + [Cavity(volt, freq, 0.0)]
    buf = pack(els, p0c=p0c)
    beta0, gamma0 = O.reference(buf)
    J = H.jacobian6(O.track, buf, np.zeros(6), h=(1e-6, 1e-7, 1e-6, 1e-7, 1e-5, 1e-7))
    A = circ / gamma0 ** 2
    B = (volt / p0c) * (2 * math.pi * freq / (beta0 * 299792458.0)) / beta0
    tr = J[4, 4] + J[5, 5]
    assert abs(tr - (2.0 - A * B)) < 1e-7
    assert abs(J[4, 5] - A) < 1e-6 * A          # slip term of the exact drift
    assert abs(J[5, 4] + B) < 1e-6 * B
    # lag = 180 deg flips the sign of the restoring force (unstable below transition)
    buf180 = pack([Drift(circ / 4)] * 4 + [Cavity(volt, freq, 180.0)], p0c=p0c)
    J180 = H.jacobian6(O.track, buf180, np.zeros(6), h=(1e-6, 1e-7, 1e-6, 1e-7, 1e-5, 1e-7))
    assert abs(J180[5, 4] - B) < 1e-6 * B


# ----------------------------- P12 curvature terms: off-momentum fixed point of a bend ring
def test_P12_weak_focusing_ring_dispersion_and_path_length():
    """[Drift(L), Bend(k0l = hxl = th, length)] x N: (x, px) = (delta*length/th, 0) is an exact
    fixed point (dispersion = bending radius of the thin model), and per cell
    dzeta = L (1 - beta0/beta) - delta*length*beta0/beta  (closed form; pins hxl*delta, the weak
    focusing term and the path-length term of the curved multipole)."""
    th, length, L, N = 2 * math.pi / 64, 3.0, 5.0, 64
    els = [Drift(L), Multipole(knl=(th,), hxl=th, length=length)] * N
    buf = pack(els)
    beta0, _ = O.reference(buf)
    for delta in (1e-3, -4e-4, 0.0):
        x0 = delta * length / th
        p = O.new_particles(buf, H.coords_from_rows([[x0, 0, 0, 0, 0, delta]]))
        O.track(buf, p, 1)
        assert abs(p["x"][0] - x0) <= 1e-13 * max(abs(x0), 1e-6)
        assert abs(p["px"][0]) < 1e-17
        d, pt = mp.mpf(delta), mp.mpf(float(p["ptau"][0]))
        b0_over_b = (1 + mp.mpf(beta0) * pt) / (1 + d)
        dz = N * (mp.mpf(L) * (1 - b0_over_b) - d * mp.mpf(length) * b0_over_b)
        assert abs(mp.mpf(float(p["zeta"][0])) - dz) <= 1e-13 * max(abs(dz), mp.mpf(1e-9))


# ----------------------------- P13 thick quadrupole (reading A18)
from xt_inputs.packed import Quadrupole  # noqa: E402


def _thin_sliced(k1, length, n):
    """n symmetric drift-kick-drift slices built from the maps pinned above (P1, P2, P6)."""
    h, kl = length / (2 * n), k1 * length / n
    return [Drift(h), Multipole(knl=(0.0, kl)), Drift(h)] * n


@pytest.mark.parametrize("k1", [0.35, -0.2])
def test_P13_thick_quadrupole_is_the_limit_of_thin_slices(k1):
    """The thick map is an exact flow; n symmetric thin slices converge to it as 1/n^2.  Pins x, px, y,
    py and the path length zeta, the delta dependence and both signs of k1.  The slices use the exact
    drift, the thick map the paraxial kinetic term (px^2 + py^2)/(2(1+delta)) (reading A18): what is left
    after Richardson extrapolation is that difference, relative p^2/2, and must scale as amplitude^3."""
    length = 3.1
    base = np.array([[1e-3, 2e-4, -5e-4, 1e-4, 0.01, 3e-4], [-2e-3, -1e-4, 1e-3, 3e-4, -0.02, -8e-4],
                     [5e-4, 0.0, 0.0, -2e-4, 0.0, 0.0]])

    def run(els, start):
        buf = pack(els)
        p = O.new_particles(buf, start)
        O.track(buf, p, 1)
        return np.stack([p[k] for k in ("x", "px", "y", "py", "zeta")], axis=1)

    residual = {}
    for amp in (1.0, 0.1):
        rows = base.copy()
        rows[:, :4] *= amp
        start = H.coords_from_rows(rows.tolist())
        thick = run([Quadrupole(k1, length)], start)
        s1, s2 = run(_thin_sliced(k1, length, 512), start), run(_thin_sliced(k1, length, 1024), start)
        residual[amp] = ((4.0 * s2 - s1) / 3.0 - thick)[:, :4]
        if amp == 0.1:                                          # paraxial difference below the slicing error
            e1, e2 = np.abs(s1 - thick)[:, :4], np.abs(s2 - thick)[:, :4]
            big = e1 > 50.0 * np.abs(residual[amp])             # slicing error well above the paraxial residual
            assert big.sum() >= 6
            assert np.all((e1[big] / e2[big] > 3.7) & (e1[big] / e2[big] < 4.4))      # second order in 1/n
            scale = amp * np.array([1e-3, 1e-4, 1e-3, 1e-4])
            assert np.max(np.abs(residual[amp]) / scale) < 2e-7   # p^2/2 with the momenta reached inside (<= 3e-4)
            slip = thick[:, 4] - rows[:, 4]
            slip_thin = ((4.0 * s2 - s1) / 3.0)[:, 4] - rows[:, 4]
            assert np.all(np.abs(slip) > 1e-11)                                       # the path length moved
            assert np.max(np.abs(slip_thin - slip) / np.abs(slip)) < 1e-6
            assert np.all(np.abs(thick[:, 0] - rows[:, 0]) > 1e-6)                    # the element did something
    ratio = residual[1.0] / residual[0.1]
    strong = np.abs(residual[1.0]) > 1e-12
    assert strong.sum() >= 6 and np.all(np.abs(ratio[strong] / 1e3 - 1.0) < 0.05)     # cubic in the amplitude


def test_P13_thick_quadrupole_matrix_symplectic_reversible():
    k1, length = 0.35, 3.1
    buf = pack([Quadrupole(k1, length)])
    J = H.jacobian6(O.track, buf, np.zeros(6))
    w = math.sqrt(k1)
    phi = w * length
    np.testing.assert_allclose(J[0:2, 0:2], [[math.cos(phi), math.sin(phi) / w],
                                             [-w * math.sin(phi), math.cos(phi)]], atol=1e-8)
    np.testing.assert_allclose(J[2:4, 2:4], [[math.cosh(phi), math.sinh(phi) / w],
                                             [w * math.sinh(phi), math.cosh(phi)]], atol=1e-8)
    line = [Drift(0.7), Quadrupole(k1, length), Drift(0.4), Quadrupole(-0.5 * k1, 1.3), Cavity(1e6, 200e6, 180.0),
            Drift(0.2)]
    for z0 in (np.zeros(6), np.array([1e-3, 2e-4, -5e-4, 1e-4, 0.01, 3e-4])):
        _check_symplectic(pack(line), z0)
    rng = np.random.default_rng(8)
    n = 32
    co = dict(x=rng.normal(0, 1e-3, n), px=rng.normal(0, 1e-4, n), y=rng.normal(0, 1e-3, n),
              py=rng.normal(0, 1e-4, n), zeta=rng.normal(0, 0.02, n), delta=rng.normal(0, 3e-4, n))
    fwd, bwd = pack(line), pack(H.reversed_lattice(line))
    p = O.new_particles(fwd, co)
    p0 = O.copy_particles(p)
    O.track(fwd, p, 2)
    H.flip_R(p)
    O.track(bwd, p, 2)
    H.flip_R(p)
    for k, scale in (("x", 1e-3), ("px", 1e-4), ("y", 1e-3), ("py", 1e-4), ("zeta", 0.02), ("delta", 3e-4)):
        # cosh / sinh amplify rounding by e^(w L) ~ 6 per pass in the defocusing plane: 1e-11, not the 1e-13 of P4
        assert np.max(np.abs(p[k] - p0[k])) < 1e-11 * scale, k


def test_P13_thick_quadrupole_rejects_degenerate_parameters():
    for bad in (Quadrupole(0.0, 1.0), Quadrupole(0.1, 0.0), Quadrupole(0.1, -1.0), Quadrupole(math.nan, 1.0)):
        with pytest.raises(ValueError):
            O.reference(pack([bad]))
    assert abs(O.s_table(pack([Quadrupole(0.1, 2.5), Drift(1.0), Marker()]))[2] - 3.5) < 1e-15


# ----------------------------- P14 thick sector bend (reading A19)
from xt_inputs.packed import Bend  # noqa: E402


def _thin_sliced_bend(k0, h, length, n):
    """n symmetric slices [drift, thin curved dipole, drift] of the maps pinned above (P1, P5 W2, P12)."""
    d = length / (2 * n)
    return [Drift(d), Multipole(knl=(k0 * length / n,), hxl=h * length / n, length=length / n), Drift(d)] * n


@pytest.mark.parametrize("k0,h,length,n", [(2.5e-3, 2.5e-3, 14.3, 4), (2.5005e-3, 2.5e-3, 14.3, 4),
                                           (-2.2004e-3, -2.2e-3, 14.3, 4), (0.05, 0.05, 8.0, 64)])
def test_P14_thick_bend_is_the_limit_of_thin_slices(k0, h, length, n):
    """The 'expanded' sector bend is the exact flow of the Hamiltonian whose kick the thin curved
    multipole applies; n symmetric slices converge to it as 1/n^2 (x, px, y, zeta: curvature, weak
    focusing, dispersion and all three path-length terms).  What Richardson extrapolation leaves is
    the exact-drift vs paraxial difference: cubic in the amplitude."""
    length = 14.3
    base = np.array([[1e-3, 2e-4, -5e-4, 1e-4, 0.01, 3e-4], [-2e-3, -1e-4, 1e-3, 3e-4, -0.02, -8e-4],
                     [5e-4, 0.0, 0.0, -2e-4, 0.0, 0.0]])

    def run(els, start):
        buf = pack(els)
        p = O.new_particles(buf, start)
        O.track(buf, p, 1)
        return np.stack([p[k] for k in ("x", "px", "y", "py", "zeta")], axis=1)

    residual = {}
    for amp in (1.0, 0.1):
        rows = base.copy()
        rows[:, :4] *= amp
        rows[:, 5] *= amp                                           # dispersion moves x by delta/h: scale it too
        start = H.coords_from_rows(rows.tolist())
        thick = run([Bend(k0, h, length)], start)
        s1, s2 = run(_thin_sliced_bend(k0, h, length, n), start), run(_thin_sliced_bend(k0, h, length, 2 * n), start)
        rich = (4.0 * s2 - s1) / 3.0
        residual[amp] = (rich - thick)[:, :3]
        if amp == 0.1:
            e1, e2 = np.abs(s1 - thick)[:, [0, 1, 2, 4]], np.abs(s2 - thick)[:, [0, 1, 2, 4]]
            big = e1 > 50.0 * np.abs(rich - thick)[:, [0, 1, 2, 4]] + 1e-16   # above the paraxial residual (y: pure drift)
            assert big.sum() >= 5
            assert np.all((e1[big] / e2[big] > 3.6) & (e1[big] / e2[big] < 4.4))      # second order in 1/n
            scale = amp * np.array([1e-3, 1e-4, 1e-3])
            assert np.max(np.abs(residual[amp]) / scale) < 1e-7
            slip, slip_thin = thick[:, 4] - rows[:, 4], rich[:, 4] - rows[:, 4]
            assert np.all(np.abs(slip) > 1e-9)                                         # h x L dominates the slip
            assert np.max(np.abs(slip_thin - slip) / np.abs(slip)) < 1e-6
            assert np.array_equal(thick[:, 3], rows[:, 3])                             # py untouched
    strong = np.abs(residual[1.0]) > 1e-11
    assert strong.sum() >= 3
    ratio = residual[1.0][strong] / residual[0.1][strong]
    # third order in (amplitude, delta): a linear error of the map would give 10, a quadratic one 100
    assert np.all((ratio > 400.0) & (ratio < 2500.0)), ratio


def test_P14_thick_bend_matrix_dispersion_symplectic_reversible():
    h, length = 2.5e-3, 14.3
    buf = pack([Bend(h, h, length)])
    J = H.jacobian6(O.track, buf, np.zeros(6))
    phi = h * length
    # textbook sector-bend matrix (x, px) and dispersion column; drift in y
    np.testing.assert_allclose(J[0:2, 0:2], [[math.cos(phi), math.sin(phi) / h], [-h * math.sin(phi), math.cos(phi)]],
                               atol=1e-8)
    np.testing.assert_allclose(J[2:4, 2:4], [[1.0, length], [0.0, 1.0]], atol=1e-8)
    beta0, _ = O.reference(buf)
    # d x / d delta = (1 - cos phi)/h, d px / d delta = sin phi; delta = pzeta * (beta0 ... ) at the origin: d delta/d pzeta = beta0/beta = 1
    assert abs(J[0, 5] - (1.0 - math.cos(phi)) / h) < 1e-6 and abs(J[1, 5] - math.sin(phi)) < 1e-7
    line = [Drift(0.7), Bend(h, h, length), Drift(0.4), Bend(1.0002 * h, h, 3.0), Cavity(1e6, 200e6, 180.0), Drift(0.2)]
    for z0 in (np.zeros(6), np.array([1e-3, 2e-4, -5e-4, 1e-4, 0.01, 3e-4])):
        _check_symplectic(pack(line), z0)
    rng = np.random.default_rng(9)
    n = 32
    co = dict(x=rng.normal(0, 1e-3, n), px=rng.normal(0, 1e-4, n), y=rng.normal(0, 1e-3, n),
              py=rng.normal(0, 1e-4, n), zeta=rng.normal(0, 0.02, n), delta=rng.normal(0, 3e-4, n))
    fwd, bwd = pack(line), pack(H.reversed_lattice(line))
    p = O.new_particles(fwd, co)
    p0 = O.copy_particles(p)
    O.track(fwd, p, 2)
    H.flip_R(p)
    O.track(bwd, p, 2)
    H.flip_R(p)
    for k, scale in (("x", 1e-3), ("px", 1e-4), ("y", 1e-3), ("py", 1e-4), ("zeta", 0.02), ("delta", 3e-4)):
        assert np.max(np.abs(p[k] - p0[k])) < 1e-12 * scale, k


def test_P14_thick_bend_rejects_degenerate_parameters():
    for bad in (Bend(0.0, 1e-3, 1.0), Bend(1e-3, 0.0, 1.0), Bend(1e-3, -1e-3, 1.0), Bend(1e-3, 1e-3, 0.0)):
        with pytest.raises(ValueError):
            O.reference(pack([bad]))
    assert abs(O.s_table(pack([Bend(1e-3, 1e-3, 2.5), Drift(1.0), Marker()]))[2] - 3.5) < 1e-15


# ----------------------------- P18 dispersion and chromaticity from tracking
def test_P18_fodo_chromaticity_and_textbook_dispersion():
    """oracle/make_optics.chromatic_optics_of against (a) the natural chromaticity of the thin-lens FODO
    cell, d mu/d delta = -2 tan(mu/2) (every focal length scales as 1 + delta), and (b) the periodic
    dispersion of a ring of thin quadrupoles and thin sector dipoles from 3x3 (x, px, delta) matrices."""
    from oracle import make_optics as MO
    n_cells, L, kq = 10, 2.0, 0.1
    cell = [Multipole(knl=(0.0, kq)), Drift(L), Multipole(knl=(0.0, -kq)), Drift(L)]
    got = MO.chromatic_optics_of(pack(cell * n_cells))
    mu = math.acos(1.0 - (L * kq) ** 2 / 2.0)
    want = -n_cells * math.tan(mu / 2.0) / math.pi
    assert abs(got["dqx"] - want) < 2e-6 * abs(want) and abs(got["dqy"] - want) < 2e-6 * abs(want)
    assert max(abs(got[k]) for k in ("dx", "dpx", "dy", "dpy")) < 1e-9                # no bends: no dispersion

    n_cells, L, kq, ell = 8, 3.0, 0.25, 1.5
    th = 2.0 * math.pi / (2 * n_cells)                                               # two dipoles per cell close the ring
    bend = Multipole(knl=(th,), hxl=th, length=ell)
    cell = [Multipole(knl=(0.0, kq)), Drift(L), bend, Drift(L), Multipole(knl=(0.0, -kq)), Drift(L), bend, Drift(L)]
    got = MO.chromatic_optics_of(pack(cell * n_cells))

    def quad(k):
        return np.array([[1.0, 0.0, 0.0], [-k, 1.0, 0.0], [0.0, 0.0, 1.0]])
    drift = np.array([[1.0, L, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]])
    dip = np.array([[1.0, 0.0, 0.0], [-th * th / ell, 1.0, th], [0.0, 0.0, 1.0]])    # px' = px + th delta - (k0 h l) x
    m = np.eye(3)
    for e in (quad(kq), drift, dip, drift, quad(-kq), drift, dip, drift):
        m = e @ m
    d = np.linalg.solve(np.eye(2) - m[:2, :2], m[:2, 2])
    assert abs(d[0]) > 1.0
    assert abs(got["dx"] - d[0]) < 1e-6 * abs(d[0]) and abs(got["dpx"] - d[1]) < 1e-6 * max(abs(d[1]), 0.1)
    assert abs(got["dy"]) < 1e-9 and abs(got["x_co"]) < 1e-12
    cosmu = 0.5 * (m[0, 0] + m[1, 1])
    q_cell = math.acos(cosmu) / (2 * math.pi)
    assert abs(got["qx_frac"] - (n_cells * q_cell) % 1.0) < 1e-8


# ----------------------------- P19 optics along the line
def test_P19_optics_along_a_fodo_ring_and_a_ring_with_dipoles():
    """oracle/make_optics.optics_along against the thin-FODO textbook: beta = 2L(1 +- sin(mu/2))/sin(mu) in the
    quadrupoles (L = half cell), alpha = -+ beta k/2 at their entrances, beta(s) = beta - 2 alpha s + gamma s^2
    in a drift, the phase grows by mu per cell; and the dispersion propagated by 3x3 matrices (P18's ring)."""
    from oracle import make_optics as MO
    n_cells, L, kq = 10, 2.0, 0.1
    cell = [Multipole(knl=(0.0, kq)), Drift(L / 2), Marker(), Drift(L / 2), Multipole(knl=(0.0, -kq)), Drift(L)]
    els = cell * n_cells
    on, rows = MO.optics_along(els, H.P0C, H.MASS0, H.Q0, list(range(len(els) + 1)))
    mu = math.acos(1.0 - (L * kq) ** 2 / 2.0)
    bmax, bmin = 2 * L * (1 + math.sin(mu / 2)) / math.sin(mu), 2 * L * (1 - math.sin(mu / 2)) / math.sin(mu)
    for c in range(n_cells):
        qf, mid, qd = rows[6 * c], rows[6 * c + 2], rows[6 * c + 4]
        assert abs(qf["betx"] - bmax) < 1e-6 and abs(qf["bety"] - bmin) < 1e-6
        assert abs(qd["betx"] - bmin) < 1e-6 and abs(qd["bety"] - bmax) < 1e-6
        assert abs(qf["alfx"] + bmax * kq / 2) < 1e-7 and abs(qd["alfx"] - bmin * kq / 2) < 1e-7
        assert abs(qf["alfy"] - bmin * kq / 2) < 1e-7 and abs(qd["alfy"] + bmax * kq / 2) < 1e-7
        # behind the thin QF: alpha = +beta k/2; half a drift further
        a1, g1 = bmax * kq / 2, (1 + (bmax * kq / 2) ** 2) / bmax
        assert abs(mid["betx"] - (bmax - 2 * a1 * (L / 2) + g1 * (L / 2) ** 2)) < 1e-6
        assert abs(mid["alfx"] - (a1 - g1 * (L / 2))) < 1e-7
        assert abs((qf["mux"] - c * mu + 1e-9) % (2 * math.pi) - 1e-9) < 1e-7 and abs((qf["muy"] - c * mu + 1e-9) % (2 * math.pi) - 1e-9) < 1e-7
        assert rows[6 * c + 2] is mid and abs(rows[6 * c + 3]["betx"] - mid["betx"]) < 1e-12     # a marker changes nothing
    end = rows[-1]
    assert abs(end["betx"] - on["betx"]) < 1e-6 and abs(end["alfx"] - on["alfx"]) < 1e-7        # periodic
    assert abs((end["mux"] - n_cells * mu) % (2 * math.pi)) < 1e-7 or abs((end["mux"] - n_cells * mu) % (2 * math.pi) - 2 * math.pi) < 1e-7

    n_cells, L, kq, ell = 8, 3.0, 0.25, 1.5
    th = 2.0 * math.pi / (2 * n_cells)
    bend = Multipole(knl=(th,), hxl=th, length=ell)
    cell = [Multipole(knl=(0.0, kq)), Drift(L), bend, Drift(L), Multipole(knl=(0.0, -kq)), Drift(L), bend, Drift(L)]
    els = cell * n_cells
    on, rows = MO.optics_along(els, H.P0C, H.MASS0, H.Q0, list(range(9)) + [len(els)])
    quad = lambda k: np.array([[1.0, 0.0, 0.0], [-k, 1.0, 0.0], [0.0, 0.0, 1.0]])
    drift = np.array([[1.0, L, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]])
    dip = np.array([[1.0, 0.0, 0.0], [-th * th / ell, 1.0, th], [0.0, 0.0, 1.0]])
    mats = [quad(kq), drift, dip, drift, quad(-kq), drift, dip, drift]
    m = np.eye(3)
    for e in mats:
        m = e @ m
    d = np.append(np.linalg.solve(np.eye(2) - m[:2, :2], m[:2, 2]), 1.0)
    for i in range(9):
        assert abs(rows[i]["dx"] - d[0]) < 1e-6 * max(abs(d[0]), 1.0) and abs(rows[i]["dpx"] - d[1]) < 1e-6, i
        assert abs(rows[i]["x"]) < 1e-12 and abs(rows[i]["dy"]) < 1e-9
        if i < 8:
            d = mats[i] @ d
    assert abs(rows[-1]["dx"] - rows[0]["dx"]) < 1e-6


# ----------------------------- P20 linear normal form with coupling
def test_P20_normal_form_uncoupled_rotated_and_closest_tune_approach():
    """oracle/make_optics.normal_form4 against (a) Courant-Snyder in an uncoupled ring: mode 1 is the
    horizontal plane, beta_y1 = beta_x2 = 0; (b) the same ring seen from a frame rotated by theta about s:
    tunes unchanged, Mais-Ripken beta_x1 = cos^2 beta_x, beta_y1 = sin^2 beta_x, beta_x2 = sin^2 beta_y,
    beta_y2 = cos^2 beta_y; (c) a thin skew quadrupole in a ring with equal tunes splits them by
    |ks| sqrt(beta_x beta_y) / (2 pi) (closest tune approach, first order in ks)."""
    from oracle import make_optics as MO
    n_cells, L, kq = 10, 2.0, 0.1
    cell = [Multipole(knl=(0.0, kq)), Drift(L), Multipole(knl=(0.0, -0.95 * kq)), Drift(L)]    # unequal strengths: Qx != Qy
    els = cell * n_cells
    on = MO.optics_of(pack(els))
    nf = MO.normal_form4(on["m"])
    assert abs(nf["betx1"] / on["betx"] - 1) < 1e-7 and abs(nf["bety2"] / on["bety"] - 1) < 1e-7
    assert abs(nf["alfx1"] - on["alfx"]) < 1e-7 and abs(nf["alfy2"] - on["alfy"]) < 1e-7
    assert nf["bety1"] < 1e-12 and nf["betx2"] < 1e-12
    assert abs(nf["q1_frac"] - on["qx_frac"]) < 1e-9 and abs(nf["q2_frac"] - on["qy_frac"]) < 1e-9
    assert abs(on["qx_frac"] - on["qy_frac"]) > 0.01

    th = 0.3
    rot = [SRotation.from_angle(-th)] + els + [SRotation.from_angle(th)]
    nfr = MO.normal_form4(MO.optics_of(pack(rot))["m"])
    c2, s2 = math.cos(th) ** 2, math.sin(th) ** 2
    assert abs(nfr["q1_frac"] - nf["q1_frac"]) < 1e-9 and abs(nfr["q2_frac"] - nf["q2_frac"]) < 1e-9
    assert abs(nfr["betx1"] - c2 * on["betx"]) < 1e-6 and abs(nfr["bety1"] - s2 * on["betx"]) < 1e-6
    assert abs(nfr["betx2"] - s2 * on["bety"]) < 1e-6 and abs(nfr["bety2"] - c2 * on["bety"]) < 1e-6
    assert abs(nfr["alfx1"] - c2 * on["alfx"]) < 1e-6 and abs(nfr["alfy2"] - c2 * on["alfy"]) < 1e-6

    # equal tunes: start in the middle of a drift of the symmetric cell, where beta_x = beta_y needs no care
    ks = 2e-5
    sym = [Multipole(knl=(0.0, kq)), Drift(L), Multipole(knl=(0.0, -kq)), Drift(L)] * n_cells
    on = MO.optics_of(pack(sym))
    assert abs(on["qx_frac"] - on["qy_frac"]) < 1e-9
    skew = [Multipole(knl=(0.0, 0.0), ksl=(0.0, ks))] + sym
    nfs = MO.normal_form4(MO.optics_of(pack(skew))["m"])
    split = abs(nfs["q1_frac"] - nfs["q2_frac"])
    want = ks * math.sqrt(on["betx"] * on["bety"]) / (2 * math.pi)
    assert abs(split / want - 1.0) < 2e-3, (split, want)
    assert abs(nfs["betx1"] / nfs["betx2"] - 1.0) < 0.05                     # fully mixed modes on the resonance
    # steps 4-5: carried along the line, the modes of an uncoupled ring are its planes
    on, rows = MO.optics_along(els, H.P0C, H.MASS0, H.Q0, list(range(0, len(els) + 1, 3)))
    for r in rows:
        assert abs(r["betx1"] / r["betx"] - 1) < 1e-7 and abs(r["bety2"] / r["bety"] - 1) < 1e-7
        assert r["bety1"] < 1e-10 and r["betx2"] < 1e-10
        for a, b in ((r["mu1"], r["mux"]), (r["mu2"], r["muy"])):
            d = (a - b) % (2 * math.pi)
            assert min(d, 2 * math.pi - d) < 1e-7
    # ... seen from the rotated frame: inside the two rotations the coordinates are the ring's own again (the
    # modes are its planes), at the start and at the end they carry the cos^2 / sin^2 shares
    on_r, rows_r = MO.optics_along(rot, H.P0C, H.MASS0, H.Q0, [0] + [1 + i for i in range(0, len(els) + 1, 3)] + [len(rot)])
    for r, rr in zip(rows, rows_r[1:-1]):
        assert abs(rr["betx1"] - r["betx"]) < 1e-5 and rr["bety1"] < 1e-9 and abs(rr["bety2"] - r["bety"]) < 1e-5
    for rr in (rows_r[0], rows_r[-1]):
        assert abs(rr["betx1"] - c2 * rows[0]["betx"]) < 1e-5 and abs(rr["bety1"] - s2 * rows[0]["betx"]) < 1e-5
        assert abs(rr["bety2"] - c2 * rows[0]["bety"]) < 1e-5 and abs(rr["betx2"] - s2 * rows[0]["bety"]) < 1e-5


# ----------------------------- P22 six-dimensional closed orbit and tunes
def test_P22_six_dimensional_closed_orbit_and_synchrotron_tune():
    """oracle/make_optics.optics6d_of: (a) drifts + cavity (pin P11's ring): cos mu_s = 1 - A B / 2 in closed
    form; (b) a cavity phased away from zero moves the fixed point to zeta = lag / kz; (c) a thin FODO ring with
    a cavity and no bends: the transverse tunes are the FODO closed form, the synchrotron tune the same formula."""
    from oracle import make_optics as MO
    p0c, volt, freq, circ = 1.0e9, 1e5, 200e6, 40.0
    buf = pack([Drift(circ / 4)] * 4 + [Cavity(volt, freq, 0.0)], p0c=p0c)
    beta0, gamma0 = O.reference(buf)
    kz = 2 * math.pi * freq / (beta0 * 299792458.0)
    A, B = circ / gamma0 ** 2, (volt / p0c) * kz / beta0
    # no transverse focusing at all: only the longitudinal 2x2 block of the 6x6 matrix is an oscillator
    J = MO.jac6(buf, np.zeros(6))
    mu_s = math.acos(1.0 - A * B / 2.0)
    assert abs(0.5 * (J[4, 4] + J[5, 5]) - math.cos(mu_s)) < 1e-9
    cell = [Multipole(knl=(0.0, 0.1)), Drift(2.0), Multipole(knl=(0.0, -0.095)), Drift(2.0)]
    for lag in (0.0, 25.0):
        buf = pack(cell * 10 + [Cavity(volt, freq, lag)], p0c=p0c)
        got = MO.optics6d_of(buf)
        np.testing.assert_allclose(got["co"][:4], 0.0, atol=1e-13)
        assert abs(got["co"][4] - math.radians(lag) / kz) < 1e-10 and abs(got["co"][5]) < 1e-13
        assert abs(got["qs"] - mu_s / (2 * math.pi)) < 1e-9
        flat = MO.optics_of(pack(cell * 10, p0c=p0c))
        assert abs(got["q1_frac"] - flat["qx_frac"]) < 1e-8 and abs(got["q2_frac"] - flat["qy_frac"]) < 1e-8
    assert abs(flat["qx_frac"] - flat["qy_frac"]) > 0.01
