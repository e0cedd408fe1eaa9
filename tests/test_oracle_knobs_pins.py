"""Pin P17 of the CPU oracle: time functions (reading A21).

The oracle rebuilds the line every turn, so what needs pinning is the bookkeeping: which coefficient, which
step, in which turn.  (a) a ramped dipole kicker in a drift-only ring: the orbit is a double sum in closed
form (exact drift, pin P1); (b) a constant table is the static line with the summed strengths, bit for bit,
curved dipole with weak focusing included; (c) step0 shifts the table, steps beyond its ends hold the last /
first value; (d) two links on one coefficient add, normal and skew are separate; (e) a sextupole knob that
follows the derivative of the dipole knob (Fig. 1): tracked = static line per turn, and the kick of turn j
is the closed-form polynomial."""
import math

import numpy as np

from oracle import knobs as K
from oracle import oracle as O
from xt_inputs.packed import Cavity, Drift, LimitRect, Multipole, pack_lattice
import helpers as H


def pack(els):
    return pack_lattice(els, H.P0C, H.MASS0, H.Q0)


def fresh(els, rows):
    return O.new_particles(pack(els), H.coords_from_rows(rows))


def test_P17_ramped_kicker_in_a_drift_ring_closed_form():
    L, g, n_turns = 3.0, 2e-5, 12
    els = [Multipole(knl=(1e-6,)), Drift(L)]
    ramp = np.array([[0.5 * j for j in range(8)]])                        # holds 3.5 from turn 7 on
    rows = [[1e-3, 2e-5, -2e-3, 1e-5, 0.0, 0.0], [0.0, 0.0, 0.0, 0.0, 0.0, 4e-4]]
    p = fresh(els, rows)
    K.track_with_knobs(els, H.P0C, H.MASS0, H.Q0, p, n_turns, ramp, [(0, 0, 0, 0, g)])
    for i, r in enumerate(rows):
        x, px, y, py, opd = r[0], r[1], r[2], r[3], 1.0 + r[5]
        for j in range(n_turns):
            px = px - (1e-6 + g * 0.5 * min(j, 7))                         # thin dipole: px' = px - k0l (pin P5)
            pz = math.sqrt(opd * opd - px * px - py * py)
            x, y = x + L * px / pz, y + L * py / pz                        # exact drift (pin P1)
        assert abs(p["x"][i] - x) < 1e-15 and abs(p["px"][i] - px) < 1e-18 and abs(p["y"][i] - y) < 1e-15
    assert np.all(p["at_turn"] == n_turns)


def test_P17_constant_table_is_the_static_line_and_links_add():
    base = [Multipole(knl=(2e-4, 0.01, 0.2), ksl=(0.0, 1e-3), hxl=2e-4, length=0.5), Drift(2.0),
            Multipole(knl=(0.0, -0.012), ksl=(0.0, 0.0, 0.0, 3.0)), Drift(2.0), Cavity(1e6, 200e6, 10.0),
            LimitRect(-0.004, 0.004, -0.004, 0.004)]
    table = np.array([[0.7] * 3, [-1.3] * 3])
    links = [(0, 0, 0, 0, 1e-5), (0, 2, 0, 1, 0.05), (0, 2, 0, 0, 0.02), (0, 1, 1, 1, 1e-4), (2, 3, 1, 0, 0.5),
             (2, 3, 0, 1, 0.25)]
    static = [Multipole(knl=(2e-4 + 1e-5 * 0.7, 0.01, (0.2 + 0.05 * -1.3) + 0.02 * 0.7), ksl=(0.0, 1e-3 + 1e-4 * -1.3),
                        hxl=2e-4, length=0.5), Drift(2.0),
              Multipole(knl=(0.0, -0.012, 0.0, 0.25 * -1.3), ksl=(0.0, 0.0, 0.0, 3.0 + 0.5 * 0.7)), Drift(2.0),
              Cavity(1e6, 200e6, 10.0), LimitRect(-0.004, 0.004, -0.004, 0.004)]
    rng = np.random.default_rng(2)
    rows = np.column_stack([rng.normal(0, 2e-3, 50), rng.normal(0, 2e-4, 50), rng.normal(0, 2e-3, 50),
                            rng.normal(0, 2e-4, 50), rng.normal(0, 0.02, 50), rng.normal(0, 5e-4, 50)]).tolist()
    a, b = fresh(base, rows), fresh(static, rows)
    K.track_with_knobs(base, H.P0C, H.MASS0, H.Q0, a, 7, table, links, step0=5)     # beyond the end: holds
    O.track(pack(static), b, 7)
    assert 0 < (b["state"] == 0).sum() < 50
    for k in a:
        assert np.array_equal(a[k], b[k], equal_nan=True), k


def test_P17_step0_shifts_the_table_and_the_ends_hold():
    els = [Multipole(knl=(0.0, 0.02)), Drift(1.5), Multipole(knl=(0.0, -0.02)), Drift(1.5)]
    f = np.array([[0.0, 1.0, -2.0, 0.5, 3.0, 1.5]])
    links = [(0, 0, 0, 0, 1e-5), (2, 1, 0, 0, 1e-3)]
    rows = [[1e-3, 0.0, 1e-3, 0.0, 0.0, 1e-4]]
    a = fresh(els, rows)
    K.track_with_knobs(els, H.P0C, H.MASS0, H.Q0, a, 4, f, links, step0=2)
    b = fresh(els, rows)
    K.track_with_knobs(els, H.P0C, H.MASS0, H.Q0, b, 4, f[:, 2:], links, step0=0)
    c = fresh(els, rows)
    K.track_with_knobs(els, H.P0C, H.MASS0, H.Q0, c, 4, np.array([[-2.0, 0.5, 3.0, 1.5, 9.0]]), links, step0=0)
    d = fresh(els, rows)
    K.track_with_knobs(els, H.P0C, H.MASS0, H.Q0, d, 6, f, links, step0=-2)          # two turns at f[0], then f[0..3]
    e = fresh(els, rows)
    K.track_with_knobs(els, H.P0C, H.MASS0, H.Q0, e, 6, np.array([[0.0, 0.0, 0.0, 1.0, -2.0, 0.5]]), links)
    for k in a:
        assert np.array_equal(a[k], b[k]) and np.array_equal(a[k], c[k]) and np.array_equal(d[k], e[k]), k
    assert not np.array_equal(a["x"], d["x"])


def test_P17_eddy_current_sextupole_follows_the_derivative_of_the_dipole():
    """Fig. 1: corrector strength I(t) and an induced sextupole proportional to dI/dt."""
    n = 10
    cur = np.sin(np.linspace(0.0, math.pi, n)) ** 2
    table = np.stack([cur, np.gradient(cur)])
    els = [Multipole(knl=(0.0, 0.0, 0.0)), Drift(1.0)]
    links = [(0, 0, 0, 0, 3e-5), (0, 2, 0, 1, 4.0)]
    rows = [[2e-3, 0.0, 1e-3, 0.0, 0.0, 0.0]]
    p = fresh(els, rows)
    x, y, px, py = 2e-3, 1e-3, 0.0, 0.0
    for j in range(n):
        K.track_with_knobs(els, H.P0C, H.MASS0, H.Q0, p, 1, table, links, step0=j)
        k0, k2 = 3e-5 * table[0][j], 4.0 * table[1][j]
        px, py = px - (k0 + 0.5 * k2 * (x * x - y * y)), py + 0.5 * k2 * (2.0 * x * y)   # thin multipole (pin P5)
        pz = math.sqrt(1.0 - px * px - py * py)
        x, y = x + px / pz, y + py / pz
        assert abs(p["x"][0] - x) < 1e-15 and abs(p["py"][0] - py) < 1e-18, j
