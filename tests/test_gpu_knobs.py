"""Time functions (reading A21) on the GPU path against the
oracle (``oracle/knobs.py``: the line rebuilt and tracked turn by turn): bit-exact in the --fmad=false build on
a cavity-free ring, 1e-12 per turn / 1e-10 over 100 turns in the production build; the image is back at its
base values afterwards."""
import numpy as np
import pytest

import helpers as H

from oracle import knobs as K
from oracle import oracle as O
from xt_inputs.packed import (Cavity, Drift, LimitEllipse, Multipole, SRotation, XYShift, pack_lattice)

pytestmark = pytest.mark.gpu
P0C, MASS0 = 450e9, 938272088.16
KEYS = ("x", "px", "y", "py", "zeta", "delta", "ptau")


@pytest.fixture(scope="module")
def X():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m gpu on the B200 box)")
    import paper_2310_00317_b200 as X
    return X


def bump_ring(cavity):
    """12 FODO cells with sextupoles; four orbit correctors (one of them a misaligned, fused record, one on a
    curved dipole with weak focusing) driven by two knobs, plus the eddy-current sextupole of Fig. 1."""
    cell = [Multipole(knl=(0.0, 0.11)), Drift(2.5), Multipole(knl=(0.0, 0.0, 0.4)), Drift(2.5),
            Multipole(knl=(0.0, -0.11)), Drift(2.5), Multipole(knl=(0.0, 0.0, -0.4)), Drift(2.5), LimitEllipse(0.007, 0.006)]
    els, idx = [], []
    for c in range(12):
        els += cell
        if c in (2, 5):
            idx.append(len(els))
            els += [Multipole(knl=(0.0, 0.0, 0.0), ksl=(0.0,)), Drift(0.3)]
        if c == 7:
            idx.append(len(els) + 2)
            els += [XYShift(1e-4, -2e-4), SRotation.from_angle(0.01), Multipole(knl=(1e-6, 0.0), ksl=(0.0, 1e-4)),
                    SRotation.from_angle(-0.01), XYShift(-1e-4, 2e-4), Drift(0.3)]
        if c == 9:
            idx.append(len(els))
            els += [Multipole(knl=(3e-4,), hxl=3e-4, length=0.4), Drift(0.3)]
    if cavity:
        els += [Cavity(1e6, 200e6, 180.0)]
    return els, idx


def knobs_for(els, idx, n_steps):
    t = np.arange(n_steps)
    cur = np.sin(np.pi * t / (n_steps - 1)) ** 2                     # corrector current
    table = np.stack([cur, np.gradient(cur), 0.3 * np.cos(0.37 * t)])
    c0, c1, c2, c3 = idx[:4]
    links = [(c0, 0, 0, 0, 4e-5), (c1, 0, 0, 0, -3e-5), (c0, 2, 0, 1, 6.0), (c1, 2, 0, 1, -5.0),
             (c2, 0, 0, 2, 1e-5), (c2, 1, 1, 0, 2e-3), (c2, 0, 1, 2, -1e-5), (c3, 0, 0, 0, 2e-5), (c0, 0, 0, 2, 1e-5)]
    return table, links


def ensemble(n, seed=5):
    rng = np.random.default_rng(seed)
    return dict(x=rng.normal(0, 1.5e-3, n), px=rng.normal(0, 1e-4, n), y=rng.normal(0, 1.5e-3, n),
                py=rng.normal(0, 1e-4, n), zeta=rng.normal(0, 0.05, n), delta=rng.normal(0, 3e-4, n))


@pytest.mark.parametrize("kind,cavity,turns", [("nofma", False, 60), ("prod", True, 1), ("prod", True, 100)])
def test_knobs_match_the_oracle(X, kind, cavity, turns):
    els, idx = bump_ring(cavity)
    assert len(idx) == 4
    table, links = knobs_for(els, idx, 48)
    buf = pack_lattice(els, P0C, MASS0, 1.0)
    co = ensemble(3000)
    ref = O.new_particles(buf, co)
    mm = np.full(3000, np.inf)
    K.track_with_knobs(els, P0C, MASS0, 1.0, ref, turns, table, links, step0=-3, threads=O.host_threads(), min_margin=mm)
    static = O.new_particles(buf, co)
    O.track(buf, static, turns, threads=O.host_threads())
    assert np.max(np.abs(static["x"] - ref["x"])) > 1e-4                 # the bump is there

    lat = X.xt_lattice_create(buf, kind=kind)
    X.xt_lattice_set_knobs(lat, table, links)
    p = X.new_particles(lat, co)
    launches = X.xt_launch_count(kind)
    X.xt_track_knobs(lat, p, turns, step0=-3)
    assert X.xt_launch_count(kind) - launches == 2 * turns + 1           # (apply, track) per turn + restore
    got = X.particles_to_host(p)
    clear = ~(mm < 1e-9)
    for k in ("state", "at_turn", "at_element"):
        assert np.array_equal(got[k][clear], ref[k][clear]), k
    if turns >= 60:
        assert 10 < (ref["state"] == 0).sum() < 2500
    if kind == "nofma":
        for k in KEYS + ("s", "rpp", "rvv"):
            assert np.array_equal(got[k], ref[k]), k
    else:
        rtol = 1e-12 if turns == 1 else 1e-10
        for k in KEYS:
            ok = np.abs(got[k] - ref[k]) <= np.maximum(rtol * np.abs(ref[k]), H.parity_atol(ref[k][clear], rtol))
            assert ok[clear].mean() > (0.999 if turns > 1 else 1.0 - 1e-12), (k, float(ok[clear].mean()))
    # the image is back at base: a plain xt_track equals a fresh lattice, bit for bit; and the knobs can be dropped
    fresh = X.xt_lattice_create(buf, kind=kind)
    a, b = X.new_particles(lat, co), X.new_particles(fresh, co)
    X.xt_track(lat, a, 3)
    X.xt_track(fresh, b, 3)
    ha, hb = X.particles_to_host(a), X.particles_to_host(b)
    for k in ha:
        assert np.array_equal(ha[k], hb[k], equal_nan=True), k
    X.xt_lattice_set_knobs(lat, table, [])
    with pytest.raises(X.XtError) as e:
        X.xt_track_knobs(lat, a, 1)
    assert e.value.code == -1
    lat.close()
    fresh.close()


def test_knob_argument_errors_and_step_clamping(X):
    els, idx = bump_ring(False)
    buf = pack_lattice(els, P0C, MASS0, 1.0)
    lat = X.xt_lattice_create(buf)
    table = np.array([[0.0, 1.0, 2.0]])
    for bad in ([(1, 0, 0, 0, 1.0)],                       # a drift
                [(idx[0], 3, 0, 0, 1.0)],                  # order beyond the element's
                [(idx[0], 0, 2, 0, 1.0)], [(idx[0], 0, 0, 1, 1.0)], [(len(els), 0, 0, 0, 1.0)]):
        with pytest.raises(X.XtError) as e:
            X.xt_lattice_set_knobs(lat, table, bad)
        assert e.value.code == -2
    with pytest.raises(X.XtError) as e:
        X.xt_lattice_set_knobs(lat, np.array([[0.0, float("nan")]]), [(idx[0], 0, 0, 0, 1.0)])
    assert e.value.code == -1
    # steps beyond the table hold its ends: 5 turns from step0 = 1 use f = 1, 2, 2, 2, 2
    X.xt_lattice_set_knobs(lat, table, [(idx[0], 0, 0, 0, 2e-5)])
    co = ensemble(64)
    p = X.new_particles(lat, co)
    X.xt_track_knobs(lat, p, 5, step0=1)
    ref = O.new_particles(buf, co)
    K.track_with_knobs(els, P0C, MASS0, 1.0, ref, 5, [[1.0, 2.0, 2.0, 2.0, 2.0]], [(idx[0], 0, 0, 0, 2e-5)])
    got = X.particles_to_host(p)
    for k in KEYS:
        assert np.all(np.abs(got[k] - ref[k]) <= np.maximum(1e-11 * np.abs(ref[k]), H.parity_atol(ref[k], 1e-11))), k
    lat.close()
