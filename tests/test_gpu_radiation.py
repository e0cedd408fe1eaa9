""""Mean" synchrotron radiation in thin multipoles (reading A22) on the GPU path against
the oracle: bit-exact in the --fmad=false build on a cavity-free positron ring, 1e-12 after one turn and 1e-10
after 100 turns in the production build with the cavity that restores the energy; and the textbook damping of
a vertical oscillation, U0/2E per turn, measured on the GPU over 3000 turns."""
import math

import numpy as np
import pytest

import helpers as H

from oracle import oracle as O
from xt_inputs.packed import Cavity, Drift, LimitEllipse, Multipole, RadMultipole, pack_lattice

pytestmark = pytest.mark.gpu
ME, R_E = 0.51099895e6, 2.8179403262e-15
KEYS = ("x", "px", "y", "py", "zeta", "delta", "ptau")


@pytest.fixture(scope="module")
def X():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m gpu on the B200 box)")
    import paper_2310_00317_b200 as X
    return X


def ring(cavity, p0c=10e9, n_cells=32, ell=40.0, L=5.0, kq=0.12):
    th = 2.0 * math.pi / (2 * n_cells)
    bend = RadMultipole(knl=(th,), hxl=th, length=ell)
    quad_f = RadMultipole(knl=(0.0, kq, 0.5), ksl=(0.0, 1e-4), length=0.5)           # quadrupoles radiate off axis
    cell = [quad_f, Drift(L), bend, Drift(L), Multipole(knl=(0.0, -kq)), Drift(L), bend, Drift(L), LimitEllipse(0.03, 0.02)]
    gamma = math.sqrt(p0c ** 2 + ME ** 2) / ME
    u0_over_e = (2.0 / 3.0) * R_E * gamma ** 3 * th * th / ell * 2 * n_cells
    els = cell * n_cells
    if cavity:
        els = els + [Cavity(3.0 * u0_over_e * p0c, 400e6, 180.0 - math.degrees(math.asin(1.0 / 3.0)))]
    return els, u0_over_e


def ensemble(n, seed=9):
    rng = np.random.default_rng(seed)
    return dict(x=rng.normal(0, 1e-3, n), px=rng.normal(0, 5e-5, n), y=rng.normal(0, 1e-3, n), py=rng.normal(0, 5e-5, n),
                zeta=rng.normal(0, 0.01, n), delta=rng.normal(0, 3e-4, n))


@pytest.mark.parametrize("kind,cavity,turns", [("nofma", False, 20), ("prod", True, 1), ("prod", True, 100)])
def test_radiating_ring_matches_the_oracle(X, kind, cavity, turns):
    els, u0 = ring(cavity)
    buf = pack_lattice(els, 10e9, ME, 1.0)
    co = ensemble(2000)
    ref = O.new_particles(buf, co)
    mm = np.full(2000, np.inf)
    O.track(buf, ref, turns, threads=O.host_threads(), min_margin=mm)
    assert (ref["state"] == 1).mean() > 0.9
    if not cavity:
        assert abs(np.mean(ref["delta"] - co["delta"]) / (-turns * u0) - 1.0) < 0.05   # the beam has lost turns x U0
    lat = X.xt_lattice_create(buf, kind=kind)
    base = None
    for ppt, block in ((0, 0), (1, 32), (2, 64), (3, 128), (4, 128)):
        p = X.new_particles(lat, co)
        X.xt_track_ex(lat, p, turns, particles_per_thread=ppt, block_size=block)
        got = X.particles_to_host(p)
        if base is None:
            base = got
            clear = ~(mm < 1e-9)
            for k in ("state", "at_turn", "at_element"):
                assert np.array_equal(got[k][clear], ref[k][clear]), k
            if kind == "nofma":
                for k in KEYS + ("rpp", "rvv", "s"):
                    assert np.array_equal(got[k], ref[k]), k
            else:
                rtol = 1e-12 if turns == 1 else 1e-10
                for k in KEYS:
                    ok = np.abs(got[k] - ref[k]) <= np.maximum(rtol * np.abs(ref[k]), H.parity_atol(ref[k][clear], rtol))
                    assert ok[clear].all(), (k, int((~ok[clear]).sum()), float(np.max(np.abs(got[k] - ref[k])[clear])))
                for k in ("rpp", "rvv"):
                    assert np.max(np.abs(got[k][clear] - ref[k][clear])) < 1e-12, k
        else:
            for k in got:
                assert np.array_equal(got[k], base[k]), (ppt, k)                     # every launch shape bit-identical
    lat.close()
    for bad in (RadMultipole(knl=(1e-3,), length=0.0), RadMultipole(knl=tuple([0.0] * 22), length=1.0)):
        with pytest.raises(X.XtError) as e:
            X.xt_lattice_create(pack_lattice([bad], 10e9, ME, 1.0))
        assert e.value.code == -2


def test_vertical_damping_rate_on_the_gpu(X):
    els, u0 = ring(True)
    els = [e for e in els if not isinstance(e, LimitEllipse)]
    buf = pack_lattice(els, 10e9, ME, 1.0)
    lat = X.xt_lattice_create(buf)
    tw = X.xt_twiss4d(lat)                                # optics with radiation: the orbit is the sawtooth one
    n = 256
    rng = np.random.default_rng(1)
    co = dict(x=np.full(n, tw["co"][0]), px=np.full(n, tw["co"][1]), y=tw["co"][2] + rng.normal(0, 1e-4, n),
              py=tw["co"][3] + rng.normal(0, 3e-6, n), zeta=np.zeros(n), delta=np.zeros(n))
    by, ay = tw["bety"], tw["alfy"]

    def action(h):
        y, py = h["y"] - tw["co"][2], (h["py"] - tw["co"][3]) / (1.0 + h["delta"])
        return np.mean(((1 + ay * ay) / by * y * y + 2 * ay * y * py + by * py * py) / 2.0)

    p = X.new_particles(lat, co)
    acts, marks = [], list(range(0, 3001, 250))
    done = 0
    for m in marks:
        X.xt_track(lat, p, m - done)
        done = m
        acts.append(action(X.particles_to_host(p)))
    lat.close()
    slope = np.polyfit(np.asarray(marks, dtype=float), np.log(acts), 1)[0]
    assert abs(slope / (-u0) - 1.0) < 0.03, (slope, u0)
