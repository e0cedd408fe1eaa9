"""Thick quadrupole on the GPU path (reading A18) against the
oracle, element by element: a FODO ring of thick quadrupoles with a cavity, sextupoles and an
aperture, 1 turn at 1e-12 and 100 turns at 1e-10; every launch shape bit-identical; losses exact.
(sin / cos / sinh / cosh differ from glibc by <= 2 ulp, so there is no bit-exact leg, as for cavities.)
"""
import numpy as np
import pytest

import helpers as H

from oracle import oracle as O
from xt_inputs.packed import Cavity, Drift, LimitEllipse, Marker, Multipole, Quadrupole, pack_lattice

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


def thick_fodo(n_cells=12, aperture=0.03):
    cell = [Quadrupole(+0.12, 0.8), Drift(1.6), Multipole(knl=(0.0, 0.0, 0.4)), Drift(0.4),
            Quadrupole(-0.12, 0.8), Drift(2.0), LimitEllipse(aperture, aperture), Marker()]
    return cell * n_cells + [Cavity(1e6, 200e6, 180.0)]


def ensemble(n, scale=1.0, seed=21):
    rng = np.random.default_rng(seed)
    return dict(x=rng.normal(0, 2e-4 * scale, n), px=rng.normal(0, 2e-5 * scale, n),
                y=rng.normal(0, 2e-4 * scale, n), py=rng.normal(0, 2e-5 * scale, n),
                zeta=rng.normal(0, 0.05, n), delta=rng.normal(0, 3e-4, n))


def close(got, ref, rtol, sel):
    H.assert_parity(got, ref, rtol, sel=sel, keys=KEYS)      # reading A8: per-coordinate floor


def test_thick_quadrupole_ring_parity(X):
    buf = pack_lattice(thick_fodo(), P0C, MASS0, 1.0)
    co = ensemble(5000)
    lat = X.xt_lattice_create(buf)
    assert lat.info["n_thick"] == 24 and lat.info["circumference"] == pytest.approx(12 * 5.6)
    for turns, rtol in ((1, 1e-12), (100, 1e-10)):
        ref = O.new_particles(buf, co)
        O.track(buf, ref, turns, threads=O.host_threads())
        p = X.new_particles(lat, co)
        X.xt_track(lat, p, turns)
        got = X.particles_to_host(p)
        assert (ref["state"] == 1).all() and np.array_equal(got["state"], ref["state"])
        assert np.array_equal(got["at_turn"], ref["at_turn"])
        close(got, ref, rtol, ref["state"] == 1)
    lat.close()


def test_thick_quadrupole_losses_shapes_and_s(X):
    """Large amplitudes in a tight aperture: losses must match the oracle exactly (outside the edge
    band), s counts the thick lengths, and every launch shape gives the same bits."""
    els = thick_fodo(aperture=0.004)
    buf = pack_lattice(els, P0C, MASS0, 1.0)
    co = ensemble(3000, scale=6.0)
    ref = O.new_particles(buf, co)
    mm = np.full(3000, np.inf)
    O.track(buf, ref, 20, threads=O.host_threads(), min_margin=mm)
    assert 0.1 < (ref["state"] == 0).mean() < 0.9
    lat = X.xt_lattice_create(buf)
    np.testing.assert_allclose(X.xt_lattice_s_table(lat), O.s_table(buf), rtol=0, atol=1e-12)
    base = None
    for ppt, block in ((0, 0), (1, 32), (2, 96), (3, 128), (4, 64)):
        p = X.new_particles(lat, co)
        X.xt_track_ex(lat, p, 20, particles_per_thread=ppt, block_size=block, compact_every=-1 if ppt else 7)
        got = X.particles_to_host(p)
        if base is None:
            base = got
            clear = mm >= 1e-9
            for k in ("state", "at_turn", "at_element"):
                assert np.array_equal(got[k][clear], ref[k][clear]), k
            lost = clear & (ref["state"] == 0)
            assert np.array_equal(got["s"][lost], ref["s"][lost])
            close(got, ref, 1e-11, clear & (ref["state"] == 1))
        else:
            for k in got:
                a, b = got[k], base[k]
                same = (a == b) | (np.isnan(a.astype(np.float64)) & np.isnan(b.astype(np.float64)))
                assert same.all(), (ppt, block, k)
    lat.close()


def test_thick_quadrupole_bad_parameters(X):
    for bad in (Quadrupole(0.0, 1.0), Quadrupole(0.1, 0.0), Quadrupole(0.1, -2.0)):
        with pytest.raises(X.XtError) as e:
            X.xt_lattice_create(pack_lattice([bad], P0C, MASS0, 1.0))
        assert e.value.code == -2
