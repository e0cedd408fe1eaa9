"""Polygon apertures and loss-location refinement (DESIGN.md reading
A20) on the GPU path against the oracle (``oracle/refine.py`` + the oracle tracker): which polygon stops a
particle is an integer decision -- compared exactly wherever the oracle's distance to the polygon edge
exceeds 1e-9 m -- and the refined records agree to 1e-12."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from oracle import refine as R
from xt_inputs.packed import (Cavity, Drift, LimitEllipse, LimitPolygon, LimitRect, Marker, Multipole, Quadrupole,
                              SRotation, XYShift, pack_lattice)

pytestmark = pytest.mark.gpu
P0C, MASS0 = 450e9, 938272088.16
KEYS = ("x", "px", "y", "py", "zeta", "delta", "ptau")
SCALE = dict(x=1e-3, px=1e-4, y=1e-3, py=1e-4, zeta=1e-2, delta=1e-4, ptau=1e-4, s=1.0)


@pytest.fixture(scope="module")
def X():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m gpu on the B200 box)")
    import paper_2310_00317_b200 as X
    return X


def ensemble(n, sx, sp, seed):
    rng = np.random.default_rng(seed)
    return dict(x=rng.normal(0, sx, n), px=rng.normal(0, sp, n), y=rng.normal(0, sx, n), py=rng.normal(0, sp, n),
                zeta=rng.normal(0, 0.03, n), delta=rng.normal(0, 5e-4, n))


def star(n, r0, r1, cx, cy, phase):
    ang = phase + 2 * np.pi * np.arange(n) / n
    r = np.where(np.arange(n) % 2 == 0, r0, r1)
    return LimitPolygon(tuple(cx + r * np.cos(ang)), tuple(cy + r * np.sin(ang)))


def test_polygon_aperture_parity_and_launch_shapes(X):
    """Convex and star-shaped polygons of 3 to 256 vertices between kicks and drifts."""
    els = [Drift(1.0), star(3, 0.014, 0.014, 0.0, 0.0, 0.3), Multipole(knl=(0.0, 0.05)), Drift(2.0),
           star(16, 0.012, 0.007, 1e-3, -5e-4, 0.1), Drift(1.5), Multipole(knl=(0.0, -0.05, 2.0)), Drift(2.5),
           star(256, 0.009, 0.0088, 0.0, 0.0, 0.0), Drift(1.0), LimitPolygon((-0.01, 0.01, 0.01, -0.01), (-0.006, -0.006, 0.006, 0.006))]
    buf = pack_lattice(els, P0C, MASS0, 1.0)
    co = ensemble(6000, 3e-3, 2e-4, 3)
    co["x"][:2] = [float("nan"), 0.0]
    ref = O.new_particles(buf, co)
    mm = np.full(6000, np.inf)
    O.track(buf, ref, 3, threads=O.host_threads(), min_margin=mm)
    lost_at = [int(((ref["state"] == 0) & (ref["at_element"] == i)).sum()) for i in (1, 4, 8, 10)]
    assert min(lost_at) > 20 and (ref["state"] == 1).sum() > 500, lost_at
    lat = X.xt_lattice_create(buf)
    clear = ~(mm < 1e-9)
    base = None
    for ppt, block in ((0, 0), (1, 32), (2, 64), (3, 128), (4, 128)):
        p = X.new_particles(lat, co)
        X.xt_track_ex(lat, p, 3, particles_per_thread=ppt, block_size=block)
        got = X.particles_to_host(p)
        if base is None:
            base = got
            for k in ("state", "at_turn", "at_element", "s"):
                assert np.array_equal(got[k][clear], ref[k][clear]), k
            assert got["state"][0] == 0 and got["at_element"][0] == 1
            for k in KEYS:
                ok = np.abs(got[k] - ref[k]) <= 1e-12 * np.maximum(np.abs(ref[k]), SCALE[k])
                assert ok[clear & ~np.isnan(ref[k])].all(), k
        else:
            for k in got:
                a, b = got[k].astype(np.float64), base[k].astype(np.float64)
                assert ((a == b) | (np.isnan(a) & np.isnan(b))).all(), (ppt, k)
    lat.close()
    for bad in (LimitPolygon((0.0, 1.0), (0.0, 1.0)), LimitPolygon(tuple(range(257)), tuple(range(257)))):
        with pytest.raises(X.XtError) as e:
            X.xt_lattice_create(pack_lattice([bad], P0C, MASS0, 1.0))
        assert e.value.code == -2


def fig4_line():
    """Rectangular and elliptical apertures, shifted and tilted differently (Fig. 4), with thin and
    thick magnets, a cavity and a nested misalignment in between; the first aperture has nothing upstream."""
    def wrapped(ap, dx, dy, th):
        return [XYShift(dx, dy), SRotation.from_angle(th), ap, SRotation.from_angle(-th), XYShift(-dx, -dy)]
    els = [Marker(), Drift(2.5), Multipole(knl=(0.0, 0.02))]
    els += wrapped(LimitRect(-0.0075, 0.0065, -0.0055, 0.006), 1e-3, -5e-4, 0.2)
    els += [Drift(3.0), Multipole(knl=(1e-5, -0.04, 0.8), ksl=(0.0, 0.004)), Drift(2.0), Quadrupole(0.05, 0.8), Drift(2.2)]
    els += wrapped(LimitEllipse(0.009, 0.006), -8e-4, 6e-4, -0.35)
    els += [Drift(1.7), Cavity(2e6, 400e6, 20.0), XYShift(2e-4, 1e-4), Multipole(knl=(0.0, 0.03)), Drift(4.1)]
    els += [SRotation.from_angle(0.5), LimitRect(-0.007, 0.007, -0.004, 0.004), LimitEllipse(0.0075, 0.0045),
            SRotation.from_angle(-0.5), XYShift(-2e-4, -1e-4), Drift(3.3), Quadrupole(-0.05, 0.8), Drift(0.4)]
    els += [LimitEllipse(0.006, 0.006)]
    return els


@pytest.mark.parametrize("ds,n_poly", [(0.1, 64), (0.013, 17)])
def test_refinement_matches_the_oracle(X, ds, n_poly):
    els = fig4_line()
    buf = pack_lattice(els, P0C, MASS0, 1.0)
    co = ensemble(5000, 2.5e-3, 3e-4, 11)
    ref = O.new_particles(buf, co)
    mm0 = np.full(5000, np.inf)
    O.track(buf, ref, 2, threads=O.host_threads(), min_margin=mm0)
    coarse = O.copy_particles(ref)
    mm = np.full(5000, np.inf)
    moved_ref = R.refine_loss_location(els, P0C, MASS0, 1.0, ref, ds, n_poly, min_margin=mm)
    apertures = [i for i, e in enumerate(els) if isinstance(e, (LimitRect, LimitEllipse))]
    per_ap = [int(((ref["state"] == 0) & (ref["at_element"] == i)).sum()) for i in apertures]
    assert min(per_ap[j] for j in (0, 1, 2, 4)) > 50 and moved_ref > 2000, (per_ap, moved_ref)
    assert (ref["s"] != coarse["s"]).sum() > 0.9 * moved_ref

    lat = X.xt_lattice_create(buf)
    p = X.new_particles(lat, co)
    X.xt_track(lat, p, 2)
    before = X.particles_to_host(p)
    clear = ~(mm0 < 1e-9) & ~(mm < 1e-9)
    for k in ("state", "at_turn", "at_element"):
        assert np.array_equal(before[k][clear], coarse[k][clear]), k
    launches = X.xt_launch_count()
    moved = X.xt_refine_loss_location(lat, p, ds, n_poly)
    assert X.xt_launch_count() - launches >= 5                  # gather, track, flip, track, scatter per aperture
    got = X.particles_to_host(p)
    assert clear.sum() > 4950 and abs(moved - moved_ref) <= (~clear).sum()
    for k in ("state", "at_turn", "at_element"):
        assert np.array_equal(got[k], before[k]), k             # refinement never touches these
    assert np.max(np.abs(got["s"][clear] - ref["s"][clear])) < 1e-9
    for k in KEYS:
        ok = np.abs(got[k] - ref[k]) <= 1e-12 * np.maximum(np.abs(ref[k]), SCALE[k])
        assert ok[clear].all(), (k, int((~ok[clear]).sum()), float(np.max(np.abs(got[k] - ref[k])[clear])))
    alive = before["state"] == 1
    for k in KEYS + ("s",):
        assert np.array_equal(got[k][alive], before[k][alive]), k   # survivors untouched, bit for bit
    # the second aperture of the rect+ellipse pair has no length upstream: its records stay
    pair = (before["state"] == 0) & (before["at_element"] == apertures[3])
    for k in KEYS + ("s",):
        assert np.array_equal(got[k][pair], before[k][pair]), k
    lat.close()


def test_refinement_argument_errors(X):
    els = [LimitEllipse(0.01, 0.01), Drift(5.0), LimitEllipse(0.005, 0.005)]
    lat = X.xt_lattice_create(pack_lattice(els, P0C, MASS0, 1.0))
    p = X.new_particles(lat, ensemble(64, 3e-3, 1e-4, 1))
    X.xt_track(lat, p, 1)
    for ds, n_poly in ((0.0, 16), (-1.0, 16), (float("nan"), 16), (0.1, 2), (0.1, 257)):
        with pytest.raises(X.XtError) as e:
            X.xt_refine_loss_location(lat, p, ds, n_poly)
        assert e.value.code == -1
    q = dict(p)
    q["at_element"] = None
    with pytest.raises(X.XtError) as e:
        X.xt_refine_loss_location(lat, q, 0.1, 16)
    assert e.value.code == -1
    assert X.xt_refine_loss_location(lat, p, 0.1, 16) > 0
    lat.close()


def test_refinement_on_the_configs4_lattice_sampled(X):
    """The dynamic-aperture ring of BASELINE.json configs[4] (8 606 elements, apertures every ~30 m), 500 100
    particles x 20 turns on the GPU; the oracle tracks and refines a sample of 600 of them one by one."""
    import torch
    from xt_inputs import configs as C
    els = C.lattice(4)
    buf = C.pack(els)
    co_all = C.particles(4)
    co = C.subsample(co_all, np.arange(0, len(co_all["x"]), 4))
    n = len(co["x"])
    ds, n_poly, turns = 0.1, 32, 20
    lat = X.xt_lattice_create(buf)
    p = X.new_particles(lat, co)
    X.xt_track(lat, p, turns)
    before = X.particles_to_host(p)
    lost = before["state"] == 0
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    moved = X.xt_refine_loss_location(lat, p, ds, n_poly)
    ev1.record()
    torch.cuda.synchronize()
    got = X.particles_to_host(p)
    lat.close()
    print("refined %d of %d lost (%d particles) in %.1f ms" % (moved, lost.sum(), n, ev0.elapsed_time(ev1)))
    assert lost.sum() > 0.3 * n and moved == lost.sum()
    assert np.all(got["s"][lost] <= before["s"][lost] + 1e-9) and np.all(got["s"][lost] > before["s"][lost] - 60.0)
    assert (got["s"][lost] < before["s"][lost] - 1e-6).mean() > 0.9
    for k in KEYS + ("s",):
        assert np.array_equal(got[k][~lost], before[k][~lost]), k
    # sample
    rng = np.random.default_rng(4)
    idx = np.sort(rng.choice(n, 600, replace=False))
    ref = O.new_particles(buf, C.subsample(co, idx))
    mm0 = np.full(600, np.inf)
    O.track(buf, ref, turns, threads=O.host_threads(), min_margin=mm0)
    mm = np.full(600, np.inf)
    R.refine_loss_location(els, C.P0C, C.MASS0, 1.0, ref, ds, n_poly, min_margin=mm)
    same = np.array_equal
    ok = ~(mm0 < 1e-9) & ~(mm < 1e-9) & (ref["state"] == got["state"][idx]) & (ref["at_turn"] == got["at_turn"][idx])
    assert ok.mean() > 0.98 and (ref["state"][ok] == 0).sum() > 150
    assert same(ref["at_element"][ok], got["at_element"][idx][ok])
    assert np.max(np.abs(ref["s"][ok] - got["s"][idx][ok])) < 1e-9
    for k in KEYS:
        a, r = got[k][idx][ok], ref[k][ok]
        good = (np.isnan(a) & np.isnan(r)) | (np.abs(a - r) <= 1e-10 * np.maximum(np.abs(r), SCALE[k]))
        assert good.mean() > 0.99, (k, float(good.mean()), float(np.nanmax(np.abs(a - r))))
    assert np.isnan(ref["x"][ok]).mean() < 0.3                     # particles born beyond |p| = 1 are lost as NaN


def test_refinement_between_polygon_apertures(X):
    """LimitPolygon apertures as the flagging and the upstream aperture (a star and a 64-gon, one of them in a
    shifted / tilted bracket), against the oracle."""
    ang = 2 * np.pi * np.arange(64) / 64
    els = [Drift(1.0), star(12, 0.0065, 0.005, 5e-4, -3e-4, 0.2), Drift(3.0), Multipole(knl=(0.0, 0.03, 1.0)), Quadrupole(0.04, 1.2),
           Drift(2.5), XYShift(-1e-3, 5e-4), SRotation.from_angle(0.4),
           LimitPolygon(tuple(0.008 * np.cos(ang)), tuple(0.005 * np.sin(ang))), SRotation.from_angle(-0.4), XYShift(1e-3, -5e-4),
           Drift(4.0), LimitRect(-0.004, 0.004, -0.003, 0.003)]
    buf = pack_lattice(els, P0C, MASS0, 1.0)
    co = ensemble(4000, 2.5e-3, 3e-4, 21)
    ref = O.new_particles(buf, co)
    mm0 = np.full(4000, np.inf)
    O.track(buf, ref, 1, threads=O.host_threads(), min_margin=mm0)
    coarse = O.copy_particles(ref)
    mm = np.full(4000, np.inf)
    moved_ref = R.refine_loss_location(els, P0C, MASS0, 1.0, ref, 0.05, 48, min_margin=mm)
    per_ap = [int(((coarse["state"] == 0) & (coarse["at_element"] == i)).sum()) for i in (1, 8, 12)]
    assert min(per_ap) > 100 and moved_ref > 1000, (per_ap, moved_ref)
    lat = X.xt_lattice_create(buf)
    p = X.new_particles(lat, co)
    X.xt_track(lat, p, 1)
    moved = X.xt_refine_loss_location(lat, p, 0.05, 48)
    got = X.particles_to_host(p)
    lat.close()
    clear = ~(mm0 < 1e-9) & ~(mm < 1e-9)
    assert clear.sum() > 3950 and abs(moved - moved_ref) <= (~clear).sum()
    assert np.array_equal(got["at_element"][clear], ref["at_element"][clear])
    assert np.max(np.abs(got["s"][clear] - ref["s"][clear])) < 1e-9
    for k in KEYS:
        ok = np.abs(got[k] - ref[k]) <= 1e-12 * np.maximum(np.abs(ref[k]), SCALE[k])
        assert ok[clear].all(), (k, int((~ok[clear]).sum()))
    # a polygon that does not surround the mean of its vertices cannot be sampled from there: reported
    bad = [Drift(1.0), LimitPolygon((0.0, 0.02, 0.02, 0.019, 0.019, 0.0), (0.0, 0.0, 0.02, 0.02, 0.001, 0.001))]
    lat = X.xt_lattice_create(pack_lattice(bad, P0C, MASS0, 1.0))
    p = X.new_particles(lat, ensemble(64, 5e-3, 1e-4, 2))
    X.xt_track(lat, p, 1)
    with pytest.raises(X.XtError) as e:
        X.xt_refine_loss_location(lat, p, 0.1, 16)
    assert e.value.code == -2
    lat.close()
