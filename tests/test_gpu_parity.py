"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the CPU
oracle on identical seeded inputs.

Tolerances (BASELINE.json north_star, reading A8): per coordinate
|gpu - ref| <= max(rtol*|ref|, atol_k), atol_k = max(1e-15, rtol x rms of that coordinate over the
compared ensemble) (helpers.parity_atol): rtol = 1e-12 after 1 turn (atol_k = 1e-15 for every
coordinate) and rtol = 1e-10 after 100 turns (stable particles, reading A9; x, y, zeta get 1e-10 of
their own scale at a zero crossing, px, py, delta, ptau keep 1e-15); lost flags / at_turn / at_element exact except
for particles within 1e-9 m of an aperture edge (A3); bit-exact in the --fmad=false
validation build on cavity-stripped lattices (A10).
"""
import numpy as np
import pytest

from oracle import oracle as O
from xt_inputs import configs as C
from xt_inputs.packed import (Cavity, Drift, LimitEllipse, LimitRect, Marker, Multipole,
                              SRotation, XYShift, pack_lattice)
import helpers as H

pytestmark = pytest.mark.gpu

FLOAT_KEYS = ("x", "px", "y", "py", "zeta", "delta", "ptau", "rpp", "rvv")
INT_KEYS = ("at_turn", "state", "at_element")
ATOL = 1e-15
THREADS = O.host_threads()


@pytest.fixture(scope="module")
def X():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m gpu on the B200 box)")
    import paper_2310_00317_b200 as X
    return X


_buf_cache = {}


def packed(cfg, strip=False):
    key = (cfg, strip)
    if key not in _buf_cache:
        els = C.lattice(cfg)
        if strip:
            els = C.strip_cavities(els)
        _buf_cache[key] = C.pack(els)
    return _buf_cache[key]


def run_both(X, buf, coords, n_turns, kind="prod", margin=False, **opts):
    """-> (gpu result dict of numpy, oracle result dict, min_margin or None)."""
    ref = O.new_particles(buf, coords)
    mm = np.full(len(ref["x"]), np.inf) if margin else None
    O.track(buf, ref, n_turns, threads=THREADS, min_margin=mm)
    lat = X.xt_lattice_create(buf, kind=kind)
    p = X.new_particles(lat, coords)
    if opts:
        X.xt_track_ex(lat, p, n_turns, **opts)
    else:
        X.xt_track(lat, p, n_turns)
    got = X.particles_to_host(p)
    lat.close()
    return got, ref, mm


def assert_close(got, ref, rtol, sel=None, keys=FLOAT_KEYS, label=None):
    """Reading A8, per-coordinate floor (helpers.assert_parity; the same helper smoke() uses)."""
    return H.assert_parity(got, ref, rtol, sel=sel, keys=keys, label=label)


def assert_bit_identical(got, ref, keys=FLOAT_KEYS + ("s",) + INT_KEYS):
    for k in keys:
        a, r = got[k], ref[k]
        if a.dtype == np.float64:
            same = (a.view(np.int64) == r.view(np.int64)) | (np.isnan(a) & np.isnan(r))
        else:
            same = a == r
        if not same.all():
            j = int(np.argmin(same))
            raise AssertionError("%s: %d/%d differ bitwise; first %d gpu=%r ref=%r" %
                                 (k, int((~same).sum()), len(same), j, a[j], r[j]))


def assert_losses_match(got, ref, mm):
    """Loss records are integers: exact, except within 1e-9 m of an aperture edge (A3)."""
    clear = mm >= 1e-9
    for k in INT_KEYS:
        bad = (got[k] != ref[k]) & clear
        assert not bad.any(), (k, int(bad.sum()), int(np.argmax(bad)))
    lost = clear & (ref["state"] == 0)
    assert np.array_equal(got["s"][lost], ref["s"][lost])
    return clear


# ----------------------------------------------------------------- init helper, lattice
def test_init_derived_and_s_table(X):
    buf = packed(3)
    coords = C.subsample(C.particles_cfg3(n=5000), slice(None))
    ref = O.new_particles(buf, coords)
    lat = X.xt_lattice_create(buf)
    p = X.particles_to_host(X.new_particles(lat, coords))
    assert_close(p, ref, 4e-16, keys=("ptau", "rpp", "rvv"))
    assert np.array_equal(X.xt_lattice_s_table(lat), O.s_table(buf))
    b0, g0 = O.reference(buf)
    assert lat.info["beta0"] == b0 and lat.info["gamma0"] == g0
    lat.close()
    latv = X.xt_lattice_create(buf, kind="nofma")
    pv = X.particles_to_host(X.new_particles(latv, coords))
    assert_bit_identical(pv, ref, keys=("ptau", "rpp", "rvv"))
    latv.close()


# ------------------------------------------------------------------------------ config 0
def test_cfg0_one_turn(X):
    got, ref, _ = run_both(X, packed(0), C.particles(0), 1)
    assert_close(got, ref, 1e-12)
    assert np.array_equal(got["at_turn"], ref["at_turn"]) and (got["state"] == 1).all()
    assert (got["s"] == 0).all()


def test_cfg0_100_turns(X):
    got, ref, _ = run_both(X, packed(0), C.particles(0), 100)
    assert_close(got, ref, 1e-10, label="configs[0] 100 turns")
    assert (got["at_turn"] == 100).all()


# --------------------------------------------------------------- worked examples (golden)
def test_worked_examples_every_element_type(X):
    g = H.load_golden()
    for line in g["lines"]:
        els = [H.element_from_json(d) for d in line["elements"]]
        buf = pack_lattice(els, H.P0C, H.MASS0, H.Q0)
        start = [H.unhex(v) for v in line["start"]]
        got, ref, _ = run_both(X, buf, H.coords_from_rows([start] * 33), 1)
        assert_close(got, ref, 1e-12)
        gotv, refv, _ = run_both(X, buf, H.coords_from_rows([start] * 33), 1, kind="nofma")
        has_cav = any(isinstance(e, Cavity) for e in els)
        if not has_cav:
            assert_bit_identical(gotv, refv)
        else:
            assert_close(gotv, refv, 1e-14)


# --------------------------------------------------------------------- bit-exact (A10)
@pytest.mark.parametrize("cfg,n,turns", [(0, 1000, 100), (2, 3000, 3), (3, 3000, 2), (4, 3000, 2)])
def test_bit_exact_nofma_cavity_stripped(X, cfg, n, turns):
    full = C.particles(cfg, n=n) if cfg in (0, 2, 3) else C.particles(cfg)
    if cfg == 4:
        idx = np.linspace(0, len(full["x"]) - 1, n).astype(np.int64)
        full = C.subsample(full, idx)
    got, ref, _ = run_both(X, packed(cfg, strip=True), full, turns, kind="nofma")
    assert_bit_identical(got, ref)


def test_bit_exact_nofma_cfg1b_with_losses(X):
    """Supplementary config[1b] (sigma_grid = 1e-3 m): the literal config[1] loses nothing."""
    coords = C.subsample(C.particles_cfg1(sigma=1e-3), slice(0, None, 97))
    got, ref, _ = run_both(X, packed(1, strip=True), coords, 600, kind="nofma")
    assert (ref["state"] == 0).sum() > 1000 and (ref["state"] == 1).sum() > 1000
    assert_bit_identical(got, ref)


# ------------------------------------------------------------------------ configs 1, 1b
def test_cfg1_literal_one_turn_and_100_turns(X):
    coords = C.subsample(C.particles_cfg1(), slice(0, None, 50))        # 20 000 particles
    got, ref, _ = run_both(X, packed(1), coords, 1)
    assert_close(got, ref, 1e-12)
    got, ref, mm = run_both(X, packed(1), coords, 100, margin=True)
    assert (ref["state"] == 1).all()
    assert_losses_match(got, ref, mm)
    assert_close(got, ref, 1e-10, label="configs[1] 100 turns")


def test_cfg1b_losses_first_100_turns(X):
    coords = C.subsample(C.particles_cfg1(sigma=1e-3), slice(0, None, 50))
    got, ref, mm = run_both(X, packed(1), coords, 100, margin=True)
    assert (ref["state"] == 0).sum() > 5000
    clear = assert_losses_match(got, ref, mm)
    # coordinates of lost particles are those AT the aperture; compare all clear particles
    # that the FMA-contracted oracle build also reproduces (A9: numerically stable ones)
    fma = O.new_particles(packed(1), coords, kind="fma")
    O.track(packed(1), fma, 100, kind="fma", threads=THREADS)
    stable = clear & (fma["state"] == ref["state"]) & (fma["at_turn"] == ref["at_turn"])
    for k in ("x", "px", "y", "py"):
        stable &= H.within(fma[k], ref[k], 1e-11, ATOL)
    assert stable.sum() > 0.5 * len(stable)
    assert_close(got, ref, 1e-10, sel=stable, keys=("x", "px", "y", "py", "zeta", "delta", "ptau"),
                 label="configs[1b] 100 turns")


# --------------------------------------------------------------------------- configs 2-4
def test_cfg2_one_turn_all_particles(X):
    got, ref, mm = run_both(X, packed(2), C.particles(2), 1, margin=True)
    assert_losses_match(got, ref, mm)
    assert_close(got, ref, 1e-12, sel=ref["state"] == 1, label="configs[2] 1 turn")


def _stable_mask(buf, coords, ref, mm, n_turns):
    fma = O.new_particles(buf, coords, kind="fma")
    O.track(buf, fma, n_turns, kind="fma", threads=THREADS)
    stable = (ref["state"] == 1) & (fma["state"] == 1) & (mm >= 1e-9)
    for k in ("x", "px", "y", "py", "zeta"):
        stable &= H.within(fma[k], ref[k], 1e-11, ATOL)
    return stable


def test_cfg2_100_turns(X):
    coords = C.subsample(C.particles(2), slice(0, None, 50))            # 2 000 particles
    got, ref, mm = run_both(X, packed(2), coords, 100, margin=True)
    assert_losses_match(got, ref, mm)
    stable = _stable_mask(packed(2), coords, ref, mm, 100)
    assert stable.sum() > 0.95 * len(stable), stable.sum()
    assert_close(got, ref, 1e-10, sel=stable, label="configs[2] 100 turns")


def test_cfg3_one_turn_and_100_turns(X):
    coords = C.particles(3, n=100_000)
    got, ref, mm = run_both(X, packed(3), coords, 1, margin=True)
    assert_losses_match(got, ref, mm)
    assert_close(got, ref, 1e-12, sel=ref["state"] == 1, label="configs[3] 1 turn")
    sub = C.subsample(coords, slice(0, 1000))
    got, ref, mm = run_both(X, packed(3), sub, 100, margin=True)
    assert_losses_match(got, ref, mm)
    stable = _stable_mask(packed(3), sub, ref, mm, 100)
    assert stable.sum() > 0.9 * len(stable), stable.sum()
    assert_close(got, ref, 1e-10, sel=stable, label="configs[3] 100 turns")


def test_cfg4_grid_losses_and_histogram(X):
    full = C.particles(4)
    idx = np.linspace(0, len(full["x"]) - 1, 6000).astype(np.int64)
    coords = C.subsample(full, idx)
    buf = packed(4)
    got, ref, mm = run_both(X, buf, coords, 60, margin=True, compact_every=20)
    assert 0.3 < (ref["state"] == 0).mean() < 0.95
    assert_losses_match(got, ref, mm)
    # survival histogram (step H) against numpy on the oracle's records, edge band removed
    import torch
    clear = mm >= 1e-9
    p = {k: torch.from_numpy(np.ascontiguousarray(got[k][clear])).cuda() for k in ("at_turn", "state", "x")}
    hist = X.xt_survival_histogram(p, 10, 6).cpu().numpy()
    lost = ref["state"][clear] == 0
    want = np.bincount(np.minimum(ref["at_turn"][clear][lost] // 10, 5), minlength=6)
    assert np.array_equal(hist[:6], want) and hist[6] == (~lost).sum()


# ----------------------------------------------------- structural invariants (P9) on GPU
def test_compaction_and_launch_chunking_do_not_change_results(X):
    coords = C.subsample(C.particles_cfg1(sigma=1e-3), slice(0, None, 211))
    buf = packed(1)
    lat = X.xt_lattice_create(buf)
    base = X.new_particles(lat, coords)
    X.xt_track_ex(lat, base, 300, compact_every=-1)
    base = X.particles_to_host(base)
    assert 0.2 < (base["state"] == 0).mean() < 0.9
    variants = [dict(compact_every=37), dict(compact_every=100, turns_per_launch=7),
                dict(compact_every=-1, turns_per_launch=1, block_size=32),
                dict(compact_every=299, block_size=256), dict(block_size=64, turns_per_launch=150)]
    for v in variants:
        p = X.new_particles(lat, coords)
        X.xt_track_ex(lat, p, 300, **v)
        assert_bit_identical(X.particles_to_host(p), base)
    # continuation: 300 = 120 + 180 (state carried only by the arrays)
    p = X.new_particles(lat, coords)
    X.xt_track(lat, p, 120)
    X.xt_track_ex(lat, p, 180, compact_every=50)
    assert_bit_identical(X.particles_to_host(p), base)
    lat.close()


def test_launch_shape_fusion_and_chunk_size_do_not_change_results(X):
    """Particles per thread, CTA size, record fusion and the staging-buffer size only change
    how the work is laid out: every variant must reproduce the default bit for bit."""
    full = C.particles(4)
    idx = np.linspace(0, len(full["x"]) - 1, 2777).astype(np.int64)     # ragged: not a multiple of 32
    coords = C.subsample(full, idx)
    buf = packed(4)
    lat = X.xt_lattice_create(buf)
    base = X.new_particles(lat, coords)
    X.xt_track_ex(lat, base, 6, compact_every=-1)
    base = X.particles_to_host(base)
    assert 0.05 < (base["state"] == 0).mean() < 0.95
    for ppt in (1, 2, 3, 4):
        for block in (32, 96, 256):
            p = X.new_particles(lat, coords)
            X.xt_track_ex(lat, p, 6, compact_every=-1, block_size=block, particles_per_thread=ppt)
            assert_bit_identical(X.particles_to_host(p), base)
    for ppt, cold in ((1, 1), (2, 1), (3, 1), (4, 1), (2, -1), (3, -1)):   # cold per-particle state in registers / shared memory
        p = X.new_particles(lat, coords)
        X.xt_track_ex(lat, p, 6, compact_every=-1, block_size=64, particles_per_thread=ppt, cold_in_registers=cold)
        assert_bit_identical(X.particles_to_host(p), base)
    with pytest.raises(X.XtError):
        X.xt_track_ex(lat, X.new_particles(lat, coords), 1, particles_per_thread=5, cold_in_registers=1)
    lat.close()
    for kw in (dict(fuse=False), dict(chunk_bytes=1024), dict(chunk_bytes=65536), dict(chunk_bytes=4224, fuse=False)):
        lat2 = X.xt_lattice_create_ex(buf, **kw)
        p = X.new_particles(lat2, coords)
        X.xt_track_ex(lat2, p, 6, compact_every=4, particles_per_thread=2)
        assert_bit_identical(X.particles_to_host(p), base)
        lat2.close()


def test_balanced_mode_is_bit_identical(X):
    """xt_track_opts.balance: persistent CTAs that draw (group of particles, block of
    turns) items from a ticket counter, the state of a group passing through HBM between its blocks.  Only
    the schedule changes: every variant reproduces the unbalanced launch bit for bit -- multi-chunk and
    single-chunk lattices, losses spread over the turns (at_turn, at_element and s of the lost included), a
    ragged last group and a ragged last block of turns, both builds, scratch from the caller's workspace."""
    import torch
    full = C.particles(4)
    idx = np.linspace(0, len(full["x"]) - 1, 5003).astype(np.int64)
    coords = C.subsample(full, idx)
    for kind in ("prod", "nofma"):
        lat = X.xt_lattice_create(packed(4), kind=kind)                 # 8 606 elements, many chunks, apertures
        base = X.new_particles(lat, coords)
        X.xt_track_ex(lat, base, 11, compact_every=-1, balance=-1)
        base = X.particles_to_host(base)
        lost = base["state"] == 0
        assert 0.05 < lost.mean() < 0.95 and len(np.unique(base["at_turn"][lost])) >= 5
        for ppt, block, bal in ((2, 128, 2), (2, 64, 3), (1, 32, 4), (3, 96, 2), (4, 128, 3), (2, 128, 1), (2, 256, 11), (1, 64, 12)):
            p = X.new_particles(lat, coords)
            X.xt_track_ex(lat, p, 11, compact_every=-1, particles_per_thread=ppt, block_size=block,
                          cold_in_registers=1, balance=bal)
            assert_bit_identical(X.particles_to_host(p), base)
        # split over several launches, each balanced; scratch taken from a caller's workspace
        ws = torch.empty(X.xt_track_workspace_bytes(len(idx)), dtype=torch.uint8, device="cuda")
        ws.fill_(0xCD)                                                  # stale bytes must not matter
        p = X.new_particles(lat, coords)
        X.xt_track_ex(lat, p, 11, compact_every=-1, particles_per_thread=2, block_size=128, cold_in_registers=1,
                      balance=2, turns_per_launch=5, workspace=ws)
        assert_bit_identical(X.particles_to_host(p), base)
        # with loss compaction: the number of groups is then a device counter and the launch has CTAs to spare
        for ppt, block, bal, every in ((2, 128, 2, 4), (3, 64, 1, 3), (1, 32, 3, 5)):
            p = X.new_particles(lat, coords)
            st = X.xt_track_ex(lat, p, 11, compact_every=every, particles_per_thread=ppt, block_size=block,
                               cold_in_registers=1, balance=bal, stats=True)
            assert st["n_passes"] >= 2
            assert_bit_identical(X.particles_to_host(p), base)
        p = X.new_particles(lat, coords)                                 # ... in a caller's workspace
        X.xt_track_ex(lat, p, 11, compact_every=4, particles_per_thread=2, block_size=128, cold_in_registers=1,
                      balance=2, workspace=ws)
        assert_bit_identical(X.particles_to_host(p), base)
        # the auto shape of a one-wave ensemble (2 per thread, registers) with the auto rule
        p = X.new_particles(lat, coords)
        X.xt_track_ex(lat, p, 11, compact_every=-1)
        assert_bit_identical(X.particles_to_host(p), base)
        with pytest.raises(X.XtError) as e:                            # needs the cold state in registers
            X.xt_track_ex(lat, X.new_particles(lat, coords), 3, cold_in_registers=-1, particles_per_thread=2, balance=1)
        assert e.value.code == -1
        with pytest.raises(X.XtError) as e:                            # forced, but the workspace cannot hold the queue
            X.xt_track_ex(lat, X.new_particles(lat, coords), 3, cold_in_registers=1, particles_per_thread=2, balance=1,
                          workspace=ws[:256])
        assert e.value.code == -1
        lat.close()
    # single-chunk lattice (warps run free inside an item), continuing a run
    coords1 = C.subsample(C.particles_cfg1(sigma=1e-3), slice(0, None, 97))
    lat = X.xt_lattice_create(packed(1))
    a, b = X.new_particles(lat, coords1), X.new_particles(lat, coords1)
    X.xt_track_ex(lat, a, 50, balance=-1)
    X.xt_track_ex(lat, b, 20, particles_per_thread=2, block_size=64, cold_in_registers=1, balance=7)
    X.xt_track_ex(lat, b, 30, particles_per_thread=1, block_size=128, cold_in_registers=1, balance=4)
    ha = X.particles_to_host(a)
    assert (ha["state"] == 0).any()
    assert_bit_identical(X.particles_to_host(b), ha)
    lat.close()


def test_balanced_mode_random_shapes(X):
    """Seeded sweep of the balanced mode over ensemble sizes (from a single particle), launch lengths (from one
    turn), item lengths, launch shapes and compaction periods, on a lattice cut into many small chunks: every
    run reproduces the static launch of the same length bit for bit (and terminates)."""
    rng = np.random.default_rng(20231000)
    full = C.particles(4)
    lat = X.xt_lattice_create_ex(packed(4), chunk_bytes=4096)
    cases = [(1, 1, 1, 32, 1, -1), (1, 9, 2, 128, 2, 3), (33, 1, 3, 32, 5, -1), (257, 2, 2, 128, 1, -1),
             (384, 7, 3, 128, 7, 2), (385, 13, 3, 128, 2, 5)]
    for _ in range(10):
        cases.append((int(rng.integers(2, 3000)), int(rng.integers(1, 30)), int(rng.integers(1, 5)),
                      int(rng.choice([32, 64, 128, 256])), int(rng.integers(1, 10)), int(rng.choice([-1, 3, 7]))))
    for n, turns, ppt, block, bal, every in cases:
        idx = np.sort(rng.choice(len(full["x"]), size=n, replace=False))
        coords = C.subsample(full, idx)
        a, b = X.new_particles(lat, coords), X.new_particles(lat, coords)
        X.xt_track_ex(lat, a, turns, compact_every=-1, balance=-1)
        X.xt_track_ex(lat, b, turns, compact_every=every, particles_per_thread=ppt, block_size=block,
                      cold_in_registers=1, balance=bal)
        try:
            assert_bit_identical(X.particles_to_host(b), X.particles_to_host(a))
        except AssertionError as e:
            raise AssertionError("case %r: %s" % ((n, turns, ppt, block, bal, every), e))
    lat.close()


def test_launch_shapes_on_a_quadrupole_sextupole_lattice(X):
    """configs[1b] (orders 1 and 2 only: the kernels with those two orders fixed; single chunk, losses): every
    launch shape and both homes of the cold state reproduce the default bit for bit, in both builds; the
    validation build equals the oracle bit for bit on the cavity-stripped lattice."""
    coords = C.subsample(C.particles_cfg1(sigma=1e-3), slice(0, None, 211))
    for kind, strip in (("prod", False), ("nofma", True)):
        buf = packed(1, strip=strip)
        lat = X.xt_lattice_create(buf, kind=kind)
        base = X.new_particles(lat, coords)
        X.xt_track_ex(lat, base, 40)
        base = X.particles_to_host(base)
        assert 0.05 < (base["state"] == 0).mean() < 0.95
        for ppt, block, cold in ((1, 32, -1), (2, 64, -1), (3, 96, -1), (4, 128, -1), (1, 64, 1), (2, 128, 1), (3, 32, 1)):
            p = X.new_particles(lat, coords)
            X.xt_track_ex(lat, p, 40, block_size=block, particles_per_thread=ppt, cold_in_registers=cold,
                          compact_every=-1 if ppt % 2 else 7)
            assert_bit_identical(X.particles_to_host(p), base)
        lat.close()
        if strip:
            ref = O.new_particles(buf, coords)
            O.track(buf, ref, 40, threads=THREADS)
            assert_bit_identical(base, ref)


def test_multi_chunk_compaction_cfg4(X):
    full = C.particles(4)
    idx = np.linspace(0, len(full["x"]) - 1, 3001).astype(np.int64)
    coords = C.subsample(full, idx)
    lat = X.xt_lattice_create(packed(4))
    a = X.new_particles(lat, coords)
    X.xt_track_ex(lat, a, 12, compact_every=-1)
    b = X.new_particles(lat, coords)
    X.xt_track_ex(lat, b, 12, compact_every=5, block_size=96)
    assert_bit_identical(X.particles_to_host(b), X.particles_to_host(a))
    lat.close()


def test_caller_workspace_and_stats(X):
    """xt_track_opts.workspace (the caller may own the scratch of step C) and .stats (CUDA-event
    record of the call): results are bit-identical to the library-allocated, untimed call; the record counts
    launches and passes and its pass sizes are the alive counts; a workspace that is too small is refused."""
    import torch
    full = C.particles(4)
    idx = np.linspace(0, len(full["x"]) - 1, 5003).astype(np.int64)
    coords = C.subsample(full, idx)
    lat = X.xt_lattice_create(packed(4))
    a = X.new_particles(lat, coords)
    X.xt_track_ex(lat, a, 12, compact_every=4)
    ha = X.particles_to_host(a)
    need = X.xt_track_workspace_bytes(len(idx))
    assert need >= 2 * 14 * 8 * len(idx)
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    ws.fill_(0xAB)                                                  # stale bytes must not matter
    b = X.new_particles(lat, coords)
    st = X.xt_track_ex(lat, b, 12, compact_every=4, workspace=ws, stats=True)
    assert_bit_identical(X.particles_to_host(b), ha)
    assert st["n_track_launches"] == 3 and st["n_passes"] == 3      # initial partition + 2 between the launches
    assert st["pass_n_in"][0] == len(idx) and st["pass_n_in"][1] == st["pass_n_out"][0]
    assert st["pass_n_in"][2] == st["pass_n_out"][1] and st["pass_n_out"][0] >= st["pass_n_out"][1] >= st["pass_n_out"][2]
    n_alive_before_last_launch = st["pass_n_out"][2]
    assert n_alive_before_last_launch >= int((ha["state"] == 1).sum()) > 0
    assert st["track_ms"] > 0 and st["compact_ms"] > 0 and st["scatter_ms"] > 0
    assert st["compact_bytes"] == 2 * 112.0 * sum(st["pass_n_in"])
    c = X.new_particles(lat, coords)
    st2 = X.xt_track_ex(lat, c, 12, compact_every=-1, stats=True)   # no compaction: one launch, no pass
    assert st2["n_track_launches"] == 1 and st2["n_passes"] == 0
    assert_bit_identical(X.particles_to_host(c), ha)
    with pytest.raises(X.XtError) as e:
        X.xt_track_ex(lat, X.new_particles(lat, coords), 12, compact_every=4, workspace=ws[:need // 2])
    assert e.value.code == -1
    lat.close()


def test_permutation_invariance_and_frozen_lost(X):
    coords = C.subsample(C.particles_cfg1(sigma=1e-3), slice(0, None, 503))
    n = len(coords["x"])
    perm = np.random.default_rng(5).permutation(n)
    lat = X.xt_lattice_create(packed(1))
    a = X.new_particles(lat, coords)
    b = X.new_particles(lat, C.subsample(coords, perm))
    X.xt_track(lat, a, 50)
    X.xt_track(lat, b, 50)
    ha, hb = X.particles_to_host(a), X.particles_to_host(b)
    assert_bit_identical({k: v for k, v in hb.items()}, {k: v[perm] for k, v in ha.items()})
    X.xt_track(lat, a, 50)
    ha2 = X.particles_to_host(a)
    lost = ha["state"] == 0
    assert lost.any()
    for k in FLOAT_KEYS + ("s",) + INT_KEYS:
        assert np.array_equal(ha2[k][lost], ha[k][lost]), k
    lat.close()


# ------------------------------------------------------------------------- edge cases
def test_edge_cases(X):
    import torch
    buf = packed(1)
    lat = X.xt_lattice_create(buf)
    # empty ensemble and zero turns are successful no-ops
    empty = X.new_particles(lat, {k: np.zeros(0) for k in C.COORDS})
    X.xt_track(lat, empty, 5)
    one = X.new_particles(lat, H.coords_from_rows([[1e-4, 0, 1e-4, 0, 0, 0]]))
    before = X.particles_to_host(one)
    X.xt_track(lat, one, 0)
    assert_bit_identical(X.particles_to_host(one), before)
    # ragged sizes around the block size
    for n in (1, 31, 33, 127, 129, 257):
        coords = C.subsample(C.particles_cfg1(sigma=1e-3), slice(0, n * 3001, 3001))
        got, ref, mm = run_both(X, buf, coords, 3, margin=True)
        assert_losses_match(got, ref, mm)
        assert_close(got, ref, 1e-12, sel=ref["state"] == 1)
    # everything lost at the first aperture; NaN is lost (A4); at_element may be NULL
    rows = [[0.5, 0, 0, 0, 0, 0], [float("nan"), 0, 0, 0, 0, 0], [0, 0, -0.02, 0, 0, 0]]
    got, ref, _ = run_both(X, buf, H.coords_from_rows(rows), 4)
    assert (got["state"] == 0).all() and (got["at_turn"] == 0).all()
    assert np.array_equal(got["at_element"], ref["at_element"]) and np.array_equal(got["s"], ref["s"])
    p = X.new_particles(lat, H.coords_from_rows(rows))
    del p["at_element"]
    X.xt_track(lat, p, 2)
    assert (p["state"] == 0).all()
    # on the edge survives, one ulp beyond is lost (P8 on the GPU)
    edge = pack_lattice([LimitRect(-0.01, 0.01, -0.01, 0.01), LimitEllipse(0.02, 0.015), Marker()],
                        H.P0C, H.MASS0, H.Q0)
    rows = [[0.01, 0, 0.01, 0, 0, 0], [np.nextafter(0.01, 1), 0, 0, 0, 0, 0], [0, 0, -0.01, 0, 0, 0],
            [0, 0, np.nextafter(-0.01, -1), 0, 0, 0]]
    got, ref, _ = run_both(X, edge, H.coords_from_rows(rows), 2)
    assert list(got["state"]) == [1, 0, 1, 0] == list(ref["state"])
    assert_bit_identical(got, ref)
    # errors: bad arguments come back as XtError, nothing is written
    with pytest.raises(X.XtError):
        X.xt_lattice_create(buf[:-8])
    with pytest.raises(X.XtError):
        X.xt_track_ex(lat, one, 1, block_size=48)
    with pytest.raises(X.XtError):
        X.xt_track(lat, one, -1)
    lat.close()
    # a marker-only / empty line is the identity apart from at_turn
    ident = X.xt_lattice_create(pack_lattice([Marker(), Marker()], H.P0C, H.MASS0, H.Q0))
    q = X.new_particles(ident, C.particles(0))
    h0 = X.particles_to_host(q)
    X.xt_track(ident, q, 7)
    h1 = X.particles_to_host(q)
    assert (h1["at_turn"] == 7).all()
    assert_bit_identical(h1, h0, keys=FLOAT_KEYS)
    ident.close()
    torch.cuda.synchronize()


def test_maximum_order_and_all_orders(X):
    rng = np.random.default_rng(11)
    els = []
    for n in range(0, 21):
        knl = tuple(rng.normal(0, 1.0, n + 1) * 10.0 ** np.arange(n + 1) * 1e-3)
        ksl = tuple(rng.normal(0, 1.0, n + 1) * 10.0 ** np.arange(n + 1) * 1e-3)
        els += [Multipole(knl=knl, ksl=ksl, hxl=(1e-3 if n % 3 == 0 else 0.0), length=0.7), Drift(0.3)]
    buf = pack_lattice(els, H.P0C, H.MASS0, H.Q0)
    coords = C.particles_cfg0(n=500, seed=77)
    for k in ("x", "y"):
        coords[k] = coords[k] * 20.0
    got, ref, _ = run_both(X, buf, coords, 1)
    assert_close(got, ref, 1e-12)
    gotv, refv, _ = run_both(X, buf, coords, 2, kind="nofma")
    assert_bit_identical(gotv, refv)


# ------------------------------------------------------- host-buffer entry point (e2e)
def test_track_host_equals_device_path(X):
    import torch
    coords = C.subsample(C.particles_cfg1(sigma=1e-3), slice(0, None, 401))
    buf = packed(1)
    lat = X.xt_lattice_create(buf)
    d = X.new_particles(lat, coords)
    host0 = X.particles_to_host(d)
    X.xt_track(lat, d, 40)
    host = {k: torch.from_numpy(v.copy()).pin_memory() for k, v in host0.items()}
    X.xt_track_host(lat, host, 40)
    assert_bit_identical({k: v.numpy() for k, v in host.items()}, X.particles_to_host(d))
    lat.close()


# ---------------------------------------- full-size launch configuration, sampled outputs
def test_full_size_cfg3_sampled_against_oracle(X):
    """BASELINE.json configs[3] at its full 10^7 particles, the launch bench.py times; the
    oracle recomputes a strided sample one by one."""
    import torch
    coords = C.particles(3)
    n = len(coords["x"])
    buf = packed(3)
    lat = X.xt_lattice_create(buf)
    p = X.new_particles(lat, coords)
    X.xt_track(lat, p, 1)
    torch.cuda.synchronize()
    idx = np.arange(0, n, n // 4000)
    got = {k: v[torch.from_numpy(idx).cuda()].cpu().numpy() for k, v in p.items()}
    alive = int((p["state"] == 1).sum().item())
    assert alive > 0.99 * n
    assert int(p["at_turn"].sum().item()) == alive
    lat.close()
    del p
    sub = C.subsample(coords, idx)
    ref = O.new_particles(buf, sub)
    mm = np.full(len(idx), np.inf)
    O.track(buf, ref, 1, threads=THREADS, min_margin=mm)
    assert_losses_match(got, ref, mm)
    assert_close(got, ref, 1e-12, sel=ref["state"] == 1)


def test_full_size_cfg1_sampled_against_oracle(X):
    """BASELINE.json configs[1] at its full 10^6 particles (single-chunk lattice: the warps run
    free, no CTA-level synchronisation), 1 turn at 1e-12 and 20 turns at 1e-10; the oracle
    recomputes a strided sample one by one."""
    import torch
    coords = C.particles(1)
    n = len(coords["x"])
    assert n == 1_000_000
    buf = packed(1)
    idx = np.arange(7, n, 250)
    sub = C.subsample(coords, idx)
    lat = X.xt_lattice_create(buf)
    for turns, rtol in ((1, 1e-12), (20, 1e-10)):
        p = X.new_particles(lat, coords)
        X.xt_track(lat, p, turns)
        torch.cuda.synchronize()
        assert int((p["state"] == 1).sum().item()) == n          # the literal config[1] loses nothing
        assert int(p["at_turn"].sum().item()) == n * turns
        got = {k: v[torch.from_numpy(idx).cuda()].cpu().numpy() for k, v in p.items()}
        ref = O.new_particles(buf, sub)
        mm = np.full(len(idx), np.inf)
        O.track(buf, ref, turns, threads=THREADS, min_margin=mm)
        assert_losses_match(got, ref, mm)
        assert_close(got, ref, rtol)
        del p
    lat.close()


def test_fp64_probes_are_ordered(X):
    """The roofline denominator and the operand-pattern probes: at most two
    vector-register operands are fastest (every row of the sweep within 2 % of the maximum), three
    distinct registers slowest, the Horner recurrence in between, faster with uniform coefficients."""
    peak, _ = X.xt_fp64_fma_peak()
    rows = X.xt_fp64_fma_peak_sweep()
    distinct, _ = X.xt_fp64_fma_probe(1)
    horner, _ = X.xt_fp64_fma_probe(2)
    horner_u, _ = X.xt_fp64_fma_probe(3)
    assert 30e12 < peak < 40e12                     # B200: 148 SM x 64 lanes x 2 x 1.965 GHz = 37.2 TFLOP/s nominal
    assert len(rows) >= 12 and min(r["tflops"] for r in rows) > 0.98 * peak / 1e12
    assert 0.5 * peak < distinct < horner < horner_u < peak
    with pytest.raises(X.XtError):
        X.xt_fp64_fma_probe(4)


def test_staging_depth_does_not_change_results(X):
    """A launch with several CTAs per SM stages one lattice chunk per bulk copy, a small ensemble
    several chunks at once: a particle must come out bit-identical whichever company it is tracked in."""
    import torch
    coords = C.particles(3, n=400_000)                         # ~2700 particles per SM: one chunk per stage
    buf = packed(3)
    lat = X.xt_lattice_create(buf)
    p = X.new_particles(lat, coords)
    X.xt_track(lat, p, 2)
    idx = np.arange(5, 400_000, 997)
    big = {k: v[torch.from_numpy(idx).cuda()].cpu().numpy() for k, v in p.items()}
    del p
    q = X.new_particles(lat, C.subsample(coords, idx))         # 402 particles: four chunks per stage
    X.xt_track(lat, q, 2)
    assert_bit_identical(X.particles_to_host(q), big)
    lat.close()


def test_particles_dead_on_entry_are_left_alone(X):
    """state == 0 on entry (lost in an earlier call, or never alive): every array of such a particle
    comes back bit for bit, whatever shares its thread or warp; the others track as if alone."""
    coords = C.subsample(C.particles(4), np.linspace(0, 2_000_399, 700).astype(np.int64))
    buf = packed(4)
    lat = X.xt_lattice_create(buf)
    ref = X.new_particles(lat, coords)
    X.xt_track(lat, ref, 3)
    ref = X.particles_to_host(ref)
    p = X.new_particles(lat, coords)
    dead = np.zeros(700, dtype=bool)
    dead[::3] = True
    dead[100:160] = True                                           # whole warps' worth in a row
    import torch
    mask = torch.from_numpy(dead).cuda()
    p["state"][mask] = 0
    p["at_turn"][mask] = 17
    p["x"][mask] = float("nan")                                    # must never be read into a live lane's result
    before = X.particles_to_host(p)
    for ppt in (1, 3, 4):
        q = {k: v.clone() for k, v in p.items()}
        X.xt_track_ex(lat, q, 3, particles_per_thread=ppt, block_size=64)
        got = X.particles_to_host(q)
        for k in got:
            a, b = got[k][dead], before[k][dead]
            same = (a == b) | (np.isnan(a.astype(np.float64)) & np.isnan(b.astype(np.float64)))
            assert same.all(), k
        assert_bit_identical({k: v[~dead] for k, v in got.items()}, {k: v[~dead] for k, v in ref.items()})
    lat.close()


def _random_line(rng, n_el):
    """A random sequence of every cavity-free thin element, biased towards the patterns the packer
    fuses (drift runs, shift/rotation wrappers, apertures behind magnets and drifts) and their
    broken variants."""
    els = []
    while len(els) < n_el:
        r = rng.random()
        if r < 0.30:
            els.append(Drift(float(rng.uniform(0.1, 3.0))))
        elif r < 0.55:
            order = int(rng.choice([0, 1, 2, 3, 4, 7, 8, 15, 20]))
            knl = rng.normal(0, 1, order + 1) * 0.02 / (np.arange(order + 1) + 1.0) * 10.0 ** np.arange(order + 1)
            ksl = rng.normal(0, 1, order + 1) * 0.02 / (np.arange(order + 1) + 1.0) * 10.0 ** np.arange(order + 1)
            if rng.random() < 0.3:
                ksl[:] = 0.0
            hxl = float(rng.choice([0.0, 0.0, 2e-3, -1e-3]))
            length = float(rng.choice([0.0, 1.7]))
            knl, ksl = knl * 2e-3, ksl * 2e-3
            knl[0] = knl[0] * 0.1 + hxl                   # a bend bends by its curvature, plus a small error
            ksl[0] *= 0.1
            els.append(Multipole(knl=tuple(knl), ksl=tuple(ksl), hxl=hxl, length=length))
        elif r < 0.63:
            els.append(XYShift(float(rng.normal(0, 1e-4)), float(rng.normal(0, 1e-4))))
        elif r < 0.71:
            els.append(SRotation.from_angle(float(rng.normal(0, 2e-3))))
        elif r < 0.79:                                   # a whole misaligned magnet
            th, dx, dy = rng.normal(0, 1e-3), rng.normal(0, 1e-4), rng.normal(0, 1e-4)
            els += [XYShift(float(dx), float(dy)), SRotation.from_angle(float(th)),
                    Multipole(knl=(0.0, float(rng.normal(0, 0.05)))), SRotation.from_angle(float(-th)),
                    XYShift(float(-dx), float(-dy))]
        elif r < 0.88:
            els.append(LimitEllipse(float(rng.uniform(0.003, 0.03)), float(rng.uniform(0.003, 0.03))))
        elif r < 0.95:
            a = float(rng.uniform(0.003, 0.03))
            els.append(LimitRect(-a, a, -0.8 * a, 1.2 * a))
        else:
            els.append(Marker())
    return els


@pytest.mark.parametrize("seed", range(16))
def test_random_lattices_bit_exact_nofma(X, seed):
    """Fuzz of step P and the dispatch: random lines through the --fmad=false build must reproduce the
    oracle bit for bit (coordinates, loss records, s), for random chunk sizes, fusion on and off and
    random launch shapes; the production build must agree within the 1-turn tolerance."""
    rng = np.random.default_rng(1000 + seed)
    els = _random_line(rng, int(rng.integers(30, 140)))
    buf = pack_lattice(els, H.P0C, H.MASS0, H.Q0)
    n = int(rng.integers(40, 700))
    amp = float(rng.choice([0.2, 0.5, 1.0]))
    co = dict(x=rng.normal(0, 1.5e-3 * amp, n), px=rng.normal(0, 1e-4 * amp, n), y=rng.normal(0, 1.5e-3 * amp, n),
              py=rng.normal(0, 1e-4 * amp, n), zeta=rng.normal(0, 0.05, n), delta=rng.normal(0, 5e-4, n))
    turns = int(rng.integers(1, 4))
    ref = O.new_particles(buf, co)
    mm = np.full(n, np.inf)
    O.track(buf, ref, turns, min_margin=mm)
    for kind in ("nofma", "prod"):
        for trial in range(3):
            kw = dict(chunk_bytes=int(rng.choice([1024, 1152, 2048, 8192, 65536])), fuse=bool(rng.random() < 0.7))
            lat = X.xt_lattice_create_ex(buf, kind=kind, **kw)
            p = X.new_particles(lat, co)
            X.xt_track_ex(lat, p, turns, particles_per_thread=int(rng.choice([0, 1, 2, 3, 4])),
                          block_size=int(rng.choice([0, 32, 64, 128, 256])), compact_every=int(rng.choice([-1, 1, 2])))
            got = X.particles_to_host(p)
            lat.close()
            if kind == "nofma":
                assert_bit_identical(got, ref)
            else:
                clear = assert_losses_match(got, ref, mm)
                assert_close(got, ref, 1e-12, sel=clear & (ref["state"] == 1))


def _random_polygon(rng):
    n = int(rng.choice([3, 4, 5, 8, 17, 60]))
    ang = 2 * np.pi * (np.arange(n) + rng.uniform(-0.3, 0.3, n) * (rng.random() < 0.5)) / n   # around the beam
    r = rng.uniform(0.006, 0.03) * (1.0 - 0.4 * rng.random(n) * (rng.random() < 0.5))     # convex-ish or star-shaped
    cx, cy = rng.normal(0, 5e-4, 2)
    from xt_inputs.packed import LimitPolygon
    return LimitPolygon(tuple(cx + r * np.cos(ang)), tuple(cy + r * np.sin(ang)))


@pytest.mark.parametrize("seed", range(8))
def test_random_lattices_with_extended_elements(X, seed):
    """The fuzz above with the elements of the widened set mixed in: polygon apertures (even seeds: still
    bit-exact in the --fmad=false build) and, on odd seeds, thick quadrupoles and sector bends (sincos / cosh
    differ from glibc by an ulp or two: 1-turn tolerance in both builds)."""
    from xt_inputs.packed import Bend, Quadrupole
    rng = np.random.default_rng(5000 + seed)
    els = _random_line(rng, int(rng.integers(30, 120)))
    thick = seed % 2 == 1
    for _ in range(int(rng.integers(3, 9))):
        at = int(rng.integers(0, len(els) + 1))
        r = rng.random()
        if not thick or r < 0.4:
            els.insert(at, _random_polygon(rng))
        elif r < 0.7:
            els.insert(at, Quadrupole(float(rng.choice([-1.0, 1.0]) * rng.uniform(0.01, 0.3)), float(rng.uniform(0.2, 3.0))))
        else:
            h = float(rng.choice([-1.0, 1.0]) * rng.uniform(1e-3, 2e-2))
            els.insert(at, Bend(h * (1.0 + float(rng.normal(0, 1e-4))), h, float(rng.uniform(0.5, 6.0))))
    buf = pack_lattice(els, H.P0C, H.MASS0, H.Q0)
    n = int(rng.integers(40, 700))
    amp = float(rng.choice([0.2, 0.5, 1.0]))
    co = dict(x=rng.normal(0, 1.5e-3 * amp, n), px=rng.normal(0, 1e-4 * amp, n), y=rng.normal(0, 1.5e-3 * amp, n),
              py=rng.normal(0, 1e-4 * amp, n), zeta=rng.normal(0, 0.05, n), delta=rng.normal(0, 5e-4, n))
    turns = int(rng.integers(1, 4))
    ref = O.new_particles(buf, co)
    mm = np.full(n, np.inf)
    O.track(buf, ref, turns, min_margin=mm)
    for kind in ("nofma", "prod"):
        for trial in range(3):
            kw = dict(chunk_bytes=int(rng.choice([2048, 8192, 65536])), fuse=bool(rng.random() < 0.7))
            lat = X.xt_lattice_create_ex(buf, kind=kind, **kw)
            p = X.new_particles(lat, co)
            X.xt_track_ex(lat, p, turns, particles_per_thread=int(rng.choice([0, 1, 2, 3, 4])),
                          block_size=int(rng.choice([0, 32, 64, 128, 256])), compact_every=int(rng.choice([-1, 1, 2])))
            got = X.particles_to_host(p)
            lat.close()
            if kind == "nofma" and not thick:
                assert_bit_identical(got, ref)
            else:
                clear = assert_losses_match(got, ref, mm)
                assert_close(got, ref, 1e-12, sel=clear & (ref["state"] == 1))
