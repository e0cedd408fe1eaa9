"""xt_track_static (include/xt.h): tracking with loss compaction whose
scratch is the library's file-scope device array, for callers that cannot call cudaMalloc.  Checked against the
existing path, xt_track_ex with a stream-ordered workspace, on the same seeded inputs.  Both run the same
kernels in the same build, so the bar is the one the launch-shape tests use: bit-identical.

Two calls in a row share the array and the second must not see the first: the second call tracks a different,
smaller ensemble (fewer tiles, other alive counts), then a third repeats the first.  The file sorts last on
purpose: the run uses -x, and this test must pass alone in a fresh process as well as after all the
others (it creates its own lattice and takes nothing from them)."""
import numpy as np
import pytest

from xt_inputs import configs as C

pytestmark = pytest.mark.gpu

KEYS = ("x", "px", "y", "py", "zeta", "delta", "ptau", "rpp", "rvv", "s", "at_turn", "state", "at_element")


@pytest.fixture(scope="module")
def X():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (run with -m gpu on the B200 box)")
    import paper_2310_00317_b200 as X
    return X


def assert_same_bits(got, ref):
    for k in KEYS:
        a, r = got[k], ref[k]
        same = (a.view(np.int64) == r.view(np.int64)) if a.dtype == np.float64 else (a == r)
        assert same.all(), "%s: %d of %d differ from xt_track_ex" % (k, int((~same).sum()), len(same))


def ensembles():
    """Amplitude scan of configs[4] (particles beyond the dynamic aperture are lost within a few turns)."""
    full = C.particles(4)
    n = len(full["x"])
    big = C.subsample(full, np.linspace(0, n - 1, 20011).astype(np.int64))
    small = C.subsample(full, np.linspace(n // 3, n - 1, 3001).astype(np.int64))
    return big, small


@pytest.mark.parametrize("kind", ["prod", "nofma"])
def test_static_workspace_tracking_equals_xt_track_ex(X, kind):
    import torch
    lat = X.xt_lattice_create(C.pack(C.lattice(4)), kind=kind)
    big, small = ensembles()
    turns, every = 14, 4                                    # 4 passes: the initial partition + 3 between launches

    def existing(coords):
        p = X.new_particles(lat, coords)
        st = X.xt_track_ex(lat, p, turns, compact_every=every, stats=True)
        return X.particles_to_host(p), st

    ref_big, st_big = existing(big)
    ref_small, st_small = existing(small)
    assert st_big["n_passes"] == 4 and st_small["n_passes"] == 4
    lost_big = int((ref_big["state"] != 1).sum())
    assert 0 < lost_big < len(big["x"]) and 0 < int((ref_small["state"] != 1).sum()) < len(small["x"])
    assert st_big["pass_n_out"][3] < st_big["pass_n_in"][0]     # the passes really retired particles

    for coords, ref in ((big, ref_big), (small, ref_small), (big, ref_big)):   # calls in a row, one shared array
        p = X.new_particles(lat, coords)
        launches = X.xt_launch_count(kind)
        X.xt_track_static(lat, p, turns, compact_every=every)
        assert X.xt_launch_count(kind) - launches == 4 + 4 + 1   # 4 passes, 4 tracking launches, the scatter
        assert_same_bits(X.particles_to_host(p), ref)

    # another launch shape through the same entry point, still the same bits
    p = X.new_particles(lat, small)
    X.xt_track_static(lat, p, turns, compact_every=every, particles_per_thread=1, block_size=64, turns_per_launch=3)
    assert_same_bits(X.particles_to_host(p), ref_small)

    # the limit: exactly XT_TRACK_STATIC_MAX_PARTICLES fits, one more is refused with a message naming the limit
    n_max = X.XT_TRACK_STATIC_MAX_PARTICLES
    assert X.xt_track_workspace_bytes(n_max, kind) <= 8 << 20
    full = C.particles(4)
    at_max = C.subsample(full, np.linspace(0, len(full["x"]) - 1, n_max).astype(np.int64))
    a, b = X.new_particles(lat, at_max), X.new_particles(lat, at_max)
    X.xt_track_ex(lat, a, 9, compact_every=4)
    X.xt_track_static(lat, b, 9, compact_every=4)
    assert_same_bits(X.particles_to_host(b), X.particles_to_host(a))
    over = C.subsample(full, np.linspace(0, len(full["x"]) - 1, n_max + 1).astype(np.int64))
    q = X.new_particles(lat, over)
    untouched = X.particles_to_host(q)
    with pytest.raises(X.XtError) as e:
        X.xt_track_static(lat, q, 9, compact_every=4)
    assert e.value.code == -1 and "XT_TRACK_STATIC_MAX_PARTICLES" in str(e.value) and str(n_max) in str(e.value)
    assert_same_bits(X.particles_to_host(q), untouched)

    # a caller-owned workspace or a stats record make no sense here and are refused (opts is passed by hand)
    import ctypes
    from paper_2310_00317_b200 import binding as B
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    o = B.xt_track_opts()
    o.compact_every = every
    o.workspace, o.workspace_bytes = ws.data_ptr(), 1024
    st = B._struct_from_tensors(p)
    rc = lat._lib.xt_track_static(lat.handle, ctypes.byref(st), len(small["x"]), turns, B._stream_ptr(None),
                                  ctypes.byref(o))
    assert rc == -1 and b"workspace" in lat._lib.xt_last_error()

    # empty ensemble and zero turns: successful no-ops, as in xt_track_ex
    X.xt_track_static(lat, X.new_particles(lat, {k: np.zeros(0) for k in C.COORDS}), 5)
    X.xt_track_static(lat, p, 0)
    assert_same_bits(X.particles_to_host(p), ref_small)
    lat.close()
