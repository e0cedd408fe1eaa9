"""CPU tests of the boundary and the host logic (no GPU, no compute call):

* both shared objects load and export every function ``include/xt.h`` declares;
* step P (the lattice packer) through ``xt_lattice_pack_host``: the device image is walked
  record by record with an independent decoder of the format documented in
  ``csrc/xt_internal.h``; counts, sizes, chunking, fusion and error codes are checked;
* argument validation of the compute entry points that needs no device;
* the multi-rank plumbing of ``bench.py`` with world_size 2 on gloo.
"""
import ctypes
import os
import re
import struct
import sys

import numpy as np
import pytest

import paper_2310_00317_b200 as X
from paper_2310_00317_b200 import binding as B
from xt_inputs import configs as C
from xt_inputs.packed import (Cavity, Drift, LimitEllipse, LimitRect, Marker, Multipole, SRotation,
                              XYShift, pack_lattice)

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
P0C, MASS0 = 450e9, 938272088.16

T_END, T_DRIFT, T_MULT, T_CAV, T_SROT, T_SHIFT, T_RECT, T_ELL, T_CMULT = range(9)
F_PRE, F_POST, F_POST2, F_MISAL, F_APER = 0x10, 0x20, 0x40, 0x80, 0x8000


def pack(els):
    return pack_lattice(els, P0C, MASS0, 1.0)


def declared_functions():
    text = open(os.path.join(ROOT, "include", "xt.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(xt_[a-z0-9_]+)\s*\(", text)))


# ------------------------------------------------------------------------------- ABI
@pytest.mark.parametrize("kind", ["prod", "nofma"])
def test_library_loads_and_exports_every_declared_symbol(kind):
    lib = X.load_library(kind)
    names = declared_functions()
    assert len(names) >= 15 and "xt_track" in names and "xt_lattice_create_ex" in names
    for name in names:
        assert hasattr(lib, name), "%s is declared in include/xt.h but not exported" % name
        assert name in B.SIGNATURES, "%s has no ctypes signature in the binding" % name
    info = X.xt_build_info(kind)
    assert "sm_100a" in info and ("fmad=false" in info) == (kind == "nofma")


def test_struct_layouts_match_the_header():
    # sizes the C compiler gives the public structs (LP64): 14 pointers; 2 x i64 + 2 x i32; ...
    assert ctypes.sizeof(B.xt_particles) == 14 * 8
    assert ctypes.sizeof(B.xt_track_opts) == 56          # + workspace ptr, bytes, stats ptr, cold_in_registers, balance
    assert ctypes.sizeof(B.xt_track_stats) == 7 * 8 + 3 * 8 * B.XT_STATS_MAX_PASSES
    assert ctypes.sizeof(B.xt_lattice_opts) == 16
    assert ctypes.sizeof(B.xt_lattice_info) == 8 * (5 + 8 + 3) + 8 * 3 + 8 + 8 + 8


def test_track_workspace_bytes_holds_step_c_and_the_queue():
    """xt_track_workspace_bytes (host arithmetic, no device): two working sets of 14 arrays for step C, and
    behind them the queue of the balanced mode for the auto shapes (one word per item: up to 256 blocks of
    turns per group of 256 particles); 256-byte granular, monotonic, 0 for an empty ensemble."""
    for kind in ("prod", "nofma"):
        assert X.xt_track_workspace_bytes(0, kind) == 0 and X.xt_track_workspace_bytes(-5, kind) == 0
        last = 0
        for n in (1, 31, 256, 257, 5003, 32768, 100000, 2000400, 10 ** 7):
            b = X.xt_track_workspace_bytes(n, kind)
            groups = -(-n // 256)
            assert b % 256 == 0 and b >= last
            assert b >= 2 * 14 * 8 * n + 8 * (-(-n // 256)) + 4 * 256 * groups
            assert b <= 2 * 14 * (8 * n + 256) + 8 * groups + 4 * 256 * groups + 2048
            last = b
    assert X.xt_track_workspace_bytes(X.XT_TRACK_STATIC_MAX_PARTICLES) <= 8 << 20


def test_compute_calls_validate_arguments_without_a_device():
    lib = X.load_library("prod")
    assert lib.xt_track(None, None, 0, 0, None) == -1                    # XT_ERR_INVALID_ARG
    assert b"NULL" in lib.xt_last_error()
    assert lib.xt_survival_histogram(None, None, 0, 0, 10, None, None) == -1
    assert lib.xt_lattice_destroy(None) == 0
    out = ctypes.c_void_p()
    assert lib.xt_lattice_create(None, 0, ctypes.byref(out)) == -1 and not out.value
    import torch
    if not torch.cuda.is_available():                                    # no CPU fallback: fails loudly
        buf = pack([Drift(1.0)])
        rc = lib.xt_lattice_create(buf, len(buf), ctypes.byref(out))
        assert rc == -3 and not out.value, "xt_lattice_create must fail with XT_ERR_CUDA without a device"
        with pytest.raises(X.XtError):
            X.xt_lattice_create(buf)


# ------------------------------------------------------------------- image decoder
def walk_image(img, chunk_bytes):
    """-> list of chunks, each a list of records (type, flags, order, elem, p0, slots[doubles])."""
    chunks, pos = [], 0
    while pos < len(img):
        start = pos
        tag, _, _ = struct.unpack_from("<IId", img, pos)
        pos += 16
        recs = []
        while tag & 0xF != T_END:
            size = tag >> 16
            nxt, elem, p0 = struct.unpack_from("<IId", img, pos)
            assert size >= 16 and size % 16 == 0
            slots = struct.unpack_from("<%dd" % ((size - 16) // 8), img, pos + 16)
            recs.append((tag & 0xF, tag & 0x80F0, (tag >> 8) & 0x7F, elem, p0, slots))
            pos += size
            tag = nxt
        assert pos - start <= chunk_bytes
        chunks.append(recs)
    assert pos == len(img)
    return chunks


def maps_of(rec):
    """Element maps a record stands for, in order, as (kind, parameters)."""
    typ, flags, order, elem, p0, s = rec
    out, k = [], 0
    if flags & F_APER:                                   # trailing LimitEllipse: {b2, a2}, {a2 b2, elem}
        inner = maps_of((typ, flags & ~F_APER, order, elem, p0, s[:-4]))
        assert s[-2] == s[-4] * s[-3] and s[-1] == int(s[-1]) > elem
        return inner + [("ellipse", (s[-4], s[-3]))]
    if typ == T_DRIFT:
        out.append(("drift", p0))
        if flags & F_POST:
            out.append(("drift", s[0]))
        return out
    if typ in (T_MULT, T_CMULT):
        # {l_pre, l_post} {l_post2, wf} [4 misalignment slots] then the coefficient pairs, highest order first
        l_pre, l_post, l_post2, wf = s[0], s[1], s[2], s[3]
        k = 4
        if typ != T_CMULT:
            assert wf == 0.0
            wf = None
        if not flags & F_PRE:
            assert l_pre == 0.0
        if not flags & F_POST:
            assert l_post == 0.0
        if not flags & F_POST2:
            assert l_post2 == 0.0
        if flags & F_PRE:
            out.append(("drift", l_pre))
        mis = s[k:k + 8] if flags & F_MISAL else None
        if mis:
            out += [("shift", mis[0:2]), ("srot", mis[2:4])]
            k += 8
        coef = s[k:k + 2 * (order + 1)]
        k += 2 * (order + 1)
        out.append(("mult", (order, p0 if typ == T_CMULT else 0.0, wf, coef)))
        if mis:
            out += [("srot", mis[4:6]), ("shift", mis[6:8])]
        if flags & F_POST:
            out.append(("drift", l_post))
        if flags & F_POST2:
            out.append(("drift", l_post2))
        assert k == len(s)
        return out
    if typ in (T_SROT, T_SHIFT) and flags & F_POST:      # half a misalignment wrapper: two transforms
        a, b = ("srot", "shift") if typ == T_SROT else ("shift", "srot")
        return [(a, s[0:2]), (b, s[2:4])]
    return [({T_CAV: "cavity", T_SROT: "srot", T_SHIFT: "shift", T_RECT: "rect", T_ELL: "ellipse"}[typ], s)]


def all_maps(img, chunk_bytes):
    return [m for ch in walk_image(img, chunk_bytes) for r in ch for m in maps_of(r)]


def expected_maps(elements, beta0):
    """What step P must encode, from the element list."""
    out = []
    for el in elements:
        if isinstance(el, Marker):
            continue
        if isinstance(el, Drift):
            out.append(("drift", el.length))
        elif isinstance(el, Multipole):
            n = el.order
            knl = list(el.knl) + [0.0] * (n + 1 - len(el.knl))
            ksl = list(el.ksl) + [0.0] * (n + 1 - len(el.ksl))
            fact = [1.0]
            for i in range(1, n + 1):
                fact.append(fact[-1] * i)
            c = [knl[i] / fact[i] for i in range(n + 1)]
            s = [ksl[i] / fact[i] for i in range(n + 1)]
            wf = None
            if el.hxl != 0.0:
                c[0] = knl[0] - el.hxl
                wf = (knl[0] * el.hxl) / el.length if el.length != 0.0 else 0.0
            coef = []
            for i in range(n, -1, -1):                       # Horner order: highest first
                coef += [c[i], s[i]]
            out.append(("mult", (n, el.hxl, wf, tuple(coef))))
        elif isinstance(el, Cavity):
            out.append(("cavity", None))
        elif isinstance(el, SRotation):
            out.append(("srot", (el.cos_z, el.sin_z)))
        elif isinstance(el, XYShift):
            out.append(("shift", (el.dx, el.dy)))
        elif isinstance(el, LimitRect):
            out.append(("rect", (el.min_x, el.max_x, el.min_y, el.max_y)))
        elif isinstance(el, LimitEllipse):
            out.append(("ellipse", (el.b * el.b, el.a * el.a)))
    return out


def assert_same_maps(got, want):
    assert len(got) == len(want)
    for i, (g, w) in enumerate(zip(got, want)):
        assert g[0] == w[0], (i, g[0], w[0])
        if w[0] == "cavity":
            continue
        if w[0] == "mult":
            assert g[1][0] == w[1][0] and g[1][1] == w[1][1], i
            assert g[1][2] == w[1][2], (i, "weak-focusing coefficient")
            assert tuple(g[1][3]) == w[1][3], (i, "Horner coefficients")
        else:
            gv = g[1] if isinstance(g[1], tuple) else (g[1],)
            wv = w[1] if isinstance(w[1], tuple) else (w[1],)
            assert tuple(gv)[:len(wv)] == tuple(wv), (i, g, w)


ALL_TYPES = [Drift(1.5), XYShift(1e-4, -2e-4), SRotation.from_angle(1e-3),
             Multipole(knl=(5e-3, 0.1, 0.5, 5.0), ksl=(0.0, 1e-3, -0.2, 1.0), hxl=5e-3, length=14.3),
             SRotation.from_angle(-1e-3), XYShift(-1e-4, 2e-4), Drift(0.25), Drift(0.75), Marker(),
             Cavity(1e6, 200e6, 180.0), Drift(1.0), LimitRect(-0.01, 0.01, -0.02, 0.02), Drift(2.0),
             Multipole(knl=(0.0, 0.1)), LimitEllipse(0.02, 0.015), Multipole(knl=(0.0, 0.0, 0.5)), Drift(3.0),
             Drift(0.5), Drift(0.125), Multipole(knl=(1e-3,), hxl=1e-3, length=0.0)]


# ------------------------------------------------------------------------ step P
def merge_drifts(maps):
    """What the PRODUCTION packer encodes: consecutive drifts as one drift of the summed length (exact
    composition; the validation build keeps every drift)."""
    out = []
    for m in maps:
        if m[0] == "drift" and out and out[-1][0] == "drift":
            out[-1] = ("drift", out[-1][1] + m[1])
        else:
            out.append(m)
    return out


@pytest.mark.parametrize("kind", ["nofma", "prod"])
@pytest.mark.parametrize("fuse", [True, False])
def test_packer_encodes_every_map_in_order_with_prescaled_coefficients(fuse, kind):
    buf = pack(ALL_TYPES)
    img, info = X.xt_lattice_pack_host(buf, kind=kind, fuse=fuse)
    assert info["n_elements"] == len(ALL_TYPES) and info["image_bytes"] == len(img)
    assert info["n_by_type"] == [1, 8, 4, 1, 2, 2, 1, 1]
    assert info["sum_order"] == 3 + 1 + 2 + 0 and info["n_curved"] == 2 and info["has_aperture"] == 1
    assert info["circumference"] == 1.5 + 0.25 + 0.75 + 1.0 + 2.0 + 3.0 + 0.5 + 0.125
    e0 = np.sqrt(P0C * P0C + MASS0 * MASS0)
    assert info["beta0"] == P0C / e0 and info["gamma0"] == e0 / MASS0
    chunks = walk_image(img, info["chunk_bytes"])
    assert len(chunks) == info["n_chunks"] == 1
    assert sum(len(c) for c in chunks) == info["n_records"]
    want = expected_maps(ALL_TYPES, info["beta0"])
    merged = kind == "prod"
    assert_same_maps(all_maps(img, info["chunk_bytes"]), merge_drifts(want) if merged else want)
    assert info["n_drift_applies"] == (5 if merged else 8)          # [0.25 0.75] and [3.0 0.5 0.125] become one each
    if fuse:
        # [D shift rot M rot shift D D], cavity, D, rect, [D M + ellipse], [M D D], [D M]
        assert info["n_records"] == 7
        assert chunks[0][4][1] == (F_PRE | F_APER)
        first = chunks[0][0]
        flags = F_PRE | F_POST | F_MISAL | (0 if merged else F_POST2)
        assert first[0] == T_CMULT and first[1] == flags and first[3] == 3
        # pre + post, D, [D M], [M D D], [D M]; merged: the last three drifts are one, behind the first of the two magnets
        assert info["n_drift_evals"] == (2 + 1 + 1 + 1 + 0 if merged else 2 + 1 + 1 + 1 + 1)
    elif not merged:
        assert info["n_records"] == len(ALL_TYPES) - 1             # the marker has no record
        assert info["n_drift_evals"] == 8
        assert [r[3] for r in chunks[0]] == [i for i, e in enumerate(ALL_TYPES) if not isinstance(e, Marker)]
    else:
        assert info["n_records"] == len(ALL_TYPES) - 1 - 3 and info["n_drift_evals"] == 5


def test_cavity_and_aperture_constants():
    buf = pack([Cavity(2e6, 400e6, 90.0), LimitEllipse(0.02, 0.015)])
    img, info = X.xt_lattice_pack_host(buf)
    (cav, ell), = walk_image(img, info["chunk_bytes"])
    beta0 = info["beta0"]
    pi = 3.14159265358979323846
    assert cav[4] == 90.0 * (pi / 180.0)                                      # lag_rad
    assert cav[5][0] == (2.0 * pi * 400e6) / (beta0 * 299792458.0)            # kz
    assert cav[5][1] == (1.0 * 2e6) / P0C                                     # vn
    a2, b2 = 0.02 * 0.02, 0.015 * 0.015
    assert ell[4] == a2 * b2 and ell[5][:2] == (b2, a2) and ell[3] == 1


@pytest.mark.parametrize("kind", ["nofma", "prod"])
@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_config_lattices_chunking_and_fusion(cfg, kind):
    els = C.lattice(cfg)
    buf = C.pack(els)
    img, info = X.xt_lattice_pack_host(buf, kind=kind)
    want = expected_maps(els, info["beta0"])
    n_drifts = sum(1 for m in want if m[0] == "drift")
    if kind == "prod":
        want = merge_drifts(want)
    assert_same_maps(all_maps(img, info["chunk_bytes"]), want)
    assert info["n_by_type"][1] == n_drifts and info["n_drift_evals"] <= n_drifts
    assert info["n_drift_applies"] == sum(1 for m in want if m[0] == "drift")
    for kw in (dict(fuse=False), dict(chunk_bytes=1024), dict(chunk_bytes=65536, fuse=False)):
        img2, info2 = X.xt_lattice_pack_host(buf, kind=kind, **kw)
        assert info2["chunk_bytes"] == kw.get("chunk_bytes", 8192)
        chunks = walk_image(img2, info2["chunk_bytes"])
        assert len(chunks) == info2["n_chunks"] and sum(len(c) for c in chunks) == info2["n_records"]
        assert_same_maps([m for ch in chunks for r in ch for m in maps_of(r)], want)
        assert info2["circumference"] == info["circumference"]
    if cfg >= 2:                                             # multi-chunk, mostly fused
        assert info["n_chunks"] > 40 and info["n_records"] < 0.5 * info["n_elements"]
        assert info["n_drift_evals"] < 0.65 * n_drifts
        if kind == "prod":                                   # [D M D][D M D]: every interior pair of drifts is one
            assert info["n_drift_applies"] < 0.56 * n_drifts


def test_empty_and_marker_only_lattices():
    for els in ([], [Marker(), Marker()]):
        img, info = X.xt_lattice_pack_host(pack(els))
        assert info["n_records"] == 0 and info["n_chunks"] == 1 and len(img) == 16
        assert walk_image(img, info["chunk_bytes"]) == [[]]


def test_bad_buffers_and_options_are_rejected():
    lib = X.load_library("prod")
    good = pack([Drift(1.0)])
    bad = [good[:-1], b"XXXX" + good[4:], good + b"\0" * 8, pack([Multipole(knl=(0.0,) * 22)]),
           pack([Drift(float("nan"))]), pack_lattice([Drift(1.0)], -1.0, MASS0, 1.0),
           good[:48] + struct.pack("<IId", 99, 0, 1.0)]
    for b in bad:
        rc = lib.xt_lattice_pack_host(b, len(b), None, None, 0, None)
        assert rc == -2, rc                                                   # XT_ERR_BAD_LATTICE
        assert lib.xt_last_error()
    for kw in (dict(chunk_bytes=1000), dict(chunk_bytes=512), dict(chunk_bytes=131072)):
        with pytest.raises(X.XtError) as e:
            X.xt_lattice_pack_host(good, **kw)
        assert e.value.code == -1
    big = pack([Multipole(knl=(0.0,) * 21, ksl=(0.0,) * 21)] * 3)              # 384-byte records
    img, info = X.xt_lattice_pack_host(big, chunk_bytes=1024)
    assert info["n_chunks"] == 2                                              # 16 + 2 x 384 fits, the third does not
    assert X.xt_lattice_pack_host(good)[1]["n_records"] == 1


# ------------------------------------------------- multi-rank plumbing (gloo, world_size 2)
def _rank_main(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.reduce_max(100.0 + 50.0 * rank, world, "cpu")                # slowest rank sets the time
    buf, coords = bench.make_inputs(0, rank)
    np.save(os.path.join(out_dir, "r%d.npy" % rank),
            np.array([ms, bench.whole_job_value(1000.0, world, ms), coords["x"][0], len(coords["x"]), len(buf)]))
    dist.barrier()
    dist.destroy_process_group()


def test_bench_rank_plumbing_world_size_2(tmp_path):
    import torch.multiprocessing as mp
    port = 29500 + (os.getpid() % 400)
    mp.spawn(_rank_main, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0, r1 = (np.load(os.path.join(str(tmp_path), "r%d.npy" % r)) for r in (0, 1))
    assert r0[0] == r1[0] == 150.0                                           # MAX over ranks on both
    assert r0[1] == r1[1] == 2 * 1000.0 / 0.150                              # whole-job aggregate
    assert r0[2] != r1[2] and r0[3] == r1[3] == 1000                         # own ensemble, same size
    assert r0[4] == r1[4]                                                    # same (replicated) lattice


def test_thick_quadrupole_is_packed_unfused():
    from xt_inputs.packed import Quadrupole
    els = [Drift(1.0), Quadrupole(0.3, 2.5), Drift(0.5), Multipole(knl=(0.0, 0.1)), Quadrupole(-0.2, 1.0)]
    img, info = X.xt_lattice_pack_host(pack(els))
    assert info["n_thick"] == 2 and info["n_by_type"][1] == 2 and info["circumference"] == 5.0
    (recs,) = walk_image(img, info["chunk_bytes"])
    kinds = [(r[0], r[1]) for r in recs]
    assert kinds == [(T_DRIFT, 0), (9, 0), (T_MULT, F_PRE), (9, 0)]            # 9 = TAG_QUAD, never fused
    assert recs[1][4] == 0.3 and recs[1][5][0] == 2.5 and recs[1][3] == 1
    lib = X.load_library("prod")
    for bad in (Quadrupole(0.0, 1.0), Quadrupole(0.1, 0.0)):
        b = pack([bad])
        assert lib.xt_lattice_pack_host(b, len(b), None, None, 0, None) == -2


def test_thick_bend_is_packed_unfused():
    from xt_inputs.packed import Bend, Quadrupole
    els = [Drift(1.0), Bend(2e-3, 2.1e-3, 3.0), Drift(0.5), Quadrupole(0.3, 1.5), Bend(1e-3, 1e-3, 2.0), Drift(1.0)]
    img, info = X.xt_lattice_pack_host(pack(els))
    assert info["n_thick"] == 3 and info["circumference"] == 9.0                # bends advance s by the arc length
    (recs,) = walk_image(img, info["chunk_bytes"])
    assert [(r[0], r[1]) for r in recs] == [(T_DRIFT, 0), (10, 0), (T_DRIFT, 0), (9, 0), (10, 0), (T_DRIFT, 0)]
    assert recs[1][4] == 2e-3 and tuple(recs[1][5][:2]) == (2.1e-3, 3.0) and recs[1][3] == 1   # p0 = k0, slot {h, length}
    assert recs[4][4] == 1e-3 and tuple(recs[4][5][:2]) == (1e-3, 2.0) and recs[4][3] == 4
    lib = X.load_library("prod")
    for bad in (Bend(0.0, 1e-3, 1.0), Bend(1e-3, 0.0, 1.0), Bend(1e-3, -1e-3, 1.0), Bend(1e-3, 1e-3, 0.0)):
        b = pack([bad])
        assert lib.xt_lattice_pack_host(b, len(b), None, None, 0, None) == -2


def test_polygon_aperture_is_packed_unfused_and_refine_rejects_bad_arguments():
    from xt_inputs.packed import LimitPolygon
    tri = LimitPolygon((0.0, 1.0, 0.0), (0.0, 0.0, 2.0))
    els = [Drift(1.0), Multipole(knl=(0.0, 0.1)), tri, Drift(0.5), LimitEllipse(0.01, 0.02)]
    img, info = X.xt_lattice_pack_host(pack(els))
    assert info["has_aperture"] == 1 and info["n_thick"] == 0
    (recs,) = walk_image(img, info["chunk_bytes"])
    assert [r[0] for r in recs][:2] == [T_MULT, 11]                             # 11 = TAG_POLY; never fused into the kick
    assert recs[1][3] == 2 and list(recs[1][5][:6]) == [0.0, 0.0, 1.0, 0.0, 0.0, 2.0]
    lib = X.load_library("prod")
    for bad in (LimitPolygon((0.0, 1.0), (0.0, 1.0)), LimitPolygon(tuple(range(257)), tuple(range(257)))):
        b = pack([bad])
        assert lib.xt_lattice_pack_host(b, len(b), None, None, 0, None) == -2
    big = pack([LimitPolygon(tuple(float(i) for i in range(256)), tuple(float(i * i) for i in range(256)))])
    assert lib.xt_lattice_pack_host(big, len(big), None, None, 0, None) > 4096
    assert lib.xt_refine_loss_location(None, None, 0, 0.1, 16, None, None) == -1  # NULL lattice: no CUDA call
    assert lib.xt_lattice_set_knobs(None, None, 1, 1, None, 0) == -1 and lib.xt_track_knobs(None, None, 0, 1, 0, None) == -1
    assert ctypes.sizeof(X.binding.xt_knob_link) == 32


def test_internal_monitor_type_is_not_a_public_element():
    body = struct.pack("<IId", 11, 0, 0.0)
    buf = struct.pack("<8sIIdddQ", b"XTLAT001", 1, 1, 450e9, 938272088.16, 1.0, 48 + len(body)) + body
    lib = X.load_library("prod")
    assert lib.xt_lattice_pack_host(buf, len(buf), None, None, 0, None) == -2
    assert lib.xt_twiss4d_line(None, 0.0, 1e-4, None, None, None, 0, None) == -1
    assert ctypes.sizeof(B.xt_twiss_row) == 21 * 8


def test_normal_form_matches_the_oracle_eigen_decomposition():
    """xt_twiss4d_normal_form is host arithmetic (reciprocal characteristic polynomial, projector eigenvectors):
    checked here, without a GPU, against oracle/make_optics.normal_form4 (numpy.linalg.eig) on one-turn matrices
    the oracle tracker produced: uncoupled, seen from a rotated frame, with a skew quadrupole, the LHC-sized ring."""
    from oracle import make_optics as MO
    from xt_inputs.packed import SRotation
    kq, L = 0.1, 2.0
    ring = [Multipole(knl=(0.0, kq)), Drift(L), Multipole(knl=(0.0, -0.95 * kq)), Drift(L)] * 10
    cases = [ring, [SRotation.from_angle(-0.3)] + ring + [SRotation.from_angle(0.3)],
             [Multipole(knl=(0.0, 0.0), ksl=(0.0, 0.004))] + ring, C.lattice(2)]
    for els in cases:
        m = MO.optics_of(pack(els))["m"]
        want, got = MO.normal_form4(m), X.xt_twiss4d_normal_form(m)
        assert got["stable"] == 1 and got["degenerate"] == 0
        # the two methods agree to rounding on a symplectic matrix; the central-difference matrix of the big
        # nonlinear ring is symplectic to 1e-5 only, and the methods split that error differently
        big = len(els) > 1000
        scale = max(want["betx1"], want["bety2"])
        for k in ("q1_frac", "q2_frac"):
            assert abs(got[k] - want[k]) < (5e-7 if big else 1e-12), k
        for k in ("betx1", "bety1", "betx2", "bety2", "alfx1", "alfy1", "alfx2", "alfy2"):
            assert abs(got[k] - want[k]) < (2e-5 if big else 1e-11) * scale, (k, got[k], want[k])
        for k in ("v1", "v2"):
            assert np.max(np.abs(got[k] - want[k])) < (2e-5 if big else 1e-11) * np.max(np.abs(want[k])), k
    # equal tunes (the symmetric FODO ring of configs[0]): flagged, not guessed; an unstable matrix: flagged
    sym = [Multipole(knl=(0.0, kq)), Drift(L), Multipole(knl=(0.0, -kq)), Drift(L)] * 10
    got = X.xt_twiss4d_normal_form(MO.optics_of(pack(sym))["m"])
    assert got["degenerate"] == 1 and got["stable"] == 1 and np.isnan(got["betx1"])
    bad = np.eye(4)
    bad[0, 0], bad[1, 1] = 2.0, 0.5
    got = X.xt_twiss4d_normal_form(bad)
    assert got["stable"] == 0 and np.isnan(got["q1_frac"])
    assert X.load_library("prod").xt_twiss4d_normal_form(None, None) == -1


def test_normal_form6_matches_the_oracle_eigen_decomposition():
    """xt_twiss6d_normal_form (host arithmetic: cubic in u = lambda + 1/lambda, projector eigenvectors) against
    oracle/make_optics.normal_form6 (numpy.linalg.eig) on 6x6 matrices the oracle tracker produced: a FODO ring
    with a cavity, the same seen from a rotated frame, and the dispersion ring of pin P24 (synchrotron tune
    1e-4: the longitudinal pair sits 5e-7 from u = 2, where the two methods split the 1e-6 asymplecticity of a
    central-difference matrix differently)."""
    from oracle import make_optics as MO
    from xt_inputs.packed import Cavity, SRotation
    cell = [Multipole(knl=(0.0, 0.1)), Drift(2.0), Multipole(knl=(0.0, -0.095)), Drift(2.0)]
    fodo = cell * 10 + [Cavity(1e5, 200e6, 0.0)]
    rot = [SRotation.from_angle(-0.3)] + fodo + [SRotation.from_angle(0.3)]
    th = 2.0 * np.pi / 16
    bend = Multipole(knl=(th,), hxl=th, length=1.5)
    ring = [Multipole(knl=(0.0, 0.25)), Drift(3.0), bend, Drift(3.0), Multipole(knl=(0.0, -0.25)), Drift(3.0), bend,
            Drift(3.0)] * 8 + [Cavity(2e4, 50e6, 180.0)]
    for els, p0c, tol in ((fodo, 1e9, 2e-8), (rot, 1e9, 2e-8), (ring, P0C, 1e-4)):
        m = MO.optics6d_of(pack_lattice(els, p0c, MASS0, 1.0))["m"]
        want, got = MO.normal_form6(m, 1.0), X.xt_twiss6d_normal_form(m, 1.0)
        assert got["stable"] == 1 and got["degenerate"] == 0
        for k, w in want.items():
            if k.startswith("v"):
                assert np.max(np.abs(got[k] - w)) < tol * np.max(np.abs(w)), k
            elif k.startswith("q"):
                assert abs(got[k] - w) < tol, (k, got[k], w)
            else:
                scale = max(abs(want["betx1"]), abs(want["bety2"])) if k[:3] in ("bet", "alf") and k[3] != "z" else 1.0
                assert abs(got[k] - w) < tol * max(abs(w), scale), (k, got[k], w)
    # rvv_co rescales the longitudinal momentum only: beta_z3 scales by 1/rvv (zeta per unit pzeta)
    a, b = X.xt_twiss6d_normal_form(m, 1.0), X.xt_twiss6d_normal_form(m, 1.0 + 1e-3)
    assert abs(b["q3_frac"] - a["q3_frac"]) < 1e-12 and abs(b["betx1"] / a["betx1"] - 1) < 1e-9
    assert abs(b["betz3"] / a["betz3"] * (1.0 + 1e-3) - 1.0) < 1e-6
    bad = np.eye(6)
    bad[0, 0], bad[1, 1] = 2.0, 0.5
    got = X.xt_twiss6d_normal_form(bad)
    assert got["stable"] == 0 and np.isnan(got["q1_frac"])
    assert X.load_library("prod").xt_twiss6d_normal_form(None, 1.0, None) == -1
    assert ctypes.sizeof(B.xt_twiss6d_modes) == 8 * (3 + 9 + 9 + 4 + 36) + 8
    assert ctypes.sizeof(B.xt_twiss6d_row) == 8 * (1 + 6 + 9 + 9 + 3 + 4)


def test_radiating_multipole_is_packed_unfused():
    from xt_inputs.packed import RadMultipole
    els = [Drift(1.0), RadMultipole(knl=(2e-3, 0.1, 6.0), ksl=(0.0, 0.01), hxl=1.5e-3, length=4.0), Drift(1.0)]
    img, info = X.xt_lattice_pack_host(pack(els))
    (recs,) = walk_image(img, info["chunk_bytes"])
    assert [r[0] for r in recs] == [T_DRIFT, 13, T_DRIFT]                         # 13 = TAG_RMULT: no drift fused into it
    slots = list(recs[1][5])
    assert recs[1][4] == 1.5e-3 and slots[:6] == [3.0, 0.0, 0.1, 0.01, 2e-3 - 1.5e-3, 0.0]   # Horner order, c[0] folded
    assert slots[6:8] == [(2e-3 * 1.5e-3) / 4.0, 4.0]
    r0 = 1.4399645478e-9 / 938272088.16
    assert abs(slots[8] / ((2.0 / 3.0) * r0 * (450e9 / 938272088.16) ** 3) - 1.0) < 1e-14
    lib = X.load_library("prod")
    for bad in (RadMultipole(knl=(1e-3,), length=0.0), RadMultipole(knl=(1e-3,), length=-2.0)):
        b = pack([bad])
        assert lib.xt_lattice_pack_host(b, len(b), None, None, 0, None) == -2
