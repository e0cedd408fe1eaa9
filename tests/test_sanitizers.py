"""ASan / UBSan runs of the two host-side parsers of the packed lattice buffer:
the oracle (oracle/xt_oracle.cpp) and the product's packer (csrc/xt_lattice.cu, compiled as plain C++).
Each is built into its own small driver (tests/sanitize/) with -fsanitize=address,undefined and fed the
same corpus: the config lattices, seeded random lines of every element type, and malformed buffers
(truncated, oversized counts, unknown types, non-finite numbers, random byte flips).  A sanitizer report
aborts the driver, which fails the test.  No GPU involved; compute-sanitizer stays closed on this pool
(DESIGN.md section 9)."""
import os
import shutil
import struct
import subprocess

import numpy as np
import pytest

from xt_inputs import configs as C
from xt_inputs.packed import (Bend, Cavity, Drift, LimitEllipse, LimitPolygon, LimitRect, Marker, Multipole,
                              Quadrupole, RadMultipole, SRotation, XYShift, pack_lattice)

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SAN = os.path.join(ROOT, "tests", "sanitize")
P0C, MASS0 = 450e9, 938272088.16
FLAGS = ["-std=c++17", "-g", "-O1", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
         "-fno-omit-frame-pointer", "-ffp-contract=off"]


def _cuda_home():
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    return os.path.dirname(os.path.dirname(os.path.realpath(nvcc)))


@pytest.fixture(scope="module")
def drivers(tmp_path_factory):
    out = tmp_path_factory.mktemp("san")
    cuda = _cuda_home()
    packer = str(out / "san_packer")
    oracle = str(out / "san_oracle")
    subprocess.run(["g++", *FLAGS, "-I", os.path.join(cuda, "include"), "-x", "c++",
                    os.path.join(ROOT, "paper_2310_00317_b200", "csrc", "xt_lattice.cu"),
                    os.path.join(SAN, "san_packer.cpp"), "-L", os.path.join(cuda, "lib64"), "-lcudart",
                    "-o", packer], check=True)
    subprocess.run(["g++", *FLAGS, os.path.join(ROOT, "oracle", "xt_oracle.cpp"),
                    os.path.join(SAN, "san_oracle.cpp"), "-o", oracle], check=True)
    return packer, oracle, corpus(out)


def random_line(rng, n):
    els = []
    for _ in range(n):
        k = int(rng.integers(0, 12))
        if k == 0:
            els.append(Drift(float(rng.uniform(0.0, 3.0))))
        elif k == 1:
            order = int(rng.integers(0, 21))
            curved = rng.random() < 0.3
            els.append(Multipole(knl=tuple(rng.normal(0, 1e-3, order + 1)), ksl=tuple(rng.normal(0, 1e-3, order + 1)),
                                 hxl=float(rng.normal(0, 1e-3)) if curved else 0.0,
                                 length=float(rng.uniform(0, 2.0)) if rng.random() < 0.8 else 0.0))
        elif k == 2:
            els.append(Cavity(float(rng.normal(0, 1e6)), float(rng.uniform(1e8, 5e8)), float(rng.uniform(0, 360))))
        elif k == 3:
            t = float(rng.normal(0, 1e-3))
            els.append(SRotation(float(np.cos(t)), float(np.sin(t))))
        elif k == 4:
            els.append(XYShift(float(rng.normal(0, 1e-4)), float(rng.normal(0, 1e-4))))
        elif k == 5:
            els.append(LimitRect(-0.01, 0.012, -0.008, 0.009))
        elif k == 6:
            els.append(LimitEllipse(0.02, 0.015))
        elif k == 7:
            els.append(Marker())
        elif k == 8:
            els.append(Quadrupole(float(rng.choice([-1, 1])) * float(rng.uniform(1e-3, 0.1)), float(rng.uniform(0.1, 3))))
        elif k == 9:
            h = float(rng.uniform(1e-4, 1e-2))
            els.append(Bend(h * float(rng.uniform(0.999, 1.001)), h, float(rng.uniform(0.5, 6))))
        elif k == 10:
            m = int(rng.integers(3, 12))
            ang = np.sort(rng.uniform(0, 2 * np.pi, m))
            els.append(LimitPolygon(tuple(0.02 * np.cos(ang)), tuple(0.015 * np.sin(ang))))
        else:
            order = int(rng.integers(0, 6))
            els.append(RadMultipole(knl=tuple(rng.normal(0, 1e-3, order + 1)), ksl=tuple(rng.normal(0, 1e-3, order + 1)),
                                    hxl=float(rng.normal(0, 1e-3)), length=float(rng.uniform(0.1, 2.0))))
    return els


def corpus(out_dir):
    rng = np.random.default_rng(4242)
    bufs = {}
    for cfg in (0, 1, 2, 3):
        bufs["cfg%d" % cfg] = C.pack(C.lattice(cfg))
    for i in range(12):
        bufs["rand%02d" % i] = pack_lattice(random_line(rng, int(rng.integers(1, 60))), P0C, MASS0, 1.0)
    bufs["empty"] = pack_lattice([], P0C, MASS0, 1.0)
    good = bufs["rand03"]
    small = pack_lattice([Drift(1.0), Multipole(knl=(0.0, 0.1)), LimitEllipse(0.02, 0.01)], P0C, MASS0, 1.0)
    # malformed: truncations, a count the buffer cannot hold (2^32 - 1 elements in 48 bytes), a
    # count larger than the records present, unknown type, order / vertex counts out of range, NaN, byte flips
    for cut in (0, 1, 7, 47, 48, 49, 56, len(small) - 1, len(small) - 8):
        bufs["cut%d" % cut] = small[:cut]
    hdr = bytearray(small[:48])
    struct.pack_into("<I", hdr, 12, 0xFFFFFFFF)
    struct.pack_into("<Q", hdr, 40, 48)
    bufs["huge_count"] = bytes(hdr)
    hdr2 = bytearray(small)
    struct.pack_into("<I", hdr2, 12, 1 << 20)
    bufs["count_gt_records"] = bytes(hdr2)

    def one_record(type_id, aux, payload):
        h = bytearray(small[:48])
        rec = struct.pack("<II", type_id, aux) + payload
        struct.pack_into("<I", h, 12, 1)
        struct.pack_into("<Q", h, 40, 48 + len(rec))
        return bytes(h) + rec

    bufs["unknown_type"] = one_record(99, 0, struct.pack("<d", 1.0))
    bufs["order_400"] = one_record(2, 400, b"\0" * 64)
    bufs["polygon_2"] = one_record(10, 2, b"\0" * 32)
    bufs["nan_drift"] = pack_lattice([Drift(float("nan"))], P0C, MASS0, 1.0)
    for i in range(24):
        b = bytearray(good)
        for _ in range(int(rng.integers(1, 6))):
            b[int(rng.integers(8, len(b)))] = int(rng.integers(0, 256))
        bufs["flip%02d" % i] = bytes(b)
    paths = []
    for name, b in bufs.items():
        path = os.path.join(str(out_dir), name + ".bin")
        with open(path, "wb") as fh:
            fh.write(b)
        paths.append(path)
    return paths


def _run(exe, paths):
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:allocator_may_return_null=1",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    res = subprocess.run([exe, *paths], capture_output=True, text=True, env=env, timeout=600)
    assert res.returncode == 0, "sanitizer report or crash:\n%s\n%s" % (res.stdout[-2000:], res.stderr[-6000:])
    assert "ERROR: AddressSanitizer" not in res.stderr and "runtime error" not in res.stderr, res.stderr[-6000:]
    return res.stdout


BAD = ("huge_count", "count_gt_records", "unknown_type", "order_400", "polygon_2", "nan_drift", "cut47", "cut56")


def test_packer_under_asan_ubsan(drivers):
    packer, _, paths = drivers
    text = _run(packer, paths)
    lines = {ln.split(" ")[0].split("/")[-1]: ln for ln in text.splitlines() if "chunk=0 fuse=0" in ln}
    assert len(lines) == len(paths)
    for ok in ("cfg0", "cfg1", "cfg2", "cfg3", "rand00", "rand11", "empty"):
        assert "bytes" in lines[ok + ".bin"], lines[ok + ".bin"]
    for bad in BAD:
        assert "rc -2" in lines[bad + ".bin"], lines[bad + ".bin"]          # XT_ERR_BAD_LATTICE, no exception


def test_oracle_under_asan_ubsan(drivers):
    _, oracle, paths = drivers
    text = _run(oracle, paths)
    lines = {ln.split(":")[0].split("/")[-1]: ln for ln in text.splitlines()}
    assert len(lines) == len(paths)
    for ok in ("cfg0", "cfg1", "cfg2", "cfg3", "rand00", "rand11", "empty"):
        assert "track rc 0" in lines[ok + ".bin"], lines[ok + ".bin"]
    for bad in BAD:
        assert "track rc 0" not in lines[bad + ".bin"], lines[bad + ".bin"]
