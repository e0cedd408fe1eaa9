"""Pin P21 of the CPU oracle: the "mean" synchrotron-radiation model in a thin multipole (PAPER.md:130,
DESIGN.md reading A22) against textbook results, not against itself:

(a) an isomagnetic ring of N thin sector dipoles loses U0 = (4 pi/3) r0 m c^2 beta^3 gamma^4 / rho per turn;
(b) the lost fraction scales as kick^2, 1/length, (beta gamma)^3, q^2/m and, in a fixed field, as (1 + delta)
    (power ~ gamma^2 B^2);
(c) a vertical betatron oscillation in a ring with radiating dipoles and a cavity that restores the energy
    damps with the rate U0/(2E) per turn in amplitude (damping partition J_y = 1);
(d) a proton at 450 GeV/c does not notice: the map is the Multipole map; zero field: identity up to the
    rounding of re-deriving delta from the energy; length <= 0 rejected."""
import math

import numpy as np
import pytest

from oracle import make_optics as MO
from oracle import oracle as O
from xt_inputs.packed import Cavity, Drift, Multipole, RadMultipole, pack_lattice
import helpers as H

ME, MMU = 0.51099895e6, 105.6583755e6          # eV
R_E = 2.8179403262e-15                         # m, classical electron radius (CODATA 2018)
P0C = 45.6e9


def loss_fraction(el, p0c=P0C, mass0=ME, q0=-1.0, delta=0.0, x=0.0):
    buf = pack_lattice([el], p0c, mass0, q0)
    p = O.new_particles(buf, H.coords_from_rows([[x, 0.0, 0.0, 0.0, 0.0, delta]]))
    beta0, _ = O.reference(buf)
    e_before = p["ptau"][0] + 1.0 / beta0
    O.track(buf, p, 1)
    return (e_before - (p["ptau"][0] + 1.0 / beta0)) / e_before, p


def test_P21_isomagnetic_ring_loses_U0():
    n = 64
    th = 2.0 * math.pi / n
    gamma = math.sqrt(P0C ** 2 + ME ** 2) / ME
    beta = P0C / math.sqrt(P0C ** 2 + ME ** 2)
    for length in (1e3, 1e5):
        rho = n * length / (2.0 * math.pi)
        u0_over_e = (4.0 * math.pi / 3.0) * R_E * beta ** 3 * gamma ** 3 / rho
        got, p = loss_fraction(RadMultipole(knl=(th,), hxl=th, length=length))
        assert abs(got * n / u0_over_e - 1.0) < 2.0 * u0_over_e / n + 1e-9, (length, got * n, u0_over_e)
        # having lost half the energy before the kick, the particle is bent by theta/(1 + delta_mid): px = theta delta_mid
        assert abs(p["px"][0] + th * got / 2.0) < 1e-3 * th * got and p["x"][0] == 0.0
        assert abs((1.0 + p["delta"][0]) ** 2 - (p["ptau"][0] ** 2 + 2 * p["ptau"][0] / beta + 1.0)) < 1e-15
    assert 7e-4 < (4.0 * math.pi / 3.0) * R_E * beta ** 3 * gamma ** 3 / (n * 1e3 / (2 * math.pi)) < 9e-4    # FCC-ee-like


def test_P21_scaling_laws():
    base, _ = loss_fraction(RadMultipole(knl=(1e-3,), length=10.0))
    assert abs(loss_fraction(RadMultipole(knl=(2e-3,), length=10.0))[0] / base - 4.0) < 2e-5
    assert abs(loss_fraction(RadMultipole(knl=(0.0,), ksl=(1e-3,), length=10.0))[0] / base - 1.0) < 1e-9
    assert abs(loss_fraction(RadMultipole(knl=(1e-3,), length=5.0))[0] / base - 2.0) < 2e-5
    bg = lambda p0c, m: p0c / m
    assert abs(loss_fraction(RadMultipole(knl=(1e-3,), length=10.0), p0c=2 * P0C)[0] / base - 8.0) < 2e-5
    want = (ME / MMU) * (bg(P0C, MMU) / bg(P0C, ME)) ** 3
    strong = RadMultipole(knl=(0.1,), length=1e-3)                                   # a muon needs a field to notice
    want *= (0.1 / 1e-3) ** 2 * (10.0 / 1e-3)
    assert abs(loss_fraction(strong, mass0=MMU)[0] / base / want - 1.0) < 2e-5
    assert abs(loss_fraction(RadMultipole(knl=(1e-3,), length=10.0), q0=-2.0)[0] / base - 4.0) < 2e-5
    # a quadrupole field radiates as the square of the offset; a fixed field takes (1 + delta) times the fraction
    q1, q2 = (loss_fraction(RadMultipole(knl=(0.0, 0.05), length=2.0), x=x)[0] for x in (1e-3, 3e-3))
    assert abs(q2 / q1 - 9.0) < 1e-4
    hi, _ = loss_fraction(RadMultipole(knl=(1e-3,), length=10.0), delta=0.02)
    assert abs(hi / base - 1.02) < 2e-5
    # curved slice: the path is longer on the outside, the same kick is spread over it
    out, _ = loss_fraction(RadMultipole(knl=(1e-3,), hxl=1e-3, length=10.0), x=0.05)
    on, _ = loss_fraction(RadMultipole(knl=(1e-3,), hxl=1e-3, length=10.0))
    k_out = 1e-3 + (1e-3 * 1e-3 / 10.0) * 0.05                                   # field kick incl. weak focusing
    assert abs(out / on - (k_out / 1e-3) ** 2 / (1.0 + 1e-4 * 0.05)) < 2e-5


def test_P21_vertical_damping_rate_is_U0_over_2E():
    # 10 GeV positrons (with q0 = +1 the cavity phase convention is the one of the proton rings of the other pins)
    p0c, n_cells, ell, L, kq = 10e9, 32, 40.0, 5.0, 0.12
    th = 2.0 * math.pi / (2 * n_cells)
    bend = RadMultipole(knl=(th,), hxl=th, length=ell)
    cell = [Multipole(knl=(0.0, kq)), Drift(L), bend, Drift(L), Multipole(knl=(0.0, -kq)), Drift(L), bend, Drift(L)]
    gamma = math.sqrt(p0c ** 2 + ME ** 2) / ME
    u0_over_e = (2.0 / 3.0) * R_E * gamma ** 3 * th * th / ell * 2 * n_cells
    assert 1e-4 < u0_over_e < 4e-4
    volt = 3.0 * u0_over_e * p0c
    lag = 180.0 - math.degrees(math.asin(1.0 / 3.0))                                 # above transition: falling slope
    els = cell * n_cells + [Cavity(volt, 400e6, lag)]
    no_rad = [Multipole(knl=e.knl, hxl=e.hxl, length=e.length) if isinstance(e, RadMultipole) else e for e in cell] * n_cells
    on = MO.optics_of(pack_lattice(no_rad, p0c, ME, 1.0))
    by, ay = on["bety"], on["alfy"]
    buf = pack_lattice(els, p0c, ME, 1.0)
    p = O.new_particles(buf, H.coords_from_rows([[0.0, 0.0, 1e-4, 0.0, 0.0, 0.0]]))
    turns, acts = 3000, []
    for _ in range(turns):
        y, py = p["y"][0], p["py"][0] / (1.0 + p["delta"][0])
        acts.append(((1 + ay * ay) / by * y * y + 2 * ay * y * py + by * py * py) / 2.0)
        O.track(buf, p, 1)
    assert p["state"][0] == 1 and abs(p["delta"][0]) < 2e-3 and abs(p["x"][0]) < 5e-3
    slope = np.polyfit(np.arange(turns), np.log(acts), 1)[0]
    assert abs(slope / (-u0_over_e) - 1.0) < 0.02, (slope, u0_over_e)                # action: twice the amplitude rate


def test_P21_proton_limit_zero_field_and_validation():
    rng = np.random.default_rng(8)
    rows = np.column_stack([rng.normal(0, 2e-3, 20), rng.normal(0, 2e-4, 20), rng.normal(0, 2e-3, 20),
                            rng.normal(0, 2e-4, 20), rng.normal(0, 0.02, 20), rng.normal(0, 5e-4, 20)]).tolist()
    kw = dict(knl=(2e-3, 0.03, 0.5, -20.0), ksl=(1e-4, 0.002, 0.0, 5.0), hxl=1.9e-3, length=1.7)
    a = O.new_particles(pack_lattice([RadMultipole(**kw)], H.P0C, H.MASS0, 1.0), H.coords_from_rows(rows))
    b = O.copy_particles(a)
    O.track(pack_lattice([RadMultipole(**kw)], H.P0C, H.MASS0, 1.0), a, 1)
    O.track(pack_lattice([Multipole(**kw)], H.P0C, H.MASS0, 1.0), b, 1)
    for k, scale in (("x", 1.0), ("px", 1e-4), ("y", 1.0), ("py", 1e-4), ("zeta", 1e-2), ("delta", 1e-3)):
        assert np.max(np.abs(a[k] - b[k])) < 1e-12 * scale, k
    assert np.all(a["delta"] <= b["delta"]) and np.any(a["delta"] < b["delta"])      # ... but it does radiate a little
    z = O.new_particles(pack_lattice([RadMultipole(knl=(0.0,), length=1.0)], P0C, ME, -1.0), H.coords_from_rows(rows))
    z0 = O.copy_particles(z)
    O.track(pack_lattice([RadMultipole(knl=(0.0,), length=1.0)], P0C, ME, -1.0), z, 1)
    for k in ("x", "y", "zeta", "ptau"):
        assert np.array_equal(z[k], z0[k]), k
    for k in ("px", "py", "delta"):                       # delta is re-derived from the energy, as behind a cavity: rounding
        assert np.max(np.abs(z[k] - z0[k])) < 4e-16 * np.max(np.abs(z0[k])) + 3e-16, k
    for bad in (RadMultipole(knl=(1e-3,), length=0.0), RadMultipole(knl=(1e-3,), length=-1.0)):
        with pytest.raises(ValueError):
            O.reference(pack_lattice([bad], P0C, ME, -1.0))
