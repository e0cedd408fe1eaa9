"""Pins P15 (LimitPolygon) and P16 (loss-location refinement, reading A20)
of the CPU oracle -- against closed forms and invariants, not against itself:

P15  even-odd polygon test  = half-plane test on convex polygons, = union of two rectangles on an
     L shape, = LimitRect on its four corners; NaN lost; vertex-count limits; margin = distance.
P16  refinement: a straight line (exact drift) leaves a round pipe, a cone, an oblique round pipe and
     a tilted elliptical pipe where the quadratic says; a rigid shift + tilt of the whole pipe moves
     nothing but the frame; re-tracking the refined record reproduces the original loss (kicks and
     a cavity in between); nested slicing orders the refined positions; no upstream aperture =
     constant cross-section from s = 0; the diamond that 4 rays cut out of a square pipe.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from oracle import refine as R
from xt_inputs.packed import (Cavity, Drift, LimitEllipse, LimitPolygon, LimitRect, Marker, Multipole,
                              SRotation, XYShift, pack_lattice)
import helpers as H


def pack(els):
    return pack_lattice(els, H.P0C, H.MASS0, H.Q0)


def particles(els, rows):
    return O.new_particles(pack(els), H.coords_from_rows(rows))


# ------------------------------------------------------------------ P15
def _decide(poly, pts):
    els = [poly]
    rows = [[x, 0.0, y_, 0.0, 0.0, 0.0] for x, y_ in pts]
    p = particles(els, rows)
    mm = np.full(len(pts), np.inf)
    O.track(pack(els), p, 1, min_margin=mm)
    return p["state"] == 1, mm, p


def test_P15_convex_polygon_is_the_intersection_of_half_planes():
    rng = np.random.default_rng(5)
    n = 7
    ang = np.sort(rng.uniform(0, 2 * np.pi, n))
    vx, vy = 0.3 + 2.0 * np.cos(ang), -0.2 + 1.5 * np.sin(ang)      # convex: points on an ellipse, ccw
    pts = rng.uniform(-2.5, 2.5, (4000, 2))
    inside, mm, _ = _decide(LimitPolygon(tuple(vx), tuple(vy)), pts)
    want = np.ones(len(pts), dtype=bool)
    for i in range(n):
        j = (i + 1) % n
        want &= (vx[j] - vx[i]) * (pts[:, 1] - vy[i]) - (vy[j] - vy[i]) * (pts[:, 0] - vx[i]) >= 0.0
    clear = mm > 1e-9
    assert clear.sum() > 3900 and 0.2 < want.mean() < 0.8
    assert np.array_equal(inside[clear], want[clear])
    # clockwise order describes the same region
    inside_cw, _, _ = _decide(LimitPolygon(tuple(vx[::-1]), tuple(vy[::-1])), pts)
    assert np.array_equal(inside_cw[clear], want[clear])


def test_P15_non_convex_polygon_rect_equivalence_margin_nan_limits():
    # an L: [0,2]x[0,1] united with [0,1]x[0,2]
    poly = LimitPolygon((0.0, 2.0, 2.0, 1.0, 1.0, 0.0), (0.0, 0.0, 1.0, 1.0, 2.0, 2.0))
    rng = np.random.default_rng(6)
    pts = rng.uniform(-0.5, 2.5, (4000, 2))
    inside, mm, _ = _decide(poly, pts)
    in_a = (pts[:, 0] >= 0) & (pts[:, 0] <= 2) & (pts[:, 1] >= 0) & (pts[:, 1] <= 1)
    in_b = (pts[:, 0] >= 0) & (pts[:, 0] <= 1) & (pts[:, 1] >= 0) & (pts[:, 1] <= 2)
    clear = mm > 1e-9
    assert np.array_equal(inside[clear], (in_a | in_b)[clear]) and 0.2 < inside.mean() < 0.5
    # the four corners of a rectangle decide like LimitRect, and the margin is the distance to the nearest side
    rect = LimitRect(-0.7, 1.1, -0.4, 0.9)
    quad = LimitPolygon((-0.7, 1.1, 1.1, -0.7), (-0.4, -0.4, 0.9, 0.9))
    pts = rng.uniform(-1.5, 1.5, (3000, 2))
    a, mm_a, pa = _decide(quad, pts)
    b, mm_b, pb = _decide(rect, pts)
    clear = mm_b > 1e-9
    assert np.array_equal(a[clear], b[clear])
    np.testing.assert_allclose(mm_a[b], mm_b[b], rtol=0, atol=1e-15)          # inside: distance to the nearest side
    for k in ("x", "y", "at_element", "at_turn", "s"):                         # the loss record is the same
        assert np.array_equal(pa[k][clear], pb[k][clear]), k
    # NaN is lost; vertex-count limits
    _, _, p = _decide(quad, [(float("nan"), 0.0), (0.0, float("nan")), (0.0, 0.0)])
    assert list(p["state"]) == [0, 0, 1]
    for bad in (LimitPolygon((0.0, 1.0), (0.0, 1.0)), LimitPolygon(tuple(range(257)), tuple(range(257)))):
        with pytest.raises(ValueError):
            O.reference(pack([bad]))
    assert O.reference(pack([LimitPolygon(tuple(np.cos(np.arange(256.0))), tuple(np.sin(np.arange(256.0))))]))


# ------------------------------------------------------------------ P16
def straight(rows):
    """Exact drift (pin P1): position after path s is (x + s px/pz, y + s py/pz)."""
    r = np.asarray(rows, dtype=float)
    pz = np.sqrt((1.0 + r[:, 5]) ** 2 - r[:, 1] ** 2 - r[:, 3] ** 2)
    return r[:, 0], r[:, 1] / pz, r[:, 2], r[:, 3] / pz


def first_grid_point(s_star, ds_piece):
    return np.ceil(s_star / ds_piece - 1e-9) * ds_piece


def lose_and_refine(els, rows, ds, n_poly, want_lost_at):
    p = particles(els, rows)
    O.track(pack(els), p, 1)
    assert np.all(p["state"] == 0) and np.all(p["at_element"] == want_lost_at), (p["state"], p["at_element"])
    coarse = O.copy_particles(p)
    mm = np.full(len(rows), np.inf)
    moved = R.refine_loss_location(els, H.P0C, H.MASS0, H.Q0, p, ds, n_poly, min_margin=mm)
    return p, coarse, moved, mm


def rays(n, seed, r_max, pmin=1.5e-3):
    rng = np.random.default_rng(seed)
    rows = []
    for _ in range(n):
        ang = rng.uniform(0, 2 * np.pi)
        rows.append([rng.uniform(-0.3, 0.3) * r_max, rng.uniform(pmin, 2 * pmin) * math.cos(ang),
                     rng.uniform(-0.3, 0.3) * r_max, rng.uniform(pmin, 2 * pmin) * math.sin(ang),
                     rng.normal(0, 0.01), rng.normal(0, 1e-3)])
    return rows


def quadratic_exit(x0, vx, y0, vy, cx0, cvx, cy0, cvy, r0, rv, ax=1.0, ay=1.0):
    """Smallest s > 0 with ((x0 + s vx - cx0 - s cvx)/ax)^2 + ((..y..)/ay)^2 = (r0 + s rv)^2."""
    px, qx = (x0 - cx0) / ax, (vx - cvx) / ax
    py, qy = (y0 - cy0) / ay, (vy - cvy) / ay
    a = qx * qx + qy * qy - rv * rv
    b = 2.0 * (px * qx + py * qy - r0 * rv)
    c = px * px + py * py - r0 * r0
    disc = np.sqrt(b * b - 4.0 * a * c)
    return (-b + disc) / (2.0 * a)          # c < 0 (starts inside), a > 0: the positive root


def check_bracket(p, rows, s_lo, s_hi, piece, s0=0.0):
    """Refined s is the first slice end at or after the exit through the polygon, which lies between
    the exits through the inscribed (s_lo) and the circumscribed (s_hi) smooth surface; the
    coordinates there are the straight line's."""
    lo, hi = first_grid_point(s_lo, piece), first_grid_point(s_hi, piece)
    s = p["s"] - s0
    assert np.all((s >= lo - 1e-9) & (s <= hi + 1e-9)), (s, lo, hi)
    assert (np.abs(lo - hi) < 1e-9).mean() > 0.8                                 # mostly a single admissible slice
    x0, vx, y0, vy = straight(rows)
    np.testing.assert_allclose(p["x"], x0 + s * vx, rtol=0, atol=1e-14)
    np.testing.assert_allclose(p["y"], y0 + s * vy, rtol=0, atol=1e-14)


def test_P16_round_pipe_cone_and_no_upstream_aperture():
    r, L, ds, n_poly = 0.02, 40.0, 0.05, 256
    rows = rays(24, 1, r)
    x0, vx, y0, vy = straight(rows)
    shrink = math.cos(math.pi / n_poly)                                          # inscribed polygon: apothem
    # round pipe between two identical circles
    els = [LimitEllipse(r, r), Drift(L), LimitEllipse(r, r)]
    p, coarse, moved, _ = lose_and_refine(els, rows, ds, n_poly, 2)
    assert moved == len(rows) and np.all(coarse["s"] == L)
    n = math.ceil(L / ds)
    check_bracket(p, rows, quadratic_exit(x0, vx, y0, vy, 0, 0, 0, 0, r * shrink, 0),
                  quadratic_exit(x0, vx, y0, vy, 0, 0, 0, 0, r, 0), L / n)
    for k in ("px", "py", "delta", "at_turn", "at_element", "state"):
        assert np.array_equal(p[k], coarse[k]), k                                 # a drift changes none of these
    # no upstream aperture: the cross-section of the flagging one from s = 0
    els = [Marker(), Drift(L), LimitEllipse(r, r)]
    p2, _, moved, _ = lose_and_refine(els, rows, ds, n_poly, 2)
    assert moved == len(rows)
    for k in ("x", "y", "s", "zeta"):
        assert np.array_equal(p2[k], p[k]), k
    # cone: radius 0.03 -> 0.01
    ru, rl = 0.03, 0.01
    els = [Drift(3.0), LimitEllipse(ru, ru), Drift(L / 2), Drift(L / 2), LimitEllipse(rl, rl)]
    rows_at_u = rows
    start = [[x0[i] - 3.0 * vx[i], rows[i][1], y0[i] - 3.0 * vy[i], rows[i][3], rows[i][4], rows[i][5]]
             for i in range(len(rows))]
    p, _, moved, _ = lose_and_refine(els, start, ds, n_poly, 4)
    assert moved == len(rows)
    piece = (L / 2) / math.ceil((L / 2) / ds)
    s_lo = quadratic_exit(x0, vx, y0, vy, 0, 0, 0, 0, ru * shrink, (rl - ru) * shrink / L)
    s_hi = quadratic_exit(x0, vx, y0, vy, 0, 0, 0, 0, ru, (rl - ru) / L)
    x0b, vxb, y0b, vyb = straight(start)
    lo, hi = first_grid_point(s_lo, piece), first_grid_point(s_hi, piece)
    s = p["s"] - 3.0
    assert np.all((s >= lo - 1e-9) & (s <= hi + 1e-9)) and np.all(s < L)
    np.testing.assert_allclose(p["x"], x0b + p["s"] * vxb, rtol=0, atol=1e-14)
    np.testing.assert_allclose(p["y"], y0b + p["s"] * vyb, rtol=0, atol=1e-14)


def test_P16_shifted_and_tilted_apertures():
    r, L, ds, n_poly = 0.02, 30.0, 0.05, 256
    rows = rays(24, 2, 0.5 * r)
    x0, vx, y0, vy = straight(rows)
    shrink = math.cos(math.pi / n_poly)
    piece = L / math.ceil(L / ds)
    # oblique round pipe: the downstream circle is displaced by (dx, dy): the centre moves linearly
    dx, dy = 0.004, -0.003
    els = [LimitEllipse(r, r), Drift(L), XYShift(dx, dy), LimitEllipse(r, r), XYShift(-dx, -dy)]
    p, _, moved, _ = lose_and_refine(els, rows, ds, n_poly, 3)
    assert moved == len(rows)
    check_bracket(p, rows, quadratic_exit(x0, vx, y0, vy, 0, dx / L, 0, dy / L, r * shrink, 0),
                  quadratic_exit(x0, vx, y0, vy, 0, dx / L, 0, dy / L, r, 0), piece)
    # elliptical pipe, both ends tilted by the same angle: an ellipse in the tilted frame.  The bracket:
    # the polygon lies between the ellipse scaled by its worst apothem ratio and the ellipse itself.
    a, b, th = 0.03, 0.012, 0.4
    c, s_ = math.cos(th), math.sin(th)
    rot, unrot = SRotation(c, s_), SRotation(c, -s_)
    els = [rot, LimitEllipse(a, b), unrot, Drift(L), rot, LimitEllipse(a, b), unrot]
    rows_t = rays(24, 3, 0.5 * b)
    p, _, moved, _ = lose_and_refine(els, rows_t, ds, n_poly, 5)
    assert moved == len(rows_t)
    x0, vx, y0, vy = straight(rows_t)
    xt, vxt = c * x0 + s_ * y0, c * vx + s_ * vy                                 # SRotation: x' = c x + s y, y' = c y - s x
    yt, vyt = c * y0 - s_ * x0, c * vy - s_ * vx
    s_hi = quadratic_exit(xt, vxt, yt, vyt, 0, 0, 0, 0, 1.0, 0, ax=a, ay=b)
    s_lo = quadratic_exit(xt, vxt, yt, vyt, 0, 0, 0, 0, 0.999, 0, ax=a, ay=b)  # 256 rays: chords within 1e-3 of the arc
    lo, hi = first_grid_point(s_lo, piece), first_grid_point(s_hi, piece)
    assert np.all((p["s"] >= lo - 1e-9) & (p["s"] <= hi + 1e-9)), (p["s"], lo, hi)
    assert np.all(hi - lo <= 2 * piece + 1e-9)
    # the loss record is in the MACHINE frame of that place (no transform element is open there)
    np.testing.assert_allclose(p["x"], x0 + p["s"] * vx, rtol=0, atol=1e-14)
    np.testing.assert_allclose(p["y"], y0 + p["s"] * vy, rtol=0, atol=1e-14)


def test_P16_rigid_motion_of_the_whole_pipe_changes_only_the_frame():
    """Fig. 4 geometry (rectangle -> ellipse, shifted and tilted differently) described twice: as is,
    and with one more shift + tilt wrapped around everything while the particles are moved along."""
    L, ds, n_poly = 12.0, 0.1, 64
    th1, th2 = 0.3, -0.2
    inner = [XYShift(1e-3, -2e-3), SRotation.from_angle(th1), LimitRect(-0.02, 0.015, -0.01, 0.012),
             SRotation.from_angle(-th1), XYShift(-1e-3, 2e-3), Drift(L / 3), Multipole(knl=(0.0, 0.01)), Drift(2 * L / 3),
             SRotation.from_angle(th2), XYShift(-2e-3, 1e-3), LimitEllipse(0.012, 0.008), XYShift(2e-3, -1e-3),
             SRotation.from_angle(-th2)]
    rows = rays(40, 4, 0.004)
    p, coarse, moved, mm = lose_and_refine(inner, rows, ds, n_poly, 10)
    assert moved == len(rows) and np.all(p["s"] > 0) and np.all(p["s"] <= L) and len(set(p["s"])) > 10
    # the same world seen from a frame shifted by D then rotated by TH; TH is a whole number of ray
    # spacings, so that the rays (fixed in the machine frame) sample the same boundary points
    D, TH = (3e-3, -1e-3), 3 * (2.0 * math.pi / n_poly)
    c, s_ = math.cos(TH), math.sin(TH)
    outer = [XYShift(*D), SRotation(c, s_)] + inner + [SRotation(c, -s_), XYShift(-D[0], -D[1])]

    def to_machine(r):          # particle coordinates such that after XYShift(D), SRotation(TH) they equal r
        x, px, y, py = r[0], r[1], r[2], r[3]
        return [c * x - s_ * y + D[0], c * px - s_ * py, s_ * x + c * y + D[1], s_ * px + c * py, r[4], r[5]]

    rows_m = [to_machine(r) for r in rows]
    p2, _, moved2, mm2 = lose_and_refine(outer, rows_m, ds, n_poly, 12)
    clear = (mm > 1e-9) & (mm2 > 1e-9)
    assert moved2 == len(rows) and clear.sum() >= 38
    np.testing.assert_allclose(p2["s"][clear], p["s"][clear], rtol=0, atol=1e-12)
    for k in ("x", "px", "y", "py", "zeta"):                                     # both records are in the local frame there
        np.testing.assert_allclose(p2[k][clear], p[k][clear], rtol=0, atol=1e-13, err_msg=k)


def test_P16_retracking_the_refined_record_reproduces_the_loss_and_slicing_nests():
    a_len, b_len, ds, n_poly = 7.0, 9.0, 0.25, 32
    kick = Multipole(knl=(1e-5, 0.02, 0.5), ksl=(0.0, 0.003))
    cav = Cavity(2e6, 400e6, 30.0)
    els = [LimitRect(-0.02, 0.02, -0.02, 0.02), Drift(a_len), kick, cav, Drift(b_len), LimitEllipse(0.012, 0.009)]
    rows = rays(40, 7, 0.006)
    p, coarse, moved, _ = lose_and_refine(els, rows, ds, n_poly, 5)
    assert moved == len(rows)
    before, after = p["s"] < a_len - 1e-9, p["s"] > a_len + 1e-9
    assert before.sum() >= 3 and after.sum() >= 10
    for i in range(len(rows)):
        s = float(p["s"][i])
        rest = [Drift(a_len - s), kick, cav, Drift(b_len)] if s < a_len - 1e-9 else [Drift(a_len + b_len - s)]
        if abs(s - a_len) <= 1e-9:
            rest = [kick, cav, Drift(b_len)]
        q = {k: v[i:i + 1].copy() for k, v in p.items()}
        q["state"][:] = 1
        O.track(pack(rest), q, 1)
        for k, scale in (("x", 1e-2), ("px", 1e-3), ("y", 1e-2), ("py", 1e-3), ("zeta", 1e-2), ("delta", 1e-3), ("ptau", 1e-3)):
            assert abs(q[k][0] - coarse[k][i]) < 2e-14 * scale, (k, i)
    # nested grids: halving ds can only move the refined position upstream, by less than the old ds
    p_half, _, _, _ = lose_and_refine(els, rows, ds / 2, n_poly, 5)
    assert np.all(p_half["s"] <= p["s"] + 1e-12) and np.all(p["s"] - p_half["s"] < ds + 1e-12)
    assert (p_half["s"] < p["s"] - 1e-12).sum() >= 5
    # survivors and particles lost elsewhere are not touched
    keep = particles(els, [[0, 0, 0, 0, 0, 0], [0.03, 0, 0, 0, 0, 0]])
    O.track(pack(els), keep, 1)
    assert list(keep["state"]) == [1, 0] and keep["at_element"][1] == 0
    snap = O.copy_particles(keep)
    assert R.refine_loss_location(els, H.P0C, H.MASS0, H.Q0, keep, ds, n_poly) == 0
    for k in snap:
        assert np.array_equal(snap[k], keep[k]), k


def test_P16_four_rays_cut_a_diamond_out_of_a_square_pipe():
    h, L, ds = 0.01, 20.0, 0.02
    els = [LimitRect(-h, h, -h, h), Drift(L), LimitRect(-h, h, -h, h)]
    rows = [[0.0, 1.2e-3, 0.0, 0.0, 0.0, 0.0], [0.001, 6e-4, -0.002, 9e-4, 0.0, 1e-3], [-0.002, -8e-4, 0.001, -7e-4, 0.0, 0.0]]
    p, _, moved, _ = lose_and_refine(els, rows, ds, 4, 2)
    assert moved == 3
    x0, vx, y0, vy = straight(rows)
    # |x| + |y| = h along a straight line that keeps its quadrant from the exit on
    sgx, sgy = np.sign(vx + 1e-300), np.sign(vy + 1e-300)
    s_star = (h - sgx * x0 - sgy * y0) / (sgx * vx + sgy * vy)
    piece = L / math.ceil(L / ds)
    np.testing.assert_allclose(p["s"], first_grid_point(s_star, piece), rtol=0, atol=1e-9)
    # with 8 rays the corners are vertices too: the first particle (on the x axis) leaves at x = h exactly
    p8, _, _, _ = lose_and_refine(els, rows[:1], ds, 8, 2)
    assert abs(p8["s"][0] - first_grid_point(h / vx[0], piece)) < 1e-9


def test_P16_polygon_apertures_as_end_points():
    """A rectangle given by its four corners and an ellipse given by 64 points on it are refined like the
    LimitRect / LimitEllipse they describe (the rays meet the same boundary; the 64-gon is inscribed, so a loss
    may be flagged one slice earlier at most), shifted and tilted brackets included."""
    L, ds, n_poly = 12.0, 0.1, 64
    th1, th2 = 0.3, -0.2
    ang = 2 * np.pi * np.arange(64) / 64

    def line(first, last):
        return [XYShift(1e-3, -2e-3), SRotation.from_angle(th1), first, SRotation.from_angle(-th1), XYShift(-1e-3, 2e-3),
                Drift(L / 3), Multipole(knl=(0.0, 0.01)), Drift(2 * L / 3), SRotation.from_angle(th2), XYShift(-2e-3, 1e-3),
                last, XYShift(2e-3, -1e-3), SRotation.from_angle(-th2)]

    rect, ell = LimitRect(-0.02, 0.015, -0.01, 0.012), LimitEllipse(0.012, 0.008)
    rect_p = LimitPolygon((-0.02, 0.015, 0.015, -0.02), (-0.01, -0.01, 0.012, 0.012))
    ell_p = LimitPolygon(tuple(0.012 * np.cos(ang)), tuple(0.008 * np.sin(ang)))
    rows = rays(40, 4, 0.004)
    ref, _, moved, mm = lose_and_refine(line(rect, ell), rows, ds, n_poly, 10)
    # the mean of the four corners is the rectangle's midpoint: same centre, same rays, same boundary points
    a, _, moved_a, mm_a = lose_and_refine(line(rect_p, ell), rows, ds, n_poly, 10)
    clear = (mm > 1e-9) & (mm_a > 1e-9)
    assert moved_a == moved and clear.sum() >= 38
    np.testing.assert_allclose(a["s"][clear], ref["s"][clear], rtol=0, atol=1e-12)
    np.testing.assert_allclose(a["x"][clear], ref["x"][clear], rtol=0, atol=1e-15)
    # the flagging aperture as a 64-gon: particles between the polygon and the ellipse are lost on it but not on
    # the ellipse, so compare the ones both lines lose there
    p = particles(line(rect, ell_p), rows)
    O.track(pack(line(rect, ell_p)), p, 1)
    assert np.all(p["state"] == 0) and np.all(p["at_element"] == 10)
    moved_b = R.refine_loss_location(line(rect, ell_p), H.P0C, H.MASS0, H.Q0, p, ds, n_poly)
    assert moved_b == len(rows)
    assert np.all(p["s"] <= ref["s"] + 1e-12) and np.all(ref["s"] - p["s"] <= ds + 1e-12)
    assert (np.abs(p["s"] - ref["s"]) < 1e-12).mean() > 0.9
