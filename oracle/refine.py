"""Loss-location refinement, CPU oracle.  TEST INFRASTRUCTURE (only tests/, smoke() and
bench.py's cpu_baseline may import it).

PAPER.md:178: aperture elements "stop the tracking for the particles found to be outside ...
which provides a localization of the losses with a few meters accuracy.  The localization is
then further improved in a post-processing stage to reach the accuracy set by the user
(typically 1 to 10 cm), using particle backtracking and a locally refined aperture model
obtained by polygonal interpolation (an example is shown in Fig. 4)" -- Fig. 4:
"the transition between a rectangular aperture and an elliptic aperture, which are shifted and
tilted with respect to each other".

The paper gives no further detail; reading A20 fixes the procedure, followed here
step by step for every lost particle whose ``at_element`` is a LimitRect / LimitEllipse / LimitPolygon ``l``:

 1. Upstream aperture ``u``: the nearest LimitRect / LimitEllipse / LimitPolygon before ``l`` in the line; if
    there is none, the start of the line (s = 0) with the cross-section of ``l`` itself.  If no
    length lies between the two, nothing is refined.
 2. Frames: XYShift / SRotation elements are changes of the reference system.  The
    frame in front of element i is the composition of all of them from the start of the line:
    local = R m + t with R = [[c, s], [-s, c]];  XYShift(dx, dy): t <- t - (dx, dy);
    SRotation(cz, sz): R <- Rz R, t <- Rz t, Rz = [[cz, sz], [-sz, cz]].
 3. Polygons: each of the two apertures is sampled on ``n_poly`` rays that leave its centre C
    (machine frame) at the machine-frame angles phi_k = 2 pi k / n_poly: V_k = C + r_k (cos phi_k,
    sin phi_k); with u = R (cos phi_k, sin phi_k) the local direction, r_k = 1/sqrt((ux/a)^2 +
    (uy/b)^2) for an ellipse and min(hx/|ux|, hy/|uy|) for a rectangle of half widths hx, hy
    about its centre; for a polygon the centre is the mean of its vertices and r_k the smallest
    positive distance at which the ray meets an edge.
 4. Backtracking: the maps are reversible (reading A11, pins P6, P13, P14): flip (px, py, zeta),
    track through the elements between u and l in reverse order (cavity lag, rotation angle and
    shifts negated; apertures dropped), flip again.  The result is the particle just after u.
 5. Forward again through the same elements with every element of length L > 0 cut into
    n = ceil(L / ds) equal pieces, a LimitPolygon after each piece: at the running position
    sloc (sum of the pieces so far) its vertices are V_k^u + lam (V_k^l - V_k^u),
    lam = sloc / (s_l - s_u), taken into the local frame of that place (v = R V + t).  The first
    polygon the particle fails gives the refined loss: its coordinates there, and
    s = s_u + sloc.  A particle that passes them all keeps its record.

All tracking is done by the oracle tracker (``oracle.track``) on lattices built here; this
file adds only the geometry of steps 2, 3 and 5.  Plain Python loops: small cases only.
"""
from __future__ import annotations

import math
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

from oracle import oracle as O
from xt_inputs import packed as PK

APERTURES = (PK.LimitRect, PK.LimitEllipse, PK.LimitPolygon)
STATE_KEYS = ("x", "px", "y", "py", "zeta", "delta", "ptau", "rpp", "rvv")


def element_length(el) -> float:
    return el.length if isinstance(el, (PK.Drift, PK.Quadrupole, PK.Bend)) else 0.0


def frames_of(elements: Sequence) -> List[Tuple[float, float, float, float]]:
    """Step 2: (c, s, tx, ty) of the frame in front of every element (and one past the end)."""
    c, s, tx, ty = 1.0, 0.0, 0.0, 0.0
    out = []
    for el in elements:
        out.append((c, s, tx, ty))
        if isinstance(el, PK.XYShift):
            tx, ty = tx - el.dx, ty - el.dy
        elif isinstance(el, PK.SRotation):
            cz, sz = el.cos_z, el.sin_z
            c, s = cz * c - sz * s, cz * s + sz * c
            tx, ty = cz * tx + sz * ty, cz * ty - sz * tx
    out.append((c, s, tx, ty))
    return out


def aperture_polygon(el, frame, n_poly: int) -> Tuple[np.ndarray, np.ndarray]:
    """Step 3: machine-frame vertices of one LimitRect / LimitEllipse seen through ``frame``."""
    c, s, tx, ty = frame
    if isinstance(el, PK.LimitRect):
        cx, cy = 0.5 * (el.min_x + el.max_x), 0.5 * (el.min_y + el.max_y)
        hx, hy = 0.5 * (el.max_x - el.min_x), 0.5 * (el.max_y - el.min_y)
    elif isinstance(el, PK.LimitPolygon):
        cx, cy = sum(el.x) / len(el.x), sum(el.y) / len(el.y)
    else:
        cx, cy = 0.0, 0.0
    # centre in the machine frame: m = R^T (local - t)
    lx, ly = cx - tx, cy - ty
    mx, my = c * lx - s * ly, s * lx + c * ly
    vx, vy = np.zeros(n_poly), np.zeros(n_poly)
    for k in range(n_poly):
        phi = (2.0 * math.pi * k) / n_poly
        dx, dy = math.cos(phi), math.sin(phi)
        ux, uy = c * dx + s * dy, c * dy - s * dx          # local direction of the ray
        if isinstance(el, PK.LimitRect):
            rx = hx / abs(ux) if ux != 0.0 else math.inf
            ry = hy / abs(uy) if uy != 0.0 else math.inf
            r = min(rx, ry)
        elif isinstance(el, PK.LimitPolygon):
            # the ray c + r u meets the edge a + t (b - a), 0 <= t <= 1, where cross(u, e) != 0:
            # r = cross(a - c, e) / cross(u, e),  t = cross(a - c, u) / cross(u, e)
            r = math.inf
            nv = len(el.x)
            for i in range(nv):
                ax, ay = el.x[i] - cx, el.y[i] - cy
                ex, ey = el.x[(i + 1) % nv] - el.x[i], el.y[(i + 1) % nv] - el.y[i]
                den = ux * ey - uy * ex
                if den == 0.0:
                    continue
                rr = (ax * ey - ay * ex) / den
                t = (ax * uy - ay * ux) / den
                if rr > 0.0 and 0.0 <= t <= 1.0 and rr < r:
                    r = rr
            assert math.isfinite(r), "the polygon does not surround the mean of its vertices"
        else:
            r = 1.0 / math.sqrt((ux / el.a) * (ux / el.a) + (uy / el.b) * (uy / el.b))
        vx[k], vy[k] = mx + r * dx, my + r * dy
    return vx, vy


def reversed_elements(elements: Sequence) -> List:
    """Step 4 (reading A11): reverse order; cavity lag, rotation angle, shifts negated; apertures dropped."""
    out = []
    for el in reversed(elements):
        if isinstance(el, APERTURES):
            continue
        if isinstance(el, PK.Cavity):
            out.append(PK.Cavity(el.voltage, el.frequency, -el.lag))
        elif isinstance(el, PK.SRotation):
            out.append(PK.SRotation(el.cos_z, -el.sin_z))
        elif isinstance(el, PK.XYShift):
            out.append(PK.XYShift(-el.dx, -el.dy))
        else:
            out.append(el)
    return out


def sliced_elements(elements: Sequence, frames: Sequence, poly_u, poly_l, seg_len: float, ds: float):
    """Step 5: the refined line between the two apertures and, per element of it, sloc."""
    out, sloc_of = [], []
    sloc = 0.0
    for el, fr in zip(elements, frames):
        if isinstance(el, APERTURES):
            continue
        length = element_length(el)
        if length > 0.0:
            n = int(math.ceil(length / ds))
            piece = length / n
            for _ in range(n):
                if isinstance(el, PK.Drift):
                    out.append(PK.Drift(piece))
                elif isinstance(el, PK.Quadrupole):
                    out.append(PK.Quadrupole(el.k1, piece))
                else:
                    out.append(PK.Bend(el.k0, el.h, piece, el.model))
                sloc_of.append(sloc)
                sloc = sloc + piece
                lam = sloc / seg_len
                c, s, tx, ty = fr                     # thick elements and drifts do not change the frame
                mx = poly_u[0] + lam * (poly_l[0] - poly_u[0])
                my = poly_u[1] + lam * (poly_l[1] - poly_u[1])
                out.append(PK.LimitPolygon(tuple(c * mx + s * my + tx), tuple(c * my - s * mx + ty)))
                sloc_of.append(sloc)
        else:
            out.append(el)
            sloc_of.append(sloc)
    return out, sloc_of


def refine_loss_location(elements: Sequence, p0c: float, mass0: float, q0: float,
                         p: Dict[str, np.ndarray], ds: float, n_poly: int,
                         min_margin: Optional[np.ndarray] = None) -> int:
    """Refine in place the records of the lost particles of ``p`` (as left by ``oracle.track``
    on ``pack_lattice(elements, ...)``).  Returns how many records were moved.  ``min_margin``
    (float64[n], optional) receives per particle the smallest distance to a polygon edge over
    the checks of step 5 (test bookkeeping: decisions closer than rounding are not compared)."""
    assert ds > 0.0 and 3 <= n_poly <= 256
    elements = list(elements)
    s_tab = O.s_table(PK.pack_lattice(elements, p0c, mass0, q0))
    frames = frames_of(elements)
    moved = 0
    lost = np.flatnonzero(p["state"] == 0)
    for l in sorted(set(int(i) for i in p["at_element"][lost])):
        if not isinstance(elements[l], APERTURES):
            continue
        u = l - 1
        while u >= 0 and not isinstance(elements[u], APERTURES):
            u -= 1
        s_u = float(s_tab[u]) if u >= 0 else 0.0
        seg_len = float(s_tab[l]) - s_u
        if not seg_len > 0.0:
            continue
        poly_l = aperture_polygon(elements[l], frames[l], n_poly)
        poly_u = aperture_polygon(elements[u], frames[u], n_poly) if u >= 0 else poly_l
        seg = elements[u + 1:l]
        idx = lost[p["at_element"][lost] == l]
        # step 4: back to just after u
        q = {k: p[k][idx].copy() for k in STATE_KEYS}
        q["s"] = np.zeros(len(idx))
        q["at_turn"] = np.zeros(len(idx), dtype=np.int64)
        q["at_element"] = np.zeros(len(idx), dtype=np.int64)
        q["state"] = np.ones(len(idx), dtype=np.int64)
        for k in ("px", "py", "zeta"):
            q[k] *= -1.0
        back = PK.pack_lattice(reversed_elements(seg) or [PK.Marker()], p0c, mass0, q0)
        O.track(back, q, 1)
        for k in ("px", "py", "zeta"):
            q[k] *= -1.0
        assert np.all(q["state"] == 1)
        q["at_turn"][:] = 0
        q["s"][:] = 0.0
        # step 5: forward through the refined aperture model
        fine, sloc_of = sliced_elements(seg, frames[u + 1:l], poly_u, poly_l, seg_len, ds)
        mm = np.full(len(idx), np.inf)
        O.track(PK.pack_lattice(fine, p0c, mass0, q0), q, 1, min_margin=mm)
        if min_margin is not None:
            min_margin[idx] = np.minimum(min_margin[idx], mm)
        hit = q["state"] == 0
        for k in STATE_KEYS:
            p[k][idx[hit]] = q[k][hit]
        p["s"][idx[hit]] = s_u + np.asarray([sloc_of[int(e)] for e in q["at_element"][hit]])
        moved += int(hit.sum())
    return moved
