"""Time functions ("knobs"), CPU oracle.  TEST INFRASTRUCTURE (only tests/, smoke() and bench.py's
cpu_baseline may import it).

PAPER.md:88: "it is possible to define 'time functions', i.e. time dependent knobs that are updated
automatically during the simulation" (Fig. 1: the dipolar strength of corrector magnets and
the sextupolar component induced by eddy currents as functions of time); a high-level
parameter controls "groups of accelerator components ... changes in the high-level parameters are
automatically propagated down to the line elements properties".

The paper gives no formula; reading A21: time advances in turns; a knob k is a table
f_k[step]; a link (element, order n, skew, knob k, gain g) adds g * f_k[step] to knl[n] (skew: ksl[n]) of
that Multipole for the turn with that step: value = base, then value = value + g * f for every link of the
coefficient in the order given (product rounded, then the sum); the turn j of a call uses
step = clamp(step0 + j, 0, n_steps - 1).  Everything derived from the coefficient follows (knl/n!, the
curvature fold and the weak-focusing term of reading A12).  Written out: rebuild the line for every turn
and track one turn with the oracle tracker.
"""
from __future__ import annotations

from typing import Dict, Sequence, Tuple

import numpy as np

from oracle import oracle as O
from xt_inputs import packed as PK

Link = Tuple[int, int, int, int, float]     # element, order, skew (0/1), knob, gain


def elements_at_step(elements: Sequence, table: np.ndarray, links: Sequence[Link], step: int):
    els = list(elements)
    for elem, order, skew, knob, gain in links:
        m = els[elem]
        assert isinstance(m, PK.Multipole) and 0 <= order <= m.order
        knl = list(m.knl) + [0.0] * (m.order + 1 - len(m.knl))
        ksl = list(m.ksl) + [0.0] * (m.order + 1 - len(m.ksl))
        term = float(gain) * float(table[knob][step])
        if skew:
            ksl[order] = ksl[order] + term
        else:
            knl[order] = knl[order] + term
        els[elem] = PK.Multipole(knl=tuple(knl), ksl=tuple(ksl), hxl=m.hxl, length=m.length)
    return els


def track_with_knobs(elements: Sequence, p0c: float, mass0: float, q0: float, p: Dict[str, np.ndarray],
                     n_turns: int, table, links: Sequence[Link], step0: int = 0, **kw) -> None:
    table = np.asarray(table, dtype=np.float64)
    assert table.ndim == 2
    n_steps = table.shape[1]
    for j in range(n_turns):
        step = min(max(step0 + j, 0), n_steps - 1)
        O.track(PK.pack_lattice(elements_at_step(elements, table, links, step), p0c, mass0, q0), p, 1, **kw)
