"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the tracking method: it only (a) serialises a
list of beam-line elements into the packed lattice buffer that both
``oracle/`` and ``paper_2310_00317_b200`` parse with their own code
(``packed.py``) and (b) builds the five synthetic workloads of BASELINE.json
(``configs.py``): lattices ("Lattice modelling and single particle
tracking": a beam line is a sequence of elements) and particle ensembles
("track particles ensembles").

It imports neither ``oracle`` nor ``paper_2310_00317_b200``.
"""
from .packed import (  # noqa: F401
    Marker, Drift, Multipole, Cavity, SRotation, XYShift, LimitRect, LimitEllipse,
    pack_lattice, unpack_lattice, ELEMENT_TYPE_IDS,
)
