"""TEST INFRASTRUCTURE: the CPU oracle of the tracking hot path.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product package
``paper_2310_00317_b200`` never does (and this package never imports it).
"""
