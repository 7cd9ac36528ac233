"""TEST INFRASTRUCTURE ONLY -- the fp64 brute-force oracle of the dyplan hot path.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product
(``paper_2607_02942_b200``) never does and shares no code with it.
"""
