"""CPU oracle for the exact-exchange hot path (TEST INFRASTRUCTURE, not product).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2501_16572_b200`` (the CUDA path) and imports nothing from it.
"""
