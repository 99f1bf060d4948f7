"""CPU oracle for the EMRI_MC hot path -- TEST INFRASTRUCTURE, not product code.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  Nothing under
``paper_2311_17174_b200/`` imports it, and it imports nothing from there.
"""
