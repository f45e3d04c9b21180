"""CPU oracle for the PRS domain-wall step (TEST INFRASTRUCTURE ONLY).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  The product package ``paper_1710_10420_b200`` never does.
"""
