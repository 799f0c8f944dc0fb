"""CPU fp64 oracle for the RPY mobility hot path -- TEST INFRASTRUCTURE, not product code.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs
of ``bench.py`` may import this package.  It imports nothing from ``paper_2510_02135_b200``.
"""
