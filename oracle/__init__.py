"""fp64 CPU oracle for the MelT / MFCCT hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  The product (``paper_2606_01009_b200``) never imports it and has no CPU
fallback.  See ``melt_oracle.c`` for the definition and its citations into PAPER.md.
"""
