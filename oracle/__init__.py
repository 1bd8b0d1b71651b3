"""CPU oracle for the SparDA decode hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with, and is never
imported by, ``paper_2606_04511_b200``.  See ``sparda_oracle.c`` for the arithmetic and its
citations, ``sparda_oracle.py`` for the thin numpy/ctypes wrapper.
"""
