"""fp64 CPU oracle of the viscoelastic FDTD step -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / reference legs
may import this package.  See ``fdtd_oracle.c`` for the arithmetic and its citations.
"""
