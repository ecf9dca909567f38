"""CPU oracle for the CC-LR hot path of arXiv:2307.14296.

TEST INFRASTRUCTURE ONLY.  Plain numpy, complex128, no blocking / fusion / packing tricks.
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package; the product (``paper_2307_14296_b200``) never does, and this package never
imports the product.  The two share no code; only ``synth/`` (seeded input generators, no method
arithmetic) serves both.

Modules
-------
bruteforce : O1 — second-quantised operators on an explicit determinant space; the literal definitions
             of Table 1 / Eq. 14.  Pins everything else on tiny inputs.
ccsd       : O2/O3 — tensor-level E(t), Omega(t) (spin-orbital CCSD residual, PAPER.md:205 cites it) and
             a DIIS ground-state solver.
cclr       : O4-O9 — sigma by exact finite differences of Omega, sigma hand-coded from S-Eq. 11-12
              with the intermediates of S-Eq. 15-28, xi / eta / Lambda /
             F.x.y, dense and iterative response solves, response functions Eq. 15-17.
packing    : the oracle's own pack / unpack between the C-ABI's packed layouts and full tensors.

Pin status: every function in ccsd and cclr is pinned by tests/test_oracle_*.py
against bruteforce, closed forms or special cases; nothing here is "parity unpinned".
"""
