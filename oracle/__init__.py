"""CPU oracle for the permutation-operator matrix P0 of arxiv/paper_1404_5253.

TEST INFRASTRUCTURE ONLY.  A plain, slow FP64 restatement of the paper's
definitions (Appendix A, eqs. A1-A15) and of the readings listed in
DESIGN.md.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it.
It shares no code with ``paper_1404_5253_b200`` (the CUDA path) and neither
imports the other.

Modules
-------
wigner    exact (rational-arithmetic) 3j / 6j / 9j / Clebsch-Gordan symbols
channels  channel enumeration (eq. 5) and the algebraic
          coefficients g of (A4)
perm      ctypes front end to ``perm_oracle.c``: overlap predicate, CSR
          pattern, the quadrature rule R(n) for (A15), sequential CSR SpMV
kernel_apply  one application of the factored kernel K = O P0 O^T V1 G1 (eq. 10, 12)

Parity pins: see the header of each module and DESIGN.md section "Oracle pins".
"""
