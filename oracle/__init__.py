"""Oracle for the PIMD/Langevin hot path of arxiv/paper_2602_13553 -- TEST INFRASTRUCTURE ONLY.

A plain, slow, FP64 numpy restatement of what the CUDA library computes, written
from /root/reference/PAPER.md (cited as PAPER.md:Lnnn) and from the readings listed in
DESIGN.md section 3 (cited as DESIGN R-n).  It shares no code with
`paper_2602_13553_b200/` and neither imports the other.  Only `tests/`,
`__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs of `bench.py`
may import it; the product path never does.

Pin status (see tests/test_oracle_*.py):
  philox.py      pinned   known-answer vectors, moments of the normals
  nm.py          pinned   orthogonality, diagonalises the ring Laplacian (PAPER.md B1-B3)
  integrator.py  pinned   closed-form harmonic propagation, variance preservation, finite-P
                          harmonic-oscillator <K>,<V>, NVE energy conservation, P=1 limit
  barostat.py    pinned   E1 = quadrature of the cell force over the kick, E4/E5 = numerical ODE, NpH enthalpy
                          (A17) conserved to second order, A12 = A11 at n = 1, closed forms, E7 variance
  compress.py    pinned   node conditions of the quintic Hermite table, 6th-order convergence, forces = -grad of
                          the compressed energy, distance to the MLP (no CUDA counterpart yet: NEXT-3)
  se_e2_a.py     backward pinned (finite differences, torch autograd, invariances, virial =
                 -dU/d(strain), continuity at r_c);  forward architecture: PARITY UNPINNED
                 against physics -- the paper prints no equation for the Deep-Potential
                 model (PAPER.md:L47, L76 only cite it), so the forward pass is "correct by
                 definition" (DESIGN R-11..R-16) and is only checked on hand-computable cases.
"""
