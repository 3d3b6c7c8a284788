"""CPU oracle for the batched LISA MBHB log-likelihood hot path (arXiv:2005.01827).

TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 numpy restatement of the method as
PAPER.md section II / II.A states it (readings listed in DESIGN.md section 4).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this package.  It shares no code with the CUDA
library under paper_2005_01827_b200/ and never imports it; the only shared
artefact is the numeric model table model_data/phenomhm_table.csv (data).

Pins (tests/test_oracle_*.py, -m "not gpu"):
  spline        P1 cubic reproduction, P2 scipy not-a-knot, P3 h^4 convergence
  inner product P4 eq. 2 identity, P5 D_L^-2 scaling and logL = 0 at injection
  phenomd       P6 Newtonian t(f), P7 Newtonian amplitude, P8 C1 continuity and
                analytic-vs-finite-difference phase derivative
  phenomhm      P13 map continuity and inspiral scaling
  response      P9 frozen-constellation time-domain brute force, P10 harmonics,
                P11 rigid triangle, P12 T-channel suppression
  chain         P14 spline-vs-direct template, P15 exact linear phase term,
                P18 independent mpmath re-evaluation of a tiny case
  sampler side  (oracle/sampler.py) Table I box, Philox known answers, stretch-move
                z density, detailed balance of move + swap on a tempered Gaussian, <d|h> linear over modes
Parity unpinned: fidelity of the model *numbers* to the published PhenomD /
PhenomHM calibration (the tables are not available offline).
"""
