"""CPU oracle for the FIESTA-4 integration hot path (arXiv:1511.03614).

TEST INFRASTRUCTURE ONLY.  This package is the plain, slow, obviously-correct
restatement of what the hot path computes.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import it.  It shares no code with `paper_1511_03614_b200/` (the CUDA
path) and never imports it; the CUDA path never imports this package.

Arithmetic: numpy `longdouble` (x87 80-bit extended on x86-64, 64-bit
mantissa), as BASELINE.json's north_star prescribes ("a plain CPU evaluator in
long double that walks the expression tree directly").  Vectorised over sample
points only; no blocking, fusion or reordering of the per-point arithmetic
beyond what each function's docstring states.

Citations are `PAPER.md:<line>` (the paper text under /root/reference at build
time) or `DESIGN.md R<n>` (a reading taken where the paper is silent).

Pin status (see tests/test_oracle_*.py, all `-m "not gpu"`):
  parser / tree walker      pinned: paper's worked example,
                            linear closed forms, brute-force Python floats
  constants P, G, PolyGamma pinned: mpmath
  monomial / bubble         pinned: closed forms  (eq. 2)
  lattice integers          pinned: brute-force Python big-int, character sums
  Philox4x32-10             pinned: cuRAND host generator (library)
  Korobov transform         pinned: scipy.special.betainc, identities
  derivatives / deformation pinned: complex-step, 1-D contour closed forms,
                            lambda-independence (Cauchy)
  det J                     pinned: cofactor expansion, numpy.linalg.det
  Vegas refine / combine    pinned: invariants, closed forms, 4-sigma coverage
  multiple-precision walk   pinned: closed forms under cancellation, agreement with
  (evaluate_mp, mixed sums)  the long-double walk, 3/2 restored by small_x (R20)
  box example end to end    pinned: the paper's printed numbers
                            and the closed form, via tests/sector_frontend.py;
                            physical-region triangle closed form (complex path)
  cubature (R21)            pinned: degrees of exactness 7 / 5 on every monomial,
                            closed forms, tiling, evaluation count, split axis
  the five BASELINE configs parity unpinned against external truth (random
                            polynomials have no closed form); covered by the
                            component pins above.
"""
