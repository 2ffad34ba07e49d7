"""Seeded synthetic inputs for the five BASELINE.json configurations.

This package only WRITES inputs (expression texts in the paper's grammar,
PAPER.md:508-519, plus rule parameters).  It holds none of the method's
arithmetic and is the one thing the oracle's callers and the CUDA path's
callers share: tests and bench.py build a workload here and hand the same texts
to `oracle/` and to `paper_1511_03614_b200`.

The texts stand in for the paper's 649-integrand four-loop database
(PAPER.md:158), which is not available; they take its shape (monomial x U^p x
F^-q x a few logarithms, PAPER.md:84-88 eq. 2, :108-110), see DESIGN.md
"Input recipe".
"""
from .generate import Workload, SectorText, make_workload, CONFIG_NAMES  # noqa: F401
from .korobov import korobov_a  # noqa: F401
