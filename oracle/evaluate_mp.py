"""Oracle step O2 at multiple precision: the same tree walk as oracle/evaluate.py on mpmath numbers.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): the product never imports this.

What it is for: the paper's default "Mixed" mode evaluates the integrand with MPFR where doubles
cancel (PAPER.md:529; knobs PAPER.md:447, :472; "-mpfr: evaluate all integration points with the
use of MPFR").  The CUDA path's stand-in for MPFR is double-double arithmetic
(R20); this module is what it is compared with: f(x) at the same double point x, every
operation carried out with `digits` significant decimal digits (default 60, far beyond the ~32 of a
double-double), point by point in plain Python.

Semantics are those of oracle/evaluate.py (R9 powers, R10 logarithm).  Constants: a numeric literal
is the nearest FP64 value of its text, as in the parser (oracle/parser.py); P, G and PolyGamma are
by default the mathematical constants at full working precision, and with const64=True their
nearest FP64 values -- DESIGN.md R20: the CUDA path's instructions carry FP64 immediates, so that is
the function its double-double walk evaluates.

Pins (tests/test_oracle_pins.py): agreement with the longdouble walk at well-conditioned points;
closed forms under catastrophic cancellation, where the longdouble walk loses every digit.
"""
from __future__ import annotations

import math

import mpmath

from .parser import Program


def _polygamma(n: int, m: int):
    # psi^(n)(m) = (-1)^(n+1) n! (zeta(n+1) - sum_{j<m} j^-(n+1))   (seven hard-coded pairs)
    tail = mpmath.mpf(0)
    for j in range(1, m):
        tail += mpmath.mpf(1) / mpmath.mpf(j) ** (n + 1)
    sign = 1 if (n + 1) % 2 == 0 else -1
    return sign * mpmath.factorial(n) * (mpmath.zeta(n + 1) - tail)


class _MPWalker:
    def __init__(self, prog: Program, x, const64: bool):
        self.prog = prog
        self.x = x
        self.const64 = const64
        self.fvals = {}

    def const(self, v):
        return mpmath.mpf(float(v)) if self.const64 else v

    def f(self, i):
        if i not in self.fvals:
            self.fvals[i] = self.walk(self.prog.funcs[i - 1])
        return self.fvals[i]

    def walk(self, node):
        op = node[0]
        if op == "num":
            return mpmath.mpf(node[1])
        if op == "x":
            return self.x[node[1] - 1]
        if op == "f":
            return self.f(node[1])
        if op == "P":
            return self.const(mpmath.pi())
        if op == "G":
            return self.const(mpmath.euler())
        if op == "pg":
            return self.const(_polygamma(node[1], node[2]))
        if op == "neg":
            return -self.walk(node[1])
        if op == "add":
            return self.walk(node[1]) + self.walk(node[2])
        if op == "sub":
            return self.walk(node[1]) - self.walk(node[2])
        if op == "mul":
            return self.walk(node[1]) * self.walk(node[2])
        if op == "div":
            a, b = self.walk(node[1]), self.walk(node[2])
            if b == 0:
                return mpmath.nan if a == 0 or mpmath.isnan(a) else mpmath.sign(a) * mpmath.inf
            return a / b
        if op == "pow":
            e, q = self.walk(node[1]), node[2]
            if float(q).is_integer():
                q = int(q)
                r = mpmath.mpf(1)
                for _ in range(abs(q)):  # R9: repeated multiplication
                    r = r * e
                if q < 0:
                    r = mpmath.inf if r == 0 else 1 / r
                return r
            if e < 0:
                return mpmath.nan
            if e == 0:
                return mpmath.mpf(0) if q > 0 else mpmath.inf
            return mpmath.power(e, mpmath.mpf(q))
        if op == "log":
            e = self.walk(node[1])
            if e < 0:
                return mpmath.nan
            if e == 0:
                return -mpmath.inf
            return mpmath.log(e)
        raise ValueError(f"unknown node {op!r}")


def evaluate_mp(prog: Program, x, digits: int = 60, const64: bool = False):
    """Values f(x_j), real mode, for points x[j, :] (FP64 coordinates) -> list of mpmath.mpf.

    Every operation is rounded to `digits` decimal digits.  Read the results inside
    `mpmath.workdps(digits)` (or convert them) to keep the precision.
    """
    out = []
    with mpmath.workdps(digits):
        for row in x:
            if len(row) != prog.nvars:
                raise ValueError(f"x must have shape [npts, {prog.nvars}]")
            pt = [mpmath.mpf(float(v)) for v in row]
            out.append(_MPWalker(prog, pt, const64).walk(prog.final))
    return out


def to_double_double(v, digits: int = 60):
    """(hi, lo): hi = the FP64 nearest v, lo = the FP64 nearest v - hi."""
    with mpmath.workdps(digits):
        if not mpmath.isfinite(v):
            return float(v), 0.0
        hi = float(v)
        if math.isinf(hi):
            return hi, 0.0
        return hi, float(v - mpmath.mpf(hi))
