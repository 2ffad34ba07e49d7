"""Oracle step O2: evaluate a parsed expression at sample points by walking the tree.

Follows PAPER.md:108 ("a sequence of quadripples (operator, first operand, second
operand, result) ... the code runs a cycle through all the operations evaluating
the function"): the value of the program is the value of the expression.  Here
the tree is walked recursively; each f[i] is evaluated once per call (the
intermediate functions of PAPER.md:511 are a DAG).  Points are the leading
array axis (the paper evaluates "multiple sampling points at the same time",
PAPER.md:110); nothing else is vectorised, reordered or fused.

Semantics (DESIGN.md readings):
  R9   p[e,q], q integer  -> repeated multiplication e*e*...*e (|q| factors, left
       to right); q<0 -> 1/(that); q=0 -> 1.
       q non-integer, real mode -> pow(e,q) (NaN for e<0);
       complex mode -> exp(q*Log e), principal Log.
  R10  l[e] -> natural log; real mode e<0 -> NaN, e=0 -> -inf; complex: principal.
  P = pi, G = Euler's gamma, PolyGamma[n,m] = psi^(n)(m) for the seven pairs of
  PAPER.md:515, from psi^(n)(m) = (-1)^(n+1) n! (zeta(n+1) - sum_{j<m} j^-(n+1)).
  R14  magnitude companion M >= |f| (running first-order error bound), used only
       to scale the per-point parity tolerance under cancellation.
"""
from __future__ import annotations

import math

import numpy as np

from .parser import Program

LD = np.longdouble
CLD = np.clongdouble

# 40 significant digits each (more than the 64-bit mantissa holds)
PI = LD("3.141592653589793238462643383279502884197")
EULER_GAMMA = LD("0.5772156649015328606065120900824024310422")
ZETA3 = LD("1.202056903159594285399738161511449990765")


def _zeta(s: int):
    if s == 2:
        return PI * PI / LD(6)
    if s == 3:
        return ZETA3
    if s == 4:
        return PI * PI * PI * PI / LD(90)
    raise ValueError(s)


def polygamma_const(n: int, m: int):
    """psi^(n)(m), n>=1, positive integer m  (closed form, see module docstring)."""
    tail = LD(0)
    for j in range(1, m):
        tail += LD(1) / LD(j) ** (n + 1)
    sign = LD(1) if (n + 1) % 2 == 0 else LD(-1)
    return sign * LD(math.factorial(n)) * (_zeta(n + 1) - tail)


def _is_complex(dtype):
    return np.issubdtype(dtype, np.complexfloating)


def _real_dtype(dtype):
    return np.empty(0, dtype=dtype).real.dtype


def _int_power(e, q: int):
    """R9: repeated multiplication, |q| factors left to right; reciprocal if q<0."""
    if q == 0:
        return np.ones_like(e)
    r = e
    for _ in range(abs(q) - 1):
        r = r * e
    if q < 0:
        r = 1 / r
    return r


class _Walker:
    def __init__(self, prog: Program, x, dtype):
        self.prog = prog
        self.x = x  # [npts, nvars], dtype
        self.dtype = dtype
        self.cplx = _is_complex(dtype)
        self.rdt = _real_dtype(dtype)
        self.fvals = {}

    def const(self, v):
        return np.full(self.x.shape[0], v, dtype=self.dtype)

    def f(self, i):
        if i not in self.fvals:
            self.fvals[i] = self.walk(self.prog.funcs[i - 1])
        return self.fvals[i]

    def walk(self, node):
        op = node[0]
        if op == "num":
            return self.const(self.rdt.type(node[1]))
        if op == "x":
            return self.x[:, node[1] - 1]
        if op == "f":
            return self.f(node[1])
        if op == "P":
            return self.const(self.rdt.type(PI))
        if op == "G":
            return self.const(self.rdt.type(EULER_GAMMA))
        if op == "pg":
            return self.const(self.rdt.type(polygamma_const(node[1], node[2])))
        if op == "neg":
            return -self.walk(node[1])
        if op == "add":
            return self.walk(node[1]) + self.walk(node[2])
        if op == "sub":
            return self.walk(node[1]) - self.walk(node[2])
        if op == "mul":
            return self.walk(node[1]) * self.walk(node[2])
        if op == "div":
            return self.walk(node[1]) / self.walk(node[2])
        if op == "pow":
            e, q = self.walk(node[1]), node[2]
            if float(q).is_integer():
                return _int_power(e, int(q))
            if self.cplx:
                return np.exp(self.rdt.type(q) * np.log(e))
            return np.power(e, self.rdt.type(q))
        if op == "log":
            return np.log(self.walk(node[1]))
        raise ValueError(f"unknown node {op!r}")


def evaluate(prog: Program, x, dtype=LD):
    """Values f(x_j) for points x[j, :] (shape [npts, nvars]); returns shape [npts].

    `dtype` is numpy longdouble (the parity oracle), clongdouble (complex mode,
    PAPER.md:477) or float64/complex128 (only for timing the same walk in double).
    """
    x = np.asarray(x, dtype=dtype)
    if x.ndim != 2 or x.shape[1] != prog.nvars:
        raise ValueError(f"x must have shape [npts, {prog.nvars}]")
    with np.errstate(all="ignore"):
        return np.asarray(_Walker(prog, x, dtype).walk(prog.final), dtype=dtype)


class _MagWalker(_Walker):
    """Walks (value, magnitude) pairs.  DESIGN.md R14.

    M >= |v| is the scale a per-point "relative 1e-12" has to be measured against when the
    expression cancels.  For sums it is R14's modulus tree; through products, quotients, powers and
    logarithms the EXCESS M - |v| (the part of M that comes from cancellation below) is carried to
    first order, the way relative rounding errors propagate:
      leaf:     |v|
      a +- b:   Ma + Mb                                    (R14: "every subtraction by addition")
      a * b:    |ab| (1 + ra + rb)  = Ma|b| + |a|Mb - |ab|         with r = M/|v| - 1
      a / b:    |a/b| (1 + ra + rb)
      e^n:      |e^n| (1 + |n| re)       (n integer; n < 0 as the reciprocal of e^|n|)
      e^q:      |e^q| (1 + |q| re)       d(e^q)/e^q = q de/e
      log e:    max(|log e|, 1) + re     d(log e) = de/e;  R14's clamp of |log| at 1
    Where nothing cancels (r = 0 at every node: C1, C2, C5, and C3 except through the logarithm
    polynomials) M = |f| up to the clamp, and the test is the plain relative one.  R14's literal
    wording (modulus tree through * and / too) multiplies the factors (1 + r) instead of adding the
    r: never smaller than this M, and for quotients and negative powers of a cancelling argument it
    is not even a bound; DESIGN.md section 3 lists this reading.
    """

    def fm(self, i):
        if i not in self.fvals:
            self.fvals[i] = self.walk(self.prog.funcs[i - 1])
        return self.fvals[i]

    def walk(self, node):  # returns (v, M)
        op = node[0]
        if op in ("num", "x", "P", "G", "pg"):
            v = _Walker.walk(self, node)
            return v, np.abs(v)
        if op == "f":
            return self.fm(node[1])
        if op == "neg":
            v, m = self.walk(node[1])
            return -v, m
        if op in ("add", "sub"):
            a, ma = self.walk(node[1])
            b, mb = self.walk(node[2])
            return (a + b if op == "add" else a - b), ma + mb
        if op == "mul":
            a, ma = self.walk(node[1])
            b, mb = self.walk(node[2])
            aa, ab = np.abs(a), np.abs(b)
            return a * b, ma * ab + aa * mb - aa * ab
        if op == "div":
            a, ma = self.walk(node[1])
            b, mb = self.walk(node[2])
            aa, ab = np.abs(a), np.abs(b)
            return a / b, ma / ab + aa * mb / (ab * ab) - aa / ab
        if op == "pow":
            e, me = self.walk(node[1])
            q = node[2]
            ae = np.abs(e)
            if float(q).is_integer():
                qi = int(q)
                v = _int_power(e, qi)
                if qi == 0:
                    return v, np.abs(v)
                n = abs(qi)
                w = np.abs(_int_power(e, n))
                mw = w + n * np.abs(_int_power(e, n - 1)) * (me - ae)   # |e|^n + n|e|^(n-1)(Me-|e|)
                return v, (mw if qi > 0 else mw / (w * w))
            if self.cplx:
                v = np.exp(self.rdt.type(q) * np.log(e))
            else:
                v = np.power(e, self.rdt.type(q))
            return v, np.abs(v) * (1 + abs(q) * (me / ae - 1))
        if op == "log":
            e, me = self.walk(node[1])
            v = np.log(e)
            return v, np.maximum(np.abs(v), 1) + (me / np.abs(e) - 1)
        raise ValueError(op)


def evaluate_with_magnitude(prog: Program, x, dtype=LD):
    """(f(x_j), M(x_j)) with M the magnitude companion of DESIGN.md R14 (see _MagWalker)."""
    x = np.asarray(x, dtype=dtype)
    with np.errstate(all="ignore"):
        v, m = _MagWalker(prog, x, dtype).walk(prog.final)
    return np.asarray(v, dtype=dtype), np.asarray(m.real if np.iscomplexobj(m) else m)
