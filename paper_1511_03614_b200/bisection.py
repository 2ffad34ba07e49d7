"""Bisection of the integration cube (the BisectionVariables option of the paper's complex mode).

PAPER.md:406: "The contour transformation cannot deal with cases where F turns to zero for the
reason that some variables are equal to 1 (for example, a factor of x-1) ... In order to handle
those singularities, set the BisectionVariables equal to the list of variables such that the
integration cube is divided into two parts.  By default, the separation point is equal to 1/2,
however this can be changed either by setting the BisectionPoint value, or by providing a list of
BisectionPoints".

For one variable x_k and separation point p

    int_0^1 f dx_k  =  p int_0^1 f(x_k = p t) dt  +  (1-p) int_0^1 f(x_k = 1 - (1-p) t) dt .

The upper half is mapped with its orientation reversed, so that the end x_k = 1 -- where the
contour deformation is pinned (its shift carries the factor x_k (1 - x_k)) and cannot move the path
away from a zero of F -- becomes t = 0 of the new integrand, the corner the decomposition into
sectors and the periodising transform are made for; the cut x_k = p becomes t = 1 in both halves.
m bisected variables give 2^m integrands.

This is a transformation of the worker-grammar TEXT, done on the host before
fiesta_compile: every occurrence of x[k] -- in the f-lines as well, so a deformation polynomial
F stays a polynomial in the new variables -- is replaced by the parenthesised substitution, and the
final expression is multiplied by the Jacobian.  No arithmetic of the integrand is done here.
"""
from __future__ import annotations

import itertools
import re
from dataclasses import dataclass, field


@dataclass
class BisectedSector:
    """One part of a bisected integrand: the fields fiesta_compile reads (binding.Context.compile)."""
    sector_id: int
    texts: list
    is_complex: bool = False
    deform_f_index: int = 0
    lam: float = 0.0
    meta: dict = field(default_factory=dict)


def _literal(v: float) -> str:
    s = repr(float(v))
    if not re.fullmatch(r"\d+\.?\d*(?:[eE][+-]?\d+)?", s):
        raise ValueError(f"separation point gives the literal {s!r}, which the worker grammar cannot carry")
    return s


def _split_block(text: str):
    body = text.strip()
    if body.endswith("|"):
        body = body[:-1]
    parts = [p.strip() for p in body.split(";")]
    if parts and parts[-1] == "":
        parts.pop()
    nvars, nf = int(parts[0]), int(parts[1])
    if len(parts) != 3 + nf:
        raise ValueError("not a worker-grammar block: <nvars>; <nf>; f-lines; final; |")
    return nvars, nf, parts[2:2 + nf], parts[2 + nf]


def bisect_text(text: str, choices) -> str:
    """choices: {variable k (1-based): (p, upper)} -> the block with x[k] substituted and the Jacobian applied."""
    nvars, nf, flines, final = _split_block(text)
    sub, jac = {}, []
    for k, (p, upper) in choices.items():
        if not (1 <= k <= nvars):
            raise ValueError(f"variable {k} out of range 1..{nvars}")
        if not (0.0 < p < 1.0):
            raise ValueError("a separation point must lie strictly between 0 and 1")
        c = _literal(1.0 - p) if upper else _literal(p)
        sub[k] = f"(1-{c}*x[{k}])" if upper else f"({c}*x[{k}])"
        jac.append(c)

    def repl(m):
        k = int(m.group(1))
        return sub.get(k, m.group(0))

    pat = re.compile(r"x\[\s*(\d+)\s*\]")
    flines = [pat.sub(repl, f) for f in flines]
    final = pat.sub(repl, final)
    if jac:
        final = "*".join(jac) + "*(" + final + ")"
    return f"{nvars};\n{nf};\n" + "".join(f + ";\n" for f in flines) + final + ";\n|"


def bisect_sector(sector, variables, points=0.5, id_base=None):
    """The 2^m parts of `sector` bisected in `variables` (1-based indices) at `points` (one number, or one
    per variable).  Part h (bit i of h set: upper half of variables[i]) gets sector_id id_base + h
    (default id_base = sector_id * 2^m): the parts draw from different random streams.
    The integrals of the parts add up to the integral of `sector`."""
    variables = list(variables)
    if len(set(variables)) != len(variables):
        raise ValueError("a variable is listed twice")
    pts = [float(points)] * len(variables) if isinstance(points, (int, float)) else [float(p) for p in points]
    if len(pts) != len(variables):
        raise ValueError("one separation point per bisected variable")
    m = len(variables)
    base = int(sector.sector_id) * (1 << m) if id_base is None else int(id_base)
    parts = []
    for h, halves in enumerate(itertools.product((False, True), repeat=m)):
        # itertools orders the first variable slowest: bit i of h belongs to variables[m-1-i]; re-index so that
        # bit i of the part number is variables[i]
        halves = halves[::-1]
        choices = {variables[i]: (pts[i], halves[i]) for i in range(m)}
        parts.append(BisectedSector(sector_id=base + h, texts=[bisect_text(t, choices) for t in sector.texts],
                                    is_complex=bool(sector.is_complex), deform_f_index=int(sector.deform_f_index),
                                    lam=float(sector.lam),
                                    meta={"bisected_from": int(sector.sector_id),
                                          "halves": {variables[i]: ("upper" if halves[i] else "lower") for i in range(m)}}))
    return parts
