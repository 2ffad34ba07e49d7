"""Oracle step O1: parse the integration worker's expression text.

Follows PAPER.md:508-519 (section 4.6, "CIntegrate options"):

    "The expression lines are the following:
       - The number of variables;
       - The number of intermediate functions;
       - A number of lines each representing an intermediate expression. If the
         second line is 0;, then this part should be missing;
       - The final expression.
     The expressions might contain algebraic operations such as +, -, *, /,
     bracket symbols, numbers with a floating point.  The integration variables
     should be referred as x[1], x[2] and so on, intermediate functions as f[1],
     f[2] and so on.  Power is represented as p[expr,exponent], natural
     logarithm as l[expr].  One can also use P for pi and G for EulerGamma.
     PolyGamma[arg1,arg2] also works ... a few values for small polygamma
     arguments are hard-coded (PolyGamma[1,1], [2,1], [2,2], [2,3], [2,4],
     [3,1], [3,2])."

Each line ends with ';', the block ends with a line '|'.
Worked example: ``1; 0; x[1]+0.2;``.

The tree is a nest of tuples:
    ('num', float)   ('x', i)   ('f', i)   ('P',)  ('G',)  ('pg', n, m)
    ('neg', a)  ('add', a, b)  ('sub', a, b)  ('mul', a, b)  ('div', a, b)
    ('pow', a, q)       q a Python float (the exponent is a numeric constant)
    ('log', a)
Operator precedence and left associativity are the usual ones; unary minus
binds tighter than * and /  (so -a*b = (-a)*b, same value).

DESIGN.md readings used here: R9 (exponent is a signed numeric constant),
number literals denote their nearest FP64 value ("doubles").
"""
from __future__ import annotations

import re
from dataclasses import dataclass

HARD_CODED_POLYGAMMA = ((1, 1), (2, 1), (2, 2), (2, 3), (2, 4), (3, 1), (3, 2))

_TOKEN = re.compile(
    r"\s*(?:(?P<num>(?:\d+\.?\d*|\.\d+)(?:[eE][+-]?\d+)?)"
    r"|(?P<name>PolyGamma|[xfplPG])"
    r"|(?P<op>[-+*/()\[\],]))"
)


class ParseError(ValueError):
    pass


@dataclass
class Program:
    """One parsed expression block: `nvars`, the f[i] trees, the final tree."""
    nvars: int
    funcs: list
    final: tuple


def _tokenize(s: str):
    pos, out = 0, []
    s = s.rstrip()
    while pos < len(s):
        m = _TOKEN.match(s, pos)
        if not m:
            raise ParseError(f"unexpected character {s[pos]!r} at column {pos + 1} in {s!r}")
        pos = m.end()
        if m.lastgroup == "num":
            out.append(("num", m.group("num")))
        elif m.lastgroup == "name":
            out.append(("name", m.group("name")))
        else:
            out.append(("op", m.group("op")))
    return out


class _ExprParser:
    def __init__(self, tokens, nvars, nfuncs_available):
        self.t, self.i = tokens, 0
        self.nvars, self.nf = nvars, nfuncs_available

    def peek(self):
        return self.t[self.i] if self.i < len(self.t) else (None, None)

    def take(self, kind=None, val=None):
        k, v = self.peek()
        if k is None or (kind and k != kind) or (val is not None and v != val):
            raise ParseError(f"expected {val or kind}, got {v!r} at token {self.i}")
        self.i += 1
        return v

    def expr(self):  # sum
        a = self.term()
        while self.peek() in (("op", "+"), ("op", "-")):
            op = self.take()
            b = self.term()
            a = ("add", a, b) if op == "+" else ("sub", a, b)
        return a

    def term(self):  # product
        a = self.unary()
        while self.peek() in (("op", "*"), ("op", "/")):
            op = self.take()
            b = self.unary()
            a = ("mul", a, b) if op == "*" else ("div", a, b)
        return a

    def unary(self):
        if self.peek() == ("op", "-"):
            self.take()
            return ("neg", self.unary())
        if self.peek() == ("op", "+"):
            self.take()
            return self.unary()
        return self.atom()

    def _index(self):
        self.take("op", "[")
        v = self.take("num")
        if not v.isdigit():
            raise ParseError(f"index must be a positive integer, got {v!r}")
        self.take("op", "]")
        return int(v)

    def _signed_number(self):
        sign = 1.0
        while self.peek() in (("op", "-"), ("op", "+")):
            if self.take() == "-":
                sign = -sign
        return sign * float(self.take("num"))

    def atom(self):
        k, v = self.peek()
        if k == "num":
            self.take()
            return ("num", float(v))  # nearest FP64 value of the literal
        if k == "op" and v == "(":
            self.take()
            e = self.expr()
            self.take("op", ")")
            return e
        if k == "name":
            self.take()
            if v == "x":
                i = self._index()
                if not 1 <= i <= self.nvars:
                    raise ParseError(f"x[{i}] out of range 1..{self.nvars}")
                return ("x", i)
            if v == "f":
                i = self._index()
                if not 1 <= i <= self.nf:
                    raise ParseError(f"f[{i}] used before it is defined (have {self.nf})")
                return ("f", i)
            if v == "p":
                self.take("op", "[")
                e = self.expr()
                self.take("op", ",")
                # exponent: a numeric constant, optionally a/b, optionally in parentheses
                paren = self.peek() == ("op", "(")
                if paren:
                    self.take()
                q = self._signed_number()
                if self.peek() == ("op", "/"):
                    self.take()
                    q = q / self._signed_number()
                if paren:
                    self.take("op", ")")
                self.take("op", "]")
                return ("pow", e, q)
            if v == "l":
                self.take("op", "[")
                e = self.expr()
                self.take("op", "]")
                return ("log", e)
            if v == "P":
                return ("P",)
            if v == "G":
                return ("G",)
            if v == "PolyGamma":
                self.take("op", "[")
                n = self.take("num")
                self.take("op", ",")
                m = self.take("num")
                self.take("op", "]")
                if not (n.isdigit() and m.isdigit()) or (int(n), int(m)) not in HARD_CODED_POLYGAMMA:
                    raise ParseError(f"PolyGamma[{n},{m}] is not one of the hard-coded values (PAPER.md:515)")
                return ("pg", int(n), int(m))
        raise ParseError(f"unexpected token {v!r} at token {self.i}")


def _parse_expr(text, nvars, nf):
    p = _ExprParser(_tokenize(text), nvars, nf)
    e = p.expr()
    if p.i != len(p.t):
        raise ParseError(f"trailing input after expression: {p.t[p.i:]!r}")
    return e


def parse(text: str) -> Program:
    """Parse one block ``<nvars>; <nfuncs>; <f1>; ...; <final>; |``."""
    body = text
    bar = body.find("|")
    if bar >= 0:
        if body[bar + 1:].strip():
            raise ParseError("text after the terminating '|'")
        body = body[:bar]
    fields = body.split(";")
    if fields[-1].strip():
        raise ParseError("every expression line must end with ';'")
    fields = [f.strip() for f in fields[:-1]]
    if len(fields) < 3:
        raise ParseError("need at least: number of variables; number of functions; final expression;")
    if not fields[0].isdigit() or not fields[1].isdigit():
        raise ParseError("the first two lines must be non-negative integers")
    nvars, nfuncs = int(fields[0]), int(fields[1])
    if len(fields) != 2 + nfuncs + 1:
        raise ParseError(f"expected {nfuncs} function lines and one final expression, got {len(fields) - 2} lines")
    funcs = []
    for k in range(nfuncs):
        funcs.append(_parse_expr(fields[2 + k], nvars, k))
    final = _parse_expr(fields[2 + nfuncs], nvars, nfuncs)
    return Program(nvars, funcs, final)
