"""A miniature algebraic front end -- TEST INFRASTRUCTURE, not part of the product.

The product starts where FIESTA's Mathematica part ends: at sector integrands in the worker grammar
(PAPER.md:506-515).  To pin the whole path against numbers the PAPER PRINTS for a Feynman integral
(the massless on-shell box: "-4.38658 + (1.3333 + 0.000019 pm7)/ep^2 -
(0.732466+0.000667 pm8)/ep"), this module derives such integrands with sympy, following the steps the
paper names: the alpha (Feynman) parameter representation of eq. (2), primary
sectors, iterated sector decomposition until U and F are non-zero at the origin, extraction of the
poles in eps by subtraction, expansion in eps.  Only what the one-loop box needs is handled: monomial
exponents >= -1 (logarithmic end-point singularities), polynomials with positive coefficients.

Nothing here evaluates an integrand numerically; the output is text for `fiesta_compile` / the oracle.
"""
from __future__ import annotations

import itertools

import sympy as sp

EPS = sp.Symbol("eps")


def _strip_monomials(poly, xs):
    """poly = prod_k x_k^m_k * rest, rest not divisible by any x_k.  Returns (m, rest)."""
    p = sp.Poly(sp.expand(poly), *xs)
    m = [min(mon[i] for mon in p.monoms()) for i in range(len(xs))]
    rest = sp.expand(poly / sp.Mul(*[x ** e for x, e in zip(xs, m)]))
    return m, rest


class Sector:
    """prod_k x_k^(A_k + B_k eps) * prod_m P_m^(c_m + d_m eps) over the unit cube in xs."""

    def __init__(self, xs, mono, factors):
        self.xs, self.mono, self.factors = list(xs), dict(mono), list(factors)

    def normalised(self):
        mono, factors = dict(self.mono), []
        for p, c, d in self.factors:
            m, rest = _strip_monomials(p, self.xs)
            for x, e in zip(self.xs, m):
                a, b = mono[x]
                mono[x] = (a + e * c, b + e * d)
            factors.append((rest, c, d))
        return Sector(self.xs, mono, factors)

    def vanishing_set(self):
        """A smallest set of variables at whose common zero some factor vanishes, or None."""
        for size in range(1, len(self.xs) + 1):
            for subset in itertools.combinations(self.xs, size):
                for p, _, _ in self.factors:
                    if sp.expand(p.subs({x: 0 for x in subset})) == 0:
                        return list(subset)
        return None


def decompose(sector):
    """Iterated sector decomposition: every returned sector's factors are non-zero at the origin."""
    done, todo = [], [sector.normalised()]
    while todo:
        s = todo.pop()
        vs = s.vanishing_set()
        if vs is None:
            done.append(s)
            continue
        for xj in vs:                                    # x_i = x_j t_i for the other members of the set
            sub = {xi: xj * xi for xi in vs if xi != xj}
            mono = dict(s.mono)
            a, b = mono[xj]
            extra_a, extra_b = len(vs) - 1, 0            # the Jacobian x_j^(|S|-1) ...
            for xi in vs:
                if xi != xj:                             # ... and the monomials of the rescaled variables
                    extra_a += mono[xi][0]
                    extra_b += mono[xi][1]
            mono[xj] = (a + extra_a, b + extra_b)
            factors = [(sp.expand(p.subs(sub, simultaneous=True)), c, d) for p, c, d in s.factors]
            todo.append(Sector(s.xs, mono, factors).normalised())
    return done


def to_text(expr, index):
    """sympy expression -> worker grammar.  index: symbol -> 1-based variable number."""
    e = expr
    if e.is_Symbol:
        return f"x[{index[e]}]"
    if e is sp.EulerGamma:
        return "G"
    if e is sp.pi:
        return "P"
    if e.is_Integer:
        return str(int(e)) if e >= 0 else f"(0-{int(-e)})"
    if e.is_Rational:
        num = str(int(e.p)) if e.p >= 0 else f"(0-{int(-e.p)})"
        return f"({num}/{int(e.q)})"
    if e.is_Add:
        return "(" + "+".join(to_text(a, index) for a in e.args) + ")"
    if e.is_Mul:
        return "(" + "*".join(to_text(a, index) for a in e.args) + ")"
    if e.is_Pow:
        base, ex = e.args
        if not ex.is_Rational:
            raise ValueError(f"exponent {ex} is not a number")
        return f"p[{to_text(base, index)},{sp.nsimplify(ex)}]" if ex.is_Integer else f"p[{to_text(base, index)},{float(ex)!r}]"
    if e.func is sp.log:
        return f"l[{to_text(e.args[0], index)}]"
    raise ValueError(f"cannot print {e!r}")


def eps_orders(sector, prefactor, orders):
    """Pole extraction and expansion of one decomposed sector.

    For the variables with x^(-1 + B eps):  int_0^1 x^(-1+B eps) g(x) dx = g(0)/(B eps) + int_0^1 x^(-1+B eps) (g(x) - g(0)) dx,
    applied to every such variable; each choice T of "taken at zero" variables is one term with the integration
    variables that remain.  Everything is then a rational function times exp(eps * logs) and is expanded to the
    requested orders of eps.  Returns a list of (remaining variables, {order: sympy integrand}).
    """
    xs = sector.xs
    poles = [x for x in xs if sector.mono[x][0] == -1]
    if any(sector.mono[x][0] < -1 for x in xs):
        raise ValueError("only logarithmic end-point singularities are handled")
    lo, hi = min(orders), max(orders)
    terms = []
    for r in range(len(poles) + 1):
        for T in itertools.combinations(poles, r):
            rest = [x for x in poles if x not in T]
            coef = sp.Integer(1)
            for x in T:
                coef = coef / sector.mono[x][1]                      # 1 / (B eps): eps^-|T| is booked below
            outer_rat = sp.Mul(*[1 / x for x in rest])
            outer_log = sp.Add(*[sector.mono[x][1] * sp.log(x) for x in rest])
            acc = {n: sp.Integer(0) for n in range(0, hi + len(T) + 1)}  # coefficient of eps^n of the bracket
            for q in range(len(rest) + 1):
                for R in itertools.combinations(rest, q):
                    zero = {x: 0 for x in list(T) + list(R)}
                    rat, lg = sp.Integer(1), outer_log
                    for x in xs:
                        if x in poles:
                            continue
                        a, b = sector.mono[x]
                        rat, lg = rat * x ** a, lg + b * sp.log(x)
                    for p, c, d in sector.factors:
                        pz = sp.expand(p.subs(zero))
                        rat, lg = rat * pz ** c, lg + d * sp.log(pz)
                    for n in acc:
                        acc[n] += (-1) ** q * rat * lg ** n / sp.factorial(n)
            pre = sp.series(prefactor, EPS, 0, hi + len(T) + 1).removeO()
            out = {}
            for m in orders:                                         # eps^m = eps^-|T| * eps^p (prefactor) * eps^n
                tot = sp.Integer(0)
                for n in acc:
                    p_ord = m + len(T) - n
                    if p_ord >= 0:
                        tot += pre.coeff(EPS, p_ord) * acc[n]
                out[m] = sp.nsimplify(coef) * outer_rat * tot
            terms.append(([x for x in xs if x not in T], out))
    return terms


def box_integrands(S=3, T=1, orders=(-2, -1, 0)):
    """The massless on-shell box (fig. 2) with indices (1,1,1,1) in d = 4 - 2 eps, Euclidean
    invariants S and T, in the normalisation of PAPER.md:293 ("(i pi^(d/2))^l and e^(-l gamma_E eps) pulled out"):

        Gamma(2 + eps) e^(gamma_E eps)  int d^4x delta(1 - sum x)  U^(2 eps) F^(-2 - eps),
        U = x1 + x2 + x3 + x4,  F = S x1 x3 + T x2 x4          (eq. (2): l = 1, a = 4).

    Returns a list of (dim, [text per order], label): finite integrals over unit cubes whose sum, order by
    order, is the coefficient of eps^order.
    """
    x = sp.symbols("x1:5", positive=True)
    U = sum(x)
    F = S * x[0] * x[2] + T * x[1] * x[3]
    pref = sp.gamma(2 + EPS) * sp.exp(sp.EulerGamma * EPS)
    out = []
    for i in range(4):                                               # primary sector i: x_i = 1 (homogeneity -4)
        rest = [v for k, v in enumerate(x) if k != i]
        start = Sector(rest, {v: (sp.Integer(0), sp.Integer(0)) for v in rest},
                       [(U.subs(x[i], 1), sp.Integer(0), sp.Integer(2)), (F.subs(x[i], 1), sp.Integer(-2), sp.Integer(-1))])
        for si, sec in enumerate(decompose(start)):
            for ti, (vs, by_order) in enumerate(eps_orders(sec, pref, orders)):
                index = {v: k + 1 for k, v in enumerate(vs)}
                texts = []
                for m in orders:
                    e = by_order[m]
                    body = "0" if e == 0 else to_text(e, index)
                    texts.append(f"{len(vs)};\n0;\n{body};\n|")
                out.append((len(vs), texts, f"primary {i + 1}, sector {si}, term {ti}"))
    return out


def triangle_integrands(s, m2=1):
    """The one-loop triangle with three equal internal masses m^2 = m2 and two light-like legs, (p1 + p2)^2 = s, in
    d = 4 (finite), from eq. (2) with l = 1, a = 3:

        J(s) = int d^3x delta(1 - sum x) 1 / (U F),   U = x1 + x2 + x3,   F = m2 U^2 - s x1 x2   (- i0).

    Above the threshold s > 4 m2 F changes sign inside the integration domain: the physical region that
    the contour deformation of PAPER.md:404 is for.  The three primary sectors need no further decomposition
    (F = m2 at the origin).  Returns [(texts, deform_f_index)]: blocks of 2 variables with f[1] = U, f[2] = F.
    """
    x = sp.symbols("x1:4", positive=True)
    U = sum(x)
    F = m2 * U ** 2 - s * x[0] * x[1]
    out = []
    for i in range(3):
        rest = [v for k, v in enumerate(x) if k != i]
        index = {v: k + 1 for k, v in enumerate(rest)}
        u_i, f_i = sp.expand(U.subs(x[i], 1)), sp.expand(F.subs(x[i], 1))
        text = f"2;\n2;\n{to_text(u_i, index)};\n{to_text(f_i, index)};\n1/(f[1]*f[2]);\n|"
        out.append(([text], 2))
    return out
