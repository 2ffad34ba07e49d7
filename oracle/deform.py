"""Oracle step O5: contour deformation and its Jacobian determinant.

The paper: "in cases where the integrand is complex, one has to perform a
contour deformation"; F enters as F - i0 (eq. 2);
`ComplexMode` "performs a contour deformation in order to avoid poles in
physical regions" with a size parameter lambda; the check is
that "the sign of the imaginary part of F is negative" (-testF).
The formula itself is not in the paper; it is BASELINE.json's north_star /
config 4 (R11, R12):

    g_k   = dF/dx_k (x)                                  (real, at the real point)
    z_k   = x_k - i*lambda*x_k*(1-x_k)*g_k
    J_kl  = delta_kl*(1 - i*lambda*(1-2x_k)*g_k) - i*lambda*x_k*(1-x_k)*d2F/dx_k dx_l
    D     = det J
    integrand(x) -> integrand(z(x)) * D          (every x in the text becomes z, R11)

Im F(z) = -lambda * sum_k x_k(1-x_k) g_k^2 + O(lambda^3) < 0, consistent with F - i0.

Derivatives are taken by differentiating the expression tree of F with the
textbook rules (sum, product, quotient by a constant, integer power), which is
the definition of dF/dx_k written out; F must be a polynomial in x.
det J: LU with partial pivoting on |.|, one matrix per point (R12).
"""
from __future__ import annotations

import numpy as np

from .evaluate import evaluate, LD, CLD
from .parser import Program

ZERO = ("num", 0.0)
ONE = ("num", 1.0)


def _is_zero(n):
    return n[0] == "num" and n[1] == 0.0


def _is_one(n):
    return n[0] == "num" and n[1] == 1.0


def _add(a, b):
    if _is_zero(a):
        return b
    if _is_zero(b):
        return a
    return ("add", a, b)


def _sub(a, b):
    if _is_zero(b):
        return a
    if _is_zero(a):
        return ("neg", b)
    return ("sub", a, b)


def _mul(a, b):
    if _is_zero(a) or _is_zero(b):
        return ZERO
    if _is_one(a):
        return b
    if _is_one(b):
        return a
    return ("mul", a, b)


def _inline(node, funcs):
    """Replace every f[i] by its defining tree (F is given as one of the f-lines)."""
    op = node[0]
    if op == "f":
        return _inline(funcs[node[1] - 1], funcs)
    if op in ("neg", "log"):
        return (op, _inline(node[1], funcs))
    if op in ("add", "sub", "mul", "div"):
        return (op, _inline(node[1], funcs), _inline(node[2], funcs))
    if op == "pow":
        return ("pow", _inline(node[1], funcs), node[2])
    return node


def _depends_on_x(node):
    op = node[0]
    if op == "x":
        return True
    if op in ("num", "P", "G", "pg"):
        return False
    if op == "pow":
        return _depends_on_x(node[1])
    return any(_depends_on_x(c) for c in node[1:])


def differentiate(node, k: int):
    """d(node)/dx_k for a polynomial tree (no f[i]; inline first)."""
    op = node[0]
    if op == "x":
        return ONE if node[1] == k else ZERO
    if op in ("num", "P", "G", "pg"):
        return ZERO
    if op == "neg":
        d = differentiate(node[1], k)
        return ZERO if _is_zero(d) else ("neg", d)
    if op == "add":
        return _add(differentiate(node[1], k), differentiate(node[2], k))
    if op == "sub":
        return _sub(differentiate(node[1], k), differentiate(node[2], k))
    if op == "mul":  # (ab)' = a'b + ab'
        a, b = node[1], node[2]
        return _add(_mul(differentiate(a, k), b), _mul(a, differentiate(b, k)))
    if op == "div":  # only division by a constant keeps a polynomial
        a, b = node[1], node[2]
        if _depends_on_x(b):
            raise ValueError("deformation polynomial F must not divide by x")
        d = differentiate(a, k)
        return ZERO if _is_zero(d) else ("div", d, b)
    if op == "pow":  # (e^q)' = q e^(q-1) e'
        e, q = node[1], node[2]
        if not _depends_on_x(e):
            return ZERO
        if not float(q).is_integer() or q < 0:
            raise ValueError("deformation polynomial F must have non-negative integer powers")
        q = int(q)
        if q == 0:
            return ZERO
        if q == 1:
            return differentiate(e, k)
        inner = e if q == 2 else ("pow", e, float(q - 1))
        return _mul(_mul(("num", float(q)), inner), differentiate(e, k))
    if op == "log":
        if _depends_on_x(node[1]):
            raise ValueError("deformation polynomial F must not contain logarithms of x")
        return ZERO
    raise ValueError(op)


def f_polynomial_tree(prog: Program, f_index: int):
    """The tree of f[f_index] with earlier f's inlined."""
    return _inline(prog.funcs[f_index - 1], prog.funcs)


def gradient_and_hessian(prog: Program, f_index: int, x, dtype=LD):
    """g[j,k] = dF/dx_k, H[j,k,l] = d2F/dx_k dx_l at the real points x[j,:]."""
    n = prog.nvars
    tree = f_polynomial_tree(prog, f_index)
    x = np.asarray(x, dtype=dtype)
    npts = x.shape[0]
    g = np.empty((npts, n), dtype=dtype)
    h = np.empty((npts, n, n), dtype=dtype)
    for k in range(1, n + 1):
        dk = differentiate(tree, k)
        g[:, k - 1] = evaluate(Program(n, [], dk), x, dtype)
        for l in range(k, n + 1):
            dkl = differentiate(dk, l)
            v = evaluate(Program(n, [], dkl), x, dtype)
            h[:, k - 1, l - 1] = v
            h[:, l - 1, k - 1] = v
    return g, h


def permanent(a):
    """per a[j,:,:] = sum over permutations of prod_k a[j,k,perm(k)]: the Leibniz formula of the
    determinant with every sign +.  For a matrix of magnitudes it is the magnitude companion (R14) of
    det; n! terms, n <= 8."""
    import itertools
    a = np.asarray(a)
    npts, n, _ = a.shape
    out = np.zeros(npts, dtype=a.dtype)
    for perm in itertools.permutations(range(n)):
        term = np.ones(npts, dtype=a.dtype)
        for k in range(n):
            term = term * a[:, k, perm[k]]
        out = out + term
    return out


def deform(prog: Program, f_index: int, lam, x, xbar=None, rdtype=LD):
    """(z, J) for real points x[j,:]; xbar = 1-x may be passed if known more accurately (R4)."""
    cdtype = CLD if rdtype == LD else np.complex128
    x = np.asarray(x, dtype=rdtype)
    xbar = rdtype(1) - x if xbar is None else np.asarray(xbar, dtype=rdtype)
    n = prog.nvars
    g, h = gradient_and_hessian(prog, f_index, x, rdtype)
    lam = rdtype(lam)
    s = x * xbar  # x_k (1 - x_k)
    z = x.astype(cdtype) - 1j * (lam * s * g).astype(cdtype)
    jac = (-1j) * (lam * s[:, :, None] * h).astype(cdtype)
    for k in range(n):
        # 1 - 2 x_k = xbar_k - x_k
        jac[:, k, k] += 1 - 1j * (lam * (xbar[:, k] - x[:, k]) * g[:, k]).astype(cdtype)
    return z, jac


def det_lu(a):
    """det of a[j,:,:] per point j by LU with partial pivoting on |.| (R12)."""
    a = np.array(a, copy=True)
    npts, n, _ = a.shape
    det = np.ones(npts, dtype=a.dtype)
    rows = np.arange(npts)
    for c in range(n):
        piv = c + np.argmax(np.abs(a[:, c:, c]), axis=1)  # row of the largest |a_ic|, i >= c
        swap = piv != c
        rc = a[rows, c, :].copy()
        rp = a[rows, piv, :].copy()
        a[rows, c, :] = rp
        a[rows, piv, :] = rc
        det = np.where(swap, -det, det)
        p = a[:, c, c]
        det = det * p
        with np.errstate(all="ignore"):
            for i in range(c + 1, n):
                m = a[:, i, c] / p
                a[:, i, c + 1:] = a[:, i, c + 1:] - m[:, None] * a[:, c, c + 1:]
    return det


def evaluate_deformed(prog: Program, f_index: int, lam, x, xbar=None, rdtype=LD):
    """integrand(z(x)) * det J(x) for every point (without the lattice weight W)."""
    cdtype = CLD if rdtype == LD else np.complex128
    z, jac = deform(prog, f_index, lam, x, xbar, rdtype)
    return evaluate(prog, z, cdtype) * det_lu(jac)


# ----------------------------------------------------------------------------- -testF and the choice of lambda

def f_at_deformed_points(prog: Program, f_index: int, lam, x, rdtype=LD):
    """F(z(x)) for real points x[j,:]: the deformation polynomial itself on the deformed contour."""
    cdtype = CLD if rdtype == LD else np.complex128
    z, _ = deform(prog, f_index, lam, x, None, rdtype)
    return evaluate(Program(prog.nvars, [], f_polynomial_tree(prog, f_index)), z, cdtype)


def test_f(prog: Program, f_index: int, lam, x, rdtype=LD):
    """PAPER.md:474 (-testF): "checks whether the sign of the imaginary part of F is negative".
    -> (number of points with Im F(z) >= 0 or NaN, max Im F(z), min |F(z)|) over the points x."""
    fz = f_at_deformed_points(prog, f_index, lam, x, rdtype)
    bad = int(np.sum(~(fz.imag < 0)))
    return bad, fz.imag.max(), np.abs(fz).min()


def select_lambda(prog: Program, f_index: int, x, lambda_max=1.0, lambda_split=4, conservative=False, rdtype=LD):
    """DESIGN.md R19, the reading of PAPER.md:404 ("tuned automatically in the interval from zero to
    MaxComplexShift", LambdaSplit candidates, LambdaIterations points, ConservativeComplexShift):
    candidates lambda_max*i/lambda_split, i = 1..lambda_split, each tested on the same points x;
    admissible = no point with Im F(z) >= 0; the admissible candidate with the largest min |F(z)| is
    chosen (first one on ties), halved if conservative.  -> (lambda or None, [(lambda_i, bad, max_im, min_abs)])."""
    scan = []
    best, best_min = None, None
    for i in range(1, lambda_split + 1):
        lam = rdtype(lambda_max) * rdtype(i) / rdtype(lambda_split)
        bad, mx, mn = test_f(prog, f_index, lam, x, rdtype)
        scan.append((lam, bad, mx, mn))
        if bad == 0 and (best is None or mn > best_min):
            best, best_min = lam, mn
    if best is None:
        return None, scan
    return (best / rdtype(2) if conservative else best), scan
