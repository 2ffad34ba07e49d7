"""Pins of the oracle against things other than itself: the paper's worked example, closed
forms, library routines (mpmath, scipy, numpy.linalg, cuRAND host), brute force.  CPU only."""
import ctypes
import itertools
import math
import os

import mpmath
import numpy as np
import pytest
import scipy.special

from conftest import golden
from oracle import points as P
from oracle.deform import (deform, det_lu, differentiate, evaluate_deformed, f_polynomial_tree,
                           gradient_and_hessian, select_lambda, test_f as oracle_test_f)
from oracle.evaluate import CLD, LD, evaluate, evaluate_with_magnitude, polygamma_const, PI, EULER_GAMMA
from oracle.integrate import (SectorSpec, combine_sectors, estimate_from_sums, integrate_lattice, integrate_mc,
                              integrate_vegas, lattice_partial_sums, neumaier_sum, vegas_combine, vegas_refine,
                              vegas_uniform_grid, exact_sum, ExactSum, mc_partial_sums, mc_points, vegas_iteration_sums)
from oracle.parser import ParseError, parse
from workloads import korobov_a

mpmath.mp.dps = 40
SEED = 20151111


def block(nvars, flines, final):
    return "\n".join([f"{nvars};", f"{len(flines)};"] + [f + ";" for f in flines] + [final + ";", "|"])


# ------------------------------------------------------------------ parser + walker

def test_paper_worked_example_integrates_to_0p7():
    g = golden("paper_worker_example.txt")
    sec = SectorSpec([g["text"] + "\n|"])
    n = 1 << 12
    val, err = integrate_lattice(sec, 8 * n, 8, P.korobov_genvec(korobov_a(n, 1), n, 1), 3, SEED)
    assert abs(float(val[0, 0]) - float(g["value"])) < 1e-12
    assert float(err[0, 0]) < 1e-10
    val, err = integrate_mc(sec, 1 << 14, SEED)
    assert abs(float(val[0, 0]) - 0.7) < 4 * float(err[0, 0])
    assert 0 < float(err[0, 0]) < 0.01      # sigma of x+0.2 is sqrt(1/12)/sqrt(N) = 2.3e-3


def test_linear_function_closed_form():
    # "-test: integrator test on a sample linear function": c0 + sum c_k/2
    rng = np.random.default_rng(1)
    n = 5
    c = [float(v) for v in rng.uniform(-2, 2, size=n + 1)]
    text = block(n, [], "+".join([f"({c[0]!r})"] + [f"({c[k + 1]!r})*x[{k + 1}]" for k in range(n)]))
    exact = c[0] + sum(c[1:]) / 2
    nl = 1 << 11
    val, err = integrate_lattice(SectorSpec([text]), 8 * nl, 8, P.korobov_genvec(korobov_a(nl, 4), nl, n), 3, SEED)
    assert abs(float(val[0, 0]) - exact) <= max(4 * float(err[0, 0]), 1e-13)
    assert float(err[0, 0]) < 5e-3


def test_walker_against_python_floats():
    # brute force: the same formula typed as a Python expression, evaluated with math.*
    text = block(3, ["x[1]*x[2]+0.5", "l[f[1]]-x[3]/(1+x[2])"],
                 "-f[2]*p[f[1],3]+p[x[3],-2]/f[1]-p[f[1],0.5]*(x[1]-2*x[2])*P+G-(-x[1])")
    prog = parse(text)
    rng = np.random.default_rng(2)
    x = rng.uniform(0.1, 0.9, size=(50, 3))
    got = evaluate(prog, x, LD)
    for j in range(50):
        a, b, c = x[j]
        f1 = a * b + 0.5
        f2 = math.log(f1) - c / (1 + b)
        ref = -f2 * f1 ** 3 + c ** -2 / f1 - f1 ** 0.5 * (a - 2 * b) * math.pi + 0.5772156649015329 - (-a)
        assert abs(float(got[j]) - ref) <= 2e-15 * max(1.0, abs(ref)) * 20


def test_operator_precedence_and_associativity():
    prog = parse(block(2, [], "1-x[1]-x[2]*2/4/x[1]+-x[2]"))
    x = np.array([[0.5, 0.25]])
    assert float(evaluate(prog, x)[0]) == 1 - 0.5 - 0.25 * 2 / 4 / 0.5 + -0.25


def test_integer_power_is_repeated_multiplication_and_negative_is_reciprocal():
    x = np.array([[LD(3) / LD(7)]], dtype=LD)
    v = x[0, 0]
    assert evaluate(parse(block(1, [], "p[x[1],4]")), x)[0] == v * v * v * v
    assert evaluate(parse(block(1, [], "p[x[1],-3]")), x)[0] == 1 / (v * v * v)
    assert evaluate(parse(block(1, [], "p[x[1],0]")), x)[0] == 1
    got = evaluate(parse(block(1, [], "p[x[1],-0.7]")), x)[0]
    # the literal -0.7 denotes its nearest FP64 value ("doubles")
    assert abs(got - LD(str(mpmath.power(mpmath.mpf(3) / 7, mpmath.mpf(-0.7))))) < 4e-19 * 2


def test_real_mode_domain_errors_give_nan():
    x = np.array([[0.25]])
    assert np.isnan(evaluate(parse(block(1, [], "l[x[1]-1]")), x)[0])
    assert np.isnan(evaluate(parse(block(1, [], "p[x[1]-1,0.5]")), x)[0])


def test_complex_mode_principal_branches():
    z = np.array([[-0.3 - 1e-3j]], dtype=CLD)
    v = evaluate(parse(block(1, [], "l[x[1]]")), z, CLD)[0]
    ref = mpmath.log(mpmath.mpc(-0.3, -1e-3))
    assert abs(complex(v) - complex(ref)) < 1e-15 and v.imag < -3.1
    v = evaluate(parse(block(1, [], "p[x[1],-2.5]")), z, CLD)[0]
    ref = mpmath.power(mpmath.mpc(-0.3, -1e-3), -2.5)
    assert abs(complex(v) - complex(ref)) < 1e-13 * abs(complex(ref))


def test_constants_against_mpmath():
    assert abs(PI - LD(str(mpmath.pi))) < 2e-19
    assert abs(EULER_GAMMA - LD(str(mpmath.euler))) < 1e-19
    for n, m in ((1, 1), (2, 1), (2, 2), (2, 3), (2, 4), (3, 1), (3, 2)):
        ref = mpmath.polygamma(n, m)
        got = polygamma_const(n, m)
        assert abs(got - LD(str(ref))) < 2e-18 * abs(float(ref)), (n, m)
        assert abs(float(evaluate(parse(block(1, [], f"PolyGamma[{n},{m}]+0*x[1]")), np.array([[0.5]]))[0])
                   - float(ref)) < 1e-15 * abs(float(ref))


@pytest.mark.parametrize("bad", [
    "1; 0; x[2];\n|",             # variable out of range
    "1; 1; f[1]; x[1];\n|",       # f used before defined
    "1; 0; x[1]+;\n|",
    "1; 0; PolyGamma[5,5];\n|",   # not hard-coded
    "1; 2; x[1]; x[1];\n|",       # wrong number of lines
    "1; 0; x[1]",                 # missing ';'
    "1; 0; p[x[1],x[1]];\n|",     # exponent must be numeric
])
def test_parse_errors(bad):
    with pytest.raises(ParseError):
        parse(bad)


# ------------------------------------------------------------------ closed forms

def _genvec(nl, dim):
    return P.korobov_genvec(korobov_a(nl, dim), nl, dim)


def test_monomial_integrals_closed_form():
    # int prod x_i^a_i = prod 1/(a_i+1) over the unit cube (BASELINE config 1's closed-form check)
    nl = 1 << 13
    for a in [(0, 1, 2, 1), (2, 2, 0, 1), (-0.45, 1, 0, -0.3)]:
        text = block(4, [], "*".join(f"p[x[{i + 1}],{ai}]" for i, ai in enumerate(a)))
        exact = np.prod([1.0 / (ai + 1) for ai in a])
        val, err = integrate_lattice(SectorSpec([text]), 8 * nl, 8, _genvec(nl, 4), 3, SEED)
        assert abs(float(val[0, 0]) - exact) <= 4 * float(err[0, 0]) + 1e-15, a
        assert float(err[0, 0]) < 2e-4 * exact, a


def test_bubble_golden_against_mpmath():
    g = golden("bubble_eps_coefficients.txt")
    eps = mpmath.mpf(0)
    coeffs = mpmath.taylor(lambda e: mpmath.gamma(1 - e) ** 2 / mpmath.gamma(2 - 2 * e), eps, 4)
    for k in range(5):
        assert abs(coeffs[k] - mpmath.mpf(g[f"c{k}"])) < mpmath.mpf("1e-15")


def test_bubble_epsilon_orders():
    # U = 1 + x1 = f[1], F = x1; order-k integrand (1+t)^-2 (2 ln(1+t) - ln t)^k / k!
    g = golden("bubble_eps_coefficients.txt")
    nl = 1 << 13
    texts = []
    for k in range(5):
        fac = math.factorial(k)
        body = "p[f[1],-2]" + (f"*p[2*l[f[1]]-l[x[1]],{k}]/{fac}" if k else "")
        texts.append(block(1, ["1+x[1]"], body))
    val, err = integrate_lattice(SectorSpec(texts), 8 * nl, 8, _genvec(nl, 1), 3, SEED)
    for k in range(5):
        exact = float(g[f"c{k}"])
        assert abs(2 * float(val[k, 0]) - exact) <= 2 * 4 * float(err[k, 0]) + 1e-14, k
        assert abs(2 * float(val[k, 0]) - exact) < 1e-9, k


def test_random_family_against_gauss_legendre_bruteforce():
    # 2-D U^p / F^q * log with random coefficients; reference = tensor Gauss-Legendre on the Python formula
    rng = np.random.default_rng(5)
    cu, cf = [float(v) for v in rng.uniform(0.5, 2, 4)], [float(v) for v in rng.uniform(0.5, 2, 4)]
    texts = [block(2, [f"{cu[0]!r}+{cu[1]!r}*x[1]+{cu[2]!r}*x[1]*x[2]+{cu[3]!r}*p[x[2],2]",
                       f"{cf[0]!r}+{cf[1]!r}*x[2]+{cf[2]!r}*x[1]*x[2]+{cf[3]!r}*p[x[1],2]"],
                   "x[1]*f[1]*p[f[2],-2.5]*l[f[2]]")]
    xs, ws = np.polynomial.legendre.leggauss(60)
    xs, ws = (xs + 1) / 2, ws / 2
    X, Y = np.meshgrid(xs, xs, indexing="ij")
    U = cu[0] + cu[1] * X + cu[2] * X * Y + cu[3] * Y ** 2
    F = cf[0] + cf[1] * Y + cf[2] * X * Y + cf[3] * X ** 2
    ref = float(np.sum(np.outer(ws, ws) * X * U * F ** -2.5 * np.log(F)))
    nl = 1 << 13
    val, err = integrate_lattice(SectorSpec(texts), 8 * nl, 8, _genvec(nl, 2), 3, SEED)
    assert abs(float(val[0, 0]) - ref) <= 4 * float(err[0, 0]) + 1e-12
    assert abs(float(val[0, 0]) - ref) < 1e-8 * abs(ref)


# ------------------------------------------------------------------ points

def test_lattice_integers_against_bigint_bruteforce():
    nl, dim, a = 1 << 9, 5, 187
    g = P.korobov_genvec(a, nl, dim)
    assert g == [pow(a, k, nl) for k in range(dim)]
    delta = P.lattice_shift(SEED, 7, 3, dim)
    t = P.lattice_t(np.arange(nl), g, nl, delta)
    for j in (0, 1, 2, 255, 511):
        for k in range(dim):
            ref = ((((j * g[k]) % nl) << 64) // nl + int(delta[k])) % (1 << 64)
            assert int(t[j, k]) == ref
    u = P.unit_from_t(t)
    for j in (0, 3, 400):
        for k in range(dim):
            assert u[j, k] == LD(2 * (int(t[j, k]) >> 12) + 1) / LD(2 ** 53)
    assert np.all((u > 0) & (u < 1))
    assert np.all(u.astype(np.float64).astype(LD) == u)      # exactly representable in FP64


def test_lattice_character_sums_vanish():
    # (1/N) sum_j exp(2 pi i h.(j g + Delta)/N) = 0 unless h.g = 0 mod N: exactness of the rank-1 rule
    nl, dim = 1 << 10, 3
    g = P.korobov_genvec(korobov_a(nl, dim), nl, dim)
    t = P.lattice_t(np.arange(nl), g, nl, P.lattice_shift(SEED, 0, 0, dim)).astype(LD) / LD(2) ** 64
    rng = np.random.default_rng(3)
    n_zero = 0
    for _ in range(40):
        h = rng.integers(-6, 7, size=dim)
        s = np.sum(np.cos(2 * PI * (t @ h.astype(LD)))) / nl
        if int(np.dot(h, g)) % nl == 0:
            continue
        n_zero += 1
        assert abs(float(s)) < 1e-13
    assert n_zero > 30


def test_philox_against_curand_host_generator():
    # cuRAND's host generator (a CPU library routine) hands out raw Philox4x32-10 words; group i of four
    # words is the block with counter (i // T, 0, i % T, 0) and key = seed, T = cuRAND's stream count.
    path = "/usr/local/cuda/lib64/libcurand.so"
    if not os.path.exists(path):
        pytest.skip("cuRAND not installed")
    lib = ctypes.CDLL(path)
    ngroups = 70000
    for seed in (0, SEED, 0xDEADBEEFCAFE1234):
        gen = ctypes.c_void_p()
        assert lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0   # CURAND_RNG_PSEUDO_PHILOX4_32_10
        assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
        out = np.zeros(4 * ngroups, dtype=np.uint32)
        assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(out.size)) == 0
        lib.curandDestroyGenerator(gen)
        out = out.reshape(-1, 4).astype(np.uint64)
        i = np.arange(ngroups)
        matched = False
        for log_t in range(10, 21):
            t = 1 << log_t
            mine = np.stack(P.philox4x32_10(i // t, 0 * i, i % t, 0 * i, seed & 0xFFFFFFFF, seed >> 32), axis=1)
            if np.array_equal(mine, out):
                matched = t < ngroups           # both c0 and c2 varied
                break
        assert matched, seed


def test_philox_stream_layout_and_moments():
    t = P.philox_t(SEED, 5, P.TAG_MC, 2, np.arange(4096), 7)
    # layout (R3): coordinate pair (2kb, 2kb+1) = words (0,1), (2,3) of the call with kblock kb
    o = P.philox4x32_10([9], [0], [5], [(1 << 28) | (2 << 20) | 2], SEED & 0xFFFFFFFF, SEED >> 32)
    assert int(t[9, 4]) == (int(o[0][0]) << 32) | int(o[1][0])
    assert int(t[9, 5]) == (int(o[2][0]) << 32) | int(o[3][0])
    u = P.unit_from_t(t).astype(np.float64)
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / u.size)
    assert abs((u ** 2).mean() - 1 / 3) < 4 * math.sqrt(4 / 45 / u.size)
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 4 / math.sqrt(4096)
    assert len(np.unique(t)) == t.size
    assert not np.array_equal(P.lattice_shift(SEED, 5, 0, 4), P.lattice_shift(SEED, 6, 0, 4))
    assert not np.array_equal(P.lattice_shift(SEED, 5, 0, 4), P.lattice_shift(SEED, 5, 1, 4))


@pytest.mark.parametrize("r", [1, 2, 3, 4])
def test_korobov_transform_against_incomplete_beta(r):
    u = np.linspace(0, 1, 1001, dtype=LD)[1:-1]
    x, xbar, w = P.korobov_transform(u, r)
    ref = scipy.special.betainc(r + 1, r + 1, u.astype(np.float64))     # phi_r = I_u(r+1, r+1)
    assert np.max(np.abs(x.astype(np.float64) - ref)) < 5e-15
    assert np.max(np.abs((x + xbar) - 1)) < 2e-19
    x2, xbar2, w2 = P.korobov_transform(LD(1) - u, r)
    assert np.max(np.abs(x2 - xbar)) < 2e-19 and np.max(np.abs(w2 - w)) < 1e-17     # phi(u)+phi(1-u)=1
    wref = math.factorial(2 * r + 1) / math.factorial(r) ** 2 * (u * (1 - u)) ** r
    assert np.max(np.abs(w - wref)) < 1e-15
    # phi' = w (central differences) and int w = 1 (Gauss-Legendre, exact for degree 2r)
    h = LD(1e-6)
    d = (P.korobov_transform(u + h, r)[0] - P.korobov_transform(u - h, r)[0]) / (2 * h)
    assert np.max(np.abs(d - w)) < 1e-9
    gx, gw = np.polynomial.legendre.leggauss(12)
    assert abs(float(np.sum(gw / 2 * np.asarray(P.korobov_transform(np.asarray((gx + 1) / 2, dtype=LD), r)[2],
                                                dtype=np.float64))) - 1) < 1e-14
    # near the faces: x = phi(u) keeps full relative accuracy, xbar does near u -> 1
    tiny = np.array([LD(2) ** -40], dtype=LD)
    xs, _, _ = P.korobov_transform(tiny, r)
    lead = math.factorial(2 * r + 1) / math.factorial(r) ** 2 / (r + 1)
    assert abs(float(xs[0]) / (lead * float(tiny[0]) ** (r + 1)) - 1) < 1e-10
    _, xb, _ = P.korobov_transform(LD(1) - tiny, r)
    assert xb[0] == xs[0]


def test_transformed_singular_integral():
    # int phi_3(u)^-0.7 w_3(u) du = int x^-0.7 dx = 1/0.3
    nl = 1 << 13
    val, err = integrate_lattice(SectorSpec([block(1, [], "p[x[1],-0.7]")]), 8 * nl, 8, _genvec(nl, 1), 3, SEED)
    assert abs(float(val[0, 0]) - 1 / 0.3) <= 4 * float(err[0, 0]) + 1e-12


# ------------------------------------------------------------------ deformation

F_TEXT = "0.7-1.3*x[1]*x[2]+0.9*p[x[3],2]*x[1]-0.4*x[2]+p[x[1]+x[3],3]/4"


def test_derivatives_against_complex_step_and_differences():
    prog = parse(block(3, [F_TEXT], "f[1]"))
    rng = np.random.default_rng(4)
    x = rng.uniform(0.05, 0.95, size=(20, 3)).astype(LD)
    g, h = gradient_and_hessian(prog, 1, x)
    step = LD("1e-30")
    for k in range(3):
        z = x.astype(CLD)
        z[:, k] += 1j * step
        cs = evaluate(prog, z, CLD).imag / step                   # Im F(x + i h e_k)/h
        assert np.max(np.abs(cs - g[:, k])) < 1e-17
        for l in range(3):
            d = LD("1e-9")
            xp, xm = x.copy(), x.copy()
            xp[:, l] += d
            xm[:, l] -= d
            fd = (gradient_and_hessian(prog, 1, xp)[0][:, k] - gradient_and_hessian(prog, 1, xm)[0][:, k]) / (2 * d)
            assert np.max(np.abs(fd - h[:, k, l])) < 1e-8
    # hand-derived gradient of F_TEXT
    a, b, c = (x[:, i] for i in range(3))
    assert np.max(np.abs(g[:, 0] - (-1.3 * b + 0.9 * c * c + 0.75 * (a + c) ** 2))) < 1e-15
    assert np.max(np.abs(g[:, 1] - (-1.3 * a - 0.4))) < 1e-15
    assert np.max(np.abs(h[:, 0, 2] - (1.8 * c + 1.5 * (a + c)))) < 1e-15


def test_det_lu_against_cofactors_and_numpy():
    rng = np.random.default_rng(6)
    for n in (1, 2, 3, 4):
        a = (rng.normal(size=(30, n, n)) + 1j * rng.normal(size=(30, n, n))).astype(CLD)
        ref = np.zeros(30, dtype=CLD)
        for perm in itertools.permutations(range(n)):                 # Leibniz formula
            sign = np.linalg.det(np.eye(n)[list(perm)])
            term = np.full(30, sign, dtype=CLD)
            for i, p in enumerate(perm):
                term = term * a[:, i, p]
            ref += term
        assert np.max(np.abs(det_lu(a) - ref) / np.abs(ref)) < 1e-15
    a = (rng.normal(size=(10, 7, 7)) + 1j * rng.normal(size=(10, 7, 7))).astype(CLD)
    ref = np.linalg.det(a.astype(np.complex128))
    assert np.max(np.abs(det_lu(a).astype(np.complex128) - ref) / np.abs(ref)) < 1e-12
    tri = np.triu(a)
    assert np.max(np.abs(det_lu(tri) - np.prod(np.diagonal(tri, axis1=1, axis2=2), axis=1))) < 1e-16
    a[:, 0, :] = 0          # singular column pivot must give 0, not NaN-free garbage
    assert np.all(det_lu(a[:, :, :]) == 0) or np.all(np.isnan(det_lu(a).real))


def test_deformation_matches_its_definition_and_jacobian_is_dz_dx():
    prog = parse(block(3, [F_TEXT], "f[1]"))
    rng = np.random.default_rng(7)
    x = rng.uniform(0.05, 0.95, size=(8, 3)).astype(LD)
    lam = 0.5
    z, jac = deform(prog, 1, lam, x)
    g, _ = gradient_and_hessian(prog, 1, x)
    assert np.max(np.abs(z - (x - 1j * LD(lam) * x * (1 - x) * g))) < 1e-18
    d = LD("1e-9")
    for l in range(3):
        xp, xm = x.copy(), x.copy()
        xp[:, l] += d
        xm[:, l] -= d
        fd = (deform(prog, 1, lam, xp)[0] - deform(prog, 1, lam, xm)[0]) / (2 * d)
        assert np.max(np.abs(fd - jac[:, :, l])) < 1e-8             # J_kl = dz_k/dx_l
    z0, j0 = deform(prog, 1, 0.0, x)
    assert np.all(z0.imag == 0) and np.all(det_lu(j0) == 1)         # lambda = 0 is the real path


def test_contour_1d_closed_forms():
    g = golden("contour_1d_closed_forms.txt")
    a = mpmath.mpf("0.3")
    assert abs(mpmath.log((1 - a) / a) - mpmath.mpf(g["inv_re"])) < 1e-17
    assert abs(2 * mpmath.sqrt(a) - mpmath.mpf(g["rsqrt_im"])) < 1e-17
    assert abs((1 - a) * mpmath.log(1 - a) + a * mpmath.log(a) - 1 - mpmath.mpf(g["log_re"])) < 1e-17
    nl = 1 << 13
    for key, final in (("inv", "1/f[1]"), ("log", "l[f[1]]"), ("rsqrt", "p[f[1],-0.5]")):
        sec = SectorSpec([block(1, ["x[1]-0.3"], final)], is_complex=True, deform_f_index=1, lam=0.5)
        val, err = integrate_lattice(sec, 8 * nl, 8, _genvec(nl, 1), 3, SEED)
        for c, part in enumerate(("re", "im")):
            exact = float(g[f"{key}_{part}"])
            assert abs(float(val[0, c]) - exact) <= 4 * float(err[0, c]) + 1e-11, (key, part)
            assert abs(float(val[0, c]) - exact) < 1e-6, (key, part)


def test_lambda_independence_for_entire_integrands():
    # Cauchy: int g(z) det J dx = int g(x) dx for polynomials g, any lambda, any polynomial F (z fixes the faces)
    nl = 1 << 12
    flines = ["0.6-1.1*x[1]*x[2]+0.8*x[3]-0.5*p[x[2],2]*x[3]"]
    final = "p[x[1],2]*x[2]+0.5*x[3]*x[1]"
    exact = 1.0 / 6 + 0.125
    for lam in (0.0, 0.3, 1.0):
        sec = SectorSpec([block(3, flines, final)], is_complex=True, deform_f_index=1, lam=lam)
        val, err = integrate_lattice(sec, 8 * nl, 8, _genvec(nl, 3), 3, SEED)
        assert abs(float(val[0, 0]) - exact) <= 4 * float(err[0, 0]) + 1e-12, lam
        assert abs(float(val[0, 1])) <= 4 * float(err[0, 1]) + 1e-12, lam
        assert float(err[0, 0]) < 1e-5


def test_c4_workload_has_negative_imaginary_f():
    # PAPER.md:474 (-testF): "the sign of the imaginary part of F is negative"
    from workloads import make_workload
    wl = make_workload("C4", nsectors=3, npoints=1 << 10)
    rng = np.random.default_rng(8)
    x = rng.uniform(0, 1, size=(2000, wl.dim)).astype(LD)
    changes = 0
    for s in wl.sectors:
        sec = SectorSpec(s.texts, s.sector_id, True, s.deform_f_index, s.lam)
        prog = sec.progs[0]
        z, _ = deform(prog, s.deform_f_index, s.lam, x)
        from oracle.parser import Program
        fz = evaluate(Program(prog.nvars, [], f_polynomial_tree(prog, s.deform_f_index)), z, CLD)
        assert np.all(fz.imag < 0)
        fx = evaluate(Program(prog.nvars, [], f_polynomial_tree(prog, s.deform_f_index)), x, LD)
        changes += int(np.any(fx < 0))
        vals = evaluate_deformed(prog, s.deform_f_index, s.lam, x)
        assert np.all(np.isfinite(vals.real)) and np.all(np.isfinite(vals.imag))


# ------------------------------------------------------------------ estimators

def test_exact_sum_against_rationals():
    """O6: the oracle's sums are the exact sum of the terms rounded once.  Pin: Python Fractions (every
    long double is a dyadic rational), math.fsum on doubles, cancelling cases, any feeding order."""
    from fractions import Fraction

    def frac(v):                      # exact value of a long double: mantissa (two exact halves) * 2^e
        m, e = np.frexp(LD(v))
        a = abs(m) * LD(2.0 ** 32)
        hi = int(np.floor(a))
        lo = int((a - LD(hi)) * LD(2.0 ** 32))
        q = Fraction((hi << 32) + lo) * Fraction(2) ** (int(e) - 64)
        return -q if m < 0 else q

    rng = np.random.default_rng(7)
    for trial in range(20):
        n = int(rng.integers(1, 400))
        v = (rng.standard_normal(n).astype(LD) * LD(3) + rng.standard_normal(n).astype(LD) * LD(2.0 ** -60)) \
            * LD(2.0) ** rng.integers(-200, 200, n).astype(LD)
        if trial % 3 == 0:            # heavy cancellation: the big terms vanish exactly
            v = np.concatenate([v, -v, rng.standard_normal(5).astype(LD) * LD(2.0 ** -300)])
            v = v[rng.permutation(v.shape[0])]
        exact = sum((frac(x) for x in v), Fraction(0))
        got = exact_sum(v)
        # rounded once: within half an ulp (2^-64 relative) of the rational sum, or exactly 0
        assert exact == 0 and got == 0 or abs(frac(got) - exact) <= abs(exact) * Fraction(1, 2 ** 64)
        acc = ExactSum()              # fed in pieces, reversed: the same number
        for piece in np.array_split(v[::-1], 7):
            acc.add(piece)
        assert acc.value() == got
    d = rng.standard_normal(5000) * 10.0 ** rng.integers(-10, 10, 5000)
    assert float(exact_sum(d.astype(LD))) == math.fsum(d)
    assert exact_sum(np.array([LD(1), LD(2) ** -70, -LD(1), LD(2) ** -70], dtype=LD)) == LD(2) ** -69
    assert np.isnan(exact_sum(np.array([LD(1), LD(np.nan)], dtype=LD)))
    assert exact_sum(np.zeros(0, dtype=LD)) == 0


def test_sums_do_not_depend_on_chunking():
    """The chunk argument of the oracle's integrators only bounds memory."""
    sec = SectorSpec([block(2, ["1+x[1]*x[2]"], "p[f[1],-2]*l[f[1]]-0.3*x[1]")], sector_id=3)
    a = lattice_partial_sums(sec, 1 << 10, 2, [1, 333], 3, SEED, chunk=1 << 14)
    b = lattice_partial_sums(sec, 1 << 10, 2, [1, 333], 3, SEED, chunk=37)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    whole = lattice_partial_sums(sec, 1 << 10, 2, [1, 333], 3, SEED, shifts=[1])
    left = lattice_partial_sums(sec, 1 << 10, 2, [1, 333], 3, SEED, shifts=[1], first=0, count=300)
    right = lattice_partial_sums(sec, 1 << 10, 2, [1, 333], 3, SEED, shifts=[1], first=300, count=724)
    assert np.allclose((left[0] + right[0]).astype(float), whole[0].astype(float), rtol=1e-17)
    assert all(np.array_equal(x, y) for x, y in zip(mc_partial_sums(sec, 1000, 5, chunk=1000), mc_partial_sums(sec, 1000, 5, chunk=64)))
    grid = vegas_uniform_grid(2, 7)
    a = vegas_iteration_sums(sec, grid, 999, 5, 2, chunk=999)
    b = vegas_iteration_sums(sec, grid, 999, 5, 2, chunk=100)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))


def test_neumaier_and_estimators():
    v = np.array([LD(1), LD(2) ** -70, -LD(1), LD(2) ** -70], dtype=LD)
    assert neumaier_sum(v) == LD(2) ** -69
    # R shifts of a constant integrand: sigma = 0
    val, err = integrate_lattice(SectorSpec([block(2, [], "2.5+0*x[1]")]), 8 * 64, 8, [1, 19], 0, SEED)
    assert float(val[0, 0]) == 2.5 and float(err[0, 0]) == 0
    # R >= 2 formula on hand numbers: Q = (1,2,3,6) -> mean 3, sigma = sqrt(14/12)
    s1 = np.array([[[10.0]], [[20.0]], [[30.0]], [[60.0]]], dtype=LD)
    value, sig = estimate_from_sums(s1, s1 * 0, 10)
    assert float(value[0, 0]) == 3 and abs(float(sig[0, 0]) - math.sqrt(14 / 12)) < 1e-15
    # R = 1: sqrt((<g^2> - <g>^2)/(N-1)) on g = (1,2,3,4): mean 2.5, <g^2> = 7.5 -> sqrt(1.25/3)
    value, sig = estimate_from_sums(np.array([[[10.0]]], dtype=LD), np.array([[[30.0]]], dtype=LD), 4)
    assert float(value[0, 0]) == 2.5 and abs(float(sig[0, 0]) - math.sqrt(1.25 / 3)) < 1e-15
    # sum the values, errors in mean square
    tot, sig = combine_sectors(np.array([[1.0, 2.0], [3.0, 4.0]]), np.array([[3.0, 0.0], [4.0, 1.0]]))
    assert list(tot) == [4.0, 6.0] and list(sig) == [5.0, 1.0]


def test_four_sigma_coverage_over_seeds():
    # the reported error must be an honest standard deviation: R = 8 shifts -> t_7 pulls
    nl = 1 << 9
    sec = SectorSpec([block(3, [], "p[x[1],2]*x[2]*p[1+x[3],-1]")])
    exact = (1 / 3) * (1 / 2) * math.log(2)
    pulls = []
    for seed in range(60):
        val, err = integrate_lattice(sec, 8 * nl, 8, _genvec(nl, 3), 3, seed)
        pulls.append((float(val[0, 0]) - exact) / float(err[0, 0]))
    pulls = np.array(pulls)
    assert np.sum(np.abs(pulls) > 4) <= 2
    assert 0.6 < np.sqrt(np.mean(pulls ** 2)) < 2.0            # t_7: sqrt(7/5) = 1.18


# ------------------------------------------------------------------ Vegas (R8)

def test_vegas_refine_flat_histogram_keeps_uniform_grid():
    grid = vegas_uniform_grid(1, 50)[0]
    new = vegas_refine(grid, np.full(50, LD(3.7)), 1.5)
    assert np.max(np.abs(new - grid)) < 1e-15
    assert new[0] == 0 and new[-1] == 1
    assert np.array_equal(vegas_refine(grid, np.zeros(50, dtype=LD), 1.5), grid)      # all-zero: unchanged


def test_vegas_refine_invariants_and_equalisation():
    rng = np.random.default_rng(9)
    grid = np.sort(np.concatenate([[0, 1], rng.uniform(0, 1, 49)])).astype(LD)
    hist = rng.uniform(0, 1, 50).astype(LD) ** 4
    hist[5] = 0
    new = vegas_refine(grid, hist, 1.5)
    assert new[0] == 0 and new[-1] == 1 and np.all(np.diff(new) > 0)
    assert abs(float(np.sum(np.diff(new))) - 1) < 1e-17
    # each new bin holds sum(m)/NB of the piecewise-constant density m_b/(width_b): brute-force check by
    # integrating that density over the new bins with fine quadrature in float64
    sm = np.empty(50)
    h = hist.astype(np.float64)
    sm[0], sm[-1] = (h[0] + h[1]) / 2, (h[-2] + h[-1]) / 2
    sm[1:-1] = (h[:-2] + h[1:-1] + h[2:]) / 3
    p = sm / sm.sum()
    m = ((1 - p) / -np.log(p)) ** 1.5
    dens = m / np.diff(grid.astype(np.float64))
    edges_old = grid.astype(np.float64)

    def mass(a, b):
        tot = 0.0
        for k in range(50):
            lo, hi = max(a, edges_old[k]), min(b, edges_old[k + 1])
            if hi > lo:
                tot += dens[k] * (hi - lo)
        return tot
    masses = [mass(float(new[i]), float(new[i + 1])) for i in range(50)]
    assert np.max(np.abs(np.array(masses) - m.sum() / 50)) < 1e-12


def test_vegas_constant_integrand_and_combination_rules():
    sec = SectorSpec([block(2, [], "1+0*x[1]")])
    tr = []
    val, sig, chi2, grid = integrate_vegas(sec, 1 << 11, SEED, nbins=16, iters=3, trace=tr)
    assert float(tr[0]["I"][0, 0]) == 1.0 and float(tr[0]["var"][0, 0]) == 0.0       # uniform 2^-4 grid: W = 1 exactly
    assert abs(float(val[0, 0]) - 1) <= 4 * float(sig[0, 0]) + 1e-15
    val, sig, chi2, grid = integrate_vegas(sec, 1 << 11, SEED, nbins=10, iters=3)    # 1/10 inexact: clamp at 0
    assert np.isfinite(float(sig[0, 0])) and float(sig[0, 0]) >= 0
    assert abs(float(val[0, 0]) - 1) <= 4 * float(sig[0, 0]) + 1e-12
    # hand numbers: I = (1, 3), var = (1, 4) -> value = (1 + 3/4)/(1 + 1/4) = 1.4, sigma^2 = 0.8, chi2 = 0.8
    v, s, c = vegas_combine(np.array([[1.0], [3.0]], dtype=LD), np.array([[1.0], [4.0]], dtype=LD))
    assert abs(float(v[0]) - 1.4) < 1e-15 and abs(float(s[0]) ** 2 - 0.8) < 1e-15 and abs(float(c[0]) - 0.8) < 1e-15
    # all-zero variances: plain mean, sigma 0; partly zero: those take the smallest positive variance
    v, s, c = vegas_combine(np.array([[1.0], [3.0]], dtype=LD), np.zeros((2, 1), dtype=LD))
    assert float(v[0]) == 2 and float(s[0]) == 0
    v, s, c = vegas_combine(np.array([[1.0], [3.0]], dtype=LD), np.array([[0.0], [4.0]], dtype=LD))
    assert float(v[0]) == 2 and abs(float(s[0]) ** 2 - 2) < 1e-15


def test_vegas_histogram_total_unbiasedness_and_adaptation():
    # separable f = prod (1-a) x_i^-a, a = 0.4: exact integral 1; ideal edges (b/NB)^(1/(1-a))
    a = 0.4
    sec = SectorSpec([block(2, [], f"{(1 - a) ** 2!r}*p[x[1],{-a}]*p[x[2],{-a}]")])
    tr = []
    val, sig, chi2, grid = integrate_vegas(sec, 1 << 13, SEED, nbins=50, iters=8, trace=tr)
    for rec in tr:
        for d in range(2):
            assert abs(float(np.sum(rec["hist"][d]) / rec["s2"][0, 0]) - 1) < 1e-15      # (iii): sum_b h = sum g^2
            assert rec["grid"][d][0] == 0 and rec["grid"][d][-1] == 1 and np.all(np.diff(rec["grid"][d]) > 0)
    assert abs(float(val[0, 0]) - 1) <= 4 * float(sig[0, 0])
    sig_it = [math.sqrt(float(r["var"][0, 0])) for r in tr]
    assert sig_it[-1] < 0.3 * sig_it[0]
    ideal = (np.arange(51) / 50) ** (1 / (1 - a))
    e0 = np.max(np.abs(tr[0]["grid"][0].astype(np.float64) - ideal))
    e1 = np.max(np.abs(grid[0].astype(np.float64) - ideal))
    assert e1 < 0.25 * e0
    # (iv) unbiased on the adapted grid: a polynomial lands within 4 sigma of its closed form
    sec2 = SectorSpec([block(2, [], "3*p[x[1],2]+x[2]")])
    val, sig, chi2, _ = integrate_vegas(sec2, 1 << 12, SEED + 1, nbins=20, iters=5)
    assert abs(float(val[0, 0]) - 1.5) <= 4 * float(sig[0, 0])


def test_magnitude_companion_bounds_the_value():
    prog = parse(block(2, ["1-x[1]+x[2]*0.5"], "l[f[1]]*(x[1]-x[2])/p[f[1],2.5]"))
    rng = np.random.default_rng(10)
    x = rng.uniform(0, 1, size=(200, 2))
    v, m = evaluate_with_magnitude(prog, x)
    assert np.all(m >= np.abs(v)) and np.all(v == evaluate(prog, x))
    # sign-definite input without real powers or logs: M = |f|
    prog = parse(block(2, ["1+x[1]+x[2]*0.5"], "x[1]*f[1]/p[f[1],3]+x[2]"))
    v, m = evaluate_with_magnitude(prog, x)
    assert np.max(np.abs(m / np.abs(v) - 1)) < 1e-17
    # a cancelling argument makes M large relative to |f|
    prog = parse(block(1, [], "(x[1]+1)-(x[1]+0.9999)"))
    v, m = evaluate_with_magnitude(prog, x[:, :1])
    assert np.all(m / np.abs(v) > 1e4)


def test_magnitude_companion_rules_on_hand_numbers():
    """The first-order rules of oracle/evaluate.py::_MagWalker on numbers worked by hand (R14)."""
    x = np.array([[0.25]], dtype=LD)
    # a = 1 - x = 0.75 with Ma = 1.25 (ra = 2/3);  b = x + 2 = 2.25, Mb = 2.25 (rb = 0)
    a, ma = 0.75, 1.25
    cases = {
        "(1-x[1])*(x[1]+2)": a * 2.25 * (1 + 2 / 3),
        "(1-x[1])/(x[1]+2)": a / 2.25 * (1 + 2 / 3),
        "(x[1]+2)/(1-x[1])": 2.25 / a * (1 + 2 / 3),
        "p[1-x[1],3]": a ** 3 * (1 + 3 * 2 / 3),
        "p[1-x[1],-2]": a ** -2 * (1 + 2 * 2 / 3),
        "p[1-x[1],-2.5]": a ** -2.5 * (1 + 2.5 * 2 / 3),
        "l[1-x[1]]": 1 + 2 / 3,                                   # |log 0.75| < 1: the clamp
        "l[p[1-x[1],20]]": abs(20 * math.log(0.75)) + 20 * 2 / 3,
        "(1-x[1])*(1-x[1])*(1-x[1])": a ** 3 * (1 + 3 * 2 / 3),   # products add the excesses
        "(1-x[1])-(x[1]+2)": ma + 2.25,
    }
    for text, want in cases.items():
        v, m = evaluate_with_magnitude(parse(block(1, [], text)), x)
        assert abs(float(m[0]) - want) < 1e-15 * want, (text, float(m[0]), want)
    # complex arguments: moduli
    z = np.array([[0.3 - 0.4j]], dtype=CLD)
    v, m = evaluate_with_magnitude(parse(block(1, [], "x[1]*x[1]-x[1]")), z, CLD)
    assert abs(float(m[0]) - (0.25 + 0.5)) < 1e-15


def test_magnitude_companion_is_sound_and_below_the_modulus_tree():
    """FP64 evaluation of the same tree differs from the long-double value by far less than 1e-12 M
    (soundness of the scale: the rounding unit is 1.1e-16), and M never exceeds R14's literal
    modulus tree for expressions without quotients of cancelling arguments."""
    rng = np.random.default_rng(12)
    x = rng.uniform(0.01, 0.99, size=(4000, 3))
    texts = ["(1-1.3*x[1]+x[2]*x[3])*(0.2-x[2]+x[1]*x[1])*l[1.01-x[3]]",
             "p[1-1.9*x[1]*x[2]+x[3],-2.5]*(x[1]-x[2])/(1+x[3])",
             "l[1+x[1]]*p[l[2-x[2]]-0.4,2]-p[x[3]-0.5,3]"]
    for t in texts:
        prog = parse(block(3, [], t))
        v, m = evaluate_with_magnitude(prog, x)
        d = evaluate(prog, x, np.float64)
        ok = np.isfinite(v.astype(float))
        assert ok.sum() > 3000
        assert np.all(m[ok] >= np.abs(v[ok]) * (1 - 1e-18))
        assert np.max(np.abs(d[ok] - v[ok].astype(float)) / m[ok].astype(float)) < 2e-14

    def modulus_tree(node, xs):                                 # R14 literally, for + - * and positive powers
        op = node[0]
        if op == "num":
            return np.full(xs.shape[0], abs(node[1]))
        if op == "x":
            return np.abs(xs[:, node[1] - 1])
        if op == "neg":
            return modulus_tree(node[1], xs)
        if op in ("add", "sub"):
            return modulus_tree(node[1], xs) + modulus_tree(node[2], xs)
        if op == "mul":
            return modulus_tree(node[1], xs) * modulus_tree(node[2], xs)
        if op == "pow":
            return modulus_tree(node[1], xs) ** int(node[2])
        raise ValueError(op)

    prog = parse(block(3, [], "(1-1.3*x[1]+x[2]*x[3])*p[0.2-x[2]+x[1]*x[1],3]-(x[1]-x[3])*(x[2]-0.5)"))
    v, m = evaluate_with_magnitude(prog, x)
    assert np.all(m.astype(float) <= modulus_tree(prog.final, x) * (1 + 1e-15))


def test_fp64_horner_of_phi_r_errs_by_its_condition_number():
    """DESIGN.md section 3 'Tolerances': the mirrored phi_r(v) = v^(r+1) sum_i c_i v^i, c_i =
    C binom(r,i) (-1)^i/(r+1+i), is an alternating sum; its FP64 Horner value differs from the exact
    one by about cond(v) = sum|c_i v^i| / |sum c_i v^i| rounding units, which is what sets the
    4e-15 (r <= 4) / 4e-14 (r = 5, 6) bars of the GPU transform test.  FP64 Horner restated here."""
    u64 = 2.0 ** -53
    v = np.concatenate([np.linspace(1e-6, 0.5, 20001), 0.5 - np.logspace(-12, -2, 2000)])
    for r in (3, 4, 5, 6):
        C = math.factorial(2 * r + 1) // math.factorial(r) ** 2
        coef = [C * math.comb(r, i) * (-1) ** i / (r + 1 + i) for i in range(r + 1)]
        poly = np.full_like(v, coef[r])
        for i in range(r - 1, -1, -1):
            poly = poly * v + coef[i]                                  # numpy float64: one rounding per operation
        exact = P._phi_small(v.astype(LD), r) / v.astype(LD) ** (r + 1)
        rel = np.abs(poly - exact.astype(float)) / np.abs(exact.astype(float))
        cond = sum(abs(c) * v ** i for i, c in enumerate(coef)) / np.abs(exact.astype(float))
        assert np.all(rel <= 2 * (r + 2) * u64 * cond)                 # the standard Horner bound
        assert cond.max() < {3: 13, 4: 33, 5: 90, 6: 250}[r]           # the condition numbers DESIGN.md quotes
        # the polynomial alone, before the v^(r+1) factor and 1 - p add their roundings: inside the bars
        assert rel.max() < (2.0e-15 if r <= 4 else 2.0e-14)
        # r = 5, 6 do need the wider bar: the polynomial's own error is already above 4e-15
        assert (rel.max() > 4e-15) == (r >= 5)


def test_testf_and_lambda_selection_closed_forms():
    """PAPER.md:474 (-testF), :404 (lambda tuned in (0, MaxComplexShift]); R19.  1-D closed forms:
    F = x - a:   F(z) = (x - a) - i lam x(1-x): Im F < 0 for every lam > 0, |F|^2 = (x-a)^2 + lam^2 s^2 grows
                 with lam, so the scan picks lambda_max;
    F = x^3 - a: z = x - i lam s 3x^2, Im F(z) = lam s g (lam^2 s^2 g^2 - 3 x^2), g = 3x^2, s = x(1-x): the
                 point x is bad exactly when lam s g >= sqrt(3) x, i.e. lam >= 1/(sqrt(3) x^2 (1-x))."""
    rng = np.random.default_rng(21)
    x = rng.uniform(0.02, 0.98, size=(4000, 1)).astype(LD)
    xs = x[:, 0]
    lin = parse(block(1, ["x[1]-0.3"], "1/f[1]"))
    for lam in (0.1, 0.5, 3.0):
        bad, mx, mn = oracle_test_f(lin, 1, lam, x)
        s = xs * (1 - xs)
        assert bad == 0
        assert abs(float(mx - np.max(-LD(lam) * s))) < 1e-18
        assert abs(float(mn - np.min(np.sqrt((xs - LD(0.3)) ** 2 + (LD(lam) * s) ** 2)))) < 1e-18
    lam, scan = select_lambda(lin, 1, x, lambda_max=2.0, lambda_split=4)
    assert float(lam) == 2.0 and [float(t[0]) for t in scan] == [0.5, 1.0, 1.5, 2.0] and all(t[1] == 0 for t in scan)
    assert float(select_lambda(lin, 1, x, 2.0, 4, conservative=True)[0]) == 1.0
    cub = parse(block(1, ["p[x[1],3]-0.2"], "1/f[1]"))
    thr = 1 / (np.sqrt(LD(3)) * xs ** 2 * (1 - xs))               # lam at which the point turns bad
    for lam in (1.0, 4.0, 6.0, 9.0):
        bad, mx, mn = oracle_test_f(cub, 1, lam, x)
        assert bad == int(np.sum(thr <= LD(lam)))
    assert oracle_test_f(cub, 1, 3.85, x)[0] == 0 and oracle_test_f(cub, 1, 4.0, x)[0] > 0    # min thr = 27/(4 sqrt 3) = 3.897.. at x = 2/3
    lam, scan = select_lambda(cub, 1, x, lambda_max=8.0, lambda_split=8)
    ok = [t for t in scan if t[1] == 0]
    assert [float(t[0]) for t in ok] == [1.0, 2.0, 3.0]            # the candidates below 3.897
    assert float(lam) == float(max(ok, key=lambda t: t[3])[0])
    none, scan = select_lambda(cub, 1, x, lambda_max=80.0, lambda_split=2)
    assert none is None and all(t[1] > 0 for t in scan)


# ------------------------------------------------------------------ multiple-precision walk (f1; R20)

def test_mp_walk_closed_forms_under_cancellation():
    """oracle/evaluate_mp.py against closed forms where the longdouble walk has no digit left."""
    from fractions import Fraction
    from oracle.evaluate_mp import evaluate_mp, to_double_double
    # ((1+x)^3 - 1 - 3x - 3x^2) / x^3 = 1 for every x != 0
    prog = parse(block(1, ["p[1+x[1],3]-1-3*x[1]-3*p[x[1],2]"], "f[1]/p[x[1],3]"))
    xs = np.array([[1e-9], [2.0 ** -20], [3.7e-7], [1e-12]])
    with mpmath.workdps(60):
        for v in evaluate_mp(prog, xs):
            assert abs(v - 1) < mpmath.mpf(10) ** -20          # numerator x^3 >= 1e-36, working precision 1e-60
    ld = evaluate(prog, xs[:1], LD)
    assert abs(float(ld[0]) - 1.0) > 1e-3                       # ... which is why the rescue exists
    # (log(1+x) - x + x^2/2) / x^3 = sum_{k>=3} (-1)^(k+1) x^(k-3) / k, summed exactly for x = 2^-30
    prog = parse(block(1, [], "(l[1+x[1]]-x[1]+p[x[1],2]/2)/p[x[1],3]"))
    x = Fraction(1, 1 << 30)
    series = sum(Fraction((-1) ** (k + 1), k) * x ** (k - 3) for k in range(3, 12))   # next term 2^-270/12
    with mpmath.workdps(60):
        v = evaluate_mp(prog, np.array([[float(x)]]))[0]
        ref = mpmath.mpf(series.numerator) / mpmath.mpf(series.denominator)
        assert abs(v - ref) < mpmath.mpf(10) ** -30             # numerator 2^-90/3 ~ 3e-28 at 1e-60: 32 digits
    # non-integer power and the (hi, lo) split
    prog = parse(block(2, [], "p[x[1]+x[2],-1.5]*x[1]"))
    with mpmath.workdps(60):
        v = evaluate_mp(prog, np.array([[0.25, 2.0]]))[0]
        assert abs(v - mpmath.mpf("0.25") / mpmath.mpf("2.25") ** mpmath.mpf("1.5")) < mpmath.mpf(10) ** -55
        hi, lo = to_double_double(v)
        assert hi == float(v) and abs(mpmath.mpf(hi) + mpmath.mpf(lo) - v) < mpmath.mpf(10) ** -31 * abs(v)


def test_mp_walk_agrees_with_longdouble_walk():
    """Well-conditioned points of generated sectors: the two walks are the same function."""
    from oracle.evaluate_mp import evaluate_mp
    from workloads import make_workload
    rng = np.random.default_rng(5)
    for name in ("C1", "C3"):
        wl = make_workload(name, nsectors=2, npoints=1 << 10)
        for s in wl.sectors:
            if s.is_complex:
                continue
            for text in s.texts:
                prog = parse(text)
                x = rng.uniform(0.05, 0.95, size=(4, prog.nvars))
                v, mag = evaluate_with_magnitude(prog, x, LD)
                with mpmath.workdps(60):
                    for j, r in enumerate(evaluate_mp(prog, x)):
                        assert abs(r - mpmath.mpf(float(v[j]))) <= 4e-16 * float(mag[j])      # float(v): one more rounding
                    # constants as their nearest doubles (the CUDA path's immediates): first order the same
                    for j, r in enumerate(evaluate_mp(prog, x, const64=True)):
                        assert abs(r - mpmath.mpf(float(v[j]))) <= 8e-16 * float(mag[j])


def test_mixed_mode_restores_closed_form():
    """integrand_values(small_x=...): int_0^1 int_0^1 ((1+x)^3-1-3x-3x^2)/x^3 (1+y) dx dy = 3/2.  The lattice rule's
    periodising transform puts points at x ~ 1e-12, where the numerator is rounding noise over x^3."""
    text = block(2, ["p[1+x[1],3]-1-3*x[1]-3*p[x[1],2]"], "f[1]/p[x[1],3]*(1+x[2])")
    sec = SectorSpec([text])
    nl = 1 << 10
    gv = P.korobov_genvec(korobov_a(nl, 2), nl, 2)
    s1, s2, _ = lattice_partial_sums(sec, nl, 4, gv, 3, 7, small_x=0.02)
    val, err = estimate_from_sums(s1, s2, nl)
    assert abs(float(val[0, 0]) - 1.5) < 1e-9 and float(err[0, 0]) < 1e-8
    s1, s2, _ = lattice_partial_sums(sec, nl, 4, gv, 3, 7)          # long double everywhere: lost
    val, err = estimate_from_sums(s1, s2, nl)
    assert abs(float(val[0, 0]) - 1.5) > 1.0
    # small_x below every coordinate: nothing is flagged, nothing changes
    a = mc_partial_sums(sec, 1 << 8, 3)
    b = mc_partial_sums(sec, 1 << 8, 3, small_x=1e-300)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


# ------------------------------------------------------------------ deterministic cubature (f4; R21)

def test_genz_malik_rule_degrees_of_exactness():
    """oracle/cubature.py: the degree-7 rule integrates every monomial of total degree <= 7 exactly over an
    arbitrary box, the embedded rule those of degree <= 5 -- which fixes every weight and node radius -- and
    neither goes one degree further."""
    from fractions import Fraction
    from oracle.cubature import genz_malik, rule_on_box
    rng = np.random.default_rng(12)
    for n in (2, 3, 5):
        off, w7, w5 = genz_malik(n)
        assert off.shape[0] == 1 + 4 * n + 2 * n * (n - 1) + 2 ** n
        assert abs(float(np.sum(w7)) - 1) < 1e-17 and abs(float(np.sum(w5)) - 1) < 1e-17
        c = np.array([Fraction(int(v), 64) for v in rng.integers(20, 44, size=n)])
        h = np.array([Fraction(int(v), 64) for v in rng.integers(2, 20, size=n)])

        def exact(a):       # prod_k int_{c-h}^{c+h} x^a dx
            out = Fraction(1)
            for k in range(n):
                out *= ((c[k] + h[k]) ** (a[k] + 1) - (c[k] - h[k]) ** (a[k] + 1)) / (a[k] + 1)
            return float(out)

        cf, hf = np.array([float(v) for v in c]), np.array([float(v) for v in h])
        worst7 = worst5 = 0.0
        for a in itertools.product(range(9), repeat=n):
            deg = sum(a)
            if deg > 8 or (n == 5 and deg > 6 and max(a) < 3 and rng.random() < 0.8):
                continue
            f = lambda x, a=a: np.prod(x ** np.array(a), axis=1)[None, :]
            i7, i5, _ = rule_on_box(f, cf, hf, (off, w7, w5))
            ex = exact(a)
            r7, r5 = abs(float(i7[0]) - ex) / ex, abs(float(i5[0]) - ex) / ex
            if deg <= 7:
                assert r7 < 1e-16, (n, a, r7)
            if deg <= 5:
                assert r5 < 1e-16, (n, a, r5)
            if deg == 8 and max(a) == 8:
                worst7 = max(worst7, r7)
            if deg == 6 and max(a) == 6:
                worst5 = max(worst5, r5)
        assert worst7 > 1e-8 and worst5 > 1e-8


def test_cubature_rounds_closed_forms_and_bookkeeping():
    from oracle.cubature import integrate_cubature, rule_on_box, sector_components
    # int_0^1 int_0^1 (1+x+y)^-2 = ln(4/3); a sector text through the oracle's evaluator
    sec = SectorSpec([block(2, ["1+x[1]+x[2]"], "p[f[1],-2]"), block(2, ["1+x[1]+x[2]"], "l[f[1]]")])
    f = sector_components(sec)
    total, err, neval, boxes = integrate_cubature(f, 2, epsrel=1e-10, maxeval=1 << 16, return_boxes=True)
    exact0 = math.log(4.0 / 3.0)
    exact1 = float(mpmath.quad(lambda x, y: mpmath.log(1 + x + y), [0, 1], [0, 1]))
    assert abs(float(total[0]) - exact0) <= float(err[0]) <= 1e-10 * exact0
    assert abs(float(total[1]) - exact1) <= float(err[1]) <= 1e-10 * exact1
    assert neval == 17 * (2 * len(boxes) - 1)                       # every split adds two boxes' worth and removes one box
    assert abs(sum(float(np.prod(2 * b["h"])) for b in boxes) - 1) < 1e-15          # the boxes tile the cube
    # maxeval is respected and reported honestly
    total2, err2, neval2, nb2 = integrate_cubature(f, 2, epsrel=1e-14, maxeval=2000)
    assert neval2 <= 2000 and float(err2[0]) > 1e-14 * exact0 and abs(float(total2[0]) - exact0) <= float(err2[0])
    # the split axis follows the fourth difference: a function of x2 alone is never cut along x1
    g = lambda x: (1 / (LD(0.05) + x[:, 1] ** 2))[None, :]
    _, _, d = rule_on_box(g, [0.5, 0.5], [0.5, 0.5])
    assert d[0] < 1e-16 * d[1] and d[1] > 0
    _, _, _, bx = integrate_cubature(g, 2, epsrel=1e-8, maxeval=1 << 15, return_boxes=True)
    assert len(bx) > 8 and all(float(b["h"][0]) == 0.5 for b in bx)
    # a peaked integrand: the boxes crowd around the peak (adaptivity), and the result is right
    peak = lambda x: (1 / (LD(1e-2) + (x[:, 0] - LD(0.3)) ** 2 + (x[:, 1] - LD(0.7)) ** 2))[None, :]
    tot, er, _, bx = integrate_cubature(peak, 2, epsrel=1e-7, maxeval=1 << 18, return_boxes=True)
    ref = float(mpmath.quad(lambda x, y: 1 / (mpmath.mpf("0.01") + (x - 0.3) ** 2 + (y - 0.7) ** 2), [0, 0.3, 1], [0, 0.7, 1]))
    assert abs(float(tot[0]) - ref) <= 10 * float(er[0]) and float(er[0]) <= 1e-7 * ref
    small = min(float(np.prod(2 * b["h"])) for b in bx)
    where = [b for b in bx if float(np.prod(2 * b["h"])) == small]
    assert all(abs(float(b["c"][0]) - 0.3) < 0.2 and abs(float(b["c"][1]) - 0.7) < 0.2 for b in where)


# ------------------------------------------------------------------ the paper's box example, end to end

def box_closed_form(S, T):
    """(1/(S T)) [4/eps^2 - 2 (ln S + ln T)/eps + 2 ln S ln T - 4 pi^2/3]: coefficients of eps^-2, eps^-1, eps^0."""
    return [4 / (S * T), -2 * (math.log(S) + math.log(T)) / (S * T), (2 * math.log(S) * math.log(T) - 4 * math.pi ** 2 / 3) / (S * T)]


def test_paper_box_example_end_to_end():
    """The massless on-shell box of PAPER.md:301-313 through a miniature front end (tests/sector_frontend.py:
    eq. (2), sector decomposition, pole subtraction, eps expansion -> 40 worker-grammar integrands of 1-3
    variables) and the oracle's lattice integrator: the numbers the paper prints, within the errors it prints,
    and the closed form they come from to 1e-9."""
    from sector_frontend import box_integrands
    g = golden("paper_box_example.txt")
    S, T = int(g["S"]), int(g["T"])
    terms = box_integrands(S, T)
    assert len(terms) == 40 and sorted({d for d, _, _ in terms}) == [1, 2, 3]
    tot, var = np.zeros(3), np.zeros(3)
    for sid, (d, texts, _) in enumerate(terms):
        nl = {1: 1 << 10, 2: 1 << 12, 3: 1 << 13}[d]
        gv = P.korobov_genvec(korobov_a(nl, d) if d > 1 else 1, nl, d)
        val, err = integrate_lattice(SectorSpec(texts, sid), 4 * nl, 4, gv, 3, SEED, rdtype=np.float64)
        tot += np.asarray(val[:, 0], dtype=float)
        var += np.asarray(err[:, 0], dtype=float) ** 2
    exact = box_closed_form(S, T)
    for k, key in enumerate(("eps_m2", "eps_m1", "eps_0")):
        assert abs(tot[k] - float(g[key])) <= 3 * float(g[key + "_err"]) + 0.5e-4, (key, tot[k])     # 0.5e-4: the printed digits
        assert abs(tot[k] - exact[k]) < 1e-9 and math.sqrt(var[k]) < 1e-9, (key, tot[k], exact[k])
    # other kinematics: the ln S ln T term
    terms = box_integrands(2, 5)
    tot = np.zeros(3)
    for sid, (d, texts, _) in enumerate(terms):
        nl = {1: 1 << 10, 2: 1 << 12, 3: 1 << 13}[d]
        gv = P.korobov_genvec(korobov_a(nl, d) if d > 1 else 1, nl, d)
        val, _ = integrate_lattice(SectorSpec(texts, sid), 4 * nl, 4, gv, 3, SEED, rdtype=np.float64)
        tot += np.asarray(val[:, 0], dtype=float)
    assert np.allclose(tot, box_closed_form(2, 5), rtol=0, atol=1e-9)


def triangle_closed_form(s, m2):
    """J(s) = int_simplex 1/(m2 - s x1 x2 - i0) above the threshold s > 4 m2: -(1/(2s)) [ln((1+b)/(1-b)) - i pi]^2,
    b = sqrt(1 - 4 m2/s) (the equal-mass scalar triangle with two light-like legs)."""
    b = math.sqrt(1 - 4 * m2 / s)
    return -(1 / (2 * s)) * (math.log((1 + b) / (1 - b)) - 1j * math.pi) ** 2


def test_physical_region_triangle_closed_form():
    """A Feynman integral in the physical region, where F changes sign inside the cube (what the contour deformation
    of PAPER.md:404 is for), in two dimensions: eq. (2) for the equal-mass triangle at s = 10 m^2, three primary
    sectors from tests/sector_frontend.py, the oracle's deformation (R11) with the deformation size chosen by its
    lambda scan (R19), against the closed form -- which is checked here, independently, by doing one integration
    analytically and the other with mpmath."""
    from sector_frontend import triangle_integrands
    s, m2 = 10, 1
    closed = triangle_closed_form(s, m2)

    def inner(x1):         # int_0^(1-x1) dx2 / (m2 - (s + i0) x1 x2) = -ln(1 - (s + i0) x1 (1-x1)/m2) / (s x1)
        a = 1 - mpmath.mpf(s) * x1 * (1 - x1) / m2
        return -(mpmath.log(abs(a)) - (1j * mpmath.pi if a < 0 else 0)) / (s * x1)

    b = math.sqrt(1 - 4 * m2 / s)
    ref = complex(mpmath.quad(inner, [0, (1 - b) / 2, (1 + b) / 2, 1]))
    assert abs(ref - closed) < 1e-14
    total = 0j
    nl = 1 << 13
    gv = P.korobov_genvec(korobov_a(nl, 2), nl, 2)
    for sid, (texts, fi) in enumerate(triangle_integrands(s, m2)):
        probe = SectorSpec(texts, sid, True, fi, 1.0)
        _, x = mc_points(probe, 5, (1 << 20) - 1, 0, 1000)
        lam, scan = select_lambda(probe.progs[0], fi, x, 1.0, 4)
        assert lam is not None and all(t[1] == 0 for t in scan)
        val, err = integrate_lattice(SectorSpec(texts, sid, True, fi, float(lam)), 4 * nl, 4, gv, 3, SEED)
        assert float(err[0, 0]) < 1e-10 and float(err[0, 1]) < 1e-10
        total += complex(float(val[0, 0]), float(val[0, 1]))
    assert abs(total - closed) < 1e-10
    # without the deformation the same integrand is not integrable on the real cube
    val, err = integrate_lattice(SectorSpec(triangle_integrands(s, m2)[0][0], 0, True, 2, 0.0), 4 * nl, 4, gv, 3, SEED)
    assert not float(err[0, 0]) < 1e-3
