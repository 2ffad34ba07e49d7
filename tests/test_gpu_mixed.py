"""GPU parity tests of the mixed-precision rescue (R20): the double-double walk
against the multiple-precision oracle walk, and the two-phase integration against the oracle's mixed
sums.  Run with `-m gpu` on the B200 box."""
import mpmath
import numpy as np
import pytest

from workloads import korobov_a, make_workload, SectorText
from oracle import integrate as OI
from oracle import points as OP
from oracle.evaluate import LD, evaluate_with_magnitude
from oracle.evaluate_mp import evaluate_mp
from oracle.parser import parse

from helpers import check_sums, genvec_of, record_margin, spec

pytestmark = pytest.mark.gpu

# (hi + lo) against the 60-digit walk: a double-double carries 2^-104 ~ 5e-32 per operation; the bar is
# 1e-30 * M(x) (M: the magnitude companion R14, which grows with the operations that cancel) for programs
# whose constants are exact in FP64, where the compiler's constant folding rounds nothing
TOL_DD = 1e-30


@pytest.fixture(scope="module")
def fb(lib):
    return lib


@pytest.fixture(scope="module")
def ctx(fb):
    c = fb.Context(0)
    yield c
    c.set_mixed(0.0)
    c.close()


def block(nvars, flines, final):
    return f"{nvars};\n{len(flines)};\n" + "".join(f + ";\n" for f in flines) + final + ";\n|"


CANCEL = block(2, ["p[1+x[1],3]-1-3*x[1]-3*p[x[1],2]"], "f[1]/p[x[1],3]*(1+x[2])")      # = 1 + x2
# The same with a second-order zero.  A double-double is 106 bits, not MPFR: it resolves the numerator down to
# ~1e-32, so the rescue holds while 1e-32 / x^2 stays small -- on the lattice rule's points (x ~ 35 u^4 down to
# ~1e-18 with weight ~ u^3) that is the case for this integrand and not for the cubic one above.
CANCEL2 = block(2, ["p[1+x[1],2]-1-2*x[1]"], "f[1]/p[x[1],2]*(1+x[2])")


def _dd_errors(ctx, text, x, const64=True):
    """max over points of |hi + lo - f_mp| / M, and of |f_double - f_mp| / M for comparison"""
    prog = ctx.compile([SectorText(sector_id=0, texts=[text])], x.shape[1])
    hi, lo = ctx.eval_points_dd(prog, 0, x)
    dbl = ctx.eval_points(prog, 0, x, tier=0).real[:, 0]
    prog.close()
    tree = parse(text)
    _, mag = evaluate_with_magnitude(tree, x, LD)
    worst_dd = worst_d = 0.0
    with mpmath.workdps(60):
        for j, ref in enumerate(evaluate_mp(tree, x, const64=const64)):
            m = mpmath.mpf(float(mag[j]))
            worst_dd = max(worst_dd, float(abs(mpmath.mpf(float(hi[j, 0])) + mpmath.mpf(float(lo[j, 0])) - ref) / m))
            if np.isfinite(dbl[j]):
                worst_d = max(worst_d, float(abs(mpmath.mpf(float(dbl[j])) - ref) / m))
    assert np.all(np.abs(lo[:, 0]) <= np.abs(hi[:, 0]) * 2.0 ** -52)     # a normalised pair
    return worst_dd, worst_d


@pytest.mark.parametrize("name,text,dim", [
    ("cubic cancellation", CANCEL, 2),
    ("log series", block(1, [], "(l[1+x[1]]-x[1]+p[x[1],2]/2)/p[x[1],3]"), 1),
    ("division, square root, powers", block(3, ["1+x[1]*x[2]+3*x[3]", "x[1]+2*x[2]*x[3]+x[1]*x[2]*x[3]"],
                                            "p[f[1],-1.5]*p[f[2],0.5]/(f[1]+f[2])+p[f[2],0.25]*l[f[1]]-p[f[1]/f[2],7]"), 3),
    ("exponent from a logarithm", block(2, ["x[1]+x[2]+0.5"], "p[f[1],-2.75]*l[f[1]]*l[f[1]]-1/f[1]+x[1]/(1+x[2])"), 2),
])
def test_dd_walk_against_multiple_precision(ctx, name, text, dim):
    rng = np.random.default_rng(3)
    x = rng.random((257, dim))
    x[:40] *= 10.0 ** -rng.uniform(1, 9, size=(40, 1))        # towards the faces, where the terms cancel
    x[40:48] = 2.0 ** -np.arange(10, 50, 5)[:, None]
    worst_dd, worst_d = _dd_errors(ctx, text, x)
    record_margin(f"dd walk: {name}", worst_dd_err_over_M=worst_dd, worst_double_err_over_M=worst_d)
    assert worst_dd <= TOL_DD
    assert worst_d > 1e4 * worst_dd      # the double walk of the same program is far from this bar


def test_dd_walk_on_generated_sectors(ctx):
    """The configurations' real sectors (Horner forms with S temporaries and shared-memory slots).  Their decimal
    coefficients pass through the compiler's FP64 constant folding, so here the bar is the FP64 one (4e-16 M);
    that every opcode of the ISA computes the right thing at full width is the previous test's business."""
    rng = np.random.default_rng(8)
    for name in ("C1", "C2", "C3", "C5"):
        wl = make_workload(name, nsectors=2, npoints=1 << 10)
        prog = ctx.compile(wl.sectors, wl.dim)
        x = rng.random((65, wl.dim))
        for si, s in enumerate(wl.sectors):
            hi, lo = ctx.eval_points_dd(prog, si, x)
            dbl = ctx.eval_points(prog, si, x, tier=0).real
            for k, text in enumerate(s.texts):
                tree = parse(text)
                _, mag = evaluate_with_magnitude(tree, x, LD)
                with mpmath.workdps(60):
                    for j, ref in enumerate(evaluate_mp(tree, x, const64=True)):
                        err = abs(mpmath.mpf(float(hi[j, k])) + mpmath.mpf(float(lo[j, k])) - ref)
                        assert err <= 4e-16 * float(mag[j]), (name, si, k, j)
                assert np.all(np.abs(hi[:, k] - dbl[:, k]) <= 1e-12 * mag)
        prog.close()


@pytest.mark.parametrize("tier", [None, 0])
@pytest.mark.parametrize("kind", ["lattice", "mc"])
def test_mixed_sums_against_oracle(fb, ctx, kind, tier):
    """Two-phase integration of an integrand that doubles cannot evaluate near x1 = 0: per-shift sums against the
    oracle's mixed sums (R15), the closed form 3/2, and -- with the mode off -- garbage.  (tier None: the default
    call, which keeps phase 1 on the interpreter while the mode is on.)"""
    if tier is None:
        tier = fb.TIER_ANY
    small_x = 0.02
    s = SectorText(sector_id=5, texts=[CANCEL2 if kind == "lattice" else CANCEL])
    prog = ctx.compile([s], 2)
    sec = spec(s)
    ctx.set_mixed(small_x)
    try:
        if kind == "lattice":
            nl = 1 << 12
            a = korobov_a(nl, 2)
            rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=4, korobov_a=a, periodize_r=3)
            gpu = ctx.partial_sums(prog, 4 * nl, rule, 77, tier=tier)[0]
            gv = OP.korobov_genvec(a, nl, 2)
            s1, s2, sa = OI.lattice_partial_sums(sec, nl, 4, gv, 3, 77, small_x=small_x)
            check_sums(gpu, s1, s2, sa, label=f"mixed lattice sums tier {tier}")
            res = ctx.integrate(prog, 4 * nl, rule, 77, tier=tier)[0]
            assert abs(res["re"][0] - 1.5) <= max(4 * res["re_err"][0], 1e-12) and res["n_nonfinite"][0] == 0
            ctx.set_mixed(0.0)
            off = ctx.partial_sums(prog, 4 * nl, rule, 77, tier=tier)[0]
            assert not np.all(np.abs(off[..., 0] - np.asarray(s1, dtype=float)) <= 1e-6 * np.abs(np.asarray(s1, dtype=float)))
        else:
            npts = 10007
            rule = fb.Rule(kind=fb.RULE_MC)
            gpu = ctx.partial_sums(prog, npts, rule, 78, tier=tier)[0, 0]
            s1, s2 = OI.mc_partial_sums(sec, npts, 78, small_x=small_x)
            assert np.allclose(gpu[..., 0], np.asarray(s1, dtype=float), rtol=1e-10)
            assert np.allclose(gpu[..., 1], np.asarray(s2, dtype=float), rtol=1e-10)
    finally:
        ctx.set_mixed(0.0)
        prog.close()


def test_mixed_vegas_iteration_against_oracle(fb, ctx):
    """Vegas with the rescue on: one iteration on a given uneven grid -- sums and the g^2 histogram, bin by bin, against
    the oracle's mixed iteration -- and a full run that reaches the closed form 3/2."""
    small_x = 0.02
    s = SectorText(sector_id=6, texts=[CANCEL])
    prog = ctx.compile([s], 2)
    sec = spec(s)
    rule = fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=16, vegas_iters=5, vegas_alpha=1.5)
    rng = np.random.default_rng(4)
    w = rng.random((2, 16)).astype(LD) ** 2 + LD(1e-2)
    grid = np.concatenate([np.zeros((2, 1), dtype=LD), np.cumsum(w, axis=1) / np.sum(w, axis=1)[:, None]], axis=1)
    grid[:, -1] = 1
    gridf = grid.astype(np.float64)
    npts = 6007
    ctx.set_mixed(small_x)
    try:
        s1, s2, hist = OI.vegas_iteration_sums(sec, gridf.astype(LD), npts, 21, 2, small_x=small_x)
        sums, h = ctx.vegas_iteration(prog, 0, npts, rule, 21, 2, gridf)
        assert np.allclose(sums[..., 0], s1.astype(float), rtol=1e-10)
        assert np.allclose(sums[..., 1], s2.astype(float), rtol=1e-10)
        hf = hist.astype(float)
        assert np.allclose(h, hf, rtol=1e-10, atol=1e-13 * hf.max())
        assert np.allclose(h.sum(axis=1), sums[0, 0, 1], rtol=1e-12)
        res = ctx.integrate(prog, 20000, rule, 22)[0]
        assert abs(res["re"][0] - 1.5) <= 4 * res["re_err"][0] and res["re_err"][0] < 0.01 and res["n_nonfinite"][0] == 0
    finally:
        ctx.set_mixed(0.0)
        prog.close()


def test_mixed_mode_with_nothing_flagged_is_bit_identical(fb, ctx):
    """small_x below every coordinate: phase 2 finds no point, the sums are the bits of the plain run; and
    small_x > 1 (every point through the double-double walk, the paper's -mpfr) agrees to FP64 accuracy."""
    wl = make_workload("C3", nsectors=3, npoints=1 << 15, n_shifts=8)
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    plain = ctx.partial_sums(prog, wl.npoints, rule, wl.seed)
    try:
        ctx.set_mixed(1e-300)
        assert np.array_equal(ctx.partial_sums(prog, wl.npoints, rule, wl.seed), plain)
        # R15's bar between two runs: sum|g| <= sqrt(N S2) (Cauchy-Schwarz) stands in for the oracle's sum|g|
        bound = 1e-10 * np.abs(plain) + 1e-13 * np.sqrt(wl.n_lattice * plain[..., 1:2])
        ctx.set_mixed(2.0)
        every = ctx.partial_sums(prog, wl.npoints, rule, wl.seed)
        assert np.all(np.abs(every - plain) <= bound) and not np.array_equal(every, plain)
        ctx.set_mixed(1e-3)
        some = ctx.partial_sums(prog, wl.npoints, rule, wl.seed)
        assert np.all(np.abs(some - plain) <= bound)
        assert np.array_equal(ctx.partial_sums(prog, wl.npoints, rule, wl.seed, tier=0), some)
        with pytest.raises(fb.FiestaError):      # the native kernels carry no mask: phase 1 is the interpreter's
            ctx.partial_sums(prog, wl.npoints, rule, wl.seed, tier=1)
    finally:
        ctx.set_mixed(0.0)
        prog.close()


def test_mixed_mode_refuses_what_it_does_not_cover(fb, ctx):
    wl = make_workload("C4", nsectors=1, npoints=1 << 12)
    prog = ctx.compile(wl.sectors, wl.dim)
    ctx.set_mixed(1e-3)
    try:
        with pytest.raises(fb.FiestaError):
            ctx.partial_sums(prog, wl.npoints, fb.Rule.from_workload(wl), wl.seed)      # complex sector: not covered
        with pytest.raises(fb.FiestaError):
            ctx.eval_points_dd(prog, 0, np.full((1, wl.dim), 0.5))
        with pytest.raises(fb.FiestaError):
            ctx.set_mixed(-1.0)
    finally:
        ctx.set_mixed(0.0)
        prog.close()
