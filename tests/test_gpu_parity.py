"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element
on the same seeded inputs.  Run with `-m gpu` on the B200 box.

Bars (BASELINE.json north_star; readings R14/R15 in DESIGN.md):
  integers t (points)         bit-exact
  per-point values            |diff| <= 1e-12 * M(x)
  per-shift sums              |diff| <= 1e-10 |S| + 1e-13 sum|g|
  closed forms                within 4 sigma of the reported error
"""
import numpy as np
import pytest

from workloads import make_workload, SectorText
from oracle import integrate as OI
from oracle import points as OP
from oracle.integrate import SectorSpec

from helpers import (LD, TOL_POINT, check_points, check_sums, genvec_of, oracle_values_and_magnitude, record_margin,
                     spec)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fb(lib):
    return lib


@pytest.fixture(scope="module")
def ctx(fb):
    c = fb.Context(0)
    yield c
    c.close()


def block(nvars, flines, final):
    return f"{nvars};\n{len(flines)};\n" + "".join(f + ";\n" for f in flines) + final + ";\n|"


def one_sector(texts, **kw):
    return SectorText(sector_id=kw.pop("sector_id", 0), texts=texts, **kw)


# ------------------------------------------------------------------------------ A1: points

@pytest.mark.parametrize("m,dim,first,count", [(13, 4, 0, 1000), (16, 4, 65000, 536), (21, 8, 12345, 777),
                                               (1, 1, 0, 2), (40, 12, (1 << 40) - 300, 300), (0, 3, 0, 1)])
def test_lattice_integers_bit_exact(fb, ctx, m, dim, first, count):
    n_l = 1 << m
    a = (0x9E3779B97F4A7C15 % n_l) | 1 if m > 0 else 1
    rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=3, korobov_a=a)
    gv = OP.korobov_genvec(a % n_l if m > 0 else 0, n_l, dim) if m > 0 else [0] * dim
    if m == 0:
        rule.genvec = gv
    for r in (0, 2):
        t = ctx.generate_points(rule, 20151111, 7, r, n_l, first, count, dim)
        delta = OP.lattice_shift(20151111, 7, r, dim)
        ref = OP.lattice_t(np.arange(first, first + count, dtype=np.uint64), gv, n_l, delta)
        assert np.array_equal(t, ref)


@pytest.mark.parametrize("dim,first,count,it", [(1, 0, 100, 0), (7, (1 << 33) + 5, 1001, 3), (12, 0, 513, 1048575)])
def test_philox_integers_bit_exact(fb, ctx, dim, first, count, it):
    rule = fb.Rule(kind=fb.RULE_MC)
    seed = 0xDEADBEEF12345678
    t = ctx.generate_points(rule, seed, 123456, it, 0, first, count, dim)
    ref = OP.philox_t(seed, 123456, OP.TAG_MC, it, np.arange(first, first + count, dtype=np.uint64), dim)
    assert np.array_equal(t, ref)


@pytest.mark.parametrize("r", [0, 1, 2, 3, 4, 5, 6])
def test_periodising_transform(fb, ctx, r):
    rng = np.random.default_rng(r)
    t = rng.integers(0, 1 << 63, size=(4001, 5), dtype=np.uint64) * np.uint64(2) + np.uint64(1)
    # the faces: u -> 0 and u -> 1
    t[0, :] = 0
    t[1, :] = np.uint64(0xFFFFFFFFFFFFFFFF)
    t[2, :] = np.uint64(1) << np.uint64(63)
    rule = fb.Rule(kind=fb.RULE_LATTICE, periodize_r=r)
    x, xbar, w = ctx.transform_points(rule, t)
    xo, xbo, wo = OP.korobov_transform(OP.unit_from_t(t), r)
    wo = np.prod(wo, axis=1)
    # x and 1-x each carry full relative accuracy at both faces (R4).  The alternating sum of
    # phi_r at v -> 1/2 has condition number ~12 (r=3) .. ~240 (r=6): DESIGN.md "Tolerances".
    tol = 4e-15 if r <= 4 else 4e-14
    assert np.max(np.abs(x - xo.astype(float)) / xo.astype(float)) < tol
    assert np.max(np.abs(xbar - xbo.astype(float)) / xbo.astype(float)) < tol
    ok = wo.astype(float) > 1e-290          # u = 2^-53 underflows FP64 for r >= 5
    assert np.max(np.abs(w[ok] - wo[ok].astype(float)) / wo[ok].astype(float)) < 2e-14


def test_mc_transform_is_identity(fb, ctx):
    rng = np.random.default_rng(5)
    t = rng.integers(0, 1 << 63, size=(100, 3), dtype=np.uint64)
    x, xbar, w = ctx.transform_points(fb.Rule(kind=fb.RULE_MC), t)
    assert np.array_equal(x, OP.unit_from_t(t).astype(float))
    assert np.all(w == 1.0)


# ------------------------------------------------------------------------------ A5: program walk

def _eval_case(ctx, wl, nsec, npts, seed, label=None, tier=None):
    prog = ctx.compile(wl.sectors, wl.dim)
    rng = np.random.default_rng(seed)
    x = rng.random((npts, wl.dim))
    # points near the faces of the cube, where the integrands vary fastest
    if npts > wl.dim:
        x[: wl.dim] = 0.5
        for k in range(wl.dim):
            x[k, k] = 1e-9
    worst = 0.0
    for si in range(nsec):
        got = ctx.eval_points(prog, si, x, tier=tier)
        if tier is not None:
            assert ctx.last_tiers() == ((1, 0) if tier == 1 else (0, 1))
        ref, mag = oracle_values_and_magnitude(spec(wl.sectors[si]), x)
        worst = max(worst, check_points(got, ref, mag, label=None if label is None else f"{label} sector {si}"))
    prog.close()
    return worst


@pytest.mark.parametrize("tier", [1, 0])
@pytest.mark.parametrize("name,nsec,npts", [("C1", 1, 2000), ("C2", 6, 1537), ("C3", 4, 1025), ("C4", 4, 700),
                                            ("C5", 4, 999)])
def test_per_point_parity_configs(ctx, name, nsec, npts, tier):
    """Per-point values of every configuration against the oracle, 1e-12 * M (R14), on BOTH forms of the
    program: tier 1 = the native kernel (the generated program body the benchmarked integration kernels
    are assembled from, in the eval kernel), tier 0 = the interpreter."""
    wl = make_workload(name, nsectors=nsec, npoints=1 << 12)
    label = f"per-point {name} {'native' if tier else 'interpreter'}"
    assert _eval_case(ctx, wl, nsec, npts, 11, label=label, tier=tier) <= 1.0


@pytest.mark.parametrize("npts", [1, 3, 511, 512, 513])
def test_per_point_ragged_counts(ctx, npts):
    wl = make_workload("C2", nsectors=1, npoints=1 << 12)
    assert _eval_case(ctx, wl, 1, npts, npts, tier=1) <= 1.0
    assert _eval_case(ctx, wl, 1, npts, npts, tier=0) <= 1.0
    wl = make_workload("C4", nsectors=1, npoints=1 << 12)
    assert _eval_case(ctx, wl, 1, npts, npts, tier=1) <= 1.0


def test_eval_zero_points(ctx):
    wl = make_workload("C1", nsectors=1, npoints=1 << 12)
    prog = ctx.compile(wl.sectors, wl.dim)
    assert ctx.eval_points(prog, 0, np.zeros((0, wl.dim))).shape == (0, 3)


# ------------------------------------------------------------------------------ A6/A7: sums

@pytest.mark.parametrize("name,nsec,npts,nsh", [("C1", 1, 1 << 16, 1), ("C1", 1, 1 << 16, 8), ("C2", 3, 1 << 15, 1),
                                                ("C3", 2, 1 << 15, 8), ("C4", 2, 1 << 14, 1), ("C4", 2, 1 << 14, 4)])
def test_lattice_partial_sums_parity(fb, ctx, name, nsec, npts, nsh):
    wl = make_workload(name, nsectors=nsec, npoints=npts, n_shifts=nsh)
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    gpu = ctx.partial_sums(prog, wl.npoints, rule, wl.seed)
    gv = genvec_of(wl)
    for si in range(nsec):
        s1, s2, sa = OI.lattice_partial_sums(spec(wl.sectors[si]), wl.n_lattice, wl.n_shifts, gv, wl.periodize_r, wl.seed)
        check_sums(gpu[si], s1, s2, sa)
    # the estimator (R5) on the device against the oracle's, from the oracle's own sums
    res = ctx.integrate(prog, wl.npoints, rule, wl.seed)
    for si in range(nsec):
        val, sig = OI.integrate_lattice(spec(wl.sectors[si]), wl.npoints, wl.n_shifts, gv, wl.periodize_r, wl.seed)[:2]
        val, sig = np.asarray(val, dtype=float), np.asarray(sig, dtype=float)
        assert np.allclose(res[si]["re"], val[:, 0], rtol=1e-9, atol=1e-13 * np.abs(val).max())
        assert np.allclose(res[si]["re_err"], sig[:, 0], rtol=1e-5, atol=1e-12 * np.abs(val).max())
        if val.shape[1] == 2:
            assert np.allclose(res[si]["im"], val[:, 1], rtol=1e-9, atol=1e-13 * np.abs(val).max())
            assert np.allclose(res[si]["im_err"], sig[:, 1], rtol=1e-5, atol=1e-12 * np.abs(val).max())
        assert np.all(res[si]["neval"] == wl.npoints) and np.all(res[si]["n_nonfinite"] == 0)


@pytest.mark.parametrize("name,nsec,npts,nsh", [("C1", 1, 1 << 16, 8), ("C2", 3, 1 << 15, 1), ("C3", 2, 1 << 15, 8),
                                                ("C5", 2, 1 << 13, 2), ("C3", 1, 64, 1), ("C2", 2, 8 * 256, 8),
                                                ("C4", 2, 1 << 13, 2)])
def test_native_and_interpreter_tiers_agree_bitwise(fb, ctx, name, nsec, npts, nsh):
    """fiesta_compile's two forms of a sector's program (interpreted fx_ins walk; the same sequence
    assembled to a native kernel) do the same operations in the same order: every partial sum and
    every result is bit-identical, and the interpreter tier on its own meets the oracle.  This is
    what lets fiesta_integrate serve a sector with whichever form is ready."""
    wl = make_workload(name, nsectors=nsec, npoints=npts, n_shifts=nsh)
    rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=nsh, korobov_a=wl.korobov_a if wl.rule == fb.RULE_LATTICE else 1129,
                   periodize_r=3)
    prog = ctx.compile(wl.sectors, wl.dim)
    a = ctx.partial_sums(prog, npts, rule, wl.seed, tier=fb.TIER_INTERPRETER)
    assert ctx.last_tiers() == (0, nsec)
    b = ctx.partial_sums(prog, npts, rule, wl.seed, tier=fb.TIER_NATIVE)
    assert ctx.last_tiers() == (nsec, 0)
    for si in range(nsec):
        ok, info = prog.native(si, fb.RULE_LATTICE)
        assert ok and "Used" in info, info
    assert a.tobytes() == b.tobytes()
    ra = ctx.integrate(prog, npts, rule, wl.seed, tier=fb.TIER_INTERPRETER)
    rb = ctx.integrate(prog, npts, rule, wl.seed, tier=fb.TIER_NATIVE)
    assert ra.tobytes() == rb.tobytes()
    assert ctx.integrate(prog, npts, rule, wl.seed).tobytes() == ra.tobytes()      # whichever is ready
    gv = OP.korobov_genvec(rule.korobov_a, npts // nsh, wl.dim)
    s1, s2, sa = OI.lattice_partial_sums(spec(wl.sectors[0]), npts // nsh, nsh, gv, 3, wl.seed)
    check_sums(a[0], s1, s2, sa)
    # a selection that mixes the order, and a sector list of one
    sel = list(range(nsec))[::-1]
    assert ctx.partial_sums(prog, npts, rule, wl.seed, sectors=sel, tier=fb.TIER_NATIVE).tobytes() == a[sel].tobytes()
    # plain MC and one Vegas iteration: the other two native kernels of the same sectors
    mc = fb.Rule(kind=fb.RULE_MC)
    a = ctx.partial_sums(prog, 5000, mc, 3, tier=fb.TIER_INTERPRETER)
    b = ctx.partial_sums(prog, 5000, mc, 3, tier=fb.TIER_NATIVE)
    assert ctx.last_tiers() == (nsec, 0) and a.tobytes() == b.tobytes()
    vr = fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=37, vegas_iters=1)
    grid = np.sort(np.random.default_rng(1).random((wl.dim, 38)), axis=1)
    grid[:, 0], grid[:, -1] = 0.0, 1.0
    sa_, ha = ctx.vegas_iteration(prog, nsec - 1, 3001, vr, 9, 2, grid, tier=fb.TIER_INTERPRETER)
    sb_, hb = ctx.vegas_iteration(prog, nsec - 1, 3001, vr, 9, 2, grid, tier=fb.TIER_NATIVE)
    assert ctx.last_tiers() == (1, 0)
    assert sa_.tobytes() == sb_.tobytes() and ha.tobytes() == hb.tobytes()
    # a full Vegas run is reproducible bit for bit, on either tier (no atomics anywhere in the histogram)
    vr3 = fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=20, vegas_iters=3)
    r1 = ctx.integrate(prog, 4096, vr3, 5, tier=fb.TIER_INTERPRETER, allow_nonfinite=True)
    r2 = ctx.integrate(prog, 4096, vr3, 5, tier=fb.TIER_NATIVE, allow_nonfinite=True)
    r3 = ctx.integrate(prog, 4096, vr3, 5, tier=fb.TIER_NATIVE, allow_nonfinite=True)
    assert r1.tobytes() == r2.tobytes() == r3.tobytes()


def test_first_call_mixes_tiers_with_identical_bits(fb, ctx):
    """fiesta_compile returns before the native kernels exist; the first fiesta_integrate serves every sector
    with whichever form is ready at its launch (the integrand is transformed once, then evaluated).
    Whatever the split was, the results are the bits of an all-native and of an all-interpreter pass."""
    wl = make_workload("C3", nsectors=48, npoints=1 << 16)
    rule = fb.Rule.from_workload(wl)
    prog = ctx.compile(wl.sectors, wl.dim)
    first = ctx.integrate(prog, wl.npoints, rule, wl.seed)           # no waiting
    n_nat, n_int = ctx.last_tiers()
    assert n_nat + n_int == 48
    assert prog.wait_native() == 48
    st = prog.native_stats()
    assert st["assembled"] + st["cache_hits"] >= 48 and st["threads"] >= 1
    allnat = ctx.integrate(prog, wl.npoints, rule, wl.seed)
    assert ctx.last_tiers() == (48, 0)
    interp = ctx.integrate(prog, wl.npoints, rule, wl.seed, tier=fb.TIER_INTERPRETER)
    assert first.tobytes() == allnat.tobytes() == interp.tobytes()
    # the same texts again: the kernels come from the cache (keyed by the program, not the sector id)
    prog2 = ctx.compile(wl.sectors[:8], wl.dim)
    assert prog2.wait_native() == 8 and prog2.native_stats()["cache_hits"] == 8


def test_native_tier_is_off_with_fiesta_jit_0(fb, ctx, monkeypatch):
    wl = make_workload("C2", nsectors=2, npoints=1 << 12)
    monkeypatch.setenv("FIESTA_JIT", "0")
    prog = ctx.compile(wl.sectors, wl.dim)
    monkeypatch.delenv("FIESTA_JIT")
    assert prog.wait_native() == 0 and prog.native(0) == (False, "")
    rule = fb.Rule.from_workload(wl)
    ctx.integrate(prog, wl.npoints, rule, wl.seed)
    assert ctx.last_tiers() == (0, 2)
    with pytest.raises(fb.FiestaError):
        ctx.eval_points(prog, 0, np.full((3, wl.dim), 0.5), tier=fb.TIER_NATIVE)


def test_mixed_real_and_complex_call(fb, ctx):
    """One fiesta_integrate call over real and complex sectors (same K): each kind on its own kernels,
    results in selection order, equal to the separate calls, on every tier."""
    wr = make_workload("C2", nsectors=2, npoints=1 << 12)           # dim 6, K = 4, real
    s = wr.sectors[1]
    cplx = SectorText(77, s.texts, is_complex=True, deform_f_index=2, lam=0.3)
    prog = ctx.compile([wr.sectors[0], cplx, wr.sectors[1]], wr.dim)
    rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=2, korobov_a=wr.korobov_a, periodize_r=3)
    for tier in (fb.TIER_INTERPRETER, fb.TIER_NATIVE, None):
        res = ctx.integrate(prog, 1 << 12, rule, 5, tier=tier)
        for i in range(3):
            one = ctx.integrate(prog, 1 << 12, rule, 5, sectors=[i], tier=tier)
            assert one.tobytes() == res[i:i + 1].tobytes()
        assert np.all(res[0]["im"] == 0) and np.all(res[2]["im"] == 0) and np.all(res[1]["im_err"] > 0)
    sec = SectorSpec(cplx.texts, 77, True, 2, 0.3)
    gv = OP.korobov_genvec(wr.korobov_a, 1 << 11, wr.dim)
    val, sig = OI.integrate_lattice(sec, 1 << 12, 2, gv, 3, 5)
    assert np.allclose(res[1]["re"], np.asarray(val, dtype=float)[:, 0], rtol=1e-9)
    assert np.allclose(res[1]["im"], np.asarray(val, dtype=float)[:, 1], rtol=1e-9, atol=1e-12 * np.abs(np.asarray(val, dtype=float)).max())


def test_sector_selection_and_order(fb, ctx):
    """sectors=[2,0] integrates those two, in that order, with streams keyed by sector_id."""
    wl = make_workload("C2", nsectors=3, npoints=1 << 12)
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    full = ctx.partial_sums(prog, wl.npoints, rule, wl.seed)
    sub = ctx.partial_sums(prog, wl.npoints, rule, wl.seed, sectors=[2, 0])
    assert np.allclose(sub[0], full[2], rtol=1e-13) and np.allclose(sub[1], full[0], rtol=1e-13)


@pytest.mark.parametrize("npts", [2, 10007, (1 << 17) + 3])
def test_mc_sums_ragged(fb, ctx, npts):
    """Plain MC (Philox) with point counts that are not multiples of the block's work quantum."""
    wl = make_workload("C1", nsectors=1, npoints=1 << 12)
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule(kind=fb.RULE_MC)
    sec = spec(wl.sectors[0])
    gpu = ctx.partial_sums(prog, npts, rule, 99)[0, 0]          # [K,1,2]
    s1 = np.zeros((sec.K, 1), dtype=LD)
    s2 = np.zeros((sec.K, 1), dtype=LD)
    for first in range(0, npts, 1 << 14):
        cnt = min(1 << 14, npts - first)
        _, x = OI.mc_points(sec, 99, 0, first, cnt)
        v = OI.integrand_values(sec, x)
        s1[:, 0] += np.sum(v, axis=1)
        s2[:, 0] += np.sum(v * v, axis=1)
    assert np.allclose(gpu[..., 0], s1.astype(float), rtol=1e-10)
    assert np.allclose(gpu[..., 1], s2.astype(float), rtol=1e-10)
    val, sig = OI.integrate_mc(sec, npts, 99)[:2]
    res = ctx.integrate(prog, npts, rule, 99)[0]
    assert np.allclose(res["re"], np.asarray(val, dtype=float)[:, 0], rtol=1e-9)
    assert np.allclose(res["re_err"], np.asarray(sig, dtype=float)[:, 0], rtol=1e-5)


def _mc_oracle(sec, npts, seed, it=0, first=0, count=None):
    s1, s2 = OI.mc_partial_sums(sec, npts, seed, it, first=first, count=count)
    return np.asarray(s1, dtype=float), np.asarray(s2, dtype=float)


@pytest.mark.parametrize("tier", [1, 0])
def test_complex_mc_and_vegas_stepwise(fb, ctx, tier):
    """fx_integrate_cplx<MC>, <Vegas> and their native kernels on a deformed C4 sector:
    plain-MC sums against the oracle, one Vegas iteration on an uneven grid (sums and the f^2 histogram, which
    takes |g|^2 = Re^2 + Im^2 summed over the orders), and the estimates of a short complex Vegas run."""
    wl = make_workload("C4", nsectors=2, npoints=1 << 12)
    prog = ctx.compile(wl.sectors, wl.dim)
    sec = spec(wl.sectors[1])
    npts = 6001
    gpu = ctx.partial_sums(prog, npts, fb.Rule(kind=fb.RULE_MC), 17, sectors=[1], tier=tier)[0, 0]     # [K, 2, 2]
    s1, s2 = _mc_oracle(sec, npts, 17)
    scale = np.abs(s1).max()
    assert np.all(np.abs(gpu[..., 0] - s1) <= 1e-10 * np.abs(s1) + 1e-13 * npts * scale)
    assert np.allclose(gpu[..., 1], s2, rtol=1e-10)
    val, sig = OI.integrate_mc(sec, npts, 17)[:2]
    res = ctx.integrate(prog, npts, fb.Rule(kind=fb.RULE_MC), 17, sectors=[1], tier=tier)[0]
    assert np.allclose(res["re"], np.asarray(val, dtype=float)[:, 0], rtol=1e-9, atol=1e-13 * scale)
    assert np.allclose(res["im"], np.asarray(val, dtype=float)[:, 1], rtol=1e-9, atol=1e-13 * scale)
    assert np.allclose(res["im_err"], np.asarray(sig, dtype=float)[:, 1], rtol=1e-5)
    rule = fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=24, vegas_iters=3)
    w = np.random.default_rng(3).random((wl.dim, 24)).astype(LD) ** 2 + LD(1e-2)
    grid = np.concatenate([np.zeros((wl.dim, 1), dtype=LD), np.cumsum(w, axis=1) / np.sum(w, axis=1)[:, None]], axis=1)
    grid[:, -1] = 1
    gridf = grid.astype(np.float64)
    s1, s2, hist = OI.vegas_iteration_sums(sec, gridf.astype(LD), 5003, 23, 4)
    sums, h = ctx.vegas_iteration(prog, 1, 5003, rule, 23, 4, gridf, tier=tier)
    s1f, s2f, hf = s1.astype(float), s2.astype(float), hist.astype(float)
    assert np.all(np.abs(sums[..., 0] - s1f) <= 1e-10 * np.abs(s1f) + 1e-13 * 5003 * np.abs(s1f).max())
    assert np.allclose(sums[..., 1], s2f, rtol=1e-10)
    assert np.allclose(h, hf, rtol=1e-10, atol=1e-14 * hf.max())
    assert np.allclose(h.sum(axis=1), sums[..., 1].sum(), rtol=1e-12)          # every dimension: sum over all |g|^2
    val, sig, chi2, g_or = OI.integrate_vegas(sec, 4096, 29, 24, 3, 1.5)
    res = ctx.integrate(prog, 4096, rule, 29, sectors=[1], tier=tier)[0]
    g, _ = ctx.vegas_grid(0, wl.dim, 24)
    assert np.max(np.abs(g - g_or.astype(float))) < 1e-11
    vf, sf = np.asarray(val, dtype=float), np.asarray(sig, dtype=float)
    assert np.allclose(res["re"], vf[:, 0], rtol=1e-9, atol=1e-12 * np.abs(vf).max())
    assert np.allclose(res["im"], vf[:, 1], rtol=1e-9, atol=1e-12 * np.abs(vf).max())
    assert np.allclose(res["re_err"], sf[:, 0], rtol=1e-6) and np.allclose(res["im_err"], sf[:, 1], rtol=1e-6)


@pytest.mark.parametrize("tier", [1, 0])
def test_vegas_with_three_orders(fb, ctx, tier):
    """Vegas on a K = 3 sector (C1): one grid per sector shared by its orders, histogram = sum over orders of g^2."""
    wl = make_workload("C1", nsectors=1, npoints=1 << 12)
    prog = ctx.compile(wl.sectors, wl.dim)
    sec = spec(wl.sectors[0])
    rule = fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=50, vegas_iters=4)
    grid = OI.vegas_uniform_grid(wl.dim, 50)
    s1, s2, hist = OI.vegas_iteration_sums(sec, grid, 7001, 31, 1)
    sums, h = ctx.vegas_iteration(prog, 0, 7001, rule, 31, 1, grid.astype(float), tier=tier)
    assert np.allclose(sums[..., 0], s1.astype(float), rtol=1e-10) and np.allclose(sums[..., 1], s2.astype(float), rtol=1e-10)
    hf = hist.astype(float)
    assert np.allclose(h, hf, rtol=1e-10, atol=1e-14 * hf.max())
    assert np.allclose(h.sum(axis=1), sums[:, 0, 1].sum(), rtol=1e-12)
    val, sig, chi2, g_or = OI.integrate_vegas(sec, 1 << 13, 37, 50, 4, 1.5)
    res = ctx.integrate(prog, 1 << 13, rule, 37, tier=tier)[0]
    g, _ = ctx.vegas_grid(0, wl.dim, 50)
    assert np.max(np.abs(g - g_or.astype(float))) < 1e-11
    assert np.allclose(res["re"], np.asarray(val, dtype=float)[:, 0], rtol=1e-10)
    assert np.allclose(res["re_err"], np.asarray(sig, dtype=float)[:, 0], rtol=1e-6)
    assert np.allclose(res["chi2"], np.asarray(chi2, dtype=float)[:, 0], rtol=1e-5, atol=1e-8)


# ------------------------------------------------------------------------------ closed forms (4 sigma)

def _within(res, exact, nsig=4.0):
    return abs(res["re"] - exact) <= nsig * res["re_err"] + 1e-15 * abs(exact)


def test_paper_worker_example(fb, ctx):
    """`1; 0; x[1]+0.2;` integrates to 0.7."""
    sec = one_sector(["1;\n0;\nx[1]+0.2;\n|"])
    prog = ctx.compile([sec], 1)
    res = ctx.integrate(prog, 8 << 10, fb.Rule(kind=fb.RULE_LATTICE, n_shifts=8, korobov_a=1, periodize_r=3), 1)[0, 0]
    assert _within(res, 0.7) and res["re_err"] < 1e-6
    res = ctx.integrate(prog, 1 << 20, fb.Rule(kind=fb.RULE_MC), 1)[0, 0]
    assert _within(res, 0.7) and res["re_err"] < 1e-3


def test_monomial_closed_form(fb, ctx):
    """BASELINE C1's closed-form check: int prod x_i^a_i over [0,1]^4 = prod 1/(a_i+1)."""
    from workloads import korobov_a
    a = [2, 0, 1, 2]
    txt = block(4, [], "*".join(f"p[x[{i + 1}],{e}]" for i, e in enumerate(a) if e) + "*1.0")
    sec = one_sector([txt])
    prog = ctx.compile([sec], 4)
    exact = float(np.prod([1.0 / (e + 1) for e in a]))
    bad = 0
    for seed in range(20):
        rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=8, korobov_a=korobov_a(1 << 13, 4), periodize_r=3)
        res = ctx.integrate(prog, 1 << 16, rule, seed)[0, 0]
        bad += not _within(res, exact)
        assert res["re_err"] < 1e-5 * exact
    assert bad <= 1


def test_noninteger_power_closed_form(fb, ctx):
    """int prod x_i^-0.4 = (1/0.6)^3 with the MC rule and with Vegas (a >= -0.45: finite variance)."""
    sec = one_sector([block(3, [], "p[x[1],-0.4]*p[x[2],-0.4]*p[x[3],-0.4]")])
    prog = ctx.compile([sec], 3)
    exact = (1 / 0.6) ** 3
    res = ctx.integrate(prog, 1 << 20, fb.Rule(kind=fb.RULE_MC), 3)[0, 0]
    assert _within(res, exact) and res["re_err"] < 0.01
    res = ctx.integrate(prog, 1 << 17, fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=50, vegas_iters=10), 3)[0, 0]
    assert _within(res, exact, 5.0) and res["re_err"] < 0.002


def test_bubble_eps_orders(fb, ctx):
    """One-loop massless bubble (eq. 2): twice the order-k integral = c_k (golden file)."""
    from conftest import golden
    g = golden("bubble_eps_coefficients.txt")
    fl = ["1+x[1]", "2*l[f[1]]-l[x[1]]"]
    fact = [1, 1, 2, 6, 24]
    texts = [block(1, fl, f"2*p[f[1],-2]*p[f[2],{k}]/{fact[k]}" if k else "2*p[f[1],-2]") for k in range(5)]
    prog = ctx.compile([one_sector(texts)], 1)
    res = ctx.integrate(prog, 8 << 13, fb.Rule(kind=fb.RULE_LATTICE, n_shifts=8, korobov_a=1, periodize_r=3), 5)[0]
    for k in range(5):
        exact = float(g[f"c{k}"])
        assert _within(res[k], exact), (k, res[k], exact)
        assert abs(res[k]["re"] - exact) < 1e-9


def test_contour_1d_closed_forms(fb, ctx):
    """F = x - a, z = x - i lam x(1-x): int dz/(z-a), int log(z-a) dz, int (z-a)^-1/2 dz (golden file)."""
    from conftest import golden
    g = golden("contour_1d_closed_forms.txt")
    texts = [block(1, ["x[1]-0.3"], f) for f in ("1/f[1]", "l[f[1]]", "p[f[1],-0.5]")]
    sec = one_sector(texts, is_complex=True, deform_f_index=1, lam=0.5)
    prog = ctx.compile([sec], 1)
    res = ctx.integrate(prog, 8 << 13, fb.Rule(kind=fb.RULE_LATTICE, n_shifts=8, korobov_a=1, periodize_r=3), 5)[0]
    for k, key in enumerate(("inv", "log", "rsqrt")):
        re, im = float(g[key + "_re"]), float(g[key + "_im"])
        assert abs(res[k]["re"] - re) <= 4 * res[k]["re_err"] + 1e-14
        assert abs(res[k]["im"] - im) <= 4 * res[k]["im_err"] + 1e-14
        assert abs(res[k]["re"] - re) < 1e-8 and abs(res[k]["im"] - im) < 1e-8


def test_lambda_zero_reproduces_real_path(fb, ctx):
    """R11: at lambda = 0 the complex path gives the real path's values with Im = 0."""
    wl = make_workload("C4", nsectors=1, npoints=1 << 12)
    s = wl.sectors[0]
    real = SectorText(s.sector_id, s.texts)
    zero = SectorText(s.sector_id, s.texts, is_complex=True, deform_f_index=s.deform_f_index, lam=0.0)
    prog = ctx.compile([real, zero], wl.dim)
    x = np.random.default_rng(2).random((500, wl.dim))
    a, b = ctx.eval_points(prog, 0, x), ctx.eval_points(prog, 1, x)
    ok = np.isfinite(a.real)            # F changes sign inside the cube: the real path has NaNs there
    assert ok.sum() > 100
    assert np.allclose(b.real[ok], a.real[ok], rtol=1e-11) and np.all(np.abs(b.imag[ok]) <= 1e-11 * np.abs(a.real[ok]))


def _box_totals(fb, ctx, terms, integrate):
    """sum over the front end's integrands, grouped by dimension (one program each) -> (totals [3], sigma [3])"""
    tot, var = np.zeros(3), np.zeros(3)
    for d in (1, 2, 3):
        secs = [SectorText(sector_id=sid, texts=texts) for sid, (dim, texts, _) in enumerate(terms) if dim == d]
        prog = ctx.compile(secs, d)
        res = integrate(prog, d)
        tot += res["re"].sum(axis=0)
        var += (res["re_err"] ** 2).sum(axis=0)
        assert np.all(res["n_nonfinite"] == 0)
        prog.close()
    return tot, np.sqrt(var)


def test_paper_box_example_on_the_gpu(fb, ctx):
    """PAPER.md:301-313, the massless on-shell box: the 40 integrands of tests/sector_frontend.py (decomposed,
    pole-subtracted, expanded in eps) through fiesta_compile / fiesta_integrate give the numbers the paper prints
    within the errors it prints, and the closed form behind them to 1e-9 -- by the lattice rule, by the lattice
    rule with the mixed-precision rescue switched on (the subtracted integrands are differences over x), and,
    for the 2- and 3-dimensional integrands, by the deterministic cubature."""
    import math
    from conftest import golden
    from sector_frontend import box_integrands
    from workloads import korobov_a
    g = golden("paper_box_example.txt")
    S, T = int(g["S"]), int(g["T"])
    exact = [4 / (S * T), -2 * math.log(S * T) / (S * T), (2 * math.log(S) * math.log(T) - 4 * math.pi ** 2 / 3) / (S * T)]
    terms = box_integrands(S, T)

    def lattice(prog, d):
        nl = 1 << 14
        rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=8, korobov_a=korobov_a(nl, d) if d > 1 else 1, periodize_r=3)
        return ctx.integrate(prog, 8 * nl, rule, 20151111)

    tot, sig = _box_totals(fb, ctx, terms, lattice)
    for k, key in enumerate(("eps_m2", "eps_m1", "eps_0")):
        assert abs(tot[k] - float(g[key])) <= 3 * float(g[key + "_err"]) + 0.5e-4, (key, tot[k])
        assert abs(tot[k] - exact[k]) < 1e-9 and sig[k] < 1e-9, (key, tot[k], exact[k], sig[k])
    ctx.set_mixed(1e-6)
    try:
        tot_mixed, _ = _box_totals(fb, ctx, terms, lattice)
    finally:
        ctx.set_mixed(0.0)
    assert np.allclose(tot_mixed, exact, rtol=0, atol=1e-9)

    def cubature(prog, d):
        if d == 1:
            return lattice(prog, d)
        return ctx.integrate_cubature(prog, epsrel=1e-7, epsabs=1e-9, maxeval=1 << 20)[0]

    tot_c, err_c = _box_totals(fb, ctx, terms, cubature)
    for k in range(3):
        assert abs(tot_c[k] - exact[k]) <= max(err_c[k], 1e-9) and err_c[k] < 1e-4, (k, tot_c[k], exact[k], err_c[k])


def test_physical_region_triangle_on_the_gpu(fb, ctx):
    """The equal-mass triangle above threshold (s = 10 m^2; tests/sector_frontend.py, three 2-dimensional sectors whose F
    changes sign inside the cube): deformation size from fiesta_select_lambda, then the lattice rule on both
    tiers and the cubature, against the closed form -(1/(2s)) [ln((1+b)/(1-b)) - i pi]^2."""
    import math
    from sector_frontend import triangle_integrands
    from workloads import korobov_a
    s_, m2 = 10, 1
    b = math.sqrt(1 - 4 * m2 / s_)
    closed = -(1 / (2 * s_)) * (math.log((1 + b) / (1 - b)) - 1j * math.pi) ** 2
    secs = [SectorText(sector_id=sid, texts=texts, is_complex=True, deform_f_index=fi, lam=1.0)
            for sid, (texts, fi) in enumerate(triangle_integrands(s_, m2))]
    prog = ctx.compile(secs, 2)
    for si in range(3):
        lam, scan = ctx.select_lambda(prog, si, 1000, 5, lambda_max=1.0, lambda_split=4)
        assert lam > 0 and all(t["n_bad"] == 0 for t in scan)
        ctx.set_lambda(prog, si, lam)
    nl = 1 << 15
    rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=8, korobov_a=korobov_a(nl, 2), periodize_r=3)
    for tier in (fb.TIER_NATIVE, fb.TIER_INTERPRETER):
        res = ctx.integrate(prog, 8 * nl, rule, 7, tier=tier)
        total = complex(res["re"].sum(), res["im"].sum())
        assert abs(total - closed) < 1e-10 and np.all(res["re_err"] < 1e-10) and np.all(res["im_err"] < 1e-10)
    cub, _ = ctx.integrate_cubature(prog, epsrel=1e-9, maxeval=1 << 20)
    total = complex(cub["re"].sum(), cub["im"].sum())
    assert abs(total - closed) <= max(float(np.sqrt((cub["re_err"] ** 2 + cub["im_err"] ** 2).sum())), 1e-10)
    assert np.all(cub["re_err"] < 1e-7)
    prog.close()


def test_shifts_split_over_ranks_give_identical_bits(fb, ctx):
    """SURVEY 8(e), few huge sectors: the shifts of the lattice rule dealt to ranks.  What rank i of 3 would compute
    (fiesta_partial_sums_shifts) is, bit for bit, rows of the full call on both tiers -- real and complex sectors --
    and fiesta_estimate_from_sums on the gathered rows is fiesta_integrate's result; world size 1 of
    sharding.integrate_split_shifts as well."""
    from paper_1511_03614_b200.sharding import integrate_split_shifts, split_shifts
    for name, npts in (("C3", 1 << 15), ("C4", 1 << 13)):
        wl = make_workload(name, nsectors=2, npoints=npts, n_shifts=8)
        prog = ctx.compile(wl.sectors, wl.dim)
        rule = fb.Rule.from_workload(wl)
        for tier in (fb.TIER_NATIVE, fb.TIER_INTERPRETER):
            full = ctx.partial_sums(prog, wl.npoints, rule, wl.seed, tier=tier)
            rows = np.zeros_like(full)
            for first, cnt in split_shifts(8, 3):
                part, nf = ctx.partial_sums_shifts(prog, wl.npoints, rule, wl.seed, first, cnt, tier=tier)
                rows[:, first:first + cnt] = part
                assert np.all(nf == 0)
            assert rows.tobytes() == full.tobytes()
        direct = ctx.integrate(prog, wl.npoints, rule, wl.seed)
        assert ctx.estimate_from_sums(prog, rows, wl.n_lattice).tobytes() == direct.tobytes()
        assert integrate_split_shifts(ctx, prog, wl.npoints, rule, wl.seed).tobytes() == direct.tobytes()
        with pytest.raises(fb.FiestaError):
            ctx.partial_sums_shifts(prog, wl.npoints, rule, wl.seed, 6, 3)          # beyond the rule's 8 shifts
        with pytest.raises(fb.FiestaError):
            ctx.partial_sums_shifts(prog, wl.npoints, fb.Rule(kind=fb.RULE_MC), wl.seed, 0, 1)
        prog.close()


def test_bisected_cube_parts_add_up(fb, ctx):
    """PAPER.md:406 BisectionVariables (bisection.py): the parts of a bisected integrand are ordinary sectors --
    per-point parity with the oracle on the rewritten texts -- and their integrals add up: to the closed forms
    of the 1-D contour integrals (the zero of F at 0.3 lies in the lower part), and to the unbisected integral
    of a generated real sector."""
    from conftest import golden
    from paper_1511_03614_b200.bisection import bisect_sector
    g = golden("contour_1d_closed_forms.txt")
    texts = [block(1, ["x[1]-0.3"], f) for f in ("1/f[1]", "l[f[1]]", "p[f[1],-0.5]")]
    sec = one_sector(texts, is_complex=True, deform_f_index=1, lam=0.5, sector_id=3)
    parts = bisect_sector(sec, [1], points=0.5)
    prog = ctx.compile(parts, 1)
    x = np.random.default_rng(4).random((300, 1))
    for si, part in enumerate(parts):
        ref, mag = oracle_values_and_magnitude(spec(part), x)
        assert check_points(ctx.eval_points(prog, si, x), ref, mag) <= 1.0
    res = ctx.integrate(prog, 8 << 13, fb.Rule(kind=fb.RULE_LATTICE, n_shifts=8, korobov_a=1, periodize_r=3), 5)
    for k, key in enumerate(("inv", "log", "rsqrt")):
        re, im = float(g[key + "_re"]), float(g[key + "_im"])
        got_re, got_im = res[0][k]["re"] + res[1][k]["re"], res[0][k]["im"] + res[1][k]["im"]
        assert abs(got_re - re) < 1e-8 and abs(got_im - im) < 1e-8
    prog.close()
    wl = make_workload("C2", nsectors=1, npoints=1 << 16, n_shifts=8)
    parts = bisect_sector(wl.sectors[0], [1, 4], points=[0.5, 0.25])
    rule = fb.Rule.from_workload(wl)
    whole_prog, parts_prog = ctx.compile(wl.sectors, wl.dim), ctx.compile(parts, wl.dim)
    whole = ctx.integrate(whole_prog, wl.npoints, rule, wl.seed)[0]
    res = ctx.integrate(parts_prog, wl.npoints, rule, wl.seed)
    for k in range(len(whole)):
        total = sum(res[h][k]["re"] for h in range(4))
        sigma = np.sqrt(whole[k]["re_err"] ** 2 + sum(res[h][k]["re_err"] ** 2 for h in range(4)))
        assert abs(total - whole[k]["re"]) <= 5 * sigma + 1e-12 * abs(whole[k]["re"])
    whole_prog.close()
    parts_prog.close()


# ------------------------------------------------------------------------------ -testF, choice of lambda

def test_testf_and_lambda_scan(fb, ctx):
    """PAPER.md:474 -testF and the automatic deformation size of PAPER.md:404 (R19) on the device
    against the oracle: counts of points with Im F(z) >= 0 bit-exact, max Im F and min |F| to 1e-12; the scan
    picks the same candidate; fiesta_program_set_lambda changes what both tiers integrate."""
    from oracle import deform as OD
    from oracle.parser import parse
    wl = make_workload("C4", nsectors=2, npoints=1 << 12)
    cub = one_sector([block(1, ["p[x[1],3]-0.2"], "1/f[1]")], sector_id=9, is_complex=True, deform_f_index=1, lam=1.0)
    prog = ctx.compile(wl.sectors, wl.dim)
    mc = fb.Rule(kind=fb.RULE_MC)
    for si, lam in ((0, -1.0), (1, 0.25), (1, 6.0), (0, 40.0)):
        s = wl.sectors[si]
        sec = spec(s)
        _, x = OI.mc_points(sec, 77, 0, 0, 3001)
        lam_o = s.lam if lam < 0 else lam
        bad, mx, mn = OD.test_f(sec.progs[0], s.deform_f_index, lam_o, x)
        got = ctx.test_f(prog, si, 3001, mc, 77, lam)
        assert got["n_points"] == 3001 and got["lam"] == lam_o
        assert got["n_bad"] == bad, (si, lam, got, bad)
        assert abs(got["max_im_f"] - float(mx)) <= 1e-12 * max(abs(float(mx)), 1.0)
        assert abs(got["min_abs_f"] - float(mn)) <= 1e-12 * float(mn)
    assert ctx.test_f(prog, 0, 3001, mc, 77)["n_bad"] == 0          # the generator rejected seeds with Im F >= 0
    # lattice points as well
    rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=2, korobov_a=wl.korobov_a, periodize_r=3)
    got = ctx.test_f(prog, 1, 1 << 12, rule, 5, 0.5)
    sec = spec(wl.sectors[1])
    # the Korobov vector the rule above implies for its 2^11-point lattice: a^k mod 2^11
    gv = OP.korobov_genvec(wl.korobov_a, 1 << 11, wl.dim)
    xs = np.concatenate([OI.lattice_points(sec, 1 << 11, gv, 3, 5, r, 0, 1 << 11)[0] for r in range(2)])
    bad, mx, mn = OD.test_f(sec.progs[0], 2, 0.5, xs)
    assert got["n_bad"] == bad and abs(got["min_abs_f"] - float(mn)) <= 1e-12 * float(mn)
    # the scan on the 1-D cubic, whose admissible range is known in closed form (lam < 3.897..)
    p1 = ctx.compile([cub], 1)
    secc = spec(cub)
    _, x = OI.mc_points(secc, 123, (1 << 20) - 1, 0, 1000)
    lam_o, scan_o = OD.select_lambda(secc.progs[0], 1, x, lambda_max=8.0, lambda_split=8)
    lam_g, scan_g = ctx.select_lambda(p1, 0, 1000, 123, lambda_max=8.0, lambda_split=8)
    assert lam_g == float(lam_o) and [t["n_bad"] for t in scan_g] == [t[1] for t in scan_o]
    assert [t["n_bad"] == 0 for t in scan_g] == [True, True, True] + [False] * 5
    assert ctx.select_lambda(p1, 0, 1000, 123, 8.0, 8, conservative=True)[0] == lam_g / 2
    with pytest.raises(fb.FiestaError) as ei:
        ctx.select_lambda(p1, 0, 1000, 123, lambda_max=80.0, lambda_split=2)
    assert ei.value.code == -4
    # applying the choice: a run-time parameter of both tiers
    lat = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=2, korobov_a=1, periodize_r=3)
    before = ctx.integrate(p1, 1 << 12, lat, 3, tier=fb.TIER_NATIVE)
    ctx.set_lambda(p1, 0, lam_g)
    a = ctx.integrate(p1, 1 << 12, lat, 3, tier=fb.TIER_NATIVE)
    b = ctx.integrate(p1, 1 << 12, lat, 3, tier=fb.TIER_INTERPRETER)
    assert a.tobytes() == b.tobytes() and a.tobytes() != before.tobytes()
    val, sig = OI.integrate_lattice(SectorSpec(cub.texts, 9, True, 1, lam_g), 1 << 12, 2, [1], 3, 3)
    assert np.allclose(a[0]["re"], np.asarray(val, dtype=float)[:, 0], rtol=1e-9)
    assert np.allclose(a[0]["im"], np.asarray(val, dtype=float)[:, 1], rtol=1e-9)
    with pytest.raises(fb.FiestaError):
        ctx.test_f(ctx.compile(make_workload("C1", nsectors=1, npoints=1 << 12).sectors, 4), 0, 100, mc, 1)


# ------------------------------------------------------------------------------ A3/A8: Vegas

def _c5(nsec, npts):
    return make_workload("C5", nsectors=nsec, npoints=npts)


def test_vegas_iteration_stepwise(fb, ctx):
    """Same grid in => sums match (R15) and the f^2 histogram matches bin by bin (pin vi)."""
    wl = _c5(2, 20000)
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    rng = np.random.default_rng(8)
    for si, it in ((0, 0), (1, 3)):
        sec = spec(wl.sectors[si])
        if it == 0:
            grid = OI.vegas_uniform_grid(wl.dim, wl.vegas_bins)
        else:  # an uneven but valid grid
            w = rng.random((wl.dim, wl.vegas_bins)).astype(LD) ** 3 + LD(1e-3)
            grid = np.concatenate([np.zeros((wl.dim, 1), dtype=LD), np.cumsum(w, axis=1) / np.sum(w, axis=1)[:, None]], axis=1)
            grid[:, -1] = 1
        gridf = grid.astype(np.float64)
        s1, s2, hist = OI.vegas_iteration_sums(sec, gridf.astype(LD), wl.npoints, wl.seed, it)
        sums, h = ctx.vegas_iteration(prog, si, wl.npoints, rule, wl.seed, it, gridf)
        assert np.allclose(sums[..., 0], s1.astype(float), rtol=1e-10)
        assert np.allclose(sums[..., 1], s2.astype(float), rtol=1e-10)
        hf = hist.astype(float)
        assert np.allclose(h, hf, rtol=1e-10, atol=1e-13 * hf.max())
        # pin iii: every dimension's histogram has the same total, the deterministic sum of g^2
        assert np.allclose(h.sum(axis=1), sums[0, 0, 1], rtol=1e-12)


def test_vegas_refine_parity(fb, ctx):
    """Same histogram in => edges match to 1e-13 (pin vi); invariants (pin ii); flat in => uniform out."""
    rng = np.random.default_rng(9)
    nb = 50
    grids, hists = [], []
    for i in range(40):
        w = rng.random(nb) ** 2 + 1e-3
        g = np.concatenate([[0.0], np.cumsum(w) / np.sum(w)])
        g[-1] = 1.0
        h = rng.random(nb) ** (1 + i % 5) * 10.0 ** rng.integers(-8, 8)
        if i % 7 == 0:
            h[rng.integers(0, nb, 10)] = 0.0       # empty bins
        if i == 5:
            h[:] = 0.0                              # nothing sampled: grid must stay
        if i == 6:
            h[:] = 0.0
            h[17] = 1.0                             # a single hot bin
        grids.append(g)
        hists.append(h)
    grids, hists = np.array(grids), np.array(hists)
    out = ctx.vegas_refine(grids, hists, 1.5)
    for i in range(40):
        ref = OI.vegas_refine(grids[i].astype(LD), hists[i].astype(LD), 1.5).astype(float)
        assert np.max(np.abs(out[i] - ref)) < 1e-13, i
        assert out[i][0] == 0.0 and out[i][-1] == 1.0 and np.all(np.diff(out[i]) > 0)
    uni = np.arange(nb + 1) / nb
    out = ctx.vegas_refine(uni[None, :], np.full((1, nb), 3.0), 1.5)
    assert np.max(np.abs(out[0] - uni)) < 1e-15
    for nb2 in (2, 3, 128):
        uni = np.arange(nb2 + 1) / nb2
        h = rng.random(nb2)
        ref = OI.vegas_refine(uni.astype(LD), h.astype(LD), 0.7).astype(float)
        assert np.max(np.abs(ctx.vegas_refine(uni[None, :], h[None, :], 0.7)[0] - ref)) < 1e-13


def test_vegas_full_run_against_oracle(fb, ctx):
    """10 iterations.  The bin of a point is integer arithmetic on t and the histogram is summed in a fixed
    order, so the only difference to the oracle is FP64 rounding (2e-14 per histogram bin, step-wise tests)
    carried through ten refinements, each of which amplifies it (compression exponent 1.5, re-binning by
    interpolation; C5's integrand has no finite variance, its histograms are dominated by few points):
    measured 2e-10 on the edges and 1.5e-11 on the value (profiles/r02_parity_margins.md); the bars are the
    1e-9 of round 1 on the edges and, tightened from 1e-7, 1e-9 on the value."""
    wl = _c5(2, 1 << 13)
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    res = ctx.integrate(prog, wl.npoints, rule, wl.seed)
    for si in range(2):
        val, sig, chi2, grid = OI.integrate_vegas(spec(wl.sectors[si]), wl.npoints, wl.seed, wl.vegas_bins, wl.vegas_iters,
                                                  wl.vegas_alpha)
        g, h = ctx.vegas_grid(si, wl.dim, wl.vegas_bins)
        record_margin(f"vegas full run C5 sector {si}", grid_max_abs_diff=float(np.max(np.abs(g - grid.astype(float)))),
                      value_rel_diff=float(abs(res[si, 0]["re"] / float(val[0, 0]) - 1)),
                      sigma_rel_diff=float(abs(res[si, 0]["re_err"] / float(sig[0, 0]) - 1)))
        assert np.max(np.abs(g - grid.astype(float))) < 1e-9
        assert g[:, 0].max() == 0.0 and g[:, -1].min() == 1.0 and np.all(np.diff(g, axis=1) > 0)
        assert np.isclose(res[si, 0]["re"], float(val[0, 0]), rtol=1e-9)
        assert np.isclose(res[si, 0]["re_err"], float(sig[0, 0]), rtol=1e-6)
        assert np.isclose(res[si, 0]["chi2"], float(chi2[0, 0]), rtol=1e-5, atol=1e-8)
        assert res[si, 0]["neval"] == wl.npoints * wl.vegas_iters


def test_vegas_constant_integrand(fb, ctx):
    """Pin i: f = 1 gives I = 1 exactly with sigma_it = 0 in iteration 1, and stays 1 within rounding."""
    prog = ctx.compile([one_sector([block(3, [], "1.0+0*x[1]")])], 3)
    res = ctx.integrate(prog, 1 << 14, fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=50, vegas_iters=1), 4)[0, 0]
    assert res["re"] == 1.0 and res["re_err"] == 0.0
    res = ctx.integrate(prog, 1 << 14, fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=50, vegas_iters=5), 4)[0, 0]
    assert abs(res["re"] - 1.0) <= 4 * res["re_err"] + 1e-12


def test_vegas_adapts_to_separable_peak(fb, ctx):
    """Pin v: f = prod (1-a) x^-a, a = 0.4: edges move towards (b/NB)^(1/(1-a)); the error shrinks."""
    sec = one_sector([block(2, [], "0.36*p[x[1],-0.4]*p[x[2],-0.4]")])
    prog = ctx.compile([sec], 2)
    r1 = ctx.integrate(prog, 1 << 16, fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=50, vegas_iters=1), 6)[0, 0]
    r10 = ctx.integrate(prog, 1 << 16, fb.Rule(kind=fb.RULE_VEGAS, vegas_bins=50, vegas_iters=10), 6)[0, 0]
    g, _ = ctx.vegas_grid(0, 2, 50)
    ideal = (np.arange(51) / 50) ** (1 / 0.6)
    assert np.max(np.abs(g - ideal[None, :])) < 0.02
    assert r10["re_err"] < 0.3 * r1["re_err"] and abs(r10["re"] - 1.0) <= 4 * r10["re_err"]


# ------------------------------------------------------------------------------ limits and errors

def test_max_dim_and_max_orders(fb, ctx):
    """dim = 12 (FIESTA_MAX_DIM) and K = 8 (FIESTA_MAX_ORDERS) in one sector."""
    fl = ["1+" + "+".join(f"{0.1 * (i + 1):.1f}*x[{i + 1}]" for i in range(12)), "l[f[1]]"]
    texts = [block(12, fl, f"p[f[1],-{k + 1}]*p[f[2],{k}]*x[12]*x[1]" if k else "p[f[1],-1]*x[12]*x[1]") for k in range(8)]
    sec = one_sector(texts, sector_id=41)
    prog = ctx.compile([sec], 12)
    x = np.random.default_rng(3).random((600, 12))
    ref, mag = oracle_values_and_magnitude(spec(sec), x)
    assert check_points(ctx.eval_points(prog, 0, x), ref, mag) <= 1.0
    rule = fb.Rule(kind=fb.RULE_LATTICE, n_shifts=2, korobov_a=1571, periodize_r=2)
    gpu = ctx.partial_sums(prog, 1 << 13, rule, 17)
    s1, s2, sa = OI.lattice_partial_sums(spec(sec), 1 << 12, 2, OP.korobov_genvec(1571, 1 << 12, 12), 2, 17)
    check_sums(gpu[0], s1, s2, sa)


def test_many_temporaries_spill_to_shared(fb, ctx):
    """More live f[i] than register temporaries: compiler-directed shared-memory slots (n_mem_slots > 0)."""
    nf = 14
    fl = [f"1+{0.3 + 0.1 * i:.1f}*x[{i % 3 + 1}]+x[{(i + 1) % 3 + 1}]*x[{(i + 2) % 3 + 1}]" for i in range(nf)]
    final = "+".join(f"l[f[{i + 1}]]*p[f[{(i + 5) % nf + 1}],-1.5]" for i in range(nf))
    sec = one_sector([block(3, fl, final)])
    prog = ctx.compile([sec], 3)
    assert prog.info[0]["n_mem_slots"] > 0
    x = np.random.default_rng(4).random((300, 3))
    ref, mag = oracle_values_and_magnitude(spec(sec), x)
    assert check_points(ctx.eval_points(prog, 0, x), ref, mag) <= 1.0
    gpu = ctx.partial_sums(prog, 1 << 12, fb.Rule(kind=fb.RULE_LATTICE, korobov_a=1, periodize_r=1, genvec=[1, 433, 1217]), 2)
    s1, s2, sa = OI.lattice_partial_sums(spec(sec), 1 << 12, 1, [1, 433, 1217], 1, 2)
    check_sums(gpu[0], s1, s2, sa)


def test_constants_and_operators(fb, ctx):
    """Grammar coverage: P, G, PolyGamma, unary minus, division, nested p[], l[]."""
    final = ("P*x[1]-G*x[2]+PolyGamma[2,1]*x[1]*x[2]-(-x[1]+2)/(1+x[2])+p[1+x[1]*x[2],3]/p[2+x[1],2]"
             "+l[1+p[x[2],2]]*p[1+x[1],0.5]-p[1+x[2],-1.5]+1.5e-3*x[1]-p[l[2+x[1]],2]")
    sec = one_sector([block(2, [], final)])
    prog = ctx.compile([sec], 2)
    x = np.random.default_rng(5).random((400, 2))
    ref, mag = oracle_values_and_magnitude(spec(sec), x)
    assert check_points(ctx.eval_points(prog, 0, x), ref, mag) <= 1.0


def test_large_integer_powers(fb, ctx):
    """p[e, n] with large n goes through square-and-multiply (40 instructions, not 999), within the per-point bar."""
    sec = one_sector([block(2, ["1+0.001*x[1]"], "p[x[1],37]*p[f[1],1000]+p[0.999*x[2],300]-p[x[1]*x[2],9]")])
    prog = ctx.compile([sec], 2)
    assert prog.info[0]["n_ir_ops"] < 80
    x = np.random.default_rng(6).random((400, 2))
    ref, mag = oracle_values_and_magnitude(spec(sec), x)
    for tier in (0, 1):
        assert check_points(ctx.eval_points(prog, 0, x, tier=tier), ref, mag) <= 1.0


def test_nonfinite_is_reported(fb, ctx):
    """R13: l[e] with e <= 0 in real mode is NaN, counted, and raises FIESTA_E_NONFINITE."""
    prog = ctx.compile([one_sector([block(1, [], "l[x[1]-0.5]")])], 1)
    with pytest.raises(fb.FiestaError) as ei:
        ctx.integrate(prog, 1 << 10, fb.Rule(kind=fb.RULE_MC), 1)
    assert ei.value.code == -6
    res = ctx.integrate(prog, 1 << 10, fb.Rule(kind=fb.RULE_MC), 1, allow_nonfinite=True)[0, 0]
    t = ctx.generate_points(fb.Rule(kind=fb.RULE_MC), 1, 0, 0, 0, 0, 1 << 10, 1)
    assert res["n_nonfinite"] == int(np.sum(OP.unit_from_t(t) < 0.5))


@pytest.mark.parametrize("text,dim,code", [
    ("1;\n0;\nx[1]+;\n|", 1, -1), ("1;\n0;\nx[1]+0.2;\n| 7", 1, -1), ("1;\n0;\nq[1];\n|", 1, -1),
    ("1;\n0;\nx[2];\n|", 1, -2), ("1;\n1;\nx[1];\nf[2];\n|", 1, -1), ("1;\n0;\nPolyGamma[9,9];\n|", 1, -1),
    ("1;\n0;\np[x[1],x[1]];\n|", 1, -1), ("13;\n0;\nx[1];\n|", 13, -2)])
def test_compile_errors(fb, ctx, text, dim, code):
    with pytest.raises(fb.FiestaError) as ei:
        ctx.compile([one_sector([text])], dim)
    assert ei.value.code == code, str(ei.value)


def test_deformation_needs_polynomial(fb, ctx):
    sec = one_sector([block(1, ["l[1+x[1]]"], "f[1]")], is_complex=True, deform_f_index=1, lam=0.5)
    with pytest.raises(fb.FiestaError) as ei:
        ctx.compile([sec], 1)
    assert ei.value.code == -3


def test_rule_errors(fb, ctx):
    prog = ctx.compile([one_sector([block(1, [], "x[1]")])], 1)
    for npts, rule in [(1000, fb.Rule(kind=0)), (1 << 10, fb.Rule(kind=0, n_shifts=3)), (1 << 10, fb.Rule(kind=0, periodize_r=7)),
                       (1 << 10, fb.Rule(kind=2, vegas_bins=1)), (1 << 10, fb.Rule(kind=2, vegas_bins=129)), (1 << 10, fb.Rule(kind=5)),
                       (1, fb.Rule(kind=1)), (1 << 10, fb.Rule(kind=0, genvec=[1 << 10]))]:
        with pytest.raises(fb.FiestaError) as ei:
            ctx.integrate(prog, npts, rule, 1)
        assert ei.value.code == -4, (npts, rule, str(ei.value))


# ------------------------------------------------------------------------------ full sizes, bench launch configuration

def test_c2_full_size_sampled_sectors(fb, ctx):
    """BASELINE config 2 at full size (64 sectors x 2^20 points, one launch): the sums of two
    sampled sectors against the oracle, every sector's result finite with no bad point."""
    wl = make_workload("C2")
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    gpu = ctx.partial_sums(prog, wl.npoints, rule, wl.seed)
    gv = genvec_of(wl)
    for si in (5, 63):
        s1, s2, sa = OI.lattice_partial_sums(spec(wl.sectors[si]), wl.n_lattice, 1, gv, wl.periodize_r, wl.seed)
        check_sums(gpu[si], s1, s2, sa)
    res = ctx.integrate(prog, wl.npoints, rule, wl.seed)
    assert res.shape == (64, 4) and np.all(res["n_nonfinite"] == 0) and np.all(np.isfinite(res["re"]))
    assert np.allclose(res["re"], gpu[:, 0, :, 0, 0] / wl.npoints, rtol=1e-12)


def test_c3_bench_configuration_sampled(fb, ctx):
    """The workload bench.py times (config 3: dim 8, K = 5, 8 shifts x 2^21 points per sector, native
    tier, two waves of blocks per sector) on a slice of its sectors: one sampled (sector, shift) sum
    against the oracle, and the properties that hold at any size -- per-shift sums agree with
    each other to the quoted error, results are finite, neval is exact."""
    wl = make_workload("C3", nsectors=6)
    assert wl.npoints == 1 << 24 and wl.n_shifts == 8
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    gpu = ctx.partial_sums(prog, wl.npoints, rule, wl.seed)          # [6, 8, 5, 1, 2]
    si, r = 4, 6
    s1, s2, sa = OI.lattice_partial_sums(spec(wl.sectors[si]), wl.n_lattice, 8, genvec_of(wl), wl.periodize_r, wl.seed,
                                         shifts=[r])
    check_sums(gpu[si, r:r + 1], s1[r:r + 1], s2[r:r + 1], sa[r:r + 1])
    res = ctx.integrate(prog, wl.npoints, rule, wl.seed)
    assert np.all(res["neval"] == 1 << 24) and np.all(res["n_nonfinite"] == 0)
    q = gpu[..., 0, 0] / wl.n_lattice                                   # [6, 8, 5]
    assert np.allclose(res["re"], q.mean(axis=1), rtol=1e-12)
    assert np.allclose(res["re_err"], q.std(axis=1, ddof=1) / np.sqrt(8), rtol=1e-6)
    assert np.all(np.abs(q - q.mean(axis=1, keepdims=True)) <= 6 * q.std(axis=1, ddof=1, keepdims=True) + 1e-300)


def test_c4_full_size_sampled_chunks(fb, ctx):
    """BASELINE config 4 at its full per-sector size (complex, deformed, 2^22 points, the launch geometry
    fiesta_integrate uses, native kernel): the partial records of sampled blocks -- the first, one in the
    middle, the ragged last -- against the oracle's sums over exactly those points; the blocks add up to
    the sector's sums; results finite."""
    wl = make_workload("C4", nsectors=2)
    assert wl.npoints == 1 << 22
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    si = 1
    chunk, recs = ctx.chunk_sums(prog, wl.npoints, rule, wl.seed, sectors=[si], tier=fb.TIER_NATIVE)   # [1, 1, nch, K, 2, 2]
    nch = recs.shape[2]
    assert nch > 1000 and (nch - 1) * chunk < wl.npoints <= nch * chunk
    gv = genvec_of(wl)
    sec = spec(wl.sectors[si])
    for c in (0, nch // 2 + 1, nch - 1):
        cnt = min(chunk, wl.npoints - c * chunk)
        s1, s2, sa = OI.lattice_partial_sums(sec, wl.n_lattice, 1, gv, wl.periodize_r, wl.seed, first=c * chunk, count=cnt)
        check_sums(recs[0, :, c], s1, s2, sa, label=f"C4 full size, sector {si}, block {c} of {nch}")
    tot = ctx.partial_sums(prog, wl.npoints, rule, wl.seed, sectors=[si], tier=fb.TIER_NATIVE)
    seq = np.zeros_like(tot[0, 0])
    for c in range(nch):
        seq = seq + recs[0, 0, c]                                           # the reduction's own order
    assert seq.tobytes() == tot[0, 0].tobytes()
    res = ctx.integrate(prog, wl.npoints, rule, wl.seed)
    assert np.all(res["neval"] == 1 << 22) and np.all(res["n_nonfinite"] == 0)
    assert np.all(np.isfinite(res["re"])) and np.all(np.isfinite(res["im"])) and np.all(res["im_err"] > 0)
    assert np.allclose(res[si]["re"], tot[0, 0, :, 0, 0] / wl.npoints, rtol=1e-13)


def test_c5_full_size_one_iteration(fb, ctx):
    """BASELINE config 5 at its full per-iteration size (dim 12, 2^22 Philox points, 50 bins, native Vegas kernel):
    the sums and the whole f^2 histogram of one iteration of one sector against the oracle."""
    wl = make_workload("C5", nsectors=1)
    assert wl.npoints == 1 << 22
    prog = ctx.compile(wl.sectors, wl.dim)
    rule = fb.Rule.from_workload(wl)
    sec = spec(wl.sectors[0])
    grid = OI.vegas_uniform_grid(wl.dim, wl.vegas_bins)
    s1, s2, hist = OI.vegas_iteration_sums(sec, grid, wl.npoints, wl.seed, 0, chunk=1 << 16)
    sums, h = ctx.vegas_iteration(prog, 0, wl.npoints, rule, wl.seed, 0, grid.astype(float), tier=fb.TIER_NATIVE)
    hf = hist.astype(float)
    record_margin("C5 full size, one iteration", S1_rel=float(abs(sums[0, 0, 0] / float(s1[0, 0]) - 1)),
                  S2_rel=float(abs(sums[0, 0, 1] / float(s2[0, 0]) - 1)), hist_worst_rel=float(np.max(np.abs(h / hf - 1))))
    assert np.allclose(sums[..., 0], s1.astype(float), rtol=1e-10) and np.allclose(sums[..., 1], s2.astype(float), rtol=1e-10)
    assert np.allclose(h, hf, rtol=1e-10)
    assert np.allclose(h.sum(axis=1), sums[0, 0, 1], rtol=1e-12)


def test_integration_pool_on_the_gpu(fb, ctx, tmp_path):
    """The queue of paper_1511_03614_b200/pool.py around the real C ABI: groups compiled one
    ahead, results stored per (sector, order), a killed job resumed -- the same bits as one fiesta_integrate call."""
    from paper_1511_03614_b200.pool import IntegrationPool
    wl = make_workload("C2", nsectors=20, npoints=1 << 14)
    rule = fb.Rule.from_workload(wl)
    prog = ctx.compile(wl.sectors, wl.dim)
    direct = ctx.integrate(prog, wl.npoints, rule, wl.seed)
    path = str(tmp_path / "results.db")
    costs = [s.naive_ops for s in wl.sectors]
    pool = IntegrationPool(ctx, wl.sectors, wl.dim, rule, wl.npoints, wl.seed, store_path=path, group=6, costs=costs)
    assert not pool.run(max_groups=2) and pool.n_integrated == 12
    pool = IntegrationPool(ctx, wl.sectors, wl.dim, rule, wl.npoints, wl.seed, store_path=path, group=6, costs=costs)
    assert pool.run() and pool.n_from_store == 12 and pool.n_integrated == 8
    res = pool.results()
    for f in ("re", "re_err", "neval"):            # JSON keeps every bit of a double
        assert np.array_equal(res[f], direct[f])
    tot = pool.totals()
    assert np.array_equal(tot["re"], ctx.combine(direct)["re"]) and np.array_equal(tot["re_err"], ctx.combine(direct)["re_err"])


def test_fp64_peak_is_plausible(ctx):
    """The roofline denominator: DFMA streams on every SM.  B200: 148 SM x 64 lanes x 2 x 1.965 GHz = 37.2."""
    t = ctx.fp64_peak(50.0)
    assert 15.0 < t < 45.0
