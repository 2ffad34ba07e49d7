"""GPU parity tests of the deterministic integrator (R21): the Genz-Malik rule on given
boxes against oracle/cubature.py, and the adaptive rounds against the oracle's rounds and closed forms.
Run with `-m gpu` on the B200 box."""
import math

import numpy as np
import pytest

from workloads import make_workload, SectorText
from oracle import cubature as OC
from oracle.integrate import LD

from helpers import spec

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


def _components(got, cplx):
    """complex [nb][K] from the binding -> [nb][ncomp] in the oracle's order (k, then Re / Im for complex sectors)"""
    if cplx:
        return np.stack([got.real, got.imag], axis=2).reshape(got.shape[0], -1)
    assert np.all(got.imag == 0.0)
    return got.real


def _random_boxes(rng, nb, n):
    h = rng.uniform(0.01, 0.25, size=(nb, n))
    c = h + rng.random((nb, n)) * (1 - 2 * h)
    boxes = np.stack([c, h], axis=1)
    boxes[0, 0], boxes[0, 1] = 0.5, 0.5              # the unit cube itself
    return boxes


@pytest.mark.parametrize("tier", [1, 0])
@pytest.mark.parametrize("name", ["C2", "C4", "C5"])
def test_rule_on_boxes_against_oracle(fb, ctx, name, tier):
    """I7, I5, fourth differences and split axis per box: real (dim 6, K = 4; dim 12) and complex deformed (dim 7)
    sectors on both forms of the program.  Bar: 1e-10 |I| + 1e-12 vol sum |w f| (the centre and l3 weights are
    negative from n = 3 / 5 on, so the rule sums cancel)."""
    wl = make_workload(name, nsectors=1, npoints=1 << 10)
    s = wl.sectors[0]
    n = wl.dim
    prog = ctx.compile([s], n)
    nb = 3 if n == 12 else 9
    boxes = _random_boxes(np.random.default_rng(n), nb, n)
    i7, i5, fourth, axis = ctx.cubature_rule(prog, 0, boxes, tier=tier)
    sec = spec(s)
    f = OC.sector_components(sec)
    cplx = sec.is_complex or sec.deform_f_index > 0
    g7, g5 = _components(i7, cplx), _components(i5, cplx)
    tables = OC.genz_malik(n)
    for b in range(boxes.shape[0]):
        c, h = boxes[b, 0].astype(LD), boxes[b, 1].astype(LD)
        r7, r5, d = OC.rule_on_box(f, c, h, tables)
        vals = np.abs(f(c[None, :] + tables[0] * h[None, :]))
        vol = float(np.prod(2 * h))
        for got, ref, w in ((g7[b], r7, tables[1]), (g5[b], r5, tables[2])):
            bound = 1e-10 * np.abs(ref.astype(float)) + 1e-12 * vol * np.sum(vals * np.abs(w)[None, :], axis=1).astype(float)
            assert np.all(np.abs(got - ref.astype(float)) <= bound), (b, got, ref)
        dd = d.astype(float)
        assert np.allclose(fourth[b], dd, rtol=1e-8, atol=1e-11 * float(np.max(np.sum(vals, axis=0))))
        top = np.sort(dd)[::-1]
        if top[0] > 1.0001 * top[1]:
            assert axis[b] == int(np.argmax(dd))
    prog.close()


@pytest.mark.parametrize("tier", [1, 0])
def test_adaptive_rounds_against_oracle_and_closed_form(fb, ctx, tier):
    """int int (1+x+y)^-2 = ln(4/3) and int int log(1+x+y) as two orders of one sector: the same rounds as the
    oracle's (same number of evaluations and boxes -- the choices are far from ties here), estimates to 1e-12,
    true error within the reported one."""
    texts = [block(2, ["1+x[1]+x[2]"], "p[f[1],-2]"), block(2, ["1+x[1]+x[2]"], "l[f[1]]")]
    s = SectorText(sector_id=0, texts=texts)
    prog = ctx.compile([s], 2)
    res, nboxes = ctx.integrate_cubature(prog, epsrel=1e-10, maxeval=1 << 16, tier=tier)
    total, err, neval, nb = OC.integrate_cubature(OC.sector_components(spec(s)), 2, epsrel=1e-10, maxeval=1 << 16)
    assert int(res[0][0]["neval"]) == neval and int(nboxes[0]) == nb
    for k in range(2):
        assert abs(res[0][k]["re"] - float(total[k])) <= 1e-12 * abs(float(total[k]))
        # the box errors are differences of two rule sums: FP64 noise of the sums, not of the error
        assert abs(res[0][k]["re_err"] - float(err[k])) <= 1e-6 * float(err[k]) + 1e-13 * abs(float(total[k]))
        assert res[0][k]["im"] == 0.0 and res[0][k]["im_err"] == 0.0 and res[0][k]["n_nonfinite"] == 0
    assert abs(res[0][0]["re"] - math.log(4.0 / 3.0)) <= res[0][0]["re_err"] <= 1e-10 * math.log(4.0 / 3.0)
    # maxeval cuts the rounds short and the reported error says so
    res2, _ = ctx.integrate_cubature(prog, epsrel=1e-14, maxeval=2000, tier=tier)
    assert res2[0][0]["neval"] <= 2000 and res2[0][0]["re_err"] > 1e-14
    assert abs(res2[0][0]["re"] - math.log(4.0 / 3.0)) <= res2[0][0]["re_err"]
    prog.close()


def test_cubature_is_reproducible_and_tier_independent(fb, ctx):
    """No random numbers, fixed summation order, and eval kernels that agree bit by bit across the tiers."""
    wl = make_workload("C2", nsectors=2, npoints=1 << 10)
    prog = ctx.compile(wl.sectors, wl.dim)
    a, na = ctx.integrate_cubature(prog, epsrel=1e-4, maxeval=60000, tier=1)
    b, nb = ctx.integrate_cubature(prog, epsrel=1e-4, maxeval=60000, tier=0)
    c, nc = ctx.integrate_cubature(prog, epsrel=1e-4, maxeval=60000)
    assert a.tobytes() == b.tobytes() == c.tobytes() and np.array_equal(na, nb) and np.array_equal(na, nc)
    assert np.all(a["neval"] <= 60000) and np.all(na >= 1)
    prog.close()


def test_cubature_agrees_with_the_lattice_rule(fb, ctx):
    """A generated sector (dim 6, 4 orders; 149 nodes per box) by both integrators."""
    wl = make_workload("C2", nsectors=1, npoints=1 << 19, n_shifts=8)
    prog = ctx.compile(wl.sectors, wl.dim)
    lat = ctx.integrate(prog, wl.npoints, fb.Rule.from_workload(wl), wl.seed)[0]
    cub, nboxes = ctx.integrate_cubature(prog, epsrel=1e-5, maxeval=1 << 21)
    for k in range(len(lat)):
        assert abs(cub[0][k]["re"] - lat[k]["re"]) <= cub[0][k]["re_err"] + 5 * lat[k]["re_err"]
        assert cub[0][k]["re_err"] <= 1e-3 * abs(cub[0][k]["re"])
    assert nboxes[0] > 10
    prog.close()


def test_cubature_on_a_deformed_sector(fb, ctx):
    """1-D closed forms do not apply (n >= 2): F = x1 - 0.3 deformed, times a smooth factor in x2:
    int dz/(z - a) * int (1+y)^2 dy = (ln((1-a)/a) + i pi) * 7/3."""
    s = SectorText(sector_id=0, texts=[block(2, ["x[1]-0.3"], "p[1+x[2],2]/f[1]")], is_complex=True, deform_f_index=1, lam=0.5)
    prog = ctx.compile([s], 2)
    res, _ = ctx.integrate_cubature(prog, epsrel=1e-9, maxeval=1 << 18)
    re, im = math.log(0.7 / 0.3) * 7.0 / 3.0, math.pi * 7.0 / 3.0
    assert abs(res[0][0]["re"] - re) <= max(res[0][0]["re_err"], 1e-12) and res[0][0]["re_err"] <= 1e-8
    assert abs(res[0][0]["im"] - im) <= max(res[0][0]["im_err"], 1e-12) and res[0][0]["im_err"] <= 1e-8
    prog.close()


def test_cubature_errors(fb, ctx):
    one = ctx.compile([SectorText(sector_id=0, texts=["1;\n0;\nx[1]+0.2;\n|"])], 1)
    with pytest.raises(fb.FiestaError):
        ctx.integrate_cubature(one)                                  # dim 1
    one.close()
    prog = ctx.compile([SectorText(sector_id=0, texts=[block(2, [], "l[x[1]-0.5]*x[2]")])], 2)
    with pytest.raises(fb.FiestaError):
        ctx.integrate_cubature(prog, maxeval=10)                     # below one rule evaluation (17 nodes)
    with pytest.raises(fb.FiestaError):
        ctx.integrate_cubature(prog)                                 # log of a negative number: NaN at nodes
    res, _ = ctx.integrate_cubature(prog, allow_nonfinite=True)
    assert res[0][0]["n_nonfinite"] > 0
    with pytest.raises(fb.FiestaError):
        ctx.cubature_rule(prog, 0, np.array([[[0.9, 0.5], [0.2, 0.5]]]))      # sticks out of the cube
    prog.close()
