"""Generators for the five BASELINE.json configurations.

Common family (shape of eq. 2, and of the epsilon-expanded
sector integrands):

    o_k(x) = M(x) * N_k(x) * U(x)^p * F(x)^-q * L_k(ln U, ln F)

M a monomial, U, F, N_k polynomials that always contain the constant monomial
(so the sector-decomposed factor never vanishes inside the cube), L_k a
polynomial in the two logarithms.  One text per (sector, order) in the worker
grammar; the K texts of a sector share their f[i] lines:

    f[1] = U, f[2] = F, f[3] = l[f[1]], f[4] = l[f[2]],
    f[5] = M * p[f[1],p] * p[f[2],-q]          final_k = f[5] * N_k * L_k

RNG: numpy default_rng([151103614, config, sector]).  Integration seed 20151111.
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

import numpy as np

from .korobov import korobov_a

CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")
BASE_SEED = 151103614
INTEGRATION_SEED = 20151111

RULE_LATTICE, RULE_MC, RULE_VEGAS = 0, 1, 2


@dataclass
class SectorText:
    sector_id: int
    texts: list                 # K blocks, each ending with '|'
    is_complex: bool = False
    deform_f_index: int = 0
    lam: float = 0.0
    naive_ops: int = 0          # operator nodes of the naive trees (f-lines once + K finals)
    meta: dict = field(default_factory=dict)


@dataclass
class Workload:
    name: str
    dim: int
    K: int
    sectors: list
    rule: int
    npoints: int                # total per sector (lattice: R * N_L; Vegas: per iteration)
    n_shifts: int = 1
    korobov_a: int = 1
    periodize_r: int = 3
    vegas_bins: int = 50
    vegas_iters: int = 10
    vegas_alpha: float = 1.5
    seed: int = INTEGRATION_SEED

    @property
    def n_lattice(self):
        return self.npoints // self.n_shifts

    @property
    def evals(self):
        """(points x sectors x orders), the unit of BASELINE.json's metric."""
        iters = self.vegas_iters if self.rule == RULE_VEGAS else 1
        return self.npoints * iters * len(self.sectors) * self.K

    @property
    def naive_ops_per_point(self):
        return float(np.mean([s.naive_ops for s in self.sectors]))


# ----------------------------------------------------------------------------- text helpers

def _num(c: float) -> str:
    s = repr(float(c))
    return f"({s})" if c < 0 else s


def _all_exponents(n: int, max_deg: int):
    """Every exponent vector with 1 <= total degree <= max_deg, in a fixed order."""
    out = []
    for deg in range(1, max_deg + 1):
        for combo in itertools.combinations_with_replacement(range(n), deg):
            e = [0] * n
            for i in combo:
                e[i] += 1
            out.append(tuple(e))
    return out


_EXP_CACHE = {}


def _draw_poly(rng, n, max_deg, n_monomials, lo, hi, neg_prob=0.0, neg_lo=0.0, neg_hi=0.0, const=None):
    """[(coef, exponents)], first the constant monomial, then distinct non-constant ones."""
    key = (n, max_deg)
    if key not in _EXP_CACHE:
        _EXP_CACHE[key] = _all_exponents(n, max_deg)
    pool = _EXP_CACHE[key]
    idx = rng.choice(len(pool), size=n_monomials - 1, replace=False)
    c0 = rng.uniform(lo, hi) if const is None else const
    mons = [(float(c0), tuple([0] * n))]
    for i in sorted(int(v) for v in idx):
        if neg_prob > 0 and rng.random() < neg_prob:
            c = rng.uniform(neg_lo, neg_hi)
        else:
            c = rng.uniform(lo, hi)
        mons.append((float(c), pool[i]))
    return mons


def _mono_text(exps) -> str:
    parts = []
    for i, e in enumerate(exps):
        if e == 1:
            parts.append(f"x[{i + 1}]")
        elif e > 1:
            parts.append(f"p[x[{i + 1}],{e}]")
    return "*".join(parts)


def _mono_ops(exps) -> int:
    nz = sum(1 for e in exps if e)
    return max(nz - 1, 0) + sum(1 for e in exps if e > 1)


_TERM_CACHE = {}


def _term_text(c, e):
    """Text and operator-node count of one term c * monomial (memoised: the C3 size loop re-renders)."""
    key = (c, e)
    hit = _TERM_CACHE.get(key)
    if hit is None:
        if len(_TERM_CACHE) > 200000:
            _TERM_CACHE.clear()
        mt = _mono_text(e)
        hit = (f"{_num(c)}*{mt}", 1 + _mono_ops(e)) if mt else (_num(c), 0)
        _TERM_CACHE[key] = hit
    return hit


def _poly_text(mons):
    """Text and operator-node count of sum_m c_m * monomial_m."""
    terms, ops = [], 0
    for c, e in mons:
        t, o = _term_text(c, e)
        terms.append(t)
        ops += o
    ops += len(terms) - 1
    return "+".join(terms), ops


def _logpoly_text(rng, max_total, lu="f[3]", lf="f[4]"):
    """L(lnU, lnF) = sum_{i+j<=max_total} c_ij lnU^i lnF^j, c ~ U[-1,1]; constant term 1."""
    terms, ops = ["1.0"], 0
    for i in range(max_total + 1):
        for j in range(max_total + 1 - i):
            if i + j == 0:
                continue
            c = float(rng.uniform(-1.0, 1.0))
            fac = []
            if i:
                fac.append(lu if i == 1 else f"p[{lu},{i}]")
                ops += 1 if i > 1 else 0
            if j:
                fac.append(lf if j == 1 else f"p[{lf},{j}]")
                ops += 1 if j > 1 else 0
            terms.append(f"{_num(c)}*" + "*".join(fac))
            ops += len(fac)
    ops += len(terms) - 1
    return "(" + "+".join(terms) + ")", ops


def _pow_text(base, q):
    if q == 1:
        return base, 0
    return f"p[{base},{_numq(q)}]", 1


def _numq(q):
    return repr(int(q)) if float(q).is_integer() else repr(float(q))


def _block(nvars, flines, final):
    lines = [f"{nvars};", f"{len(flines)};"] + [f"{f};" for f in flines] + [f"{final};", "|"]
    return "\n".join(lines)


def _family_sector(n, a_exp, u_mons, f_mons, p, q, numerators, logpolys):
    """Texts and naive op count for the common family.  numerators: list of K monomial lists or None."""
    ut, uo = _poly_text(u_mons)
    ft, fo = _poly_text(f_mons)
    mt = _mono_text(a_exp)
    up, upo = _pow_text("f[1]", p)
    fq, fqo = _pow_text("f[2]", -q)
    pref = "*".join(([mt] if mt else []) + [up, fq])
    pref_ops = (_mono_ops(a_exp) + 1 if mt else 0) + upo + fqo + 1
    flines = [ut, ft, "l[f[1]]", "l[f[2]]", pref]
    ops = uo + fo + 2 + pref_ops
    texts = []
    for k, (num, (lt, lo)) in enumerate(zip(numerators, logpolys)):
        final = "f[5]"
        if num is not None:
            nt, no = _poly_text(num)
            final += f"*({nt})"
            ops += no + 1
        if lt is not None:
            final += f"*{lt}"
            ops += lo + 1
        texts.append(_block(n, flines, final))
    return texts, ops


# ----------------------------------------------------------------------------- the configs

def _c1(nsectors, rng_of):
    n, K = 4, 3
    secs = []
    for s in range(nsectors):
        rng = rng_of(s)
        a = tuple(int(v) for v in rng.integers(0, 3, size=n))
        u = _draw_poly(rng, n, 2, 6, 0.5, 2.0)
        f = _draw_poly(rng, n, 2, 6, 0.5, 2.0)
        logs = [(None, 0), ("f[3]", 0), ("f[4]", 0)]
        texts, ops = _family_sector(n, a, u, f, 1, 2, [None] * K, logs)
        secs.append(SectorText(s, texts, naive_ops=ops, meta=dict(a=a, u=u, f=f, p=1, q=2)))
    return n, K, secs


def _c2(nsectors, rng_of):
    n, K = 6, 4
    secs = []
    for s in range(nsectors):
        rng = rng_of(s)
        a = tuple(int(v) for v in rng.integers(0, 2, size=n))
        u = _draw_poly(rng, n, 3, int(rng.integers(12, 21)), 0.1, 3.0)
        f = _draw_poly(rng, n, 4, int(rng.integers(12, 21)), 0.1, 3.0)
        p = int(rng.integers(1, 3))
        q = int(rng.integers(1, 4))
        logs = [(None, 0)] + [_logpoly_text(rng, min(k, 2)) for k in range(1, K)]
        texts, ops = _family_sector(n, a, u, f, p, q, [None] * K, logs)
        secs.append(SectorText(s, texts, naive_ops=ops, meta=dict(a=a, p=p, q=q)))
    return n, K, secs


def _c3(nsectors, rng_of, target_ops=1000):
    n, K = 8, 5
    secs = []
    for s in range(nsectors):
        rng = rng_of(s)
        a = tuple(int(v) for v in rng.integers(0, 2, size=n))
        f = _draw_poly(rng, n, 5, int(rng.integers(36, 45)), 0.1, 3.0)
        u = _draw_poly(rng, n, 4, int(rng.integers(26, 35)), 0.1, 3.0)
        q = 2.0 + 0.5 * (s % 4)
        logs = [(None, 0)] + [_logpoly_text(rng, min(k, 3)) for k in range(1, K)]
        nmon = [int(rng.integers(20, 31)) for _ in range(K)]
        nums = [_draw_poly(rng, n, 3, m, 0.1, 3.0) for m in nmon]
        texts, ops = _family_sector(n, a, u, f, 1, q, nums, logs)
        # add / drop numerator monomials until the naive-tree count is target +- 5 %
        guard = 0
        while abs(ops - target_ops) > 0.05 * target_ops and guard < 200:
            k = guard % K
            if ops < target_ops:
                pool = _EXP_CACHE[(n, 3)]
                have = {e for _, e in nums[k]}
                cand = pool[int(rng.integers(len(pool)))]
                if cand not in have:
                    nums[k].append((float(rng.uniform(0.1, 3.0)), cand))
            elif len(nums[k]) > 2:
                nums[k].pop()
            texts, ops = _family_sector(n, a, u, f, 1, q, nums, logs)
            guard += 1
        secs.append(SectorText(s, texts, naive_ops=ops, meta=dict(a=a, q=q, nmon=[len(m) for m in nums])))
    return n, K, secs


def _poly_eval_f64(mons, x):
    """Plain FP64 value of a monomial list at points x[j,:] (generator-side input validation only)."""
    out = np.zeros(x.shape[0], dtype=x.dtype)
    for c, e in mons:
        term = np.full(x.shape[0], c, dtype=x.dtype)
        for i, ei in enumerate(e):
            for _ in range(ei):
                term = term * x[:, i]
        out = out + term
    return out


def _poly_diff(mons, k):
    out = []
    for c, e in mons:
        if e[k] > 0:
            e2 = list(e)
            e2[k] -= 1
            out.append((c * e[k], tuple(e2)))
    return out


def _c4_accept(f_mons, n, lam, rng):
    """Input validation of DESIGN.md's C4 recipe: no cube vertex with |F| < 0.1
    and Im F(z) < 0 on 2^14 probe points."""
    verts = np.array(list(itertools.product([0.0, 1.0], repeat=n)))
    if np.min(np.abs(_poly_eval_f64(f_mons, verts))) < 0.1:
        return False
    x = rng.random((1 << 14, n))
    z = x.astype(np.complex128)
    for k in range(n):
        gk = _poly_eval_f64(_poly_diff(f_mons, k), x)
        z[:, k] = x[:, k] - 1j * lam * x[:, k] * (1.0 - x[:, k]) * gk
    fz = _poly_eval_f64(f_mons, z)
    return bool(np.all(fz.imag < 0))


def _c4(nsectors, rng_of, lam=0.5):
    n, K = 7, 4
    secs = []
    for s in range(nsectors):
        rng = rng_of(s)
        tries = 0
        while True:
            f = _draw_poly(rng, n, 3, int(rng.integers(28, 33)), 0.1, 3.0, neg_prob=0.3, neg_lo=-2.0, neg_hi=-0.1)
            tries += 1
            if _c4_accept(f, n, lam, rng):
                break
        a = tuple(int(v) for v in rng.integers(0, 2, size=n))
        u = _draw_poly(rng, n, 2, int(rng.integers(12, 17)), 0.1, 3.0)
        q = 2.0 if s % 2 == 0 else 2.5
        logs = [(None, 0)] + [_logpoly_text(rng, min(k, 2)) for k in range(1, K)]
        texts, ops = _family_sector(n, a, u, f, 1, q, [None] * K, logs)
        secs.append(SectorText(s, texts, is_complex=True, deform_f_index=2, lam=lam, naive_ops=ops,
                               meta=dict(a=a, q=q, tries=tries, f=f)))
    return n, K, secs


def _c5(nsectors, rng_of):
    n, K = 12, 1
    secs = []
    for s in range(nsectors):
        rng = rng_of(s)
        sing = sorted(int(v) for v in rng.choice(n, size=4, replace=False))
        num = _draw_poly(rng, n, 2, 12, 0.1, 3.0)
        den = _draw_poly(rng, n, 2, 13, 0.1, 3.0)
        nt, no = _poly_text(num)
        dt, do = _poly_text(den)
        sing_t = "*".join(f"p[x[{i + 1}],-0.7]" for i in sing)
        final = f"{sing_t}*f[1]/f[2]"
        ops = no + do + 4 + 3 + 2
        secs.append(SectorText(s, [_block(n, [nt, dt], final)], naive_ops=ops, meta=dict(singular=sing)))
    return n, K, secs


_FULL = {
    "C1": dict(S=1, npoints=1 << 16, R=1),
    "C2": dict(S=64, npoints=1 << 20, R=1),
    "C3": dict(S=2000, npoints=1 << 24, R=8),
    "C4": dict(S=500, npoints=1 << 22, R=1),
    "C5": dict(S=200, npoints=1 << 22, R=1),
}


def make_workload(name: str, nsectors: int | None = None, npoints: int | None = None,
                  n_shifts: int | None = None, first_sector: int = 0) -> Workload:
    """Build config `name` (C1..C5).  nsectors / npoints / n_shifts override the full sizes
    (reduced parity cases); sector s always gets the same texts whatever the overrides."""
    if name not in _FULL:
        raise ValueError(f"unknown config {name!r}")
    cfg = _FULL[name]
    S = cfg["S"] if nsectors is None else nsectors
    npts = cfg["npoints"] if npoints is None else npoints
    R = cfg["R"] if n_shifts is None else n_shifts
    ci = CONFIG_NAMES.index(name) + 1

    def rng_of(s):
        return np.random.default_rng([BASE_SEED, ci, first_sector + s])

    n, K, secs = {"C1": _c1, "C2": _c2, "C3": _c3, "C4": _c4, "C5": _c5}[name](S, rng_of)
    for s in secs:
        s.sector_id += first_sector
    if name == "C5":
        return Workload(name, n, K, secs, RULE_VEGAS, npts, vegas_bins=50, vegas_iters=10, vegas_alpha=1.5)
    return Workload(name, n, K, secs, RULE_LATTICE, npts, n_shifts=R,
                    korobov_a=korobov_a(npts // R, n), periodize_r=3)
