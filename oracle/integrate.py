"""Oracle steps O6-O8: sums, estimates and errors, Vegas.

What the paper fixes: each integrand yields a value and an error estimate
"produced by the integrator"; per-order totals are sums of the values and the
errors are combined "using the mean-square norm ... treat this number as the
delta value (standard deviation)".  Vegas (Cuba) is the default
integrator.  The estimators and Vegas internals are not in the
paper; they are DESIGN.md readings R5-R8, restated here step by step.

A sector is described by plain data (no CUDA-path types):
    SectorSpec(texts=[K expression blocks], sector_id, is_complex,
               deform_f_index, lam)
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import points as P
from .deform import evaluate_deformed
from .evaluate import evaluate, LD, CLD
from .parser import parse

U64 = np.uint64


@dataclass
class SectorSpec:
    texts: list                 # K expression blocks in the paper's grammar
    sector_id: int = 0
    is_complex: bool = False    # PAPER.md:477 (-complex)
    deform_f_index: int = 0     # >=1: f[deform_f_index] is the polynomial F of the deformation
    lam: float = 0.0
    progs: list = field(default_factory=list)

    def __post_init__(self):
        if not self.progs:
            self.progs = [parse(t) for t in self.texts]
        self.dim = self.progs[0].nvars
        self.K = len(self.progs)


def neumaier_sum(values):
    """Compensated sum of a 1-D long-double array in index order (kept for small arrays)."""
    s = values.dtype.type(0)
    c = values.dtype.type(0)
    for v in values:
        t = s + v
        if abs(s) >= abs(v):
            c += (s - t) + v
        else:
            c += (v - t) + s
        s = t
    return s + c


_BIAS = 16600  # long double exponents lie in (-16446, 16385): value = integer * 2^-(_BIAS+64)


class ExactSum:
    """O6: sum_j v_j as the plain definition -- the EXACT sum of the terms, rounded once at the end.

    Every finite long double is an integer times a power of two, v = M * 2^(e-64) with
    |M| < 2^64 (np.frexp).  The integers M are added without rounding (numpy int64 per
    exponent value, then Python integers), so the order of the terms, and how a caller feeds
    them in pieces, cannot change the result.  NaN / Inf terms make the sum NaN / Inf.
    """

    def __init__(self):
        self.total = 0          # exact sum = total * 2^-(_BIAS+64)
        self.special = LD(0)    # plain sum of the non-finite terms (propagates NaN / Inf)
        self.has_special = False

    def add(self, values):
        v = np.asarray(values, dtype=LD).ravel()
        fin = np.isfinite(v)
        if not np.all(fin):
            self.special = self.special + np.sum(v[~fin])
            self.has_special = True
            v = v[fin]
        for i in range(0, v.shape[0], 1 << 20):
            self._add_finite(v[i:i + (1 << 20)])
        return self

    def _add_finite(self, v):
        if v.shape[0] == 0:
            return
        m, e = np.frexp(v)                       # v = m * 2^e, 0.5 <= |m| < 1 (or m = 0)
        a = np.abs(m) * LD(2.0 ** 32)
        hi = np.floor(a)                         # top 32 bits of the 64-bit integer mantissa
        lo = (a - hi) * LD(2.0 ** 32)            # low 32 bits; both conversions are exact
        sign = np.where(m < 0, -1.0, 1.0)
        e0 = int(e.min())
        idx = (e - e0).astype(np.int64)
        # per exponent, sums of at most 2^20 integers < 2^32: exact in float64
        shi = np.bincount(idx, weights=hi.astype(np.float64) * sign)
        slo = np.bincount(idx, weights=lo.astype(np.float64) * sign)
        for k in np.nonzero((shi != 0) | (slo != 0))[0]:
            part = (int(shi[k]) << 32) + int(slo[k])
            self.total += part << (int(k) + e0 + _BIAS)

    def value(self):
        if self.has_special:
            return self.special
        n = abs(self.total)
        if n == 0:
            return LD(0)
        shift = max(n.bit_length() - 64, 0)
        q, rem = n >> shift, n & ((1 << shift) - 1)
        if shift and (rem > (1 << (shift - 1)) or (rem == (1 << (shift - 1)) and (q & 1))):
            q += 1                               # round to nearest, ties to even
        x = LD(float(q >> 32)) * LD(2.0 ** 32) + LD(float(q & 0xFFFFFFFF))   # halves < 2^33: exact
        x = np.ldexp(x, shift - _BIAS - 64)
        return -x if self.total < 0 else x


def exact_sum(values):
    """Exact sum of an array of long doubles, rounded once (see ExactSum)."""
    return ExactSum().add(values).value()


def integrand_values(sec: SectorSpec, x, xbar=None, rdtype=LD, small_x=0.0):
    """o_k at the points, shape [K, npts]; complex dtype if the sector is complex.

    With deformation every x becomes z(x) and the result is multiplied by det J (R11).
    The lattice / Vegas weight W is NOT included.

    small_x > 0 (real sectors; the paper's "Mixed" mode, with its SmallX knob,
    PAPER.md:447; R20): a point whose FP64 coordinates have min_k x_k < small_x takes its
    value from the multiple-precision walk (oracle/evaluate_mp.py, FP64 constants) at that FP64
    point, rounded to FP64.
    """
    cdtype = CLD if rdtype == LD else np.complex128
    out = []
    for prog in sec.progs:
        if sec.deform_f_index > 0:
            out.append(evaluate_deformed(prog, sec.deform_f_index, sec.lam, x, xbar, rdtype))
        elif sec.is_complex:
            out.append(evaluate(prog, np.asarray(x, dtype=rdtype).astype(cdtype), cdtype))
        else:
            out.append(evaluate(prog, x, rdtype))
    if small_x > 0.0:
        if sec.is_complex or sec.deform_f_index > 0:
            raise ValueError("the mixed mode is defined for real sectors")
        from .evaluate_mp import evaluate_mp
        x64 = np.asarray(x, dtype=np.float64)
        flagged = np.nonzero(np.min(x64, axis=1) < small_x)[0]
        for k, prog in enumerate(sec.progs):
            for j, v in zip(flagged, evaluate_mp(prog, x64[flagged], const64=True)):
                out[k][j] = rdtype(float(v))
    return np.stack(out)


def _components(g):
    """Real sectors: [g]; complex: [Re g, Im g] (each its own estimate, R5)."""
    return [g.real, g.imag] if np.iscomplexobj(g) else [g]


def lattice_points(sec: SectorSpec, n_lattice, genvec, r_periodize, seed, shift_index, first, count, rdtype=LD):
    """x, xbar, W (product of w_r) of lattice points j = first..first+count-1 of one shift."""
    j = np.arange(first, first + count, dtype=U64)
    delta = P.lattice_shift(seed, sec.sector_id, shift_index, sec.dim)
    t = P.lattice_t(j, genvec, n_lattice, delta)
    u = P.unit_from_t(t, rdtype)
    x, xbar, w = P.korobov_transform(u, r_periodize)
    return x, xbar, np.prod(w, axis=1)


def lattice_partial_sums(sec: SectorSpec, n_lattice, n_shifts, genvec, r_periodize, seed, chunk=1 << 14, rdtype=LD,
                         shifts=None, first=0, count=None, small_x=0.0):
    """S1[r,k,c] = sum_j g, S2[r,k,c] = sum_j g^2, SA[r,k,c] = sum_j |g|, g = W*o_k component c.

    Shapes [R, K, C], C = 1 (real) or 2 (Re, Im).  Each sum is the exact sum of its terms rounded
    once (O6, ExactSum); `chunk` only bounds the memory of one evaluation and cannot change a result.
    `shifts`: optional subset of shift indices to compute (the other rows stay 0); `first`, `count`:
    optional sub-range j = first..first+count-1 of the lattice; both are used to sample pieces of a
    full-size run.  `small_x`: the mixed mode of integrand_values.
    """
    ncomp = 2 if (sec.is_complex or sec.deform_f_index > 0) else 1
    s1 = np.zeros((n_shifts, sec.K, ncomp), dtype=rdtype)
    s2 = np.zeros_like(s1)
    sa = np.zeros_like(s1)
    last = n_lattice if count is None else first + count
    for r in (range(n_shifts) if shifts is None else shifts):
        acc = [[[ExactSum(), ExactSum(), ExactSum()] for _ in range(ncomp)] for _ in range(sec.K)]
        for f0 in range(first, last, chunk):
            cnt = min(chunk, last - f0)
            x, xbar, w = lattice_points(sec, n_lattice, genvec, r_periodize, seed, r, f0, cnt, rdtype)
            vals = integrand_values(sec, x, xbar, rdtype, small_x)
            for k in range(sec.K):
                for c, comp in enumerate(_components(vals[k])):
                    g = w * comp
                    acc[k][c][0].add(g)
                    acc[k][c][1].add(g * g)
                    acc[k][c][2].add(np.abs(g))
        for k in range(sec.K):
            for c in range(ncomp):
                s1[r, k, c] = acc[k][c][0].value()
                s2[r, k, c] = acc[k][c][1].value()
                sa[r, k, c] = acc[k][c][2].value()
    return s1, s2, sa


def estimate_from_sums(s1, s2, n_per_shift):
    """(value, sigma) from per-shift sums (R5).

    R >= 2 shifts:  Q_r = S1_r/N_L, value = mean_r Q_r,
                    sigma = sqrt( sum_r (Q_r - value)^2 / (R (R-1)) ).
    R == 1 (or plain MC): value = <g>, sigma = sqrt( (<g^2> - <g>^2) / (N-1) ), clamped at 0.
    Leading axis of s1, s2 is the shift index.
    """
    dt = s1.dtype.type
    nshift = s1.shape[0]
    q = s1 / dt(n_per_shift)
    if nshift >= 2:
        value = np.sum(q, axis=0) / dt(nshift)
        var = np.sum((q - value) ** 2, axis=0) / dt(nshift * (nshift - 1))
    else:
        value = q[0]
        var = (s2[0] / dt(n_per_shift) - value * value) / dt(n_per_shift - 1)
    return value, np.sqrt(np.maximum(var, 0))


def integrate_lattice(sec: SectorSpec, npoints, n_shifts, genvec, r_periodize, seed, chunk=1 << 14, rdtype=LD):
    """value[K,C], sigma[K,C] of one sector; npoints = R * N_L total (R6)."""
    n_lattice = npoints // n_shifts
    s1, s2, _ = lattice_partial_sums(sec, n_lattice, n_shifts, genvec, r_periodize, seed, chunk, rdtype)
    return estimate_from_sums(s1, s2, n_lattice)


def mc_points(sec: SectorSpec, seed, iteration, first, count, rdtype=LD):
    """y[j,:] uniform in the cube from the Philox MC stream (R3), as (t integers, y)."""
    j = np.arange(first, first + count, dtype=U64)
    t = P.philox_t(seed, sec.sector_id, P.TAG_MC, iteration, j, sec.dim)
    return t, P.unit_from_t(t, rdtype)


def mc_partial_sums(sec: SectorSpec, npoints, seed, iteration=0, chunk=1 << 14, rdtype=LD, first=0, count=None,
                    small_x=0.0):
    """Plain MC (x = u, W = 1): S1[k,c] = sum_j o_k, S2[k,c] = sum_j o_k^2 over points first..first+count-1
    of the Philox MC stream (default: all npoints); exact sums rounded once (O6)."""
    ncomp = 2 if (sec.is_complex or sec.deform_f_index > 0) else 1
    acc = [[[ExactSum(), ExactSum()] for _ in range(ncomp)] for _ in range(sec.K)]
    last = npoints if count is None else first + count
    for f0 in range(first, last, chunk):
        cnt = min(chunk, last - f0)
        _, y = mc_points(sec, seed, iteration, f0, cnt, rdtype)
        vals = integrand_values(sec, y, None, rdtype, small_x)
        for k in range(sec.K):
            for c, comp in enumerate(_components(vals[k])):
                acc[k][c][0].add(comp)
                acc[k][c][1].add(comp * comp)
    s1 = np.array([[acc[k][c][0].value() for c in range(ncomp)] for k in range(sec.K)], dtype=rdtype)
    s2 = np.array([[acc[k][c][1].value() for c in range(ncomp)] for k in range(sec.K)], dtype=rdtype)
    return s1, s2


def integrate_mc(sec: SectorSpec, npoints, seed, chunk=1 << 14, rdtype=LD):
    """Plain Monte Carlo: x = u, W = 1; value, sigma per (order, component) (R5)."""
    s1, s2 = mc_partial_sums(sec, npoints, seed, 0, chunk, rdtype)
    return estimate_from_sums(s1[None], s2[None], npoints)


# ----------------------------------------------------------------------------- Vegas (R8)

def vegas_uniform_grid(dim, nbins, rdtype=LD):
    return np.tile(np.arange(nbins + 1, dtype=rdtype) / rdtype(nbins), (dim, 1))


def vegas_bin_and_frac(t, nbins, rdtype=LD):
    """b = floor(y*NB) and frac = y*NB - b with y = (2s+1)/2^53, s = t>>12: exact integers (R8)."""
    s = np.asarray(t, dtype=U64) >> U64(12)
    prod = (U64(2) * s + U64(1)) * U64(nbins)   # < 2^53 * NB < 2^64 for NB < 2048
    b = (prod >> U64(53)).astype(np.int64)
    rem = prod & U64((1 << 53) - 1)
    return b, rem.astype(rdtype) * rdtype(2.0 ** -53)


def vegas_map(t, grid, rdtype=LD):
    """x[j,d] = xi_b + frac*(xi_{b+1}-xi_b), W[j] = prod_d NB*(xi_{b+1}-xi_b), bins b[j,d]."""
    dim, nb1 = grid.shape
    nbins = nb1 - 1
    b, frac = vegas_bin_and_frac(t, nbins, rdtype)
    x = np.empty(b.shape, dtype=rdtype)
    w = np.ones(b.shape[0], dtype=rdtype)
    for d in range(dim):
        lo = grid[d][b[:, d]]
        width = grid[d][b[:, d] + 1] - lo
        x[:, d] = lo + frac[:, d] * width
        w = w * (rdtype(nbins) * width)
    return x, w, b


def vegas_refine(grid_d, hist_d, alpha):
    """New edges of one dimension from its histogram (R8, sub-steps i-iv)."""
    dt = grid_d.dtype.type
    nb = hist_d.shape[0]
    h = hist_d
    # (i) smooth
    sm = np.empty_like(h)
    sm[0] = (h[0] + h[1]) / dt(2)
    sm[-1] = (h[-2] + h[-1]) / dt(2)
    sm[1:-1] = (h[:-2] + h[1:-1] + h[2:]) / dt(3)
    tot = np.sum(sm)
    if not tot > 0:
        return grid_d.copy()
    # (ii) normalise
    p = sm / tot
    # (iii) compress
    m = np.zeros_like(p)
    mid = (p > 0) & (p < 1)
    with np.errstate(all="ignore"):
        m[mid] = ((dt(1) - p[mid]) / (-np.log(p[mid]))) ** dt(alpha)
    m[p >= 1] = dt(1)
    # (iv) re-bin: equal sum(m)/NB in every new bin, linear interpolation inside old bins
    cum = np.zeros(nb + 1, dtype=grid_d.dtype)
    for b in range(nb):
        cum[b + 1] = cum[b] + m[b]
    new = np.empty_like(grid_d)
    new[0] = dt(0)
    new[nb] = dt(1)
    for i in range(1, nb):
        target = dt(i) * cum[nb] / dt(nb)
        k = int(np.sum(cum[1:nb] <= target))      # cum[k] <= target < cum[k+1]
        new[i] = grid_d[k] + (target - cum[k]) / m[k] * (grid_d[k + 1] - grid_d[k])
    return new


def vegas_iteration_sums(sec: SectorSpec, grid, npoints, seed, iteration, chunk=1 << 14, rdtype=LD, small_x=0.0):
    """S1[K,C], S2[K,C] and histogram h[dim, NB] (sum over orders/components of g^2) of one iteration.
    `small_x`: the mixed mode of integrand_values (decided on the mapped point x).

    All three are exact sums of their terms rounded once (O6, ExactSum): the histogram bin h[d][b]
    is the sum of g^2 over the points whose coordinate d falls in bin b."""
    ncomp = 2 if (sec.is_complex or sec.deform_f_index > 0) else 1
    nbins = grid.shape[1] - 1
    acc = [[[ExactSum(), ExactSum()] for _ in range(ncomp)] for _ in range(sec.K)]
    hacc = [[ExactSum() for _ in range(nbins)] for _ in range(sec.dim)]
    for first in range(0, npoints, chunk):
        cnt = min(chunk, npoints - first)
        t, _ = mc_points(sec, seed, iteration, first, cnt, rdtype)
        x, w, b = vegas_map(t, grid, rdtype)
        vals = integrand_values(sec, x, None, rdtype, small_x)
        g2 = np.zeros(cnt, dtype=rdtype)
        for k in range(sec.K):
            for c, comp in enumerate(_components(vals[k])):
                g = w * comp
                acc[k][c][0].add(g)
                acc[k][c][1].add(g * g)
                g2 = g2 + g * g
        for d in range(sec.dim):
            order = np.argsort(b[:, d], kind="stable")
            bs, gs = b[order, d], g2[order]
            cuts = np.searchsorted(bs, np.arange(nbins + 1))
            for bb in range(nbins):
                if cuts[bb + 1] > cuts[bb]:
                    hacc[d][bb].add(gs[cuts[bb]:cuts[bb + 1]])
    s1 = np.array([[acc[k][c][0].value() for c in range(ncomp)] for k in range(sec.K)], dtype=rdtype)
    s2 = np.array([[acc[k][c][1].value() for c in range(ncomp)] for k in range(sec.K)], dtype=rdtype)
    hist = np.array([[hacc[d][bb].value() for bb in range(nbins)] for d in range(sec.dim)], dtype=rdtype)
    return s1, s2, hist


def vegas_combine(i_it, var_it):
    """Weighted average over iterations, sigma, chi2 (R8).  Arrays [iters, ...]."""
    dt = i_it.dtype.type
    var = np.maximum(var_it, 0)
    pos = var > 0
    value = np.empty(i_it.shape[1:], dtype=i_it.dtype)
    sigma = np.empty_like(value)
    chi2 = np.empty_like(value)
    for idx in np.ndindex(value.shape):
        v = var[(slice(None),) + idx]
        i = i_it[(slice(None),) + idx]
        if not np.any(v > 0):
            value[idx], sigma[idx], chi2[idx] = np.sum(i) / dt(len(i)), dt(0), dt(0)
            continue
        v = np.where(v > 0, v, np.min(v[v > 0]))
        wgt = dt(1) / v
        value[idx] = np.sum(i * wgt) / np.sum(wgt)
        sigma[idx] = dt(1) / np.sqrt(np.sum(wgt))
        chi2[idx] = np.sum((i - value[idx]) ** 2 * wgt)
    return value, sigma, chi2


def integrate_vegas(sec: SectorSpec, npoints_per_iter, seed, nbins=50, iters=10, alpha=1.5, chunk=1 << 14,
                    rdtype=LD, trace=None, small_x=0.0):
    """Classic Lepage Vegas as restated in DESIGN.md R8.  Returns value, sigma, chi2 [K,C], final grid.

    `trace`, if a list, receives per iteration a dict(grid=, s1=, s2=, hist=, I=, var=).
    """
    grid = vegas_uniform_grid(sec.dim, nbins, rdtype)
    n = rdtype(npoints_per_iter)
    i_list, v_list = [], []
    for it in range(iters):
        s1, s2, hist = vegas_iteration_sums(sec, grid, npoints_per_iter, seed, it, chunk, rdtype, small_x)
        i_it = s1 / n
        var_it = (s2 / n - i_it * i_it) / (n - rdtype(1))
        i_list.append(i_it)
        v_list.append(var_it)
        if trace is not None:
            trace.append(dict(grid=grid.copy(), s1=s1, s2=s2, hist=hist.copy(), I=i_it, var=var_it))
        grid = np.stack([vegas_refine(grid[d], hist[d], alpha) for d in range(sec.dim)])
    value, sigma, chi2 = vegas_combine(np.stack(i_list), np.stack(v_list))
    return value, sigma, chi2, grid


def combine_sectors(values, sigmas):
    """Sum over sectors (leading axis): sum of values, sqrt of the sum of sigma^2."""
    return np.sum(values, axis=0), np.sqrt(np.sum(np.asarray(sigmas) ** 2, axis=0))
