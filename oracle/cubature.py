"""Oracle for the deterministic integrator (R21): a Cuhre-like globally adaptive
cubature on the same integrand evaluator.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): the product never imports this.

The paper integrates through the Cuba library, whose Cuhre is "a deterministic algorithm which uses one
of several cubature rules of polynomial degree in a globally adaptive subdivision scheme"
(`CurrentIntegrator -> cuhreCuba`).  The paper does not spell the algorithm out; the
reading R21 fixes it as the classic scheme of Genz and Malik (J. Comput. Appl. Math. 6 (1980) 295),
restated here step by step in long double:

  rule       on a box with centre c and half-widths h (n >= 2 dimensions) the degree-7 rule I7 with its
             embedded degree-5 rule I5 on the same 1 + 4n + 2n(n-1) + 2^n nodes; err = |I7 - I5| per
             component (order k, Re / Im);
  split axis the axis with the largest fourth divided difference
                 D_i = sum_comp | f(c + l2 h_i e_i) + f(c - l2 h_i e_i) - 2 f(c)
                                  - (l2/l3)^2 ( f(c + l3 h_i e_i) + f(c - l3 h_i e_i) - 2 f(c) ) |,
             ties to the lowest index;
  rounds     start from the unit cube.  After every round I = sum I7 and E = sum err over the current boxes.
             Stop when E <= max(epsabs, epsrel |I|) for every component, or when the next round would exceed
             maxeval integrand evaluations.  Otherwise order the boxes by e = sum_comp err, largest first
             (ties: the older box), take the shortest prefix that carries at least half of sum e -- cut to
             what maxeval still allows -- and halve each of its boxes along its split axis; the two
             halves (lower first) go to the end of the list.

Cuhre proper splits one box per step from a heap and uses a family of null rules for err; halving the worst
half of the error per round is the breadth-first version a GPU wants, with the same fixed point.
"""
from __future__ import annotations

import itertools

import numpy as np

from .integrate import LD, SectorSpec, integrand_values

L2 = np.sqrt(LD(9) / LD(70))
L3 = np.sqrt(LD(9) / LD(10))
L5 = np.sqrt(LD(9) / LD(19))


def genz_malik(n: int):
    """(offsets [NN, n] in units of the half-widths, w7 [NN], w5 [NN]); weights sum to 1 (a mean over the box).

    Node order: centre; +-l2 along axis 0, 1, ...; +-l3 along axis 0, 1, ...; for every pair i < j the four
    (+-l3, +-l3) (signs ++, -+, +-, --); the 2^n corners (+-l5, ..., +-l5), bit k of the corner number set:
    coordinate k negative."""
    if n < 2:
        raise ValueError("the Genz-Malik rule needs n >= 2")
    w1 = LD(12824 - 9120 * n + 400 * n * n) / LD(19683)
    w2 = LD(980) / LD(6561)
    w3 = LD(1820 - 400 * n) / LD(19683)
    w4 = LD(200) / LD(19683)
    w5 = LD(6859) / LD(19683) / LD(2 ** n)
    e1 = LD(729 - 950 * n + 50 * n * n) / LD(729)
    e2 = LD(245) / LD(486)
    e3 = LD(265 - 100 * n) / LD(1458)
    e4 = LD(25) / LD(729)
    off, w7, w5l = [np.zeros(n, dtype=LD)], [w1], [e1]
    for lam, a, b in ((L2, w2, e2), (L3, w3, e3)):
        for i in range(n):
            for s in (1, -1):
                v = np.zeros(n, dtype=LD)
                v[i] = s * lam
                off.append(v)
                w7.append(a)
                w5l.append(b)
    for i, j in itertools.combinations(range(n), 2):
        for sj in (1, -1):
            for si in (1, -1):
                v = np.zeros(n, dtype=LD)
                v[i], v[j] = si * L3, sj * L3
                off.append(v)
                w7.append(w4)
                w5l.append(e4)
    for corner in range(2 ** n):
        v = np.array([-L5 if (corner >> k) & 1 else L5 for k in range(n)], dtype=LD)
        off.append(v)
        w7.append(w5)
        w5l.append(LD(0))
    return np.stack(off), np.array(w7, dtype=LD), np.array(w5l, dtype=LD)


def rule_on_box(f, c, h, tables=None):
    """f: points [npts, n] -> values [ncomp, npts].  Returns I7 [ncomp], I5 [ncomp], D [n] for the box (c, h)."""
    c, h = np.asarray(c, dtype=LD), np.asarray(h, dtype=LD)
    n = c.shape[0]
    off, w7, w5 = tables or genz_malik(n)
    vals = f(c[None, :] + off * h[None, :])
    vol = np.prod(2 * h)
    i7 = vol * np.sum(vals * w7[None, :], axis=1)
    i5 = vol * np.sum(vals * w5[None, :], axis=1)
    f0 = vals[:, 0]
    ratio = (L2 / L3) ** 2
    d = np.zeros(n, dtype=LD)
    for i in range(n):
        a = vals[:, 1 + 2 * i] + vals[:, 2 + 2 * i] - 2 * f0
        b = vals[:, 1 + 2 * n + 2 * i] + vals[:, 2 + 2 * n + 2 * i] - 2 * f0
        d[i] = np.sum(np.abs(a - ratio * b))
    return i7, i5, d


def sector_components(sec: SectorSpec):
    """The integrand of a sector as f(points) -> [ncomp, npts] real components: order k, then Re / Im."""
    cplx = sec.is_complex or sec.deform_f_index > 0

    def f(x):
        v = integrand_values(sec, x)
        if cplx:
            return np.concatenate([np.stack([v[k].real, v[k].imag]) for k in range(sec.K)]).astype(LD)
        return np.asarray(v, dtype=LD)
    return f


def integrate_cubature(f, n, epsrel=1e-6, epsabs=0.0, maxeval=1 << 20, return_boxes=False):
    """The rounds described in the module docstring.  Returns (I [ncomp], E [ncomp], neval, nboxes)."""
    tables = genz_malik(n)
    nn = tables[0].shape[0]
    boxes = []          # dicts: c, h, i7, err, axis
    fresh = [(np.full(n, LD(0.5)), np.full(n, LD(0.5)))]
    neval = 0
    while True:
        for c, h in fresh:
            i7, i5, d = rule_on_box(f, c, h, tables)
            boxes.append({"c": c, "h": h, "i7": i7, "err": np.abs(i7 - i5), "axis": int(np.argmax(d))})
        neval += nn * len(fresh)
        total = np.sum([b["i7"] for b in boxes], axis=0)
        err = np.sum([b["err"] for b in boxes], axis=0)
        if np.all(err <= np.maximum(LD(epsabs), LD(epsrel) * np.abs(total))):
            break
        room = (maxeval - neval) // (2 * nn)
        if room < 1:
            break
        e = np.array([float(np.sum(b["err"])) for b in boxes])
        order = sorted(range(len(boxes)), key=lambda i: (-e[i], i))
        chosen, acc, half = [], 0.0, 0.5 * float(np.sum(e))
        for i in order:
            if len(chosen) >= room:
                break
            chosen.append(i)
            acc += e[i]
            if acc >= half:
                break
        fresh = []
        for i in chosen:
            b = boxes[i]
            a = b["axis"]
            for s in (-1, 1):
                c, h = b["c"].copy(), b["h"].copy()
                h[a] = h[a] / 2
                c[a] = c[a] + s * h[a]
                fresh.append((c, h))
        keep = set(chosen)
        boxes = [b for i, b in enumerate(boxes) if i not in keep]
    if return_boxes:
        return total, err, neval, boxes
    return total, err, neval, len(boxes)
