"""Shared by the GPU parity tests: oracle-side quantities for a workload sector.

Only tests import this.  It calls `oracle/` (CPU, long double) and never the CUDA path.
"""
import numpy as np

from oracle import deform as OD
from oracle import evaluate as OE
from oracle import integrate as OI
from oracle import points as OP
from oracle.integrate import SectorSpec

LD = np.longdouble
CLD = np.clongdouble

# Tolerances of BASELINE.json's north_star, with the readings R14 / R15 of DESIGN.md.
TOL_POINT = 1e-12    # |f_gpu - f_orc| <= TOL_POINT * M(x), M = magnitude companion (R14)
TOL_SUM = 1e-10      # |S_gpu - S_orc| <= TOL_SUM * |S_orc| + TOL_SUM_ABS * sum|g|   (R15)
TOL_SUM_ABS = 1e-13


def spec(s):
    return SectorSpec(s.texts, s.sector_id, s.is_complex, s.deform_f_index, s.lam)


def oracle_values_and_magnitude(sec, x):
    """o_k(x) [npts, K] (complex128-compatible long double) and M_k(x) [npts, K] (R14).

    Deformed sectors: the value is o_k(z) * det J.  The companion of det J is the permanent of |J|
    (Leibniz's formula with every term by its modulus: R14's rule on the determinant's definition),
    combined with the companion of o_k(z) by the product rule of oracle/evaluate.py."""
    x = np.asarray(x, dtype=LD)
    vals, mags = [], []
    z = det = dperm = None
    for prog in sec.progs:
        if sec.deform_f_index > 0:
            if z is None:      # the K texts share their f-lines: z and det J are common to the orders
                z, jac = OD.deform(prog, sec.deform_f_index, sec.lam, x, None, LD)
                det = OD.det_lu(jac)
                dperm = OD.permanent(np.abs(jac))
            v, m = OE.evaluate_with_magnitude(prog, z, CLD)
            av, ad = np.abs(v), np.abs(det)
            vals.append(v * det)
            mags.append(m * ad + av * dperm - av * ad)
        elif sec.is_complex:
            v, m = OE.evaluate_with_magnitude(prog, x.astype(CLD), CLD)
            vals.append(v)
            mags.append(m)
        else:
            v, m = OE.evaluate_with_magnitude(prog, x, LD)
            vals.append(v)
            mags.append(m)
    return np.stack(vals, axis=1), np.stack(mags, axis=1).astype(np.float64)


def check_points(got, ref, mag, tol=TOL_POINT, label=None):
    """got complex128 [npts,K]; ref long double (complex) [npts,K]; returns the worst ratio err/(tol*M).
    With a label, the margins (worst err/(tol*M), worst and median plain relative error err/|f|, median
    and worst M/|f|) are appended to gpurun_out/parity_margins.jsonl (R14: "the plain relative error is
    reported as well")."""
    d = np.abs(np.asarray(got, dtype=CLD) - np.asarray(ref, dtype=CLD)).astype(np.float64)
    ratio = d / (tol * mag)
    if label is not None:
        af = np.abs(np.asarray(ref, dtype=CLD)).astype(np.float64)
        ok = af > 0
        record_margin(label, npts=int(d.shape[0]), worst_err_over_tolM=float(np.max(ratio)),
                      worst_plain_rel=float(np.max(d[ok] / af[ok])), median_plain_rel=float(np.median(d[ok] / af[ok])),
                      median_M_over_f=float(np.median(mag[ok] / af[ok])), p90_M_over_f=float(np.percentile(mag[ok] / af[ok], 90)),
                      max_M_over_f=float(np.max(mag[ok] / af[ok])))
    return float(np.max(ratio))


def record_margin(label, **numbers):
    """Append one JSON line to gpurun_out/parity_margins.jsonl (scratch; summarised under profiles/)."""
    import json
    import os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = os.path.join(root, "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_margins.jsonl"), "a") as fh:
            fh.write(json.dumps(dict(label=label, **numbers)) + "\n")
    except OSError:
        pass


def genvec_of(wl):
    return OP.korobov_genvec(wl.korobov_a, wl.n_lattice, wl.dim)


def check_sums(gpu, s1, s2, sa, label=None):
    """gpu [R,K,C,2]; oracle s1,s2,sa [R,K,C].  Asserts R15."""
    s1f, s2f, saf = (np.asarray(a, dtype=np.float64) for a in (s1, s2, sa))
    e1 = np.abs(gpu[..., 0] - s1f)
    e2 = np.abs(gpu[..., 1] - s2f)
    if label is not None:
        record_margin(label, worst_S1_err_over_tol=float(np.max(e1 / (TOL_SUM * np.abs(s1f) + TOL_SUM_ABS * saf))),
                      worst_S1_plain_rel=float(np.max(e1 / np.abs(s1f))), worst_S2_rel=float(np.max(e2 / s2f)))
    assert np.all(e1 <= TOL_SUM * np.abs(s1f) + TOL_SUM_ABS * saf), (e1.max(), np.abs(s1f).min())
    assert np.all(e2 <= TOL_SUM * s2f), (e2 / s2f).max()
