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
    """o_k(x) [npts, K] (complex128-compatible long double) and M_k(x) [npts, K]."""
    x = np.asarray(x, dtype=LD)
    vals, mags = [], []
    for prog in sec.progs:
        if sec.deform_f_index > 0:
            z, jac = OD.deform(prog, sec.deform_f_index, sec.lam, x, None, LD)
            det = OD.det_lu(jac)
            v, m = OE.evaluate_with_magnitude(prog, z, CLD)
            # |det J| <= prod_k sum_l |J_kl| bounds the magnitude of the determinant's own rounding
            dm = np.prod(np.sum(np.abs(jac), axis=2), axis=1)
            vals.append(v * det)
            mags.append(m * dm)
        elif sec.is_complex:
            v, m = OE.evaluate_with_magnitude(prog, x.astype(CLD), CLD)
            vals.append(v)
            mags.append(m)
        else:
            v, m = OE.evaluate_with_magnitude(prog, x, LD)
            vals.append(v)
            mags.append(m)
    return np.stack(vals, axis=1), np.stack(mags, axis=1).astype(np.float64)


def check_points(got, ref, mag, tol=TOL_POINT):
    """got complex128 [npts,K]; ref long double (complex) [npts,K]; returns the worst ratio err/(tol*M)."""
    d = np.abs(np.asarray(got, dtype=CLD) - np.asarray(ref, dtype=CLD)).astype(np.float64)
    ratio = d / (tol * mag)
    return float(np.max(ratio))


def genvec_of(wl):
    return OP.korobov_genvec(wl.korobov_a, wl.n_lattice, wl.dim)


def check_sums(gpu, s1, s2, sa):
    """gpu [R,K,C,2]; oracle s1,s2,sa [R,K,C].  Asserts R15."""
    s1f, s2f, saf = (np.asarray(a, dtype=np.float64) for a in (s1, s2, sa))
    e1 = np.abs(gpu[..., 0] - s1f)
    assert np.all(e1 <= TOL_SUM * np.abs(s1f) + TOL_SUM_ABS * saf), (e1.max(), np.abs(s1f).min())
    e2 = np.abs(gpu[..., 1] - s2f)
    assert np.all(e2 <= TOL_SUM * s2f), (e2 / s2f).max()
