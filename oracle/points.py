"""Oracle steps O3/O4: sample points on the unit cube.

The paper fixes only the domain: the unit cube with Lebesgue measure
("integrating x + 0.2 from 0 to 1") and that Vegas-type Monte
Carlo from the Cuba library draws the points.  It is
silent on the rule itself; BASELINE.json's north_star names it ("rank-1 Korobov
lattice with random shift and periodising transform, or Philox MC").  The
definitions below are DESIGN.md readings R1-R4.  Everything up to the 64-bit
integer t is exact integer arithmetic, so the CUDA path can be compared on t
bit for bit.

R1  rank-1 lattice, N_L = 2^m points, generating vector g_k = a^k mod N_L
    (Korobov form), k = 0..n-1, or an explicit vector.
R2  t_{j,k} = (((j*g_k) mod N_L) << (64-m)) + Delta_{r,k}   (mod 2^64)
    u = (2*(t >> 12) + 1) * 2^-53   in (0,1), exactly representable in FP64.
R3  Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), key = 64-bit seed as
    (lo32, hi32), counter = (j lo32, j hi32, sector_id, tag<<28 | kblock<<20 | it):
      tag 0 = lattice shift stream (j = 0, it = shift index r),
      tag 1 = Monte-Carlo stream   (j = point index, it = iteration index).
    One call yields coordinates 2*kblock and 2*kblock+1:
      t_even = out0*2^32 + out1,  t_odd = out2*2^32 + out3.
R4  Korobov periodising transform of weight r:
      w_r(u) = (2r+1)!/(r!)^2 u^r (1-u)^r,   phi_r(u) = int_0^u w_r,
    evaluated mirrored: v = min(u,1-u), p = phi_r(v); x = p (u<=1/2) or 1-p.
    r = 0: x = u, w = 1.
"""
from __future__ import annotations

import math

import numpy as np

LD = np.longdouble
U32 = np.uint32
U64 = np.uint64
MASK32 = 0xFFFFFFFF

PHILOX_M0 = 0xD2511F53
PHILOX_M1 = 0xCD9E8D57
PHILOX_W0 = 0x9E3779B9
PHILOX_W1 = 0xBB67AE85


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox4x32 with 10 rounds on arrays of 32-bit words (held in uint64).

    Round (Salmon et al., SC'11, sect. 3.3):  (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2,
    c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0); the key is bumped by (W0, W1) between rounds.
    """
    c0, c1, c2, c3 = (np.asarray(c, dtype=U64) & U64(MASK32) for c in (c0, c1, c2, c3))
    k0 = U64(int(k0) & MASK32)
    k1 = U64(int(k1) & MASK32)
    for rnd in range(10):
        if rnd > 0:
            k0 = U64((int(k0) + PHILOX_W0) & MASK32)
            k1 = U64((int(k1) + PHILOX_W1) & MASK32)
        p0 = U64(PHILOX_M0) * c0  # < 2^64, exact in uint64
        p1 = U64(PHILOX_M1) * c2
        hi0, lo0 = p0 >> U64(32), p0 & U64(MASK32)
        hi1, lo1 = p1 >> U64(32), p1 & U64(MASK32)
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
    return c0, c1, c2, c3


TAG_SHIFT = 0
TAG_MC = 1


def _counter_word3(tag: int, kblock: int, it: int) -> int:
    if not (0 <= tag < 16 and 0 <= kblock < 256 and 0 <= it < (1 << 20)):
        raise ValueError("tag < 16, kblock < 256, iteration/shift index < 2^20 required")
    return (tag << 28) | (kblock << 20) | it


def philox_t(seed: int, sector_id: int, tag: int, it: int, j, dim: int):
    """64-bit integers t[j, k], k < dim, from the Philox stream (R3).  j: uint64 array."""
    j = np.atleast_1d(np.asarray(j, dtype=U64))
    out = np.empty((j.shape[0], dim), dtype=U64)
    jlo, jhi = j & U64(MASK32), j >> U64(32)
    sec = np.full_like(j, sector_id & MASK32)
    for kb in range((dim + 1) // 2):
        w3 = np.full_like(j, _counter_word3(tag, kb, it))
        o0, o1, o2, o3 = philox4x32_10(jlo, jhi, sec, w3, seed & MASK32, (seed >> 32) & MASK32)
        out[:, 2 * kb] = (o0 << U64(32)) | o1
        if 2 * kb + 1 < dim:
            out[:, 2 * kb + 1] = (o2 << U64(32)) | o3
    return out


def lattice_shift(seed: int, sector_id: int, r: int, dim: int):
    """Delta_{r,k}: the 64-bit random shift of shift index r (R3, tag 0, j = 0)."""
    return philox_t(seed, sector_id, TAG_SHIFT, r, np.zeros(1, dtype=U64), dim)[0]


def korobov_genvec(a: int, n_lattice: int, dim: int):
    """g_k = a^k mod N_L, k = 0..dim-1  (R1)."""
    g, out = 1, []
    for _ in range(dim):
        out.append(g)
        g = (g * a) % n_lattice
    return out


def lattice_t(j, genvec, n_lattice: int, shift):
    """t[j, k] = (((j*g_k) mod N_L) << (64-m)) + Delta_k  mod 2^64, N_L = 2^m  (R2)."""
    m = n_lattice.bit_length() - 1
    if n_lattice != 1 << m or not 0 <= m <= 40:
        raise ValueError("lattice size must be a power of two, at most 2^40")
    j = np.atleast_1d(np.asarray(j, dtype=U64))
    out = np.empty((j.shape[0], len(genvec)), dtype=U64)
    for k, g in enumerate(genvec):
        if not 0 <= g < n_lattice:
            raise ValueError("generating vector entries must lie in [0, N_L)")
        # j < 2^40 and g < 2^40 could overflow 64 bits; reduce j first, the product of
        # two m-bit numbers is taken modulo 2^64 and then modulo 2^m, which is exact.
        jm = j & U64(n_lattice - 1)
        with np.errstate(over="ignore"):
            r = (jm * U64(g)) & U64(n_lattice - 1)
            out[:, k] = (r << U64(64 - m)) + U64(int(shift[k])) if m > 0 else np.full_like(r, int(shift[k]))
    return out


def unit_from_t(t, dtype=LD):
    """u = (2*(t>>12)+1) * 2^-53  (R2): 52 bits, mid-point offset, never 0 or 1."""
    s = np.asarray(t, dtype=U64) >> U64(12)
    # s < 2^52 converts exactly to FP64 and to long double.
    return (dtype(2) * s.astype(dtype) + dtype(1)) * dtype(2.0 ** -53)


def _phi_small(v, r: int):
    """phi_r(v) = C * sum_i binom(r,i) (-1)^i v^(r+1+i)/(r+1+i), C = (2r+1)!/(r!)^2."""
    c = math.factorial(2 * r + 1) // (math.factorial(r) ** 2)
    dt = v.dtype.type
    acc = np.zeros_like(v)
    for i in range(r + 1):
        coef = dt(c * math.comb(r, i) * (-1) ** i) / dt(r + 1 + i)
        acc = acc + coef * v ** (r + 1 + i)
    return acc


def korobov_transform(u, r: int):
    """(x, xbar, w) for x = phi_r(u), xbar = 1 - x, w = w_r(u), elementwise  (R4)."""
    u = np.asarray(u)
    dt = u.dtype.type
    if r == 0:
        return u, dt(1) - u, np.ones_like(u)
    if r < 0:
        raise ValueError("r >= 0")
    ubar = dt(1) - u  # exact: u = odd*2^-53
    v = np.minimum(u, ubar)
    p = _phi_small(v, r)
    big = dt(1) - p
    left = u <= ubar
    x = np.where(left, p, big)
    xbar = np.where(left, big, p)
    c = math.factorial(2 * r + 1) // (math.factorial(r) ** 2)
    w = dt(c) * (u * ubar) ** r
    return x, xbar, w
