// fx_math.cuh -- scalar helpers of the device path: complex FP64 arithmetic, Philox4x32-10,
// lattice integers, the Korobov periodising transform and the Vegas grid map.
// Definitions: DESIGN.md R2 (integers t and u), R3 (Philox counter layout), R4 (transform),
// R8 (Vegas map), R9/R10 (principal log / power).  The paper itself fixes only the unit-cube
// domain and the complex mode.
#ifndef FX_MATH_CUH
#define FX_MATH_CUH

#include <stdint.h>

struct cplx {
  double re, im;
};

// ---- overloaded arithmetic used by the interpreter handlers (T = double or cplx) ----------
__device__ __forceinline__ double t_fma(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ double t_fma_c(double a, double b, double c) { return fma(a, b, c); }  // c real
__device__ __forceinline__ double t_fma_rc(double r, double c, double a) { return fma(r, c, a); }  // r*c + a
__device__ __forceinline__ double t_mul(double a, double b) { return a * b; }
__device__ __forceinline__ double t_mulc(double a, double c) { return a * c; }
__device__ __forceinline__ double t_add(double a, double b) { return a + b; }
__device__ __forceinline__ double t_addc(double a, double c) { return a + c; }
__device__ __forceinline__ double t_sub(double a, double b) { return a - b; }
__device__ __forceinline__ double t_rsubc(double c, double a) { return c - a; }
__device__ __forceinline__ double t_div(double a, double b) { return a / b; }
__device__ __forceinline__ double t_divc(double a, double c) { return a / c; }
__device__ __forceinline__ double t_rdivc(double c, double a) { return c / a; }
__device__ __forceinline__ double t_neg(double a) { return -a; }
__device__ __forceinline__ double t_log(double a) { return log(a); }
__device__ __forceinline__ double t_exp(double a) { return exp(a); }
__device__ __forceinline__ double t_sqrt(double a) { return sqrt(a); }
__device__ __forceinline__ double t_from_real(double a, double) { return a; }

__device__ __forceinline__ cplx t_fma(cplx a, cplx b, cplx c) {
  cplx r;
  r.re = fma(a.re, b.re, fma(-a.im, b.im, c.re));
  r.im = fma(a.re, b.im, fma(a.im, b.re, c.im));
  return r;
}
__device__ __forceinline__ cplx t_fma_c(cplx a, cplx b, double c) {
  cplx r;
  r.re = fma(a.re, b.re, fma(-a.im, b.im, c));
  r.im = fma(a.re, b.im, a.im * b.re);
  return r;
}
__device__ __forceinline__ cplx t_fma_rc(cplx r, double c, cplx a) {
  cplx o;
  o.re = fma(r.re, c, a.re);
  o.im = fma(r.im, c, a.im);
  return o;
}
__device__ __forceinline__ cplx t_mul(cplx a, cplx b) {
  cplx r;
  r.re = fma(a.re, b.re, -a.im * b.im);
  r.im = fma(a.re, b.im, a.im * b.re);
  return r;
}
__device__ __forceinline__ cplx t_mulc(cplx a, double c) { return cplx{a.re * c, a.im * c}; }
__device__ __forceinline__ cplx t_add(cplx a, cplx b) { return cplx{a.re + b.re, a.im + b.im}; }
__device__ __forceinline__ cplx t_addc(cplx a, double c) { return cplx{a.re + c, a.im}; }
__device__ __forceinline__ cplx t_sub(cplx a, cplx b) { return cplx{a.re - b.re, a.im - b.im}; }
__device__ __forceinline__ cplx t_rsubc(double c, cplx a) { return cplx{c - a.re, -a.im}; }
__device__ __forceinline__ cplx t_div(cplx a, cplx b) {
  double d = fma(b.re, b.re, b.im * b.im);
  double inv = 1.0 / d;
  cplx r;
  r.re = fma(a.re, b.re, a.im * b.im) * inv;
  r.im = fma(a.im, b.re, -a.re * b.im) * inv;
  return r;
}
__device__ __forceinline__ cplx t_divc(cplx a, double c) { return cplx{a.re / c, a.im / c}; }
__device__ __forceinline__ cplx t_rdivc(double c, cplx a) {
  double d = fma(a.re, a.re, a.im * a.im);
  double s = c / d;
  return cplx{a.re * s, -a.im * s};
}
__device__ __forceinline__ cplx t_neg(cplx a) { return cplx{-a.re, -a.im}; }
// principal branch: arg in (-pi, pi]  (R10)
__device__ __forceinline__ cplx t_log(cplx a) {
  return cplx{0.5 * log(fma(a.re, a.re, a.im * a.im)), atan2(a.im, a.re)};
}
__device__ __forceinline__ cplx t_exp(cplx a) {
  double e = exp(a.re), s, c;
  sincos(a.im, &s, &c);
  return cplx{e * c, e * s};
}
__device__ __forceinline__ cplx t_sqrt(cplx a) {
  double m = sqrt(fma(a.re, a.re, a.im * a.im));
  if (m == 0.0) return cplx{0.0, a.im};
  double t = sqrt(0.5 * (m + fabs(a.re)));
  if (a.re >= 0.0) return cplx{t, a.im / (2.0 * t)};
  return cplx{fabs(a.im) / (2.0 * t), copysign(t, a.im)};
}
__device__ __forceinline__ cplx t_from_real(double a, cplx) { return cplx{a, 0.0}; }

// ---- Philox4x32-10 (Salmon et al., SC'11), R3 -------------------------------------
struct philox_out {
  uint32_t v[4];
};

__device__ __forceinline__ philox_out philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                                    uint32_t k1) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0;
    c1 = lo1;
    c2 = n2;
    c3 = lo0;
    k0 += W0;
    k1 += W1;
  }
  philox_out o;
  o.v[0] = c0;
  o.v[1] = c1;
  o.v[2] = c2;
  o.v[3] = c3;
  return o;
}

// The same ten rounds with the round keys (k0 + r W0, k1 + r W1), r = 0..9, given: rk[2r], rk[2r+1].
// The evaluation kernels take them from their launch parameters (constant bank): the key schedule is
// the same for every call of a launch and costs nothing per point that way.
__device__ __forceinline__ philox_out philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                       const uint32_t *rk) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
    uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
    uint32_t n0 = hi1 ^ c1 ^ rk[2 * r], n2 = hi0 ^ c3 ^ rk[2 * r + 1];
    c0 = n0;
    c1 = lo1;
    c2 = n2;
    c3 = lo0;
  }
  philox_out o;
  o.v[0] = c0;
  o.v[1] = c1;
  o.v[2] = c2;
  o.v[3] = c3;
  return o;
}

#define FX_TAG_SHIFT 0u
#define FX_TAG_MC 1u

// t for coordinates 2*kb and 2*kb+1 of point j: counter (j lo, j hi, sector_id, tag<<28|kb<<20|it).
__device__ __forceinline__ void philox_t_pair(uint64_t seed, uint32_t sector_id, uint32_t tag, uint32_t it, uint64_t j,
                                              uint32_t kb, uint64_t &t_even, uint64_t &t_odd) {
  philox_out o = philox4x32_10((uint32_t)j, (uint32_t)(j >> 32), sector_id, (tag << 28) | (kb << 20) | it,
                               (uint32_t)seed, (uint32_t)(seed >> 32));
  t_even = ((uint64_t)o.v[0] << 32) | o.v[1];
  t_odd = ((uint64_t)o.v[2] << 32) | o.v[3];
}

__device__ __forceinline__ void philox_t_pair_rk(const uint32_t *rk, uint32_t sector_id, uint32_t tag, uint32_t it,
                                                 uint64_t j, uint32_t kb, uint64_t &t_even, uint64_t &t_odd) {
  philox_out o = philox4x32_10_rk((uint32_t)j, (uint32_t)(j >> 32), sector_id, (tag << 28) | (kb << 20) | it, rk);
  t_even = ((uint64_t)o.v[0] << 32) | o.v[1];
  t_odd = ((uint64_t)o.v[2] << 32) | o.v[3];
}

// u = (2*(t>>12)+1) * 2^-53 in (0,1)   (R2)
// Built from the bits instead of an int64 -> double conversion (a slow multi-instruction sequence on
// the conversion pipe): with s = t>>12 < 2^52, d = 1 + s*2^-52 is the double with mantissa s;
// d - 1 = s*2^-52 exactly, and adding 2^-53 gives (2s+1)*2^-53, which has 53 significant bits: exact.
__device__ __forceinline__ double unit_from_t(uint64_t t) {
  const double d = __longlong_as_double((long long)(0x3FF0000000000000ull | (t >> 12)));
  return (d - 1.0) + 0x1p-53;
}

// lattice integer: (((j*g) mod N_L) << (64-m)) + delta, N_L = 2^m   (R2)
__device__ __forceinline__ uint64_t lattice_t(uint64_t j, uint64_t g, int m, uint64_t delta) {
  if (m == 0) return delta;
  uint64_t mask = (m >= 64) ? ~0ull : ((1ull << m) - 1ull);
  return (((j * g) & mask) << (64 - m)) + delta;
}

// Korobov periodising transform of weight r (R4), mirrored about 1/2.
struct fx_transform {
  int r;          // 0..6
  double cw;      // (2r+1)!/(r!)^2
  double coef[7]; // phi_r(v) = v^(r+1) * sum_i coef[i] v^i
  double cwd;     // cw^dim (integrate kernels: the weight of a point is cw^dim * (prod_k u_k(1-u_k))^r)
};

// From the lattice integer t itself:
//   - u > 1/2 iff the top bit of t is set, and 1-u = (2(2^52-1-s)+1) 2^-53 has the complemented
//     mantissa, so v = min(u, 1-u) comes from one XOR (no FP64 compare/select), and one exact add turns
//     the mantissa into v (d - (1 - 2^-53) with d = 1 + m 2^-52: the result (2m+1) 2^-53 is representable);
//   - x = phi_r(u) and xbar = 1 - x both from v, whichever side u is on (R4: full relative accuracy at both faces);
//   - instead of w = cw (u(1-u))^r it returns s = u(1-u): the caller multiplies the s of all
//     coordinates and raises the product to r once per point, W = cw^dim (prod s)^r, which saves
//     3 multiplications per coordinate and differs from prod w by rounding only (R4).
template <int R>
__device__ __forceinline__ void korobov_xs_r(const fx_transform &tf, uint64_t t, double &x, double &xbar, double &s) {
  const bool left = (long long)t >= 0;
  const uint64_t tm = left ? t : ~t;
  const double d = __longlong_as_double((long long)(0x3FF0000000000000ull | (tm >> 12)));
  const double v = d - (1.0 - 0x1p-53);
  const double vbar = 1.0 - v;
  if constexpr (R == 0) {
    x = left ? v : vbar;
    xbar = left ? vbar : v;
    s = 1.0;
  } else {
    double poly = tf.coef[R];
#pragma unroll
    for (int i = R - 1; i >= 0; --i) poly = fma(poly, v, tf.coef[i]);
    double vp;
    if constexpr (R == 3) {  // v^4 by squaring: one multiplication fewer (and one rounding fewer) than v*v*v*v
      const double v2 = v * v;
      vp = v2 * v2;
    } else {
      vp = v;
#pragma unroll
      for (int i = 0; i < R; ++i) vp *= v;
    }
    const double p = vp * poly;
    const double big = 1.0 - p;
    x = left ? p : big;
    xbar = left ? big : p;
    s = fma(-v, v, v);  // = v (1-v) rounded once, the same number as v * vbar (vbar = 1-v is exact)
  }
}

__device__ __forceinline__ void korobov_xs(const fx_transform &tf, uint64_t t, double &x, double &xbar, double &s) {
  switch (tf.r) {
    case 0: korobov_xs_r<0>(tf, t, x, xbar, s); break;
    case 1: korobov_xs_r<1>(tf, t, x, xbar, s); break;
    case 2: korobov_xs_r<2>(tf, t, x, xbar, s); break;
    case 3: korobov_xs_r<3>(tf, t, x, xbar, s); break;
    case 4: korobov_xs_r<4>(tf, t, x, xbar, s); break;
    case 5: korobov_xs_r<5>(tf, t, x, xbar, s); break;
    default: korobov_xs_r<6>(tf, t, x, xbar, s); break;
  }
}

// W = cw^dim * S^r from S = prod_k u_k(1-u_k)
__device__ __forceinline__ double korobov_weight(const fx_transform &tf, double S) {
  if (tf.r == 3) return tf.cwd * (S * S * S);
  if (tf.r == 0) return 1.0;
  double sp = S;
  for (int i = 1; i < tf.r; ++i) sp *= S;
  return tf.cwd * sp;
}

// Vegas map of one coordinate (R8): exact integer bin and fraction, then the edges.
__device__ __forceinline__ void vegas_map_coord(uint64_t t, int nbins, const double *edges /* [NB+1] */, double &x,
                                                double &wfac, int &bin) {
  uint64_t s = t >> 12;
  uint64_t prod = (2ull * s + 1ull) * (uint64_t)nbins;  // < 2^53 * NB
  bin = (int)(prod >> 53);
  // rem < 2^53 as a double, exactly and without the slow int64 -> double conversion: the high 21 and
  // the low 32 bits become the mantissas of 2^84 + hi 2^32 and 2^52 + lo; the two offsets are taken off
  // first (hi 2^32 - 2^52 is exact), then lo is added (hi 2^32 + lo < 2^53 is exact)
  const uint64_t rem = prod & ((1ull << 53) - 1ull);
  const double dhi = __hiloint2double(0x45300000, (int)(uint32_t)(rem >> 32));
  const double dlo = __hiloint2double(0x43300000, (int)(uint32_t)rem);
  const double frac = __dadd_rn(__dadd_rn(dhi, -(0x1p84 + 0x1p52)), dlo) * 0x1p-53;
  double lo = edges[bin];
  double width = edges[bin + 1] - lo;
  x = fma(frac, width, lo);
  wfac = (double)nbins * width;
}

#endif
