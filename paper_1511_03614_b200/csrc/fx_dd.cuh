// fx_dd.cuh -- double-double arithmetic for the mixed-precision rescue.
//
// The paper's default "Mixed" mode evaluates the integrand with MPFR in the parts of the integration
// cube where doubles cancel (knobs SmallX, MPThreshold, PrecisionShift, MPPrecision,
// MPMin; -mpfr evaluates every point that way).  On the GPU the higher
// precision is a pair of doubles (hi, lo), value hi + lo with |lo| <= ulp(hi)/2: about 106 bits,
// built from the error-free transformations two_sum (Knuth) and two_prod (FMA), as in Dekker's and
// Hida-Li-Bailey's double-double arithmetic, restated here.  The translation units are compiled with
// -fmad=false, so the compiler cannot contract the transformations away.
#ifndef FX_DD_CUH
#define FX_DD_CUH

struct dd {
  double hi, lo;
};

__device__ __forceinline__ dd dd_from(double a) { return dd{a, 0.0}; }

// s + e = a + b exactly
__device__ __forceinline__ dd dd_two_sum(double a, double b) {
  const double s = a + b, bb = s - a;
  return dd{s, (a - (s - bb)) + (b - bb)};
}
// the same for |a| >= |b|
__device__ __forceinline__ dd dd_quick_two_sum(double a, double b) {
  const double s = a + b;
  return dd{s, b - (s - a)};
}
// p + e = a * b exactly
__device__ __forceinline__ dd dd_two_prod(double a, double b) {
  const double p = a * b;
  return dd{p, fma(a, b, -p)};
}

__device__ __forceinline__ dd dd_neg(dd a) { return dd{-a.hi, -a.lo}; }

__device__ __forceinline__ dd dd_add(dd a, dd b) {
  dd s = dd_two_sum(a.hi, b.hi);
  const dd t = dd_two_sum(a.lo, b.lo);
  s.lo += t.hi;
  s = dd_quick_two_sum(s.hi, s.lo);
  s.lo += t.lo;
  return dd_quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_sub(dd a, dd b) { return dd_add(a, dd_neg(b)); }
__device__ __forceinline__ dd dd_add_d(dd a, double b) {
  dd s = dd_two_sum(a.hi, b);
  s.lo += a.lo;
  return dd_quick_two_sum(s.hi, s.lo);
}

__device__ __forceinline__ dd dd_mul(dd a, dd b) {
  dd p = dd_two_prod(a.hi, b.hi);
  p.lo += a.hi * b.lo + a.lo * b.hi;
  return dd_quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b) {
  dd p = dd_two_prod(a.hi, b);
  p.lo += a.lo * b;
  return dd_quick_two_sum(p.hi, p.lo);
}
// a * 2^k, exact
__device__ __forceinline__ dd dd_ldexp(dd a, int k) { return dd{ldexp(a.hi, k), ldexp(a.lo, k)}; }

// long division: three quotient digits
__device__ __forceinline__ dd dd_div(dd a, dd b) {
  const double q1 = a.hi / b.hi;
  dd r = dd_sub(a, dd_mul_d(b, q1));
  const double q2 = r.hi / b.hi;
  r = dd_sub(r, dd_mul_d(b, q2));
  const double q3 = r.hi / b.hi;
  const dd q = dd_quick_two_sum(q1, q2);
  return dd_add_d(q, q3);
}

// Karp-Markstein: with x ~ 1/sqrt(a), sqrt(a) = a x + (a - (a x)^2) x / 2
__device__ __forceinline__ dd dd_sqrt(dd a) {
  if (a.hi <= 0.0) return dd{a.hi == 0.0 ? 0.0 : __longlong_as_double(0x7ff8000000000000ll), 0.0};
  const double x = 1.0 / sqrt(a.hi);
  const double ax = a.hi * x;
  const dd ax2 = dd_two_prod(ax, ax);
  const double corr = dd_sub(a, ax2).hi * (x * 0.5);
  return dd_two_sum(ax, corr);
}

// exp: a = m ln2 + 512 r;  exp(r) by its Taylor series (|r| < ln2/1024: 1e-33 after the r^9 term), squared
// nine times, scaled by 2^m
__device__ inline dd dd_exp(dd a) {
  if (!(a.hi > -709.0)) return dd{a.hi != a.hi ? a.hi : 0.0, 0.0};
  if (a.hi >= 709.0) return dd{__longlong_as_double(0x7ff0000000000000ll), 0.0};
  const dd ln2 = dd{6.93147180559945286e-01, 2.31904681384629956e-17};
  const double inv_fact[7][2] = {{1.66666666666666657e-01, 9.25185853854297066e-18}, {4.16666666666666644e-02, 2.31296463463574266e-18},
                                 {8.33333333333333322e-03, 1.15648231731787138e-19}, {1.38888888888888894e-03, -5.30054395437357706e-20},
                                 {1.98412698412698413e-04, 1.72095582934207053e-22}, {2.48015873015873016e-05, 2.15119478667758816e-23},
                                 {2.75573192239858925e-06, -1.85839327404647208e-22}};
  const double m = floor(a.hi / ln2.hi + 0.5);
  const dd r = dd_ldexp(dd_sub(a, dd_mul_d(ln2, m)), -9);
  dd p = dd_mul(r, r);
  dd s = dd_add(r, dd_ldexp(p, -1));  // r + r^2/2
  p = dd_mul(p, r);
#pragma unroll 1
  for (int i = 0; i < 7; ++i) {
    s = dd_add(s, dd_mul(p, dd{inv_fact[i][0], inv_fact[i][1]}));
    p = dd_mul(p, r);
  }
#pragma unroll 1
  for (int i = 0; i < 9; ++i) s = dd_add(dd_ldexp(s, 1), dd_mul(s, s));  // exp(2r) - 1 = 2 s + s^2
  s = dd_add_d(s, 1.0);
  return dd_ldexp(s, (int)m);
}

// log: one Newton step on exp from the double logarithm, x <- x + a exp(-x) - 1
__device__ inline dd dd_log(dd a) {
  if (!(a.hi > 0.0)) {
    if (a.hi == 0.0) return dd{-__longlong_as_double(0x7ff0000000000000ll), 0.0};
    return dd{__longlong_as_double(0x7ff8000000000000ll), 0.0};
  }
  const double x = log(a.hi);
  const dd t = dd_mul(a, dd_exp(dd{-x, 0.0}));
  return dd_add(dd_from(x), dd_add_d(t, -1.0));
}

#endif
