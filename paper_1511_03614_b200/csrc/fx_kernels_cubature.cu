// fx_kernels_cubature.cu -- the deterministic integrator (R21): node
// generation and per-box reduction of the Genz-Malik degree-7 rule with its embedded degree-5 rule
// (A. C. Genz, A. A. Malik, J. Comput. Appl. Math. 6 (1980) 295), the building block of a
// Cuhre-like globally adaptive cubature ("cuhreCuba").  The integrand values at the
// nodes come from the SAME evaluation kernels as everywhere else (the eval kernels of both tiers,
// fiesta_abi_integrate.inc eval_device); the adaptive loop is on the host (fiesta_abi_cubature.inc).
//
// Node order of a box (centre c, half-widths h), NN = 1 + 4n + 2n(n-1) + 2^n nodes:
//   0                        c
//   1 .. 2n                  c +- l2 h_i e_i          (axis i = 0, 1, ..; + before -)
//   2n+1 .. 4n               c +- l3 h_i e_i
//   4n+1 .. 4n+2n(n-1)       c +- l3 h_i e_i +- l3 h_j e_j   pairs i < j in lexicographic order; signs (i,j) = ++, -+, +-, --
//   the last 2^n             c + (+-l5 h_0, .., +-l5 h_{n-1}); bit k of the corner number set: minus
#include <math.h>

#include "fx_kernels.h"

namespace {

__device__ __forceinline__ int gm_class(int q, int n, int &local) {  // 0 centre, 1 l2, 2 l3, 3 pairs, 4 corners
  if (q == 0) { local = 0; return 0; }
  if (q <= 2 * n) { local = q - 1; return 1; }
  if (q <= 4 * n) { local = q - 1 - 2 * n; return 2; }
  const int np4 = 2 * n * (n - 1);
  if (q <= 4 * n + np4) { local = q - 1 - 4 * n; return 3; }
  local = q - 1 - 4 * n - np4;
  return 4;
}

__global__ void k_gm_nodes(const double *boxes, uint64_t nboxes, int n, int nn, fx_gm_tables tb, double *x) {
  const uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nboxes * (uint64_t)nn) return;
  const uint64_t b = idx / nn;
  const int q = (int)(idx % nn);
  const double *c = boxes + b * 2 * n, *h = c + n;
  double *out = x + idx * n;
  int local;
  const int cls = gm_class(q, n, local);
  int i = -1, j = -1;
  double si = 0.0, sj = 0.0, lam = 0.0;
  if (cls == 1 || cls == 2) {
    i = local >> 1;
    si = (local & 1) ? -1.0 : 1.0;
    lam = cls == 1 ? tb.l2 : tb.l3;
  } else if (cls == 3) {
    int pair = local >> 2;
    i = 0;
    while (pair >= n - 1 - i) {
      pair -= n - 1 - i;
      ++i;
    }
    j = i + 1 + pair;
    si = (local & 1) ? -1.0 : 1.0;
    sj = (local & 2) ? -1.0 : 1.0;
    lam = tb.l3;
  }
  for (int k = 0; k < n; ++k) {
    double s = 0.0, l = lam;
    if (cls == 4) {
      s = ((local >> k) & 1) ? -1.0 : 1.0;
      l = tb.l5;
    } else if (k == i) {
      s = si;
    } else if (k == j) {
      s = sj;
    }
    out[k] = s == 0.0 ? c[k] : c[k] + (s * l) * h[k];
  }
}

// one block per box: I7, |I7 - I5| per component, fourth differences, split axis.  A thread takes the nodes
// q = tid, tid + 128, .. with all components of a node at once (they are contiguous); lanes are added by a
// shuffle tree, the four warps in order: a fixed assignment and order, so the sums are reproducible.
__global__ void __launch_bounds__(128) k_gm_reduce(const double *vals /*[box][node][ncomp]*/, const double *boxes, int n, int nn,
                                                   int ncomp, fx_gm_tables tb, double *rec /*[box][FX_GM_REC]*/,
                                                   double *i5_out /*[box][ncomp] or NULL*/, double *d_out /*[box][n] or NULL*/) {
  __shared__ double sh[2][16][4];
  __shared__ double sh_d[FX_NXMAX];
  const uint64_t b = blockIdx.x;
  const double *v = vals + b * (uint64_t)nn * ncomp;
  const double *h = boxes + b * 2 * n + n;
  double vol = 1.0;
  for (int k = 0; k < n; ++k) vol *= 2.0 * h[k];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double *r = rec + b * FX_GM_REC;
  unsigned bad = 0;
  double s7[16], s5[16];
#pragma unroll
  for (int c = 0; c < 16; ++c) s7[c] = s5[c] = 0.0;
  for (int q = threadIdx.x; q < nn; q += 128) {
    int local;
    const int cls = gm_class(q, n, local);
    const double w7 = tb.w7[cls], w5 = tb.w5[cls];
    const double *f = v + (size_t)q * ncomp;
#pragma unroll
    for (int c = 0; c < 16; ++c) {
      if (c < ncomp) {
        const double fv = f[c];
        bad += isfinite(fv) ? 0u : 1u;
        s7[c] = fma(w7, fv, s7[c]);
        s5[c] = fma(w5, fv, s5[c]);
      }
    }
  }
#pragma unroll
  for (int c = 0; c < 16; ++c) {
    if (c < ncomp) {  // block-uniform
      double a = s7[c], e = s5[c];
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, off);
        e += __shfl_down_sync(0xffffffffu, e, off);
      }
      if (lane == 0) {
        sh[0][c][warp] = a;
        sh[1][c][warp] = e;
      }
    }
  }
  __syncthreads();
  if (threadIdx.x < ncomp) {
    const int c = threadIdx.x;
    const double i7 = vol * (((sh[0][c][0] + sh[0][c][1]) + sh[0][c][2]) + sh[0][c][3]);
    const double i5 = vol * (((sh[1][c][0] + sh[1][c][1]) + sh[1][c][2]) + sh[1][c][3]);
    r[c] = i7;
    r[16 + c] = fabs(i7 - i5);
    if (i5_out) i5_out[b * ncomp + c] = i5;
  }
  // fourth divided differences along the axes, summed over the components
  if (threadIdx.x < n) {
    const int i = threadIdx.x;
    double d = 0.0;
    for (int c = 0; c < ncomp; ++c) {
      const double f0 = v[c];
      const double a = v[(size_t)(1 + 2 * i) * ncomp + c] + v[(size_t)(2 + 2 * i) * ncomp + c] - 2.0 * f0;
      const double e = v[(size_t)(1 + 2 * n + 2 * i) * ncomp + c] + v[(size_t)(2 + 2 * n + 2 * i) * ncomp + c] - 2.0 * f0;
      d += fabs(a - tb.ratio * e);
    }
    sh_d[i] = d;
    if (d_out) d_out[b * n + i] = d;
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) bad += __shfl_down_sync(0xffffffffu, bad, off);
  __shared__ unsigned sh_bad[4];
  __shared__ double sh_err[16];
  if (lane == 0) sh_bad[warp] = bad;
  if (threadIdx.x < ncomp) sh_err[threadIdx.x] = r[16 + threadIdx.x];  // this thread wrote it above
  __syncthreads();
  if (threadIdx.x == 0) {
    int axis = 0;
    for (int i = 1; i < n; ++i)
      if (sh_d[i] > sh_d[axis]) axis = i;  // ties: the lowest index
    for (int c = ncomp; c < 16; ++c) r[c] = r[16 + c] = 0.0;
    double e = 0.0;
    for (int c = 0; c < ncomp; ++c) e += sh_err[c];
    r[32] = (double)axis;
    r[33] = (double)(sh_bad[0] + sh_bad[1] + sh_bad[2] + sh_bad[3]);
    r[34] = e;
    r[35] = 0.0;
  }
}

}  // namespace

fx_gm_tables fx_gm_make_tables(int n) {
  fx_gm_tables t;
  const double dn = (double)n;
  t.l2 = sqrt(9.0 / 70.0);
  t.l3 = sqrt(9.0 / 10.0);
  t.l5 = sqrt(9.0 / 19.0);
  t.ratio = 1.0 / 7.0;  // (l2 / l3)^2
  t.w7[0] = (12824.0 - 9120.0 * dn + 400.0 * dn * dn) / 19683.0;
  t.w7[1] = 980.0 / 6561.0;
  t.w7[2] = (1820.0 - 400.0 * dn) / 19683.0;
  t.w7[3] = 200.0 / 19683.0;
  t.w7[4] = 6859.0 / 19683.0 / ldexp(1.0, n);
  t.w5[0] = (729.0 - 950.0 * dn + 50.0 * dn * dn) / 729.0;
  t.w5[1] = 245.0 / 486.0;
  t.w5[2] = (265.0 - 100.0 * dn) / 1458.0;
  t.w5[3] = 25.0 / 729.0;
  t.w5[4] = 0.0;
  return t;
}

int fx_gm_nodes_per_box(int n) { return 1 + 4 * n + 2 * n * (n - 1) + (1 << n); }

cudaError_t fx_launch_gm_nodes(const double *boxes, uint64_t nboxes, int n, double *x, cudaStream_t st) {
  const int nn = fx_gm_nodes_per_box(n);
  const uint64_t total = nboxes * (uint64_t)nn;
  if (total == 0) return cudaSuccess;
  k_gm_nodes<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(boxes, nboxes, n, nn, fx_gm_make_tables(n), x);
  return cudaGetLastError();
}

cudaError_t fx_launch_gm_reduce(const double *vals, const double *boxes, uint64_t nboxes, int n, int ncomp, double *rec,
                                double *i5_out, double *d_out, cudaStream_t st) {
  if (nboxes == 0) return cudaSuccess;
  k_gm_reduce<<<(unsigned)nboxes, 128, 0, st>>>(vals, boxes, n, fx_gm_nodes_per_box(n), ncomp, fx_gm_make_tables(n), rec, i5_out,
                                                d_out);
  return cudaGetLastError();
}
