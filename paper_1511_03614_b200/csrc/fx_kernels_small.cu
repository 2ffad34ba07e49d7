// fx_kernels_small.cu -- the small kernels around the evaluation kernel: second level of the
// deterministic reduction, estimators (A9; R5; "treat
// this number as the delta value (standard deviation)"), Vegas grid refinement and combination
// (A8/A9; R8), the parity hooks for points, and the FP64 peak micro-benchmark.
#include "../../include/fiesta_b200.h"
#include "fx_kernels.h"
#include "fx_math.cuh"

namespace {

__global__ void k_reduce_chunks(const double *partials, double *sums, int nrows, int nchunks) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;  // row*FX_ACC_SLOTS + slot
  if (i >= nrows * FX_ACC_SLOTS) return;
  const int row = i / FX_ACC_SLOTS, slot = i % FX_ACC_SLOTS;
  double s = 0.0;
  for (int c = 0; c < nchunks; ++c) s += partials[((size_t)row * nchunks + c) * FX_ACC_SLOTS + slot];
  sums[i] = s;
}

// Vegas: the blocks' histograms of a sector, added in block order (deterministic)
__global__ void k_reduce_hist(const double *hist_part, double *hist, int nsectors, int nchunks, int cells) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;  // sector*cells + cell
  if (i >= (size_t)nsectors * cells) return;
  const size_t s = i / cells, cell = i % cells;
  double t = 0.0;
  for (int c = 0; c < nchunks; ++c) t += hist_part[(s * nchunks + c) * cells + cell];
  hist[i] = t;
}

// slot layout of one sums row: real sector: [k][S1,S2]; complex: [k][c][S1,S2]
__device__ __forceinline__ int slot_of(int k, int c, int ncomp) { return (k * ncomp + c) * 2; }

__global__ void k_estimate(const double *sums, const fx_sector_dev *sectors, const int32_t *sel, int nsel, int R,
                           uint64_t n_per_shift, const unsigned long long *nonfinite, fx_result_dev *results,
                           int Kstride) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nsel * Kstride) return;
  const int s = i / Kstride, k = i % Kstride;
  const fx_sector_dev sec = sectors[sel[s]];
  fx_result_dev out = {0, 0, 0, 0, 0, 0ull, 0ull};
  if (k < sec.K) {
    const int ncomp = sec.is_complex ? 2 : 1;
    const double n = (double)n_per_shift;
    for (int c = 0; c < ncomp; ++c) {
      const int sl = slot_of(k, c, ncomp);
      double value, var;
      if (R >= 2) {
        double mean = 0.0;
        for (int r = 0; r < R; ++r) mean += sums[((size_t)s * R + r) * FX_ACC_SLOTS + sl] / n;
        mean /= (double)R;
        double ss = 0.0;
        for (int r = 0; r < R; ++r) {
          double d = sums[((size_t)s * R + r) * FX_ACC_SLOTS + sl] / n - mean;
          ss = fma(d, d, ss);
        }
        value = mean;
        var = ss / ((double)R * (double)(R - 1));
      } else {
        const double s1 = sums[(size_t)s * FX_ACC_SLOTS + sl], s2 = sums[(size_t)s * FX_ACC_SLOTS + sl + 1];
        value = s1 / n;
        var = (s2 / n - value * value) / (n - 1.0);
      }
      const double sigma = sqrt(fmax(var, 0.0));
      if (c == 0) {
        out.re = value;
        out.re_err = sigma;
      } else {
        out.im = value;
        out.im_err = sigma;
      }
    }
    out.neval = (unsigned long long)n_per_shift * (unsigned long long)R;
    out.n_nonfinite = nonfinite[s];
  }
  results[i] = out;
}

// per iteration: slot pair (S1,S2) -> (I_it, var_it) in place layout
__global__ void k_vegas_iter_stats(const double *sums, double *iter_stats, int nsel, uint64_t npoints) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;  // s*(FX_ACC_SLOTS/2) + pair
  if (i >= nsel * (FX_ACC_SLOTS / 2)) return;
  const int s = i / (FX_ACC_SLOTS / 2), pr = i % (FX_ACC_SLOTS / 2);
  const double n = (double)npoints;
  const double s1 = sums[(size_t)s * FX_ACC_SLOTS + 2 * pr], s2 = sums[(size_t)s * FX_ACC_SLOTS + 2 * pr + 1];
  const double I = s1 / n;
  iter_stats[(size_t)s * FX_ACC_SLOTS + 2 * pr] = I;
  iter_stats[(size_t)s * FX_ACC_SLOTS + 2 * pr + 1] = (s2 / n - I * I) / (n - 1.0);
}

__global__ void k_vegas_combine(const double *iter_stats, int iters, const fx_sector_dev *sectors, const int32_t *sel,
                                int nsel, uint64_t npoints, const unsigned long long *nonfinite, fx_result_dev *results,
                                int Kstride) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nsel * Kstride) return;
  const int s = i / Kstride, k = i % Kstride;
  const fx_sector_dev sec = sectors[sel[s]];
  fx_result_dev out = {0, 0, 0, 0, 0, 0ull, 0ull};
  if (k < sec.K) {
    const int ncomp = sec.is_complex ? 2 : 1;
    for (int c = 0; c < ncomp; ++c) {
      const int sl = slot_of(k, c, ncomp);
      const size_t stride = (size_t)nsel * FX_ACC_SLOTS;
      const double *st = iter_stats + (size_t)s * FX_ACC_SLOTS + sl;
      double vmin = 0.0;
      bool any = false;
      for (int it = 0; it < iters; ++it) {
        double v = fmax(st[it * stride + 1], 0.0);
        if (v > 0.0 && (!any || v < vmin)) {
          vmin = v;
          any = true;
        }
      }
      double value, sigma, chi2;
      if (!any) {
        double m = 0.0;
        for (int it = 0; it < iters; ++it) m += st[it * stride];
        value = m / (double)iters;
        sigma = 0.0;
        chi2 = 0.0;
      } else {
        double sw = 0.0, swi = 0.0;
        for (int it = 0; it < iters; ++it) {
          double v = fmax(st[it * stride + 1], 0.0);
          if (!(v > 0.0)) v = vmin;
          const double w = 1.0 / v;
          sw += w;
          swi = fma(st[it * stride], w, swi);
        }
        value = swi / sw;
        sigma = 1.0 / sqrt(sw);
        chi2 = 0.0;
        for (int it = 0; it < iters; ++it) {
          double v = fmax(st[it * stride + 1], 0.0);
          if (!(v > 0.0)) v = vmin;
          const double d = st[it * stride] - value;
          chi2 += d * d / v;
        }
      }
      if (c == 0) {
        out.re = value;
        out.re_err = sigma;
        out.chi2 = chi2;
      } else {
        out.im = value;
        out.im_err = sigma;
        out.chi2 += chi2;
      }
    }
    out.neval = (unsigned long long)npoints * (unsigned long long)iters;
    out.n_nonfinite = nonfinite[s];
  }
  results[i] = out;
}

// One thread per grid: smooth, normalise, compress, re-bin (R8 i-iv).
__global__ void k_vegas_refine(const double *grid_in, const double *hist, double *grid_out, int ngrids, int nb,
                               double alpha) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ngrids) return;
  const double *xi = grid_in + (size_t)g * (nb + 1);
  const double *h = hist + (size_t)g * nb;
  double *out = grid_out + (size_t)g * (nb + 1);
  double m[FIESTA_MAX_BINS], old[FIESTA_MAX_BINS + 1];
  for (int b = 0; b <= nb; ++b) old[b] = xi[b];
  double tot = 0.0;
  for (int b = 0; b < nb; ++b) {
    double sm;
    if (nb == 1) sm = h[0];
    else if (b == 0) sm = (h[0] + h[1]) / 2.0;
    else if (b == nb - 1) sm = (h[nb - 2] + h[nb - 1]) / 2.0;
    else sm = (h[b - 1] + h[b] + h[b + 1]) / 3.0;
    m[b] = sm;
    tot += sm;
  }
  if (!(tot > 0.0)) {
    for (int b = 0; b <= nb; ++b) out[b] = old[b];
    return;
  }
  double cum_total = 0.0;
  for (int b = 0; b < nb; ++b) {
    const double p = m[b] / tot;
    double v = 0.0;
    if (p >= 1.0) v = 1.0;
    else if (p > 0.0) v = pow((1.0 - p) / (-log(p)), alpha);
    m[b] = v;
    cum_total += v;
  }
  out[0] = 0.0;
  out[nb] = 1.0;
  int k = 0;
  double cum_k = 0.0;  // sum of m[0..k)
  for (int i = 1; i < nb; ++i) {
    const double target = (double)i * cum_total / (double)nb;
    // advance while cum[k+1] <= target (k stays < nb-1)
    while (k < nb - 1 && cum_k + m[k] <= target) {
      cum_k += m[k];
      ++k;
    }
    out[i] = old[k] + (target - cum_k) / m[k] * (old[k + 1] - old[k]);
  }
}

__global__ void k_vegas_init_grid(double *grid, int ngrids, int nb) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ngrids * (nb + 1)) return;
  grid[i] = (double)(i % (nb + 1)) / (double)nb;
}

struct genvec_arg {
  uint64_t g[FX_NXMAX];
};

__global__ void k_generate_points(int rule, uint64_t seed, uint32_t sector_id, uint32_t shift_or_iter, int log2_n,
                                  genvec_arg gv, uint64_t first, uint64_t count, int dim, uint64_t *t_out) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  const uint64_t j = first + i;
  for (int kb = 0; kb < (dim + 1) / 2; ++kb) {
    uint64_t te, to;
    if (rule == FIESTA_RULE_LATTICE) {
      uint64_t de, dod;
      philox_t_pair(seed, sector_id, FX_TAG_SHIFT, shift_or_iter, 0ull, kb, de, dod);
      te = lattice_t(j, gv.g[2 * kb], log2_n, de);
      to = (2 * kb + 1 < dim) ? lattice_t(j, gv.g[2 * kb + 1], log2_n, dod) : 0ull;
    } else {
      philox_t_pair(seed, sector_id, FX_TAG_MC, shift_or_iter, j, kb, te, to);
    }
    t_out[i * dim + 2 * kb] = te;
    if (2 * kb + 1 < dim) t_out[i * dim + 2 * kb + 1] = to;
  }
}

__global__ void k_transform_points(int rule, fx_transform tf, const uint64_t *t, uint64_t count, int dim, double *x,
                                   double *xbar, double *w) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= count) return;
  // the integrate kernels' own arithmetic (fx_make_points): korobov_xs per coordinate, one weight per point
  double S = 1.0;
  for (int k = 0; k < dim; ++k) {
    double xx, xb, ss;
    if (rule == FIESTA_RULE_LATTICE) korobov_xs(tf, t[i * dim + k], xx, xb, ss);
    else {
      xx = unit_from_t(t[i * dim + k]);
      xb = 1.0 - xx;
      ss = 1.0;
    }
    x[i * dim + k] = xx;
    xbar[i * dim + k] = xb;
    S *= ss;
  }
  w[i] = rule == FIESTA_RULE_LATTICE ? korobov_weight(tf, S) : 1.0;
}

// 16 independent DFMA chains per thread, 256 threads/block: the FP64 pipe limit (2 flops per DFMA).
__global__ void __launch_bounds__(256) k_fp64_peak(double *sink, int iters) {
  double a[16];
  const double b = 1.0000001 + 1e-9 * threadIdx.x, c = 1e-9 * (blockIdx.x + 1);
#pragma unroll
  for (int i = 0; i < 16; ++i) a[i] = 1.0 + i * 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int rep = 0; rep < 8; ++rep)
#pragma unroll
      for (int i = 0; i < 16; ++i) a[i] = fma(a[i], b, c);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += a[i];
  if (s == 123.456) sink[0] = s;
}

inline unsigned blocks_for(size_t n, int t) { return (unsigned)((n + t - 1) / t); }

}  // namespace

cudaError_t fx_launch_reduce_chunks(const double *partials, double *sums, int nrows, int nchunks, cudaStream_t st) {
  k_reduce_chunks<<<blocks_for((size_t)nrows * FX_ACC_SLOTS, 128), 128, 0, st>>>(partials, sums, nrows, nchunks);
  return cudaGetLastError();
}

cudaError_t fx_launch_reduce_hist(const double *hist_part, double *hist, int nsectors, int nchunks, int cells,
                                  cudaStream_t st) {
  k_reduce_hist<<<blocks_for((size_t)nsectors * cells, 128), 128, 0, st>>>(hist_part, hist, nsectors, nchunks, cells);
  return cudaGetLastError();
}

cudaError_t fx_launch_estimate(const double *sums, const fx_sector_dev *sectors, const int32_t *sel, int nsel, int R,
                               uint64_t n_per_shift, const unsigned long long *nonfinite, fx_result_dev *results,
                               int Kstride, cudaStream_t st) {
  k_estimate<<<blocks_for((size_t)nsel * Kstride, 128), 128, 0, st>>>(sums, sectors, sel, nsel, R, n_per_shift,
                                                                      nonfinite, results, Kstride);
  return cudaGetLastError();
}

cudaError_t fx_launch_vegas_iter_stats(const double *sums, double *iter_stats, int it, int nsel, uint64_t npoints,
                                       cudaStream_t st) {
  k_vegas_iter_stats<<<blocks_for((size_t)nsel * (FX_ACC_SLOTS / 2), 128), 128, 0, st>>>(
      sums, iter_stats + (size_t)it * nsel * FX_ACC_SLOTS, nsel, npoints);
  return cudaGetLastError();
}

cudaError_t fx_launch_vegas_combine(const double *iter_stats, int iters, const fx_sector_dev *sectors,
                                    const int32_t *sel, int nsel, uint64_t npoints,
                                    const unsigned long long *nonfinite, fx_result_dev *results, int Kstride,
                                    cudaStream_t st) {
  k_vegas_combine<<<blocks_for((size_t)nsel * Kstride, 128), 128, 0, st>>>(iter_stats, iters, sectors, sel, nsel,
                                                                           npoints, nonfinite, results, Kstride);
  return cudaGetLastError();
}

cudaError_t fx_launch_vegas_refine(const double *grid_in, const double *hist, double *grid_out, int ngrids, int nbins,
                                   double alpha, cudaStream_t st) {
  k_vegas_refine<<<blocks_for(ngrids, 64), 64, 0, st>>>(grid_in, hist, grid_out, ngrids, nbins, alpha);
  return cudaGetLastError();
}

cudaError_t fx_launch_vegas_init_grid(double *grid, int ngrids, int nbins, cudaStream_t st) {
  k_vegas_init_grid<<<blocks_for((size_t)ngrids * (nbins + 1), 128), 128, 0, st>>>(grid, ngrids, nbins);
  return cudaGetLastError();
}

cudaError_t fx_launch_generate_points(int rule, uint64_t seed, int sector_id, int shift_or_iter, uint64_t n_lattice,
                                      int log2_n, const uint64_t *genvec_host, uint64_t first, uint64_t count, int dim,
                                      uint64_t *t_dev, cudaStream_t st) {
  (void)n_lattice;
  genvec_arg gv{};
  if (genvec_host)
    for (int k = 0; k < dim; ++k) gv.g[k] = genvec_host[k];
  if (count == 0) return cudaSuccess;
  k_generate_points<<<blocks_for(count, 128), 128, 0, st>>>(rule, seed, (uint32_t)sector_id, (uint32_t)shift_or_iter,
                                                            log2_n, gv, first, count, dim, t_dev);
  return cudaGetLastError();
}

cudaError_t fx_launch_transform_points(int rule, const fx_transform_host &tf, const uint64_t *t_dev, uint64_t count,
                                       int dim, double *x_dev, double *xbar_dev, double *w_dev, cudaStream_t st) {
  if (count == 0) return cudaSuccess;
  fx_transform t;
  t.r = tf.r;
  t.cw = tf.cw;
  for (int i = 0; i < 7; ++i) t.coef[i] = tf.coef[i];
  t.cwd = 1.0;
  for (int k = 0; k < dim; ++k) t.cwd *= tf.cw;
  k_transform_points<<<blocks_for(count, 128), 128, 0, st>>>(rule, t, t_dev, count, dim, x_dev, xbar_dev, w_dev);
  return cudaGetLastError();
}

cudaError_t fx_launch_fp64_peak(double *sink_dev, int iters, int blocks, cudaStream_t st) {
  k_fp64_peak<<<blocks, 256, 0, st>>>(sink_dev, iters);
  return cudaGetLastError();
}
