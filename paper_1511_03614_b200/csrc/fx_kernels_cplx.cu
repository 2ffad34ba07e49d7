// fx_kernels_cplx.cu -- evaluation kernels for complex sectors ("-complex"), with
// the contour deformation of the physical region (formula DESIGN.md R11):
//     g_k  = dF/dx_k (x)                                  real program (FX_STM outputs)
//     z_k  = x_k - i*lambda*x_k*(1-x_k)*g_k
//     J_kl = delta_kl (1 - i*lambda*(1-2x_k) g_k) - i*lambda*x_k(1-x_k) d2F/dx_k dx_l
//     o_k(z) * det J                                      complex program, LU with partial pivoting
// Compiled once per dimension N (-DFX_N=1..8) so the N x N elimination is fully unrolled on
// registers.  SURVEY 8(a) steps A4, A5 (complex), A6, A7.
#ifndef FX_N
#error "compile with -DFX_N=<dimension 1..8>"
#endif
#define FX_WANT(is_cplx, nx, p) ((nx) == FX_N && (p) == 1)  // real (deformation program) and complex, P = 2
#define FX_NO_MIXED_MASK  // fiesta_set_mixed: phase 1 runs on the real interpreter kernels only
#include "fx_device_common.cuh"
#include "fx_deform.cuh"

#define FX_CAT2(a, b) a##b
#define FX_CAT(a, b) FX_CAT2(a, b)

// one named namespace per dimension: the objects of all dimensions are linked into one library
namespace FX_CAT(fx_cplx_n, FX_N) {

constexpr int N = FX_N;
constexpr int P = FX_P_CPLX;
constexpr int NGH = N + N * (N + 1) / 2;  // gradient + upper Hessian slots written by the deform program

struct NoSink {
  __device__ __forceinline__ void operator()(int, double (&)[P]) {}
};

// x (real, registers) -> X = z(x) (complex) and det J per point.  sh_deform == nullptr: z = x, det = 1.
__device__ __forceinline__ void fx_deform_points(const fx_ins *sh_deform, double lambda, double (&x)[N][P],
                                                 double (&xbar)[N][P], const fx_mem<double> M, cplx (&X)[N][P],
                                                 cplx (&det)[P]) {
  if (sh_deform == nullptr) {
#pragma unroll
    for (int k = 0; k < N; ++k) FX_PLOOP { X[k][p] = cplx{x[k][p], 0.0}; }
    FX_PLOOP { det[p] = cplx{1.0, 0.0}; }
    return;
  }
  NoSink ns;
  fx_run<double, N, P>(sh_deform, x, M, ns);  // M[0..NGH) = gradient, upper Hessian
#pragma unroll
  for (int k = 0; k < N; ++k) FX_PLOOP {
      M.st(NGH + k, p, P, x[k][p]);
      M.st(NGH + N + k, p, P, xbar[k][p]);
    }
#pragma unroll 1
  for (int p = 0; p < P; ++p) {  // one matrix at a time: 2*N*N doubles in registers
    double xv[N], xbv[N], zi[N];
#pragma unroll
    for (int k = 0; k < N; ++k) {
      xv[k] = M.ld(NGH + k, p, P);
      xbv[k] = M.ld(NGH + N + k, p, P);
    }
    const cplx d = fx_jacobian_det<N>(lambda, xv, xbv, [&](int slot) { return M.ld(slot, p, P); }, zi);
#pragma unroll
    for (int k = 0; k < N; ++k) M.st(k, p, P, zi[k]);
    if constexpr (P == 1) {
      det[0] = d;  // the elimination is over: its result stays in registers
    } else {
      M.st(NGH + 2 * N, p, P, d.re);
      M.st(NGH + 2 * N + 1, p, P, d.im);
    }
  }
  // x is re-read from its slot: nothing but J has to stay in registers across the elimination
#pragma unroll
  for (int k = 0; k < N; ++k) FX_PLOOP { X[k][p] = cplx{M.ld(NGH + k, p, P), M.ld(k, p, P)}; }
  if constexpr (P != 1) FX_PLOOP { det[p] = cplx{M.ld(NGH + 2 * N, p, P), M.ld(NGH + 2 * N + 1, p, P)}; }
}

struct IntegrateSinkCplx {
  double *acc;
  const cplx (&Wd)[P];  // weight * det J
  unsigned valid;
  unsigned nonfinite;
  double (&h2)[P];
  __device__ __forceinline__ void operator()(int k, cplx (&A)[P]) {
    double s1r = acc[(4 * k) * FX_THREADS], s2r = acc[(4 * k + 1) * FX_THREADS];
    double s1i = acc[(4 * k + 2) * FX_THREADS], s2i = acc[(4 * k + 3) * FX_THREADS];
    FX_PLOOP {
      cplx g = t_mul(Wd[p], A[p]);
      if (!((valid >> p) & 1u)) g = cplx{0.0, 0.0};
      nonfinite += (isfinite(g.re) && isfinite(g.im)) ? 0u : 1u;
      s1r += g.re;
      s2r = fma(g.re, g.re, s2r);
      s1i += g.im;
      s2i = fma(g.im, g.im, s2i);
      h2[p] = fma(g.re, g.re, fma(g.im, g.im, h2[p]));
    }
    acc[(4 * k) * FX_THREADS] = s1r;
    acc[(4 * k + 1) * FX_THREADS] = s2r;
    acc[(4 * k + 2) * FX_THREADS] = s1i;
    acc[(4 * k + 3) * FX_THREADS] = s2i;
  }
};

template <int RULE>
__global__ void __launch_bounds__(FX_THREADS) fx_integrate_cplx(const __grid_constant__ fx_integrate_params prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int b = blockIdx.x;
  const int chunk = b % prm.nchunks;
  const int r = (b / prm.nchunks) % prm.n_shifts;
  const int sel_idx = fx_sel_index(prm, b / (prm.nchunks * prm.n_shifts));
  const fx_sector_dev sec = prm.sectors[prm.sel[sel_idx]];
  constexpr bool vegas = RULE == FIESTA_RULE_VEGAS;
  // the accumulator area holds what the call's complex sectors need (4 K slots), not the record's 32: one more resident block
  const fx_smem_layout L = fx_layout(prm.prog_ins_max, prm.mem_doubles, N, prm.nbins, vegas,
                                     prm.acc_slots_cplx > 0 ? prm.acc_slots_cplx : FX_ACC_SLOTS);
  fx_ins *sh_prog = reinterpret_cast<fx_ins *>(smem + L.prog);
  fx_ins *sh_deform = sec.deform_len ? sh_prog + sec.main_len : nullptr;
  double *sh_mem = reinterpret_cast<double *>(smem + L.mem);
  double *sh_acc = reinterpret_cast<double *>(smem + L.acc);
  uint64_t *sh_delta = reinterpret_cast<uint64_t *>(smem + L.delta);
  double *sh_grid = reinterpret_cast<double *>(smem + L.grid);
  double *sh_hist = reinterpret_cast<double *>(smem + L.hist);
  double *sh_wsum = reinterpret_cast<double *>(smem + L.wsum);

  fx_copy_program(sh_prog, prm.arena + sec.main_off, sec.main_len);
  if (sec.deform_len) fx_copy_program(sh_deform, prm.arena + sec.deform_off, sec.deform_len);
  fx_block_setup(prm, N, (uint32_t)sec.sector_id, r, sel_idx, sh_delta, sh_grid, sh_hist);
  const int nslots = 4 * sec.K;
  for (int s = 0; s < nslots; ++s) sh_acc[s * FX_THREADS + threadIdx.x] = 0.0;
  __syncthreads();

  const uint64_t c0 = (uint64_t)chunk * prm.chunk;
  const uint64_t c1 = min(c0 + prm.chunk, prm.n_per_shift);
  const fx_mem<double> Mr{sh_mem + threadIdx.x, FX_THREADS};
  const fx_mem<cplx> Mc{sh_mem + threadIdx.x, FX_THREADS};
  unsigned nonfinite = 0;
  for (uint64_t it = c0; it < c1; it += (uint64_t)FX_THREADS * P) {  // block-uniform trip count (see the real kernel)
    const uint64_t base = it + (uint64_t)threadIdx.x * P;
    double x[N][P], xbar[N][P], W[P], h2[P];
    uint32_t bins[(N + 3) / 4][P];
    unsigned valid;
    fx_make_points<RULE, N, P, true>(prm, N, (uint32_t)sec.sector_id, sh_delta, sh_grid, base, c1, x, xbar, W, valid, bins);
    cplx X[N][P], Wd[P];
    fx_deform_points(sh_deform, sec.lambda, x, xbar, Mr, X, Wd);
    FX_PLOOP {
      Wd[p] = t_mulc(Wd[p], W[p]);
      h2[p] = 0.0;
    }
    IntegrateSinkCplx sink{sh_acc + threadIdx.x, Wd, valid, 0u, h2};
    fx_run<cplx, N, P>(sh_prog, X, Mc, sink);
    nonfinite += sink.nonfinite;
    if (vegas) fx_hist_points<N, P>(sh_hist, N, prm.nbins, valid, bins, h2);
  }
  __syncthreads();
  fx_block_reduce(sh_acc, sh_wsum, nslots, fx_partial_record(prm, sel_idx, r, chunk));
  fx_block_finish(prm, N, sel_idx, chunk, nonfinite, sh_hist);
}

// -testF: "instead of the integration, the code checks whether the sign of the imaginary
// part of F is negative".  The sector's F(z) program is walked at the rule's points, deformed with
// lambda (the sector's, or the candidate of a lambda scan); per block one record:
// points with Im F(z) >= 0 (or NaN), max Im F(z), min |F(z)|^2, points looked at.
struct TestFSink {
  unsigned valid;
  unsigned bad;
  double max_im, min_abs2;
  __device__ __forceinline__ void operator()(int, cplx (&A)[P]) {
    FX_PLOOP {
      if ((valid >> p) & 1u) {
        bad += (A[p].im < 0.0) ? 0u : 1u;
        max_im = fmax(max_im, A[p].im);
        min_abs2 = fmin(min_abs2, fma(A[p].re, A[p].re, A[p].im * A[p].im));
      }
    }
  }
};

template <int RULE>
__global__ void __launch_bounds__(FX_THREADS) fx_testf_cplx(const __grid_constant__ fx_integrate_params prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int b = blockIdx.x;
  const int chunk = b % prm.nchunks;
  const int r = (b / prm.nchunks) % prm.n_shifts;
  const int sel_idx = fx_sel_index(prm, b / (prm.nchunks * prm.n_shifts));
  const fx_sector_dev sec = prm.sectors[prm.sel[sel_idx]];
  const fx_smem_layout L = fx_layout(prm.prog_ins_max, prm.mem_doubles, N, prm.nbins, false);
  fx_ins *sh_prog = reinterpret_cast<fx_ins *>(smem + L.prog);
  fx_ins *sh_deform = sh_prog + sec.testf_len;
  double *sh_mem = reinterpret_cast<double *>(smem + L.mem);
  uint64_t *sh_delta = reinterpret_cast<uint64_t *>(smem + L.delta);
  double *sh_red = reinterpret_cast<double *>(smem + L.acc);
  fx_copy_program(sh_prog, prm.arena + sec.testf_off, sec.testf_len);
  fx_copy_program(sh_deform, prm.arena + sec.deform_off, sec.deform_len);
  fx_block_setup(prm, N, (uint32_t)sec.sector_id, r, sel_idx, sh_delta, nullptr, nullptr);
  __syncthreads();
  const double lambda = prm.lambda_override >= 0.0 ? prm.lambda_override : sec.lambda;
  const uint64_t c0 = (uint64_t)chunk * prm.chunk;
  const uint64_t c1 = min(c0 + prm.chunk, prm.n_per_shift);
  const fx_mem<double> Mr{sh_mem + threadIdx.x, FX_THREADS};
  const fx_mem<cplx> Mc{sh_mem + threadIdx.x, FX_THREADS};
  TestFSink sink{0u, 0u, -INFINITY, INFINITY};
  unsigned seen = 0;
  for (uint64_t base = c0 + (uint64_t)threadIdx.x * P; base < c1; base += (uint64_t)FX_THREADS * P) {
    double x[N][P], xbar[N][P], W[P];
    uint32_t bins[(N + 3) / 4][P];
    unsigned valid;
    fx_make_points<RULE, N, P, true>(prm, N, (uint32_t)sec.sector_id, sh_delta, nullptr, base, c1, x, xbar, W, valid, bins);
    cplx X[N][P], det[P];
    fx_deform_points(sh_deform, lambda, x, xbar, Mr, X, det);
    sink.valid = valid;
    seen += __popc(valid);
    fx_run<cplx, N, P>(sh_prog, X, Mc, sink);
  }
  // block reduction in a fixed order: lanes by shuffle tree, warps in order
  double v[4] = {(double)sink.bad, sink.max_im, sink.min_abs2, (double)seen};
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    v[0] += __shfl_down_sync(0xffffffffu, v[0], off);
    v[1] = fmax(v[1], __shfl_down_sync(0xffffffffu, v[1], off));
    v[2] = fmin(v[2], __shfl_down_sync(0xffffffffu, v[2], off));
    v[3] += __shfl_down_sync(0xffffffffu, v[3], off);
  }
  __syncthreads();
  if ((threadIdx.x & 31) == 0)
    for (int q = 0; q < 4; ++q) sh_red[(threadIdx.x >> 5) * 4 + q] = v[q];
  __syncthreads();
  if (threadIdx.x == 0) {
    double o[4] = {0.0, -INFINITY, INFINITY, 0.0};
    for (int w = 0; w < FX_THREADS / 32; ++w) {
      o[0] += sh_red[w * 4];
      o[1] = fmax(o[1], sh_red[w * 4 + 1]);
      o[2] = fmin(o[2], sh_red[w * 4 + 2]);
      o[3] += sh_red[w * 4 + 3];
    }
    for (int q = 0; q < 4; ++q) prm.testf_out[(size_t)b * 4 + q] = o[q];
  }
}

struct EvalSinkCplx {
  double *out;
  int K;
  unsigned valid;
  const cplx (&det)[P];
  __device__ __forceinline__ void operator()(int k, cplx (&A)[P]) {
    FX_PLOOP {
      if ((valid >> p) & 1u) {
        const cplx v = t_mul(det[p], A[p]);
        out[((size_t)p * K + k) * 2] = v.re;
        out[((size_t)p * K + k) * 2 + 1] = v.im;
      }
    }
  }
};

__global__ void __launch_bounds__(FX_THREADS) fx_eval_cplx(const __grid_constant__ fx_eval_params prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  const fx_sector_dev sec = prm.sectors[prm.sector];
  fx_ins *sh_prog = reinterpret_cast<fx_ins *>(smem);
  fx_ins *sh_deform = sec.deform_len ? sh_prog + sec.main_len : nullptr;
  double *sh_mem = reinterpret_cast<double *>(smem + (size_t)prm.prog_ins_max * 16);
  fx_copy_program(sh_prog, prm.arena + sec.main_off, sec.main_len);
  if (sec.deform_len) fx_copy_program(sh_deform, prm.arena + sec.deform_off, sec.deform_len);
  __syncthreads();
  const uint64_t first = ((uint64_t)blockIdx.x * FX_THREADS + threadIdx.x) * P;
  if (first >= prm.npts) return;
  double x[N][P], xbar[N][P];
  unsigned valid = 0;
  FX_PLOOP {
    const bool ok = first + p < prm.npts;
    if (ok) valid |= 1u << p;
#pragma unroll
    for (int k = 0; k < N; ++k) {
      x[k][p] = ok ? prm.x[(first + p) * N + k] : 0.5;
      xbar[k][p] = 1.0 - x[k][p];
    }
  }
  const fx_mem<double> Mr{sh_mem + threadIdx.x, FX_THREADS};
  const fx_mem<cplx> Mc{sh_mem + threadIdx.x, FX_THREADS};
  cplx X[N][P], det[P];
  fx_deform_points(sh_deform, sec.lambda, x, xbar, Mr, X, det);
  EvalSinkCplx sink{prm.out + first * sec.K * 2, sec.K, valid, det};
  fx_run<cplx, N, P>(sh_prog, X, Mc, sink);
}

}  // namespace
using namespace FX_CAT(fx_cplx_n, FX_N);

cudaError_t FX_CAT(fx_launch_integrate_cplx_n, FX_N)(const fx_integrate_params &prm, int nsectors, size_t smem,
                                                     cudaStream_t st) {
  const unsigned grid = (unsigned)((size_t)nsectors * prm.n_shifts * prm.nchunks);
  cudaError_t e;
#define FX_LAUNCH(RULE)                                                                                                \
  {                                                                                                                    \
    e = cudaFuncSetAttribute(fx_integrate_cplx<RULE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);         \
    if (e != cudaSuccess) return e;                                                                                    \
    fx_integrate_cplx<RULE><<<grid, FX_THREADS, smem, st>>>(prm);                                                        \
  }
  if (prm.rule == FIESTA_RULE_LATTICE) FX_LAUNCH(FIESTA_RULE_LATTICE)
  else if (prm.rule == FIESTA_RULE_MC) FX_LAUNCH(FIESTA_RULE_MC)
  else FX_LAUNCH(FIESTA_RULE_VEGAS)
#undef FX_LAUNCH
  return cudaGetLastError();
}

cudaError_t FX_CAT(fx_launch_eval_cplx_n, FX_N)(const fx_eval_params &prm, size_t smem, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(fx_eval_cplx, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  const uint64_t per_block = (uint64_t)FX_THREADS * P;
  const unsigned grid = (unsigned)((prm.npts + per_block - 1) / per_block);
  if (grid == 0) return cudaSuccess;
  fx_eval_cplx<<<grid, FX_THREADS, smem, st>>>(prm);
  return cudaGetLastError();
}

cudaError_t FX_CAT(fx_launch_testf_cplx_n, FX_N)(const fx_integrate_params &prm, int nsectors, size_t smem, cudaStream_t st) {
  const unsigned grid = (unsigned)((size_t)nsectors * prm.n_shifts * prm.nchunks);
  cudaError_t e;
#define FX_LAUNCH(RULE)                                                                                            \
  {                                                                                                                \
    e = cudaFuncSetAttribute(fx_testf_cplx<RULE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);         \
    if (e != cudaSuccess) return e;                                                                                \
    fx_testf_cplx<RULE><<<grid, FX_THREADS, smem, st>>>(prm);                                                        \
  }
  if (prm.rule == FIESTA_RULE_LATTICE) FX_LAUNCH(FIESTA_RULE_LATTICE)
  else FX_LAUNCH(FIESTA_RULE_MC)
#undef FX_LAUNCH
  return cudaGetLastError();
}
