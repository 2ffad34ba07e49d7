// fx_jit_template_cplx.cu -- the evaluation kernels of complex sectors ("-complex", with
// the contour deformation of PAPER.md:53, :404; R11) with BOTH program walks left open.
//
// Same scheme as fx_jit_template.cu (which see): build.py compiles this file to PTX once per
// dimension N and MODE; fx_jit.cpp replaces the two marker lines, per sector, by
//   FXJIT_DEFORM  the sector's real gradient/Hessian program (dF/dx_k, d2F/dx_k dx_l of the
//                 deformation polynomial) lowered to PTX: reads x[0..N), writes gh[0..NGH);
//   FXJIT_BODY    the sector's main program lowered to PTX on (re, im) register pairs -- the same
//                 instruction sequences as the interpreter's complex handlers -- reading z[k].
// Between the two, the Jacobian and its determinant are built in registers by the same code as in
// the interpreter kernel (fx_deform.cuh).  One point per thread and pass (a 7 x 7 complex Jacobian is
// 98 doubles).  The kernel is otherwise fx_integrate_cplx / fx_eval_cplx (fx_kernels_cplx.cu).
//
// Marker operand order (fx_jit.cpp parses it):
//   FXJIT_DEFORM  gh[0..NGH) x[0..N)
//   FXJIT_BODY    integrate: [h2 if Vegas] valid acc Wd.re Wd.im z[0].re z[0].im z[1].re ...
//                 eval:      valid out det.re det.im z[0].re z[0].im ...
// build.py passes the operand lists as macros: FXJ_DFMT / FXJ_FMT ("%0 %1 ..."), FXJ_GH_OUTS
// ("=d"(gh[0]), ...), FXJ_X_INS ("d"(xv[0]), ...), FXJ_Z_INS ("d"(xv[0]), "d"(zi[0]), ...).
#define FX_WANT(is_cplx, nx, p) 0  // no interpreter fast path in this translation unit
#define FX_NO_MIXED_MASK  // fiesta_set_mixed: phase 1 runs on the real interpreter kernels only
#include "fx_device_common.cuh"
#include "fx_deform.cuh"

#if !defined(FX_N) || !defined(FXJ_MODE)
#error "compile with -DFX_N=1..8 -DFXJ_MODE=0..3"
#endif

// library-backed complex operations (CUDA math inside): the generated code calls these
extern "C" __device__ __noinline__ cplx fxj_clog(double re, double im) { return t_log(cplx{re, im}); }
extern "C" __device__ __noinline__ cplx fxj_cexp(double re, double im) { return t_exp(cplx{re, im}); }
extern "C" __device__ __noinline__ cplx fxj_csqrt(double re, double im) { return t_sqrt(cplx{re, im}); }

constexpr int N = FX_N;
constexpr int NGH = N + N * (N + 1) / 2;

// x -> Im z and det J through the sector's gradient/Hessian program (left open)
__device__ __forceinline__ cplx fxj_deform(double lambda, const double (&xv)[N], const double (&xbv)[N], double (&zi)[N]) {
  double gh[NGH];
  asm volatile("FXJIT_DEFORM " FXJ_DFMT ";" : FXJ_GH_OUTS : FXJ_X_INS);
  return fx_jacobian_det<N>(lambda, xv, xbv, [&](int slot) { return gh[slot]; }, zi);
}

#if FXJ_MODE != 3

constexpr int FXJ_RULE = FXJ_MODE;

extern "C" __global__ void __launch_bounds__(FX_THREADS, FXJ_CBLOCKS)
    fxj_integrate(const __grid_constant__ fx_integrate_params prm) {
  constexpr int P = FX_P_CPLX;
  static_assert(P == 1, "one point per thread");
  constexpr bool vegas = FXJ_RULE == FIESTA_RULE_VEGAS;
  extern __shared__ __align__(16) unsigned char smem[];
  const fx_block_id id0 = fx_block_coords(prm);
  const int chunk = id0.chunk, r = id0.r, sel_idx = id0.sel_idx;
  const fx_sector_dev sec = prm.sectors[prm.sel[sel_idx]];
  const fxj_smem_layout L = fxj_layout(N, prm.nbins, vegas, fxj_acc_slots(vegas, true, sec.K));
  double *sh_acc = reinterpret_cast<double *>(smem + L.acc);
  uint64_t *sh_delta = reinterpret_cast<uint64_t *>(smem + L.delta);
  double *sh_grid = reinterpret_cast<double *>(smem + L.grid);
  double *sh_hist = reinterpret_cast<double *>(smem + L.hist);
  double *sh_wsum = reinterpret_cast<double *>(smem + L.wsum);

  fx_block_setup(prm, N, (uint32_t)sec.sector_id, r, sel_idx, sh_delta, sh_grid, sh_hist);
  const int nslots = 4 * sec.K;
  for (int s = 0; s < nslots; ++s) sh_acc[s * FX_THREADS + threadIdx.x] = 0.0;
  unsigned *sh_nf = reinterpret_cast<unsigned *>(smem + L.nf);  // non-finite values seen by this thread (the body counts)
  sh_nf[2 * threadIdx.x] = 0u;
  __syncthreads();

  const uint64_t c0 = (uint64_t)chunk * prm.chunk;
  const uint64_t c1 = min(c0 + prm.chunk, prm.n_per_shift);
  const uint32_t acc = (uint32_t)__cvta_generic_to_shared(sh_acc + threadIdx.x);
  const bool deform = sec.deform_len != 0;
#pragma unroll 1
  for (uint64_t it = c0; it < c1; it += (uint64_t)FX_THREADS * P) {  // block-uniform trip count
    const uint64_t base = it + (uint64_t)threadIdx.x * P;
    __syncthreads();  // the block's warps share one instruction stream (see fx_jit_template.cu)
    double x[N][P], xbar[N][P], W[P];
    uint32_t bins[(N + 3) / 4][P];
    unsigned valid;
    fx_make_points<FXJ_RULE, N, P>(prm, N, (uint32_t)sec.sector_id, sh_delta, sh_grid, base, c1, x, xbar, W, valid, bins);
    double xv[N], xbv[N], zi[N];
#pragma unroll
    for (int k = 0; k < N; ++k) {
      xv[k] = x[k][0];
      xbv[k] = xbar[k][0];
      zi[k] = 0.0;
    }
    cplx det{1.0, 0.0};
    if (deform) det = fxj_deform(sec.lambda, xv, xbv, zi);
    const cplx Wd = t_mulc(det, W[0]);
#if FXJ_MODE == 2
    double h2[P] = {0.0};
    asm volatile("FXJIT_BODY " FXJ_FMT ";"
                 : "+d"(h2[0])
                 : "r"(valid), "r"(acc), "d"(Wd.re), "d"(Wd.im), FXJ_Z_INS
                 : "memory");
    fx_hist_points<N, P>(sh_hist, N, prm.nbins, valid, bins, h2);
#else
    asm volatile("FXJIT_BODY " FXJ_FMT ";"
                 :
                 : "r"(valid), "r"(acc), "d"(Wd.re), "d"(Wd.im), FXJ_Z_INS
                 : "memory");
#endif
  }
  if (prm.nsel < 0) {  // never true: keeps the library wrappers in the PTX
    const cplx a = fxj_clog(sh_acc[0], sh_acc[1]), e = fxj_cexp(sh_acc[2], sh_acc[3]), q = fxj_csqrt(sh_acc[4], sh_acc[5]);
    sh_acc[threadIdx.x] = a.re + a.im + e.re + e.im + q.re + q.im;
  }
  __syncthreads();
  const fx_block_id id1 = fx_block_coords(prm);  // again, rather than kept across the loop
  const unsigned nonfinite = sh_nf[2 * threadIdx.x];
  fx_block_reduce(sh_acc, sh_wsum, 4 * prm.sectors[prm.sel[id1.sel_idx]].K, fx_partial_record(prm, id1.sel_idx, id1.r, id1.chunk));
  fx_block_finish(prm, N, id1.sel_idx, id1.chunk, nonfinite, sh_hist);
}

#else  // FXJ_MODE == 3: both program bodies on the caller's points (fiesta_eval_points, native tier)

extern "C" __global__ void __launch_bounds__(FX_THREADS) fxj_eval(const __grid_constant__ fx_eval_params prm) {
  const fx_sector_dev sec = prm.sectors[prm.sector];
  const uint64_t first = (uint64_t)blockIdx.x * FX_THREADS + threadIdx.x;
  if (first < prm.npts) {
    double xv[N], xbv[N], zi[N];
#pragma unroll
    for (int k = 0; k < N; ++k) {
      xv[k] = prm.x[first * N + k];
      xbv[k] = 1.0 - xv[k];
      zi[k] = 0.0;
    }
    cplx det{1.0, 0.0};
    if (sec.deform_len != 0) det = fxj_deform(sec.lambda, xv, xbv, zi);
    const unsigned valid = 1u;
    double *out = prm.out + first * sec.K * 2;  // [point][K][re, im]
    asm volatile("FXJIT_BODY " FXJ_FMT ";" : : "r"(valid), "l"(out), "d"(det.re), "d"(det.im), FXJ_Z_INS : "memory");
  }
  if (prm.npts == ~0ull) {  // never true: keeps the library wrappers in the PTX
    const cplx a = fxj_clog(prm.out[0], prm.out[1]), e = fxj_cexp(prm.out[2], prm.out[3]), q = fxj_csqrt(prm.out[4], prm.out[5]);
    prm.out[0] = a.re + a.im + e.re + e.im + q.re + q.im;
  }
}

#endif
