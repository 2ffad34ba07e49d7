// fx_jit_template.cu -- the evaluation kernels of real sectors with the program walk left OPEN.
//
// build.py compiles this file to PTX (one per NX and MODE), not to SASS.  The kernels are the same
// as fx_integrate_real / fx_eval_real (points made on the device, periodising transform or Vegas
// map, accumulation, block-level reduction, histogram: SURVEY 8(a) A1-A3, A6-A8) except that where
// the interpreter walks the instruction program (A5, "a cycle through all the
// operations") they carry ONE marker line of inline assembly naming the registers of x[k][p], W[p],
// the valid mask and the accumulator address.  fx_jit.cpp replaces that line, per sector, by the
// sector's fx_ins program lowered to straight-line PTX on virtual registers -- the same operations
// in the same order with the same roundings (.rn, explicit fma) as the interpreter's handlers --
// and assembles the result for sm_100a with the in-process PTX assembler.  The "internal form" of
// an integrand is then native code: no fetch, no decode, no indirect branch, and ptxas does the
// register allocation over all P points at once.
//
// MODE 0 lattice, 1 plain MC, 2 Vegas (fiesta rule kinds), 3 eval (caller's points: the parity
// hook fiesta_eval_points runs the SAME generated program body as the integration kernels).
//
// Marker operand order (fx_jit.cpp parses it):
//   integrate: [h2[0..P) if Vegas] valid acc W[0..P) x[0][0..P) x[1][..) ...
//   eval:      valid out x[0][0..P) ...
#define FX_WANT(is_cplx, nx, p) 0  // no interpreter fast path in this translation unit
#define FX_NO_MIXED_MASK  // fiesta_set_mixed: phase 1 runs on the real interpreter kernels only
#include "fx_device_common.cuh"

#ifndef FXJ_NX
#error "compile with -DFXJ_NX=4|8|12"
#endif
#ifndef FXJ_MODE
#error "compile with -DFXJ_MODE=0..3"
#endif

// FP64 log/exp are library routines (CUDA math); the generated code calls these two
extern "C" __device__ __noinline__ double fxj_log(double a) { return log(a); }
extern "C" __device__ __noinline__ double fxj_exp(double a) { return exp(a); }

struct fxj_xs {
  double x, s;
};
// weights other than the default r = 3: one out-of-line copy
static __device__ __noinline__ fxj_xs fxj_transform_any(const fx_transform *tf, uint64_t t) {
  fxj_xs c;
  double xb;
  korobov_xs(*tf, t, c.x, xb, c.s);
  return c;
}

// Lattice points of one pass, inline (2 points x NX coordinates; with 4 points live inlining was slower) and
// without xbar = 1-x, which real programs never read.  Same arithmetic and order as
// fx_make_points<FIESTA_RULE_LATTICE>: x and W are bit-identical -- except that it knows nothing of the mixed
// mode's mask (fx_flag_mask): with fiesta_set_mixed on, phase 1 runs on the interpreter kernels.  (The per-point branch on the weight
// also keeps ptxas from interleaving all 2 NX transforms at once, which costs it spills.)
template <int NX, int P>
__device__ __forceinline__ void fxj_make_points(const fx_integrate_params &prm, int dim, const uint64_t *sh_delta,
                                                uint64_t j0, uint64_t jend, double (&x)[NX][P], double (&W)[P],
                                                unsigned &valid) {
  valid = 0;
  FX_PLOOP {
    W[p] = 1.0;
    if (j0 + p < jend) valid |= 1u << p;
  }
  const fx_transform *tf = reinterpret_cast<const fx_transform *>(sh_delta + FX_NXMAX);
  const bool r3 = tf->r == 3;
#pragma unroll
  for (int k = 0; k < NX; ++k) {
    if (k < dim) {
      const uint64_t G = fx_lattice_steps(sh_delta)[k];
      const uint64_t d = sh_delta[k];
      FX_PLOOP {
        const uint64_t t = (j0 + p) * G + d;
        double xb, sv;
        if (r3) {
          korobov_xs_r<3>(*tf, t, x[k][p], xb, sv);
        } else {
          const fxj_xs c = fxj_transform_any(tf, t);
          x[k][p] = c.x;
          sv = c.s;
        }
        W[p] *= sv;
      }
    } else {
      FX_PLOOP { x[k][p] = 0.5; }
    }
  }
  FX_PLOOP { W[p] = korobov_weight(*tf, W[p]); }
}

// FXJ_FMT ("%0 %1 ... %(n-1)": the marker line lists every operand once, in order) and the operand lists
// FXJ_XS ("d"(x[0][0]), ...), FXJ_WS ("d"(W[0]), ...), FXJ_H2S ("+d"(h2[0]), ...) come from build.py
#if !defined(FXJ_FMT) || !defined(FXJ_XS) || !defined(FXJ_WS) || !defined(FXJ_H2S)
#error "build.py passes FXJ_FMT, FXJ_XS, FXJ_WS, FXJ_H2S"
#endif

#if FXJ_MODE != 3

constexpr int FXJ_RULE = FXJ_MODE;
// resident blocks per SM the register allocation is held to: the most for which the assembler reports
// no spill on the configurations' programs (lattice: 6 x 80 registers at NX <= 8; plain MC carries
// the Philox state on top: 5 x 96; Vegas also the bins and h2: 4 x 128)
constexpr int FXJ_BLOCKS = FXJ_MODE == 2 ? (FXJ_P_VEGAS == 1 ? 7 : 4) : FXJ_MODE == 1 ? (FXJ_NX <= 8 ? 5 : 4) : (FXJ_NX <= 8 ? 6 : 4);

extern "C" __global__ void __launch_bounds__(FX_THREADS, FXJ_BLOCKS)
    fxj_integrate(const __grid_constant__ fx_integrate_params prm) {
  constexpr int PB = FX_P_REAL;  // points per thread and batch: the interpreter's
  constexpr int P = FXJ_P_OF(FXJ_MODE);  // points per pass of the program body
  constexpr int NX = FXJ_NX;
  constexpr bool vegas = FXJ_RULE == FIESTA_RULE_VEGAS;
  static_assert(PB % P == 0, "a batch is a whole number of passes");
  extern __shared__ __align__(16) unsigned char smem[];
  const fx_block_id id0 = fx_block_coords(prm);
  const int chunk = id0.chunk, r = id0.r, sel_idx = id0.sel_idx;
  const fx_sector_dev sec = prm.sectors[prm.sel[sel_idx]];
  const int dim = prm.dim;
  const fxj_smem_layout L = fxj_layout(dim, prm.nbins, vegas, fxj_acc_slots(vegas, false, sec.K));
  double *sh_acc = reinterpret_cast<double *>(smem + L.acc);
  uint64_t *sh_delta = reinterpret_cast<uint64_t *>(smem + L.delta);
  double *sh_grid = reinterpret_cast<double *>(smem + L.grid);
  double *sh_hist = reinterpret_cast<double *>(smem + L.hist);
  double *sh_wsum = reinterpret_cast<double *>(smem + L.wsum);

  fx_block_setup(prm, dim, (uint32_t)sec.sector_id, r, sel_idx, sh_delta, sh_grid, sh_hist);
  const int nslots = 2 * sec.K;
  for (int s = 0; s < nslots; ++s) sh_acc[s * FX_THREADS + threadIdx.x] = 0.0;
  unsigned *sh_nf = reinterpret_cast<unsigned *>(smem + L.nf);  // non-finite values seen by this thread (the body counts)
  sh_nf[2 * threadIdx.x] = 0u;
  if (threadIdx.x == 96) {
    const uint64_t c0 = (uint64_t)chunk * prm.chunk;
    const uint64_t c1 = min(c0 + prm.chunk, prm.n_per_shift);
    uint64_t *rg = fx_block_range(sh_delta);
    rg[0] = c0;
    rg[1] = c1;
    rg[2] = (c1 - c0 + (uint64_t)FX_THREADS * PB - 1) / ((uint64_t)FX_THREADS * PB) * (PB / P);
  }
  __syncthreads();

  // The trip count is the same for every thread of the block (points past the end are masked by
  // `valid`), so the block can re-align its warps at every pass: a sector's native code is ~45 KB
  // of straight-line instructions, far beyond the instruction caches, and warps that drift apart
  // each stream it from L2 on their own; in step they share one stream.
  //
  // A thread owns the same PB = 4 consecutive points per batch as in the interpreter kernel, but
  // walks the program over them in two passes of P = 2.  With 4 points live (64 registers of x
  // alone, 4 copies of every temporary) ptxas, held to 128 registers, serialises the points into
  // dependent chains and over-subscribes the uniform registers the immediates live in; with 2 it
  // interleaves both chains in 80 registers and 6 blocks are resident instead of 4.  Outputs are
  // accumulated (and, for Vegas, histogrammed) in point order either way, so the sums are
  // unchanged (bit-identical to the interpreter's).
  //
  // Pass q covers the points c0 + (q / (PB/P)) * 512 + PB tid + P (q % (PB/P)) + {0..P-1} (a chunk has at most 2^17 points).
  // Only q is carried across the program body: the block's range, the thread index and the
  // accumulator address are read again in every pass (volatile), so that the register allocation
  // of the body has no loop invariants to hold -- or to spill.
#pragma unroll 1
  for (uint32_t q = 0;; ++q) {
    const uint64_t *rg = fx_block_range(sh_delta);
    if (q >= (uint32_t)fx_lds_volatile(rg + 2)) break;
    {
      const unsigned tid = fx_tid_volatile();
      const uint64_t c1 = fx_lds_volatile(rg + 1);
      const uint64_t base = fx_lds_volatile(rg) + (uint64_t)((q / (PB / P)) * (FX_THREADS * PB) + tid * PB + (q % (PB / P)) * P);
      const uint32_t acc = (uint32_t)__cvta_generic_to_shared(sh_acc) + tid * 8u;
      __syncthreads();
      double x[NX][P], W[P];
      unsigned valid;
#if FXJ_MODE == 0
      fxj_make_points<NX, P>(prm, dim, sh_delta, base, c1, x, W, valid);
      asm volatile("FXJIT_BODY " FXJ_FMT ";"
                   :
                   : "r"(valid), "r"(acc), FXJ_WS, FXJ_XS
                   : "memory");
#else
      double xbar[NX][P];
      uint32_t bins[(NX + 3) / 4][P];
      fx_make_points<FXJ_RULE, NX, P, true>(prm, dim, (uint32_t)sec.sector_id, sh_delta, sh_grid, base, c1, x, xbar, W, valid,
                                      bins);
#if FXJ_MODE == 2
      double h2[P];
      FX_PLOOP { h2[p] = 0.0; }
      asm volatile("FXJIT_BODY " FXJ_FMT ";"
                   : FXJ_H2S
                   : "r"(valid), "r"(acc), FXJ_WS, FXJ_XS
                   : "memory");
      fx_hist_points<NX, P>(sh_hist, dim, prm.nbins, valid, bins, h2);
#else
      asm volatile("FXJIT_BODY " FXJ_FMT ";"
                   :
                   : "r"(valid), "r"(acc), FXJ_WS, FXJ_XS
                   : "memory");
#endif
#endif
    }
  }
  if (prm.nsel < 0) {  // never true: keeps the two library wrappers in the PTX
    sh_acc[threadIdx.x] = fxj_log(sh_acc[threadIdx.x]);
    sh_acc[threadIdx.x + FX_THREADS] = fxj_exp(sh_acc[threadIdx.x + FX_THREADS]);
  }
  __syncthreads();
  const fx_block_id id1 = fx_block_coords(prm);  // again, rather than kept across the loop
  const unsigned nonfinite = sh_nf[2 * threadIdx.x];
  fx_block_reduce(sh_acc, sh_wsum, 2 * prm.sectors[prm.sel[id1.sel_idx]].K, fx_partial_record(prm, id1.sel_idx, id1.r, id1.chunk));
  fx_block_finish(prm, dim, id1.sel_idx, id1.chunk, nonfinite, sh_hist);
}

#else  // FXJ_MODE == 3: the program body on the caller's points (fiesta_eval_points, native tier)

extern "C" __global__ void __launch_bounds__(FX_THREADS) fxj_eval(const __grid_constant__ fx_eval_params prm) {
  constexpr int P = FXJ_P_OF(FXJ_MODE);
  constexpr int NX = FXJ_NX;
  const fx_sector_dev sec = prm.sectors[prm.sector];
  const uint64_t first = ((uint64_t)blockIdx.x * FX_THREADS + threadIdx.x) * P;
  if (first < prm.npts) {
    double x[NX][P];
    unsigned valid = 0;
    FX_PLOOP {
      const bool ok = first + p < prm.npts;
      if (ok) valid |= 1u << p;
#pragma unroll
      for (int k = 0; k < NX; ++k) x[k][p] = (ok && k < prm.dim) ? prm.x[(first + p) * prm.dim + k] : 0.5;
    }
    double *out = prm.out + first * sec.K * 2;  // [point][K][re, im]
    asm volatile("FXJIT_BODY " FXJ_FMT ";" : : "r"(valid), "l"(out), FXJ_XS : "memory");
  }
  if (prm.npts == ~0ull) {  // never true: keeps the two library wrappers in the PTX
    prm.out[0] = fxj_log(prm.out[0]);
    prm.out[1] = fxj_exp(prm.out[1]);
  }
}

#endif
