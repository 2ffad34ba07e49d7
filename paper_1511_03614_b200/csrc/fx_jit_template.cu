// fx_jit_template.cu -- the evaluation kernel of real sectors with the program walk left OPEN.
//
// build.py compiles this file to PTX (one per NX), not to SASS.  The kernel is the same as
// fx_integrate_real (points made on the device, periodising transform, accumulation, block-level
// reduction: SURVEY 8(a) A1, A2, A6, A7) except that where the interpreter walks the instruction
// program (A5, "a cycle through all the operations") it carries ONE marker line of
// inline assembly naming the registers of x[k][p], W[p], the valid mask and the accumulator
// address.  fiesta_compile (fx_jit.cpp) replaces that line, per sector, by the sector's fx_ins
// program lowered to straight-line PTX on virtual registers -- the same operations in the same
// order with the same roundings (.rn, explicit fma) as the interpreter's handlers -- and assembles
// the result for sm_100a with the in-process PTX assembler.  The "internal form" of an integrand
// is then native code: no fetch, no decode, no indirect branch, and ptxas does the register
// allocation over all P points at once.
//
// Marker operand order (fx_jit.cpp parses it): nonfinite, valid, acc, W[0..P), x[0][0..P), x[1][..), ...
#define FX_WANT(is_cplx, nx, p) 0  // no interpreter fast path in this translation unit
#include "fx_device_common.cuh"

#ifndef FXJ_NX
#error "compile with -DFXJ_NX=4|8|12"
#endif
#ifndef FXJ_RULE
#define FXJ_RULE FIESTA_RULE_LATTICE
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
// fx_make_points<FIESTA_RULE_LATTICE>: x and W are bit-identical.
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
      const uint64_t G = prm.log2_n ? (prm.genvec[k] << (64 - prm.log2_n)) : 0ull;
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

#define FXJ_X2(k) "d"(x[k][0]), "d"(x[k][1])
#if FXJ_NX == 4
#define FXJ_FMT "%0 %1 %2 %3 %4 %5 %6 %7 %8 %9 %10 %11 %12"
#define FXJ_XS FXJ_X2(0), FXJ_X2(1), FXJ_X2(2), FXJ_X2(3)
#elif FXJ_NX == 8
#define FXJ_FMT "%0 %1 %2 %3 %4 %5 %6 %7 %8 %9 %10 %11 %12 %13 %14 %15 %16 %17 %18 %19 %20"
#define FXJ_XS FXJ_X2(0), FXJ_X2(1), FXJ_X2(2), FXJ_X2(3), FXJ_X2(4), FXJ_X2(5), FXJ_X2(6), FXJ_X2(7)
#else
#define FXJ_FMT \
  "%0 %1 %2 %3 %4 %5 %6 %7 %8 %9 %10 %11 %12 %13 %14 %15 %16 %17 %18 %19 %20 %21 %22 %23 %24 %25 %26 %27 %28"
#define FXJ_XS                                                                                             \
  FXJ_X2(0), FXJ_X2(1), FXJ_X2(2), FXJ_X2(3), FXJ_X2(4), FXJ_X2(5), FXJ_X2(6), FXJ_X2(7), FXJ_X2(8), FXJ_X2(9), \
      FXJ_X2(10), FXJ_X2(11)
#endif

extern "C" __global__ void __launch_bounds__(FX_THREADS, FXJ_NX <= 8 ? 6 : 4)
    fxj_integrate(const __grid_constant__ fx_integrate_params prm) {
  constexpr int PB = FX_P_REAL;  // points per thread and batch: the interpreter's
  constexpr int P = FXJ_P;       // points per pass of the program body
  constexpr int NX = FXJ_NX;
  static_assert(P == 2 && PB % P == 0, "the marker lists 2 points per variable");
  extern __shared__ __align__(16) unsigned char smem[];
  const int b = blockIdx.x;
  const int chunk = b % prm.nchunks;
  const int r = (b / prm.nchunks) % prm.n_shifts;
  const int sel_idx = prm.sel_base + b / (prm.nchunks * prm.n_shifts);
  const fx_sector_dev sec = prm.sectors[prm.sel[sel_idx]];
  const int dim = prm.dim;
  const fxj_smem_layout L = fxj_layout();
  double *sh_acc = reinterpret_cast<double *>(smem + L.acc);
  uint64_t *sh_delta = reinterpret_cast<uint64_t *>(smem + L.delta);
  double *sh_wsum = reinterpret_cast<double *>(smem + L.wsum);

  fx_block_setup(prm, dim, (uint32_t)sec.sector_id, r, sel_idx, sh_delta, nullptr, nullptr);
  const int nslots = 2 * sec.K;
  for (int s = 0; s < nslots; ++s) sh_acc[s * FX_THREADS + threadIdx.x] = 0.0;
  __syncthreads();

  const uint64_t c0 = (uint64_t)chunk * prm.chunk;
  const uint64_t c1 = min(c0 + prm.chunk, prm.n_per_shift);
  unsigned nonfinite = 0;
  const uint32_t acc = (uint32_t)__cvta_generic_to_shared(sh_acc + threadIdx.x);
  // The trip count is the same for every thread of the block (points past the end are masked by
  // `valid`), so the block can re-align its warps at every pass: a sector's native code is ~45 KB
  // of straight-line instructions, far beyond the instruction caches, and warps that drift apart
  // each stream it from L2 on their own; in step they share one stream.
#pragma unroll 1
  for (uint64_t it = c0; it < c1; it += (uint64_t)FX_THREADS * PB) {
    // A thread owns the same PB = 4 consecutive points per batch as in the interpreter kernel, but
    // walks the program over them in two passes of P = 2.  With 4 points live (64 registers of x
    // alone, 4 copies of every temporary) ptxas, held to 128 registers, serialises the points into
    // dependent chains and over-subscribes the uniform registers the immediates live in; with 2 it
    // interleaves both chains in 80 registers and 6 blocks are resident instead of 4.  Outputs are
    // accumulated in point order either way, so the sums are unchanged (bit-identical to the
    // interpreter's).
#pragma unroll 1
    for (int h = 0; h < PB / P; ++h) {
      const uint64_t base = it + (uint64_t)threadIdx.x * PB + (uint64_t)h * P;
      __syncthreads();
      double x[NX][P], W[P];
      unsigned valid;
      fxj_make_points<NX, P>(prm, dim, sh_delta, base, c1, x, W, valid);
      asm volatile("FXJIT_BODY " FXJ_FMT ";"
                   : "+r"(nonfinite)
                   : "r"(valid), "r"(acc), "d"(W[0]), "d"(W[1]), FXJ_XS
                   : "memory");
    }
  }
  if (prm.nsel < 0) {  // never true: keeps the two library wrappers in the PTX
    sh_acc[threadIdx.x] = fxj_log(sh_acc[threadIdx.x]);
    sh_acc[threadIdx.x + FX_THREADS] = fxj_exp(sh_acc[threadIdx.x + FX_THREADS]);
  }
  __syncthreads();
  double *out = prm.partials + (((size_t)sel_idx * prm.n_shifts + r) * prm.nchunks + chunk) * FX_ACC_SLOTS;
  fx_block_reduce(sh_acc, sh_wsum, nslots, out);
  fx_block_finish(prm, dim, sel_idx, nonfinite, nullptr);
}
