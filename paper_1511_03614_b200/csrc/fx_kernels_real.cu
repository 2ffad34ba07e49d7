// fx_kernels_real.cu -- evaluation kernels for real (Euclidean) sectors: lattice / MC / Vegas
// points made on the device, program walk, accumulation of sum g and sum g^2 per order
// (SURVEY 8(a) A1-A3, A5-A7, A8 histogram part).  Replaces the reference's CUDA kernel of
// PAPER.md:118-126 (thread per point, temporaries in GPU memory, points uploaded per batch).
#define FX_WANT(is_cplx, nx, p) ((is_cplx) == 0 && (p) == 4)  // fast-path variants this file instantiates
#include "fx_device_common.cuh"

namespace {

// accumulator slots of a launch: what the call's real sectors need (make_plan), not the record's 32
// (2 K_max accumulators + FX_P_REAL weights + 1 counter: fiesta_abi_integrate.inc make_plan)
__host__ __device__ inline int fx_real_acc_slots(const fx_integrate_params &prm) {
  return prm.acc_slots_real > 0 ? prm.acc_slots_real : FX_ACC_SLOTS;
}

template <int P, bool VEGAS>
struct IntegrateSinkReal {
  double *acc;      // &acc[0][tid], slot stride FX_THREADS
  const double *W;  // &W[0][tid] in shared memory, stride FX_THREADS: read here, at the outputs, instead of held in
                    // 2 P registers across the walk (that is what lets 4 blocks of 128 registers be resident)
  unsigned valid;
  unsigned nonfinite;
  double *h2;       // Vegas: &h2[0][tid] in shared memory (sum over the orders of g^2, for the histogram)
  __device__ __forceinline__ void operator()(int k, double (&A)[P]) {
    double s1 = acc[(2 * k) * FX_THREADS], s2 = acc[(2 * k + 1) * FX_THREADS];
    FX_PLOOP {
      double g = W[p * FX_THREADS] * A[p];
      if (!((valid >> p) & 1u)) g = 0.0;
      nonfinite += isfinite(g) ? 0u : 1u;
      s1 += g;
      s2 = fma(g, g, s2);
      if constexpr (VEGAS) h2[p * FX_THREADS] = fma(g, g, h2[p * FX_THREADS]);
    }
    acc[(2 * k) * FX_THREADS] = s1;
    acc[(2 * k + 1) * FX_THREADS] = s2;
  }
};

template <int NX, int RULE>
__global__ void __launch_bounds__(FX_THREADS, NX <= 4 ? 4 : NX <= 8 ? (RULE == FIESTA_RULE_LATTICE ? 4 : 3) : 3) fx_integrate_real(const __grid_constant__ fx_integrate_params prm) {
  constexpr int P = FX_P_REAL;
  extern __shared__ __align__(16) unsigned char smem[];
  const int b = blockIdx.x;
  const int chunk = b % prm.nchunks;
  const int r = (b / prm.nchunks) % prm.n_shifts;
  const int sel_idx = fx_sel_index(prm, b / (prm.nchunks * prm.n_shifts));
  const fx_sector_dev sec = prm.sectors[prm.sel[sel_idx]];
  const int dim = prm.dim;
  constexpr bool vegas = RULE == FIESTA_RULE_VEGAS;
  const fx_smem_layout L = fx_layout(prm.prog_ins_max, prm.mem_doubles, dim, prm.nbins, vegas, fx_real_acc_slots(prm));
  fx_ins *sh_prog = reinterpret_cast<fx_ins *>(smem + L.prog);
  double *sh_mem = reinterpret_cast<double *>(smem + L.mem);
  double *sh_acc = reinterpret_cast<double *>(smem + L.acc);
  uint64_t *sh_delta = reinterpret_cast<uint64_t *>(smem + L.delta);
  double *sh_grid = reinterpret_cast<double *>(smem + L.grid);
  double *sh_hist = reinterpret_cast<double *>(smem + L.hist);
  double *sh_wsum = reinterpret_cast<double *>(smem + L.wsum);

  fx_copy_program(sh_prog, prm.arena + sec.main_off, sec.main_len);
  fx_block_setup(prm, dim, (uint32_t)sec.sector_id, r, sel_idx, sh_delta, sh_grid, sh_hist);
  const int nslots = 2 * sec.K;
  for (int s = 0; s < nslots; ++s) sh_acc[s * FX_THREADS + threadIdx.x] = 0.0;
  // behind the accumulators: this thread's P weights and its count of non-finite values; for Vegas also the
  // points' sums of g^2 and their bins, which are needed only after the walk
  constexpr int NBW = (NX + 3) / 4;                       // 32-bit words of bins per point
  constexpr int XTRA = vegas ? P + (NBW * P + 1) / 2 : 0;  // doubles per thread (make_plan reserves them)
  double *sh_w = sh_acc + (size_t)(fx_real_acc_slots(prm) - (P + 1 + XTRA)) * FX_THREADS + threadIdx.x;
  unsigned *sh_nf = reinterpret_cast<unsigned *>(sh_w + P * FX_THREADS);
  double *sh_h2 = sh_w + (P + 1) * FX_THREADS;
  uint32_t *sh_bins = reinterpret_cast<uint32_t *>(sh_acc + (size_t)(fx_real_acc_slots(prm) - (NBW * P + 1) / 2) * FX_THREADS) + threadIdx.x;
  *sh_nf = 0u;
  __syncthreads();

  const uint64_t c0 = (uint64_t)chunk * prm.chunk;
  const uint64_t c1 = min(c0 + prm.chunk, prm.n_per_shift);
  const fx_mem<double> M{sh_mem + threadIdx.x, FX_THREADS};
  // the trip count is the same for every thread of the block (points past the end are masked by
  // `valid`): the Vegas histogram update is a warp-collective operation
  for (uint64_t it = c0; it < c1; it += (uint64_t)FX_THREADS * P) {
    const uint64_t base = it + (uint64_t)threadIdx.x * P;
    __syncthreads();  // the block's warps walk the program in step: one instruction stream through the caches
    double x[NX][P], xbar[NX][P], W[P];
    unsigned valid;
    {
      uint32_t bins[NBW][P];
      fx_make_points<RULE, NX, P, RULE == FIESTA_RULE_VEGAS>(prm, dim, (uint32_t)sec.sector_id, sh_delta, sh_grid, base, c1, x, xbar, W, valid, bins);
      FX_PLOOP {
        sh_w[p * FX_THREADS] = W[p];
        if constexpr (vegas) {
          sh_h2[p * FX_THREADS] = 0.0;
#pragma unroll
          for (int q = 0; q < NBW; ++q) sh_bins[(q * P + p) * FX_THREADS] = bins[q][p];
        }
      }
    }
    IntegrateSinkReal<P, vegas> sink{sh_acc + threadIdx.x, sh_w, valid, 0u, sh_h2};
    fx_run<double, NX, P>(sh_prog, x, M, sink);
    *sh_nf += sink.nonfinite;
    if constexpr (vegas) {
      uint32_t bins[NBW][P];
      double h2[P];
      FX_PLOOP {
        h2[p] = sh_h2[p * FX_THREADS];
#pragma unroll
        for (int q = 0; q < NBW; ++q) bins[q][p] = sh_bins[(q * P + p) * FX_THREADS];
      }
      fx_hist_points<NX, P>(sh_hist, dim, prm.nbins, valid, bins, h2);
    }
  }
  __syncthreads();
  const unsigned nonfinite = *sh_nf;
  const fx_block_id id1 = fx_block_coords(prm);  // computed again (volatile read of the block index) rather than kept across the walk
  fx_block_reduce(sh_acc, sh_wsum, 2 * prm.sectors[prm.sel[id1.sel_idx]].K, fx_partial_record(prm, id1.sel_idx, id1.r, id1.chunk));
  fx_block_finish(prm, prm.dim, id1.sel_idx, id1.chunk, nonfinite, sh_hist);
}

template <int P>
struct EvalSinkReal {
  double *out;  // &out[first point of this thread][0][0]
  int K;
  unsigned valid;
  __device__ __forceinline__ void operator()(int k, double (&A)[P]) {
    FX_PLOOP {
      if ((valid >> p) & 1u) {
        out[((size_t)p * K + k) * 2] = A[p];
        out[((size_t)p * K + k) * 2 + 1] = 0.0;
      }
    }
  }
};

template <int NX>
__global__ void __launch_bounds__(FX_THREADS) fx_eval_real(const __grid_constant__ fx_eval_params prm) {
  constexpr int P = FX_P_REAL;
  extern __shared__ __align__(16) unsigned char smem[];
  const fx_sector_dev sec = prm.sectors[prm.sector];
  fx_ins *sh_prog = reinterpret_cast<fx_ins *>(smem);
  double *sh_mem = reinterpret_cast<double *>(smem + (size_t)prm.prog_ins_max * 16);
  fx_copy_program(sh_prog, prm.arena + sec.main_off, sec.main_len);
  __syncthreads();
  const uint64_t first = ((uint64_t)blockIdx.x * FX_THREADS + threadIdx.x) * P;
  if (first >= prm.npts) return;
  double x[NX][P];
  unsigned valid = 0;
  FX_PLOOP {
    const bool ok = first + p < prm.npts;
    if (ok) valid |= 1u << p;
#pragma unroll
    for (int k = 0; k < NX; ++k) x[k][p] = (ok && k < prm.dim) ? prm.x[(first + p) * prm.dim + k] : 0.5;
  }
  const fx_mem<double> M{sh_mem + threadIdx.x, FX_THREADS};
  EvalSinkReal<P> sink{prm.out + first * sec.K * 2, sec.K, valid};
  fx_run<double, NX, P>(sh_prog, x, M, sink);
}

template <typename K>
cudaError_t set_smem(K kernel, size_t bytes) {
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

}  // namespace

size_t fx_integrate_cplx_smem_bytes(const fx_integrate_params &prm) {
  return fx_layout(prm.prog_ins_max, prm.mem_doubles, prm.dim, prm.nbins, prm.rule == FIESTA_RULE_VEGAS,
                   prm.acc_slots_cplx > 0 ? prm.acc_slots_cplx : FX_ACC_SLOTS).total;
}

size_t fx_integrate_smem_bytes(const fx_integrate_params &prm) {
  return fx_layout(prm.prog_ins_max, prm.mem_doubles, prm.dim, prm.nbins, prm.rule == FIESTA_RULE_VEGAS).total;
}

cudaError_t fx_launch_integrate_real(const fx_integrate_params &prm, int nsectors, cudaStream_t st) {
  const size_t smem = fx_layout(prm.prog_ins_max, prm.mem_doubles, prm.dim, prm.nbins, prm.rule == FIESTA_RULE_VEGAS,
                                fx_real_acc_slots(prm)).total;
  const unsigned grid = (unsigned)((size_t)nsectors * prm.n_shifts * prm.nchunks);
  cudaError_t e;
#define FX_LAUNCH2(NX, RULE)                                                            \
  {                                                                                     \
    if ((e = set_smem(fx_integrate_real<NX, RULE>, smem)) != cudaSuccess) return e;     \
    fx_integrate_real<NX, RULE><<<grid, FX_THREADS, smem, st>>>(prm);                     \
  }
#define FX_LAUNCH(NX)                                                  \
  {                                                                    \
    if (prm.rule == FIESTA_RULE_LATTICE) FX_LAUNCH2(NX, FIESTA_RULE_LATTICE) \
    else if (prm.rule == FIESTA_RULE_MC) FX_LAUNCH2(NX, FIESTA_RULE_MC)      \
    else FX_LAUNCH2(NX, FIESTA_RULE_VEGAS)                                   \
  }
  if (prm.dim <= 4) FX_LAUNCH(4)
  else if (prm.dim <= 8) FX_LAUNCH(8)
  else FX_LAUNCH(12)
#undef FX_LAUNCH
#undef FX_LAUNCH2
  return cudaGetLastError();
}

cudaError_t fx_launch_eval_real(const fx_eval_params &prm, cudaStream_t st) {
  const size_t smem = (size_t)prm.prog_ins_max * 16 + (size_t)prm.mem_doubles * 8;
  const uint64_t per_block = (uint64_t)FX_THREADS * FX_P_REAL;
  const unsigned grid = (unsigned)((prm.npts + per_block - 1) / per_block);
  if (grid == 0) return cudaSuccess;
  cudaError_t e;
#define FX_LAUNCH(NX)                                                        \
  {                                                                          \
    if ((e = set_smem(fx_eval_real<NX>, smem)) != cudaSuccess) return e;     \
    fx_eval_real<NX><<<grid, FX_THREADS, smem, st>>>(prm);                     \
  }
  if (prm.dim <= 4) FX_LAUNCH(4)
  else if (prm.dim <= 8) FX_LAUNCH(8)
  else FX_LAUNCH(12)
#undef FX_LAUNCH
  return cudaGetLastError();
}
