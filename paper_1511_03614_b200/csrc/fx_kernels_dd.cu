// fx_kernels_dd.cu -- the mixed-precision rescue of real sectors (R20).
//
// The paper's default "Mixed" mode re-evaluates the integrand with MPFR in the parts of the
// integration cube where doubles cancel (-SmallX and the other knobs PAPER.md:447,
// :472; "-mpfr: evaluate all integration points with the use of MPFR").  Here the
// higher precision is double-double (fx_dd.cuh, ~106 bits) and the decision is the SmallX one: a
// point with min_k x_k < small_x is "flagged".  The interpreter's evaluation kernels mask flagged
// points out of their sums and histograms (phase 1); fx_rescue_real below makes the same points again, evaluates
// the flagged ones by walking the SAME instruction program on (hi, lo) pairs, and adds them to the
// same per-block partial records before the chunk reduction runs (phase 2).  The points, their
// weights and the order of the sums stay those of phase 1; only f(x) is computed more precisely.
//
// The walk is a plain C++ switch over the ISA of fx_isa.h: flagged points are rare, so this kernel's
// speed is set by making the points again, not by the walk.
#define FX_WANT(is_cplx, nx, p) 0  // no interpreter fast path in this translation unit
#include "fx_device_common.cuh"
#include "fx_dd.cuh"

namespace {

struct fx_mem_dd {  // spill slots in shared memory: [slot][hi, lo][thread]
  double *base;     // &M[0][0][tid]
  __device__ __forceinline__ dd ld(int slot) const { return dd{base[(2 * slot) * FX_THREADS], base[(2 * slot + 1) * FX_THREADS]}; }
  __device__ __forceinline__ void st(int slot, dd v) const {
    base[(2 * slot) * FX_THREADS] = v.hi;
    base[(2 * slot + 1) * FX_THREADS] = v.lo;
  }
};

// Walk `prog` (shared memory) for one point; R[0..NX) hold x, R[FX_NXMAX..] the S temporaries.
// `sink(k, A)` receives output k.  Operation by operation the same program as fx_run.
template <class Sink>
__device__ __noinline__ void fx_run_dd(const fx_ins *prog, dd (&R)[FX_NR], const fx_mem_dd M, Sink &sink) {
  dd A[FX_L];
#pragma unroll
  for (int d = 0; d < FX_L; ++d) A[d] = dd_from(0.0);
  for (int pc = 0;; ++pc) {
    const fx_ins ins = prog[pc];
    const int op = ins.op, aux = ins.aux;
    const double imm = ins.imm;
    if (op < FX_LDC) {  // (level, register) families
      const int fam = op / FX_LR, d = (op % FX_LR) / FX_NR;
      const dd r = R[op % FX_NR];
      switch (fam * FX_LR) {
        case FX_MULC_R: A[d] = dd_mul_d(r, imm); break;
        case FX_MUL_R: A[d] = dd_mul(A[d], r); break;
        case FX_FMA_AR_C: A[d] = dd_add_d(dd_mul(A[d], r), imm); break;
        case FX_FMA_RC_A: A[d] = dd_add(dd_mul_d(r, imm), A[d]); break;
        case FX_FMA_UP: A[d] = dd_add(dd_mul(A[d + 1], r), A[d]); break;
        case FX_ADD_R: A[d] = dd_add(A[d], r); break;
        case FX_LD_R: A[d] = r; break;
        case FX_FMA_AR_M: A[d] = dd_add(dd_mul(A[d], r), M.ld(aux)); break;
      }
    } else if (op < FX_SUB_R) {  // level families
      const int d = (op - FX_LDC) % FX_L;
      switch (op - d) {
        case FX_LDC: A[d] = dd_from(imm); break;
        case FX_ADDC: A[d] = dd_add_d(A[d], imm); break;
        case FX_MULC: A[d] = dd_mul_d(A[d], imm); break;
        case FX_ADD_UP: A[d] = dd_add(A[d], A[d + 1]); break;
        case FX_MUL_UP: A[d] = dd_mul(A[d], A[d + 1]); break;
        case FX_LDM: A[d] = M.ld(aux); break;
        case FX_STM: M.st(aux, A[d]); break;
        case FX_ADDM: A[d] = dd_add(A[d], M.ld(aux)); break;
        case FX_MULM: A[d] = dd_mul(A[d], M.ld(aux)); break;
        case FX_FMA_MC_A: A[d] = dd_add(dd_mul_d(M.ld(aux), imm), A[d]); break;
        case FX_FMA_AM_C: A[d] = dd_add_d(dd_mul(A[d], M.ld(aux)), imm); break;
        case FX_FMA_UPC: A[d] = dd_add(dd_mul_d(A[d + 1], imm), A[d]); break;
      }
    } else if (op < FX_RSUBC) {  // level-0 register families
      const int r = (op - FX_SUB_R) % FX_NR;
      switch (op - r) {
        case FX_SUB_R: A[0] = dd_sub(A[0], R[r]); break;
        case FX_RSUB_R: A[0] = dd_sub(R[r], A[0]); break;
        case FX_DIV_R: A[0] = dd_div(A[0], R[r]); break;
        case FX_RDIV_R: A[0] = dd_div(R[r], A[0]); break;
        case FX_ST_S: R[FX_NXMAX + r] = A[0]; break;  // r = j < FX_NS
      }
    } else {
      switch (op) {
        case FX_RSUBC: A[0] = dd_add_d(dd_neg(A[0]), imm); break;
        case FX_DIVC: A[0] = dd_div(A[0], dd_from(imm)); break;
        case FX_RDIVC: A[0] = dd_div(dd_from(imm), A[0]); break;
        case FX_SUBM: A[0] = dd_sub(A[0], M.ld(aux)); break;
        case FX_RSUBM: A[0] = dd_sub(M.ld(aux), A[0]); break;
        case FX_DIVM: A[0] = dd_div(A[0], M.ld(aux)); break;
        case FX_RDIVM: A[0] = dd_div(M.ld(aux), A[0]); break;
        case FX_NEG: A[0] = dd_neg(A[0]); break;
        case FX_SQR: A[0] = dd_mul(A[0], A[0]); break;
        case FX_LOG: A[0] = dd_log(A[0]); break;
        case FX_EXP: A[0] = dd_exp(A[0]); break;
        case FX_SQRT: A[0] = dd_sqrt(A[0]); break;
        case FX_OUT: sink(aux, A[0]); break;
        case FX_END: return;
        default: __trap();
      }
    }
  }
}

template <typename K>
cudaError_t set_smem(K kernel, size_t bytes) {
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// ---- parity hook: the dd walk on the caller's points (fiesta_eval_points_dd) -----------------------

struct EvalSinkDD {
  double *out;  // &out[point][0][0]: [K][hi, lo]
  __device__ __forceinline__ void operator()(int k, dd a) {
    out[2 * k] = a.hi;
    out[2 * k + 1] = a.lo;
  }
};

__global__ void __launch_bounds__(FX_THREADS) fx_eval_dd(const __grid_constant__ fx_eval_params prm) {
  extern __shared__ __align__(16) unsigned char smem[];
  const fx_sector_dev sec = prm.sectors[prm.sector];
  fx_ins *sh_prog = reinterpret_cast<fx_ins *>(smem);
  double *sh_mem = reinterpret_cast<double *>(smem + (size_t)prm.prog_ins_max * 16);
  fx_copy_program(sh_prog, prm.arena + sec.main_off, sec.main_len);
  __syncthreads();
  const uint64_t j = (uint64_t)blockIdx.x * FX_THREADS + threadIdx.x;
  if (j >= prm.npts) return;
  dd R[FX_NR];
  for (int k = 0; k < FX_NR; ++k) R[k] = dd_from(k < prm.dim ? prm.x[j * prm.dim + k] : 0.5);
  EvalSinkDD sink{prm.out + j * sec.K * 2};
  fx_run_dd(sh_prog, R, fx_mem_dd{sh_mem + threadIdx.x}, sink);
}

// ---- phase 2: flagged points of a batch, added to its partial records ------------------------------

struct RescueSink {
  double *acc;  // &acc[0][tid], slot stride FX_THREADS
  double W;
  unsigned nonfinite;
  double h2;    // sum over the orders of g^2: what the Vegas histogram collects
  __device__ __forceinline__ void operator()(int k, dd a) {
    const double g = W * a.hi;  // the value rounded to double, as the sums are
    nonfinite += isfinite(g) ? 0u : 1u;
    acc[(2 * k) * FX_THREADS] += g;
    acc[(2 * k + 1) * FX_THREADS] = fma(g, g, acc[(2 * k + 1) * FX_THREADS]);
    h2 = fma(g, g, h2);
  }
};

constexpr int FX_RQ = 64;  // entries of a warp's queue of flagged point indices

struct fx_rescue_smem {
  uint32_t prog, mem, acc, delta, queue, wsum, rec, grid, hist, total;
};
__host__ __device__ inline fx_rescue_smem fx_rescue_layout(int prog_ins, int mem_doubles, int dim, int nbins, bool vegas) {
  fx_rescue_smem L;
  uint32_t o = 0;
  L.prog = o;
  o += (uint32_t)prog_ins * 16u;
  L.mem = o;
  o += (uint32_t)mem_doubles * 8u;
  L.acc = o;
  o += FX_ACC_SLOTS * FX_THREADS * 8u;
  L.delta = o;
  o += FX_NXMAX * 8u + FX_TF_BYTES;
  L.queue = o;
  o += (FX_THREADS / 32) * FX_RQ * 8u;
  L.wsum = o;
  o += FX_ACC_SLOTS * (FX_THREADS / 32) * 8u;
  L.rec = o;
  o += FX_ACC_SLOTS * 8u;
  L.grid = o;
  o += vegas ? (uint32_t)dim * (nbins + 1) * 8u : 0u;
  L.hist = o;
  o += vegas ? (FX_THREADS / 32) * (uint32_t)dim * nbins * 8u : 0u;  // one histogram per warp, as in phase 1
  L.total = o;
  return L;
}

template <int NX, int RULE>
__global__ void __launch_bounds__(FX_THREADS) fx_rescue_real(const __grid_constant__ fx_integrate_params prm) {
  constexpr bool vegas = RULE == FIESTA_RULE_VEGAS;
  extern __shared__ __align__(16) unsigned char smem[];
  const fx_block_id id = fx_block_coords(prm);
  const fx_sector_dev sec = prm.sectors[prm.sel[id.sel_idx]];
  const int dim = prm.dim;
  const fx_rescue_smem L = fx_rescue_layout(prm.prog_ins_max, prm.mem_doubles, dim, prm.nbins, vegas);
  fx_ins *sh_prog = reinterpret_cast<fx_ins *>(smem + L.prog);
  double *sh_mem = reinterpret_cast<double *>(smem + L.mem);
  double *sh_acc = reinterpret_cast<double *>(smem + L.acc);
  uint64_t *sh_delta = reinterpret_cast<uint64_t *>(smem + L.delta);
  uint64_t *sh_queue = reinterpret_cast<uint64_t *>(smem + L.queue) + (threadIdx.x >> 5) * FX_RQ;
  double *sh_wsum = reinterpret_cast<double *>(smem + L.wsum);
  double *sh_rec = reinterpret_cast<double *>(smem + L.rec);
  double *sh_grid = reinterpret_cast<double *>(smem + L.grid);
  double *sh_hist = reinterpret_cast<double *>(smem + L.hist);

  fx_copy_program(sh_prog, prm.arena + sec.main_off, sec.main_len);
  fx_block_setup(prm, dim, (uint32_t)sec.sector_id, id.r, id.sel_idx, sh_delta, sh_grid, sh_hist);
  const int nslots = 2 * sec.K;
  for (int s = 0; s < nslots; ++s) sh_acc[s * FX_THREADS + threadIdx.x] = 0.0;
  __syncthreads();

  const uint64_t c0 = (uint64_t)id.chunk * prm.chunk;
  const uint64_t c1 = min(c0 + prm.chunk, prm.n_per_shift);
  const unsigned lane = threadIdx.x & 31u;
  const fx_mem_dd M{sh_mem + threadIdx.x};
  unsigned nonfinite = 0, queued = 0;  // queued: warp-uniform

  // one queued point per lane: made again from its index, evaluated in double-double
  auto drain = [&](unsigned n) {
    uint32_t bins[(NX + 3) / 4][1];
    double h2[1] = {0.0};
#pragma unroll
    for (int q = 0; q < (NX + 3) / 4; ++q) bins[q][0] = 0;
    if (lane < n) {
      double x[NX][1], xbar[NX][1], W[1];
      unsigned valid;
      fx_make_points<RULE, NX, 1>(prm, dim, (uint32_t)sec.sector_id, sh_delta, sh_grid, sh_queue[lane], c1, x, xbar, W, valid, bins);
      dd R[FX_NR];
#pragma unroll
      for (int k = 0; k < FX_NR; ++k) R[k] = dd_from(0.5);
#pragma unroll
      for (int k = 0; k < NX; ++k) R[k] = dd_from(x[k][0]);
      RescueSink sink{sh_acc + threadIdx.x, W[0], 0u, 0.0};
      fx_run_dd(sh_prog, R, M, sink);
      nonfinite += sink.nonfinite;
      h2[0] = sink.h2;
    }
    __syncwarp();
    // Vegas: the rescued points' g^2 go to the warp's histogram by the same warp-collective, fixed-order update as in phase 1
    if constexpr (vegas) fx_hist_points<NX, 1>(sh_hist, dim, prm.nbins, lane < n ? 1u : 0u, bins, h2);
  };

  // the same trip count for every thread: the queue is a warp-collective structure
  for (uint64_t it = c0; it < c1; it += FX_THREADS) {
    const uint64_t j = it + threadIdx.x;
    double x[NX][1], xbar[NX][1], W[1];
    uint32_t bins[(NX + 3) / 4][1];
    unsigned valid;
    fx_make_points<RULE, NX, 1>(prm, dim, (uint32_t)sec.sector_id, sh_delta, sh_grid, j, c1, x, xbar, W, valid, bins);
    const bool flag = j < c1 && fx_flag_mask<NX, 1>(x, dim, prm.small_x);  // (fx_make_points cleared the flagged bit of `valid`)
    const unsigned m = __ballot_sync(0xffffffffu, flag);
    if (flag) sh_queue[queued + __popc(m & ((1u << lane) - 1u))] = j;
    queued += __popc(m);
    __syncwarp();
    if (queued >= 32u) {
      drain(32u);
      const uint64_t keep = lane + 32u < queued ? sh_queue[lane + 32u] : 0ull;
      __syncwarp();
      sh_queue[lane] = keep;
      queued -= 32u;
      __syncwarp();
    }
  }
  drain(queued);
  __syncthreads();
  fx_block_reduce(sh_acc, sh_wsum, nslots, sh_rec);
  __syncthreads();
  if (threadIdx.x < FX_ACC_SLOTS) fx_partial_record(prm, id.sel_idx, id.r, id.chunk)[threadIdx.x] += sh_rec[threadIdx.x];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) nonfinite += __shfl_down_sync(0xffffffffu, nonfinite, off);
  if (lane == 0 && nonfinite) atomicAdd(prm.nonfinite + id.sel_idx, (unsigned long long)nonfinite);
  if constexpr (vegas) {  // the warps' histograms in warp order, added to the record phase 1 wrote for this block
    const int cells = dim * prm.nbins;
    double *h = prm.hist_part + ((size_t)(id.sel_idx - prm.batch_base) * prm.nchunks + id.chunk) * cells;
    for (int i = threadIdx.x; i < cells; i += blockDim.x) {
      double v = 0.0;
      for (int w = 0; w < FX_THREADS / 32; ++w) v += sh_hist[w * cells + i];
      h[i] += v;
    }
  }
}

}  // namespace

size_t fx_eval_dd_smem_bytes(const fx_eval_params &prm) { return (size_t)prm.prog_ins_max * 16 + (size_t)prm.mem_doubles * 8; }

// prm.mem_doubles = 2 * n_mem_main * FX_THREADS; out[npts][K][hi, lo]
cudaError_t fx_launch_eval_dd(const fx_eval_params &prm, cudaStream_t st) {
  const size_t smem = fx_eval_dd_smem_bytes(prm);
  const unsigned grid = (unsigned)((prm.npts + FX_THREADS - 1) / FX_THREADS);
  if (grid == 0) return cudaSuccess;
  cudaError_t e;
  if ((e = set_smem(fx_eval_dd, smem)) != cudaSuccess) return e;
  fx_eval_dd<<<grid, FX_THREADS, smem, st>>>(prm);
  return cudaGetLastError();
}

size_t fx_rescue_smem_bytes(const fx_integrate_params &prm) {
  return fx_rescue_layout(prm.prog_ins_max, prm.mem_doubles, prm.dim, prm.nbins, prm.rule == FIESTA_RULE_VEGAS).total;
}

// prm.mem_doubles = 2 * max n_mem_main * FX_THREADS; launch_map / sel_base as for the evaluation kernels
cudaError_t fx_launch_rescue_real(const fx_integrate_params &prm, int nsectors, cudaStream_t st) {
  const size_t smem = fx_rescue_smem_bytes(prm);
  const unsigned grid = (unsigned)((size_t)nsectors * prm.n_shifts * prm.nchunks);
  cudaError_t e;
#define FX_LAUNCH2(NX, RULE)                                                      \
  {                                                                               \
    if ((e = set_smem(fx_rescue_real<NX, RULE>, smem)) != cudaSuccess) return e;  \
    fx_rescue_real<NX, RULE><<<grid, FX_THREADS, smem, st>>>(prm);                \
  }
#define FX_LAUNCH(NX)                                                        \
  {                                                                          \
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
