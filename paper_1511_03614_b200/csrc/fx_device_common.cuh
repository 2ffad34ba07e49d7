// fx_device_common.cuh -- pieces shared by the real and the complex evaluation kernels:
// shared-memory layout, on-device point generation (no HBM traffic for
// points, contrast PAPER.md:118 where points are uploaded per batch), accumulation (A6) and the
// block-level half of the deterministic two-level reduction (A7).
#ifndef FX_DEVICE_COMMON_CUH
#define FX_DEVICE_COMMON_CUH

#include "../../include/fiesta_b200.h"
#include "fx_interp.cuh"
#include "fx_kernels.h"

struct fx_smem_layout {
  uint32_t prog, mem, acc, delta, tf, grid, hist, wsum, total;
};

__host__ __device__ inline fx_smem_layout fx_layout(int prog_ins, int mem_doubles, int dim, int nbins, bool vegas,
                                                    int acc_slots = FX_ACC_SLOTS) {
  fx_smem_layout L;
  uint32_t o = 0;
  L.prog = o;
  o += (uint32_t)prog_ins * 16u;
  L.mem = o;
  o += (uint32_t)mem_doubles * 8u;
  L.acc = o;
  o += (uint32_t)acc_slots * FX_THREADS * 8u;
  L.delta = o;
  o += FX_NXMAX * 8u;
  L.tf = o;
  o += FX_TF_BYTES;  // fx_transform (80 bytes) for the per-coordinate helper, then the lattice steps G_k
  L.grid = o;
  o += vegas ? (uint32_t)dim * (nbins + 1) * 8u : 0u;
  L.hist = o;
  o += vegas ? (FX_THREADS / 32) * (uint32_t)dim * nbins * 8u : 0u;  // one histogram per warp
  L.wsum = o;
  o += FX_ACC_SLOTS * (FX_THREADS / 32) * 8u;
  L.total = o;
  return L;
}

__device__ __forceinline__ void fx_copy_program(fx_ins *dst, const fx_ins *src, int n) {
  const uint4 *s = reinterpret_cast<const uint4 *>(src);
  uint4 *d = reinterpret_cast<uint4 *>(dst);
  for (int i = threadIdx.x; i < n; i += blockDim.x) d[i] = s[i];
}

// the lattice steps G_k live in shared memory behind the transform (fx_layout / fxj_layout): loop
// invariants the evaluation kernels need not hold in registers across the program walk
__device__ __forceinline__ uint64_t *fx_lattice_steps(uint64_t *sh_delta) {
  return sh_delta + FX_NXMAX + 80 / 8;
}
__device__ __forceinline__ const uint64_t *fx_lattice_steps(const uint64_t *sh_delta) {
  return sh_delta + FX_NXMAX + 80 / 8;
}
// ... and behind them the block's point range [c0, c1) and its pass count (native kernels): read back
// through volatile loads in every pass, so that they are not held in registers across the program body
__device__ __forceinline__ uint64_t *fx_block_range(uint64_t *sh_delta) { return sh_delta + FX_NXMAX + 80 / 8 + FX_NXMAX; }
__device__ __forceinline__ uint64_t fx_lds_volatile(const uint64_t *p) {
  uint64_t v;
  asm volatile("ld.volatile.shared.u64 %0, [%1];" : "=l"(v) : "r"((uint32_t)__cvta_generic_to_shared(p)));
  return v;
}
__device__ __forceinline__ unsigned fx_tid_volatile() {
  unsigned t;
  asm volatile("mov.u32 %0, %%tid.x;" : "=r"(t));
  return t;
}

// Out-of-line helpers: the evaluation kernels call them once per coordinate.  Keeping one copy of
// each (instead of NX*P inlined copies) keeps the per-batch code outside the program walk small, so
// it does not evict the walk's handlers from the 32 KB instruction cache (profiles/r01_*.md).
struct fx_coord {
  double x, xbar, w;
};
struct fx_tpair {
  uint64_t e, o;
};

// all P points of one coordinate per call: P independent dependency chains (int->double, Horner,
// powers) overlap
template <int P>
struct fx_coordP {
  double x[P], xbar[P], s[P];  // s = u(1-u): the point's weight is cw^dim (prod_k s_k)^r (korobov_weight)
};
template <int P>
struct fx_tP {
  uint64_t t[P];
};
template <int P>
__device__ __forceinline__ fx_coordP<P> fx_lattice_coord_body(fx_tP<P> t, const fx_transform *tf /* shared memory */) {
  fx_coordP<P> c;
  if (tf->r == 3) {  // the default weight: no switch
#pragma unroll
    for (int p = 0; p < P; ++p) korobov_xs_r<3>(*tf, t.t[p], c.x[p], c.xbar[p], c.s[p]);
  } else {
#pragma unroll
    for (int p = 0; p < P; ++p) korobov_xs(*tf, t.t[p], c.x[p], c.xbar[p], c.s[p]);
  }
  return c;
}

template <int P>
static __device__ __noinline__ fx_coordP<P> fx_lattice_coord(fx_tP<P> t, const fx_transform *tf) {
  return fx_lattice_coord_body<P>(t, tf);
}

__device__ __forceinline__ fx_tpair fx_philox_pair_body(const uint32_t *rk, uint32_t sector_id, uint32_t tag, uint32_t it,
                                                        uint64_t j, uint32_t kb) {
  fx_tpair r;
  philox_t_pair_rk(rk, sector_id, tag, it, j, kb, r.e, r.o);
  return r;
}
static __device__ __noinline__ fx_tpair fx_philox_pair(const uint32_t *rk, uint32_t sector_id, uint32_t tag, uint32_t it,
                                                       uint64_t j, uint32_t kb) {
  return fx_philox_pair_body(rk, sector_id, tag, it, j, kb);
}

struct fx_vcoord {
  double x, w;
  int bin;
};
__device__ __forceinline__ fx_vcoord fx_vegas_coord_body(uint64_t t, int nbins, const double *edges) {
  fx_vcoord c;
  vegas_map_coord(t, nbins, edges, c.x, c.w, c.bin);
  return c;
}
static __device__ __noinline__ fx_vcoord fx_vegas_coord(uint64_t t, int nbins, const double *edges) {
  return fx_vegas_coord_body(t, nbins, edges);
}

// Mixed precision (R20): the points with some coordinate below small_x, as a bit mask.
// The evaluation kernels leave them out of their sums; fx_rescue_real (fx_kernels_dd.cu) evaluates
// exactly these in double-double.  One function, so that the two phases cannot disagree on a point.
template <int NX, int P>
__device__ __forceinline__ unsigned fx_flag_mask(const double (&x)[NX][P], int dim, double small_x) {
  unsigned m = 0;
  FX_PLOOP {
    bool f = false;
#pragma unroll
    for (int k = 0; k < NX; ++k) f = f || (k < dim && x[k][p] < small_x);
    m |= f ? 1u << p : 0u;
  }
  return m;
}

// Points j0..j0+P-1 of (sector, shift r / iteration) -> real x, xbar = 1-x, weight W, Vegas bins.
// RULE is a compile-time constant: each rule has its own kernel instantiation.  INL: the per-coordinate
// helpers inline instead of out of line -- an out-of-line call makes the kernel save the values it
// has live across the call to local memory, which the kernels with many such values (Vegas with 4
// points per thread; all complex kernels) avoid this way at the price of longer code.
template <int RULE, int NX, int P, bool INL = false>
__device__ __forceinline__ void fx_make_points(const fx_integrate_params &prm, int dim, uint32_t sector_id,
                                               const uint64_t *sh_delta, const double *sh_grid, uint64_t j0,
                                               uint64_t jend, double (&x)[NX][P], double (&xbar)[NX][P],
                                               double (&W)[P], unsigned &valid, uint32_t (&bins)[(NX + 3) / 4][P]) {
  valid = 0;
  FX_PLOOP {
    W[p] = 1.0;
    if (j0 + p < jend) valid |= 1u << p;
  }
#pragma unroll
  for (int q = 0; q < (NX + 3) / 4; ++q) FX_PLOOP { bins[q][p] = 0; }
  if constexpr (RULE == FIESTA_RULE_LATTICE) {
    const fx_transform *tf = reinterpret_cast<const fx_transform *>(sh_delta + FX_NXMAX);  // fx_layout: tf follows delta
#pragma unroll
    for (int k = 0; k < NX; ++k) {
      if (k < dim) {
        // t_j = ((j g) mod 2^m) << (64-m) + Delta = j * (g << (64-m)) + Delta  (mod 2^64)
        const uint64_t G = fx_lattice_steps(sh_delta)[k];
        fx_tP<P> tt;
        FX_PLOOP { tt.t[p] = (j0 + p) * G + sh_delta[k]; }
        const fx_coordP<P> c = INL ? fx_lattice_coord_body<P>(tt, tf) : fx_lattice_coord<P>(tt, tf);
        FX_PLOOP {
          x[k][p] = c.x[p];
          xbar[k][p] = c.xbar[p];
          W[p] *= c.s[p];
        }
      } else {
        FX_PLOOP {
          x[k][p] = 0.5;
          xbar[k][p] = 0.5;
        }
      }
    }
    FX_PLOOP { W[p] = korobov_weight(*tf, W[p]); }  // W held prod_k u_k(1-u_k) until here
  } else {
#pragma unroll
    for (int kb = 0; kb < (NX + 1) / 2; ++kb) {
      FX_PLOOP {
        fx_tpair tp{0ull, 0ull};
        if (2 * kb < dim)
          tp = INL ? fx_philox_pair_body(prm.philox_rk, sector_id, FX_TAG_MC, (uint32_t)prm.iteration, j0 + p, kb)
                   : fx_philox_pair(prm.philox_rk, sector_id, FX_TAG_MC, (uint32_t)prm.iteration, j0 + p, kb);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int k = 2 * kb + h;
          if (k < NX) {
            const uint64_t t = h ? tp.o : tp.e;
            if (k < dim) {
              if constexpr (RULE == FIESTA_RULE_VEGAS) {
                const double *edges = sh_grid + k * (prm.nbins + 1);
                const fx_vcoord c = INL ? fx_vegas_coord_body(t, prm.nbins, edges) : fx_vegas_coord(t, prm.nbins, edges);
                x[k][p] = c.x;
                xbar[k][p] = 1.0 - c.x;
                W[p] *= c.w;
                bins[k / 4][p] |= (uint32_t)c.bin << (8 * (k % 4));
              } else {
                const double u = unit_from_t(t);
                x[k][p] = u;
                xbar[k][p] = 1.0 - u;
              }
            } else {
              x[k][p] = 0.5;
              xbar[k][p] = 0.5;
            }
          }
        }
      }
    }
  }
#ifndef FX_NO_MIXED_MASK  // the native templates and the complex kernels never run with the mixed mode on
  if (prm.small_x > 0.0) valid &= ~fx_flag_mask<NX, P>(x, dim, prm.small_x);  // block-uniform branch
#endif
}

// block start: shift Delta_{r,k} from the Philox shift stream (R3), Vegas grid and histogram
__device__ __forceinline__ void fx_block_setup(const fx_integrate_params &prm, int dim, uint32_t sector_id, int r,
                                               int sel_idx, uint64_t *sh_delta, double *sh_grid, double *sh_hist) {
  if (threadIdx.x < (FX_NXMAX + 1) / 2) {
    uint64_t te = 0, to = 0;
    if (prm.rule == FIESTA_RULE_LATTICE)
      philox_t_pair_rk(prm.philox_rk, sector_id, FX_TAG_SHIFT, (uint32_t)(prm.shift_base + r), 0ull, threadIdx.x, te, to);
    sh_delta[2 * threadIdx.x] = te;
    sh_delta[2 * threadIdx.x + 1] = to;
  }
  if (threadIdx.x >= 64 && threadIdx.x < 64 + FX_NXMAX)  // t_j = j * G_k + Delta_k (mod 2^64), G_k = g_k << (64-m)
    fx_lattice_steps(sh_delta)[threadIdx.x - 64] =
        (prm.rule == FIESTA_RULE_LATTICE && prm.log2_n) ? (prm.genvec[threadIdx.x - 64] << (64 - prm.log2_n)) : 0ull;
  if (threadIdx.x == 32) {  // fx_layout puts the transform right after the shifts
    fx_transform *tf = reinterpret_cast<fx_transform *>(sh_delta + FX_NXMAX);
    tf->r = prm.tf.r;
    tf->cw = prm.tf.cw;
    for (int i = 0; i < 7; ++i) tf->coef[i] = prm.tf.coef[i];
    double cwd = 1.0;
    for (int k = 0; k < dim; ++k) cwd *= prm.tf.cw;
    tf->cwd = cwd;
  }
  if (prm.rule == FIESTA_RULE_VEGAS) {
    const double *g = prm.grid + (size_t)sel_idx * dim * (prm.nbins + 1);
    for (int i = threadIdx.x; i < dim * (prm.nbins + 1); i += blockDim.x) sh_grid[i] = g[i];
    for (int i = threadIdx.x; i < (FX_THREADS / 32) * dim * prm.nbins; i += blockDim.x) sh_hist[i] = 0.0;
  }
}

// Vegas histogram (R8): h[k][bin_k] += v for one point per lane and every
// dimension k, into the WARP's own histogram in shared memory.  Without atomics and in a fixed order,
// so that the histogram -- like the sums -- is bit-reproducible:
//   - in step k of a point, lane l handles dimension (k + l) mod n: the lanes l < n work on different
//     dimensions, and only the lanes l, l + n, l + 2n, ... (same dimension) can meet in a cell, which
//     happens when their points fall into the same bin;
//   - so the lanes take ceil(32 / n) turns per step -- turn t: the lanes t n <= l < (t + 1) n do a plain
//     read-modify-write of their cell -- with a warp barrier after every turn.  Two lanes never touch
//     one cell in the same turn, and a cell receives its contributions in step order, then lane order.
// (An earlier form found out by shuffles which lanes actually meet -- with 12 dimensions and 50 bins a
// second turn was needed in 5 % of the steps -- and took turns by that rank: the same order of additions,
// but two shuffles, a vote and a loop per step; the fixed turns are 4-7 % faster at 4-8 dimensions and
// took the 12-dimensional C5 from 1.50 to 1.9e10 evaluations/s.)
template <int NX, int P>
__device__ __forceinline__ void fx_hist_points(double *sh_hist, int dim, int nbins, unsigned valid,
                                               const uint32_t (&bins)[(NX + 3) / 4][P], const double (&h2)[P]) {
  const unsigned lane = threadIdx.x & 31u;
  double *wh = sh_hist + (size_t)(threadIdx.x >> 5) * dim * nbins;
  const unsigned d0 = lane % (unsigned)dim;
  const unsigned turn = lane / (unsigned)dim;
  FX_PLOOP {  // point by point: the order both tiers use
    const bool ok = (valid >> p) & 1u;
    unsigned d = d0;
#pragma unroll 1
    for (int k = 0; k < dim; ++k) {
      uint32_t w = bins[0][p];
      if constexpr ((NX + 3) / 4 > 1) w = d >= 4 ? bins[1][p] : w;
      if constexpr ((NX + 3) / 4 > 2) w = d >= 8 ? bins[2][p] : w;
      const unsigned cell = d * (unsigned)nbins + ((w >> (8 * (d & 3u))) & 0xffu);
      if (dim >= 11) {  // three turns, unrolled
#pragma unroll
        for (unsigned t = 0; t < 3; ++t) {
          if (ok && turn == t) wh[cell] += h2[p];
          __syncwarp();
        }
      } else {
#pragma unroll 1
        for (unsigned t = 0; t * (unsigned)dim < 32u; ++t) {
          if (ok && turn == t) wh[cell] += h2[p];
          __syncwarp();
        }
      }
      d = d + 1u == (unsigned)dim ? 0u : d + 1u;
    }
  }
}

// block end: acc[slot][tid] -> one partial per slot, fixed order (lanes by shuffle tree, then warps in order)
__device__ __forceinline__ void fx_block_reduce(const double *sh_acc, double *sh_wsum, int nslots, double *out) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int s = 0; s < nslots; ++s) {
    double v = sh_acc[s * FX_THREADS + threadIdx.x];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    if (lane == 0) sh_wsum[s * (FX_THREADS / 32) + warp] = v;
  }
  __syncthreads();
  if (threadIdx.x < FX_ACC_SLOTS) {  // every slot of the record is written: the buffer is never cleared
    double t = 0.0;
    if (threadIdx.x < nslots)
      for (int w = 0; w < FX_THREADS / 32; ++w) t += sh_wsum[threadIdx.x * (FX_THREADS / 32) + w];
    out[threadIdx.x] = t;
  }
}

// block end: non-finite count (an integer: atomics keep it exact), and the block's histogram = the
// warps' histograms added in warp order, written to this block's own record (fx_launch_reduce_hist
// adds the records in block order)
__device__ __forceinline__ void fx_block_finish(const fx_integrate_params &prm, int dim, int sel_idx, int chunk,
                                                unsigned nonfinite, const double *sh_hist) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) nonfinite += __shfl_down_sync(0xffffffffu, nonfinite, off);
  if ((threadIdx.x & 31) == 0 && nonfinite) atomicAdd(prm.nonfinite + sel_idx, (unsigned long long)nonfinite);
  if (prm.rule == FIESTA_RULE_VEGAS) {
    const int cells = dim * prm.nbins;
    double *h = prm.hist_part + ((size_t)(sel_idx - prm.batch_base) * prm.nchunks + chunk) * cells;
    __syncthreads();
    for (int i = threadIdx.x; i < cells; i += blockDim.x) {
      double v = 0.0;
      for (int w = 0; w < FX_THREADS / 32; ++w) v += sh_hist[w * cells + i];
      h[i] = v;
    }
  }
}

// Which (sector, shift, chunk) this block works on.  The block index is read through a volatile asm,
// so a kernel that asks again after its point loop gets a recomputation there instead of three
// registers held (or spilled to local memory) across the whole program walk.
struct fx_block_id {
  int chunk, r, sel_idx;
};
__device__ __forceinline__ fx_block_id fx_block_coords(const fx_integrate_params &prm) {
  unsigned b;
  asm volatile("mov.u32 %0, %%ctaid.x;" : "=r"(b));
  fx_block_id id;
  id.chunk = (int)(b % (unsigned)prm.nchunks);
  id.r = (int)((b / (unsigned)prm.nchunks) % (unsigned)prm.n_shifts);
  id.sel_idx = fx_sel_index(prm, (int)(b / ((unsigned)prm.nchunks * (unsigned)prm.n_shifts)));
  return id;
}

// where this block's partial record goes
__device__ __forceinline__ double *fx_partial_record(const fx_integrate_params &prm, int sel_idx, int r, int chunk) {
  return prm.partials + (((size_t)(sel_idx - prm.batch_base) * prm.n_shifts + r) * prm.nchunks + chunk) * FX_ACC_SLOTS;
}

#endif
