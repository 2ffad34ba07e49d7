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

__host__ __device__ inline fx_smem_layout fx_layout(int prog_ins, int mem_doubles, int dim, int nbins, bool vegas) {
  fx_smem_layout L;
  uint32_t o = 0;
  L.prog = o;
  o += (uint32_t)prog_ins * 16u;
  L.mem = o;
  o += (uint32_t)mem_doubles * 8u;
  L.acc = o;
  o += FX_ACC_SLOTS * FX_THREADS * 8u;
  L.delta = o;
  o += FX_NXMAX * 8u;
  L.tf = o;
  o += 80u;  // fx_transform (80 bytes), kept in shared memory for the per-coordinate helper
  L.grid = o;
  o += vegas ? (uint32_t)dim * (nbins + 1) * 8u : 0u;
  L.hist = o;
  o += vegas ? (uint32_t)dim * nbins * 8u : 0u;
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
static __device__ __noinline__ fx_coordP<P> fx_lattice_coord(fx_tP<P> t, const fx_transform *tf /* shared memory */) {
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

static __device__ __noinline__ fx_tpair fx_philox_pair(uint64_t seed, uint32_t sector_id, uint32_t tag, uint32_t it, uint64_t j,
                                                uint32_t kb) {
  fx_tpair r;
  philox_t_pair(seed, sector_id, tag, it, j, kb, r.e, r.o);
  return r;
}

struct fx_vcoord {
  double x, w;
  int bin;
};
static __device__ __noinline__ fx_vcoord fx_vegas_coord(uint64_t t, int nbins, const double *edges) {
  fx_vcoord c;
  vegas_map_coord(t, nbins, edges, c.x, c.w, c.bin);
  return c;
}

// Points j0..j0+P-1 of (sector, shift r / iteration) -> real x, xbar = 1-x, weight W, Vegas bins.
// RULE is a compile-time constant: each rule has its own kernel instantiation.
template <int RULE, int NX, int P>
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
        const uint64_t G = prm.log2_n ? (prm.genvec[k] << (64 - prm.log2_n)) : 0ull;
        fx_tP<P> tt;
        FX_PLOOP { tt.t[p] = (j0 + p) * G + sh_delta[k]; }
        const fx_coordP<P> c = fx_lattice_coord<P>(tt, tf);
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
        if (2 * kb < dim) tp = fx_philox_pair(prm.seed, sector_id, FX_TAG_MC, (uint32_t)prm.iteration, j0 + p, kb);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int k = 2 * kb + h;
          if (k < NX) {
            const uint64_t t = h ? tp.o : tp.e;
            if (k < dim) {
              if constexpr (RULE == FIESTA_RULE_VEGAS) {
                const fx_vcoord c = fx_vegas_coord(t, prm.nbins, sh_grid + k * (prm.nbins + 1));
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
}

// block start: shift Delta_{r,k} from the Philox shift stream (R3), Vegas grid and histogram
__device__ __forceinline__ void fx_block_setup(const fx_integrate_params &prm, int dim, uint32_t sector_id, int r,
                                               int sel_idx, uint64_t *sh_delta, double *sh_grid, double *sh_hist) {
  if (threadIdx.x < (FX_NXMAX + 1) / 2) {
    uint64_t te = 0, to = 0;
    if (prm.rule == FIESTA_RULE_LATTICE)
      philox_t_pair(prm.seed, sector_id, FX_TAG_SHIFT, (uint32_t)r, 0ull, threadIdx.x, te, to);
    sh_delta[2 * threadIdx.x] = te;
    sh_delta[2 * threadIdx.x + 1] = to;
  }
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
    for (int i = threadIdx.x; i < dim * prm.nbins; i += blockDim.x) sh_hist[i] = 0.0;
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
  if (threadIdx.x < nslots) {
    double t = 0.0;
    for (int w = 0; w < FX_THREADS / 32; ++w) t += sh_wsum[threadIdx.x * (FX_THREADS / 32) + w];
    out[threadIdx.x] = t;
  }
}

__device__ __forceinline__ void fx_block_finish(const fx_integrate_params &prm, int dim, int sel_idx, unsigned nonfinite,
                                                const double *sh_hist) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) nonfinite += __shfl_down_sync(0xffffffffu, nonfinite, off);
  if ((threadIdx.x & 31) == 0 && nonfinite) atomicAdd(prm.nonfinite + sel_idx, (unsigned long long)nonfinite);
  if (prm.rule == FIESTA_RULE_VEGAS) {
    double *h = prm.hist + (size_t)sel_idx * dim * prm.nbins;
    for (int i = threadIdx.x; i < dim * prm.nbins; i += blockDim.x) {
      double v = sh_hist[i];
      if (v != 0.0) atomicAdd(h + i, v);
    }
  }
}

#endif
