// fx_kernels.h -- launch interface between the C ABI (host) and the sm_100a kernels.
#ifndef FX_KERNELS_H
#define FX_KERNELS_H

#include <cuda_runtime.h>
#include <stdint.h>

#include "fx_isa.h"

#define FX_THREADS 128   // threads per block of the evaluation kernels
#define FX_P_REAL 4      // points per thread, real programs
#define FX_P_CPLX 1      // points per thread, complex programs
#define FX_TF_BYTES (80u + FX_NXMAX * 8u + 32u)  // shared memory: fx_transform, the lattice steps G_k, the block's point range
#define FX_ACC_SLOTS 32  // per-(sector,shift,chunk) partial record: [K<=8][C<=2][S1,S2]

struct fx_sector_dev {       // one compiled sector in the device arena
  uint32_t main_off;         // instruction index of the main program in the arena
  uint32_t main_len;         // instructions incl. FX_END and one pad
  uint32_t deform_off;
  uint32_t deform_len;       // 0: no deformation
  int32_t K;
  int32_t is_complex;
  int32_t sector_id;
  int32_t n_mem_main;        // spill slots (scalars of the program's type)
  int32_t n_mem_deform;      // spill slots (doubles) incl. the gradient/Hessian outputs
  int32_t n_mem_testf;       // spill slots (complex) of the F(z) program
  double lambda;
  uint32_t testf_off;        // F(z) program of a deformed sector (fiesta_test_f); 0 length: none
  uint32_t testf_len;
};

struct fx_transform_host {
  int r;
  double cw;
  double coef[7];
};

struct fx_integrate_params {
  const fx_ins *arena;
  const fx_sector_dev *sectors;
  const int32_t *sel;        // device: selected sector indices [nsel]
  int32_t nsel;
  int32_t dim;
  int32_t rule;              // FIESTA_RULE_*
  int32_t n_shifts;          // R (lattice) or 1
  uint64_t n_per_shift;      // N_L (lattice) or points per iteration (MC / Vegas)
  int32_t log2_n;            // m (lattice)
  uint64_t chunk;            // points per block
  int32_t nchunks;
  int32_t iteration;         // Vegas iteration / MC stream index
  uint64_t genvec[FX_NXMAX];
  fx_transform_host tf;
  uint64_t seed;
  uint32_t philox_rk[20];    // Philox round keys of `seed`: (lo32 + r W0, hi32 + r W1), r = 0..9 (R3)
  int32_t nbins;
  const double *grid;        // Vegas: [nsel][dim][nbins+1]
  double *hist_part;         // Vegas: per-block histograms of this batch [batch sector][nchunks][dim][nbins]
  double *partials;          // partial records of this batch [batch sector][R][nchunks][FX_ACC_SLOTS]
  unsigned long long *nonfinite;  // [nsel]
  int32_t mem_doubles;       // shared-memory spill doubles per block (all threads)
  int32_t prog_ins_max;      // instructions reserved in shared memory (main + deform)
  // A launch covers some sectors of one batch of the call (a batch = consecutive positions
  // batch_base .. of the selection; its partial records are what `partials` / `hist_part` point to).
  // Block q / (nchunks * n_shifts) = launch-local sector number j; its position in the selection is
  // launch_map[j] (interpreter launches over the sectors of the batch that have no native kernel yet)
  // or sel_base + j when launch_map is NULL (one native kernel per sector).
  const int32_t *launch_map;
  int32_t sel_base;
  int32_t batch_base;        // position in the selection of the batch's first sector
  // fiesta_test_f (PAPER.md:474 -testF): one record per block, [bad points, max Im F(z), min |F(z)|^2, points]
  double *testf_out;
  double lambda_override;    // >= 0: use instead of the sector's lambda (the lambda scan); < 0: the sector's own
  // mixed precision (fiesta_set_mixed; R20): points with some x_k < small_x are left out of the sums
  // here and evaluated in double-double by fx_launch_rescue_real.  0: off.
  double small_x;
  int32_t shift_base;        // lattice: the block's shift r stands for shift shift_base + r of the rule (a rank's share of the shifts)
  int32_t acc_slots_real;    // accumulator slots per thread the real interpreter kernel reserves in shared memory: 2 K of the
                             // call's real sectors + FX_P_REAL + 1 (0: FX_ACC_SLOTS).  Less shared memory per block = one more resident block.
  int32_t acc_slots_cplx;    // the same for the complex interpreter kernel: 4 K of the call's complex sectors (0: FX_ACC_SLOTS)
};

// position in the selection of the sector a block works on
static inline __host__ __device__ int fx_sel_index(const fx_integrate_params &prm, int launch_sector) {
  return prm.launch_map ? prm.launch_map[launch_sector] : prm.sel_base + launch_sector;
}

struct fx_eval_params {
  const fx_ins *arena;
  const fx_sector_dev *sectors;
  int32_t sector;
  int32_t dim;
  uint64_t npts;
  const double *x;           // device [npts][dim]
  double *out;               // device [npts][K][2]
  int32_t mem_doubles;
  int32_t prog_ins_max;
};

size_t fx_integrate_smem_bytes(const fx_integrate_params &p);
size_t fx_integrate_cplx_smem_bytes(const fx_integrate_params &p);  // fx_integrate_cplx: accumulator area sized by acc_slots_cplx

// Shared-memory layout of the native kernels (fx_jit_template*.cu): accumulators (sum g, sum g^2 per
// output component: FXJ_ACC_SLOTS slots, one column per thread), the lattice shifts, the transform
// parameters (fx_block_setup puts them right after the shifts), Vegas grid and per-warp histograms,
// the block reduction's per-warp sums.  No program and no spill slots: both are registers.
#define FXJ_ACC_SLOTS 32
#define FXJ_P 2  // points per thread and pass of the native program body (two passes per batch of FX_P_REAL)
#ifndef FXJ_P_VEGAS
#define FXJ_P_VEGAS 1  // ... of the Vegas kernels: 12 x[] + bins + Philox state per point; one point keeps 6 blocks resident
#endif
#define FXJ_P_OF(mode) ((mode) == 2 ? FXJ_P_VEGAS : FXJ_P)
struct fxj_smem_layout {
  uint32_t acc, nf, delta, tf, grid, hist, wsum, total;
};
// accumulator slots of a native kernel: a fixed 16 (real) / 32 (complex) for the lattice and MC kernels (every
// shared-memory offset is then a compile-time constant), exactly 2K / 4K for the Vegas kernels, whose
// per-warp histograms want the room
static inline __host__ __device__ int fxj_acc_slots(bool vegas, bool cplx, int K) {
  return vegas ? (cplx ? 4 : 2) * K : (cplx ? FXJ_ACC_SLOTS : 16);
}
static inline __host__ __device__ fxj_smem_layout fxj_layout(int dim, int nbins, bool vegas, int acc_slots) {
  fxj_smem_layout L;
  L.acc = 0;
  L.nf = (uint32_t)acc_slots * FX_THREADS * 8u;  // per-thread count of non-finite values, right behind the accumulators
  L.delta = L.nf + FX_THREADS * 8u;
  L.tf = L.delta + FX_NXMAX * 8u;
  L.grid = L.tf + FX_TF_BYTES;
  L.hist = L.grid + (vegas ? (uint32_t)dim * (nbins + 1) * 8u : 0u);
  L.wsum = L.hist + (vegas ? (FX_THREADS / 32) * (uint32_t)dim * nbins * 8u : 0u);
  L.total = L.wsum + (uint32_t)acc_slots * (FX_THREADS / 32) * 8u;
  return L;
}

// S[row][FX_ACC_SLOTS] = sum over chunks of the partials of nrows (sector, shift) rows, fixed order
cudaError_t fx_launch_reduce_chunks(const double *partials, double *sums, int nrows, int nchunks, cudaStream_t st);
// Vegas: hist[sector][dim*nbins] = sum over the blocks' histograms, fixed order
cudaError_t fx_launch_reduce_hist(const double *hist_part, double *hist, int nsectors, int nchunks, int cells,
                                  cudaStream_t st);

struct fx_result_dev {
  double re, re_err, im, im_err, chi2;
  unsigned long long neval, n_nonfinite;
};
// lattice / MC estimator (R5) -> results[nsel][K]
cudaError_t fx_launch_estimate(const double *sums, const fx_sector_dev *sectors, const int32_t *sel, int nsel, int R,
                               uint64_t n_per_shift, const unsigned long long *nonfinite, fx_result_dev *results,
                               int Kstride, cudaStream_t st);
// Vegas: per-iteration (I, var) from the sums of one iteration -> iter_stats[it][nsel][FX_ACC_SLOTS]
cudaError_t fx_launch_vegas_iter_stats(const double *sums, double *iter_stats, int it, int nsel, uint64_t npoints,
                                       cudaStream_t st);
cudaError_t fx_launch_vegas_combine(const double *iter_stats, int iters, const fx_sector_dev *sectors,
                                    const int32_t *sel, int nsel, uint64_t npoints,
                                    const unsigned long long *nonfinite, fx_result_dev *results, int Kstride,
                                    cudaStream_t st);
// refine ngrids independent (grid[NB+1], hist[NB]) pairs (R8 i-iv); in place allowed
cudaError_t fx_launch_vegas_refine(const double *grid_in, const double *hist, double *grid_out, int ngrids, int nbins,
                                   double alpha, cudaStream_t st);
cudaError_t fx_launch_vegas_init_grid(double *grid, int ngrids, int nbins, cudaStream_t st);

cudaError_t fx_launch_generate_points(int rule, uint64_t seed, int sector_id, int shift_or_iter, uint64_t n_lattice,
                                      int log2_n, const uint64_t *genvec_host, uint64_t first, uint64_t count, int dim,
                                      uint64_t *t_dev, cudaStream_t st);
cudaError_t fx_launch_transform_points(int rule, const fx_transform_host &tf, const uint64_t *t_dev, uint64_t count,
                                       int dim, double *x_dev, double *xbar_dev, double *w_dev, cudaStream_t st);
// double-double walk (fx_kernels_dd.cu): mem_doubles = 2 * n_mem_main * FX_THREADS
cudaError_t fx_launch_eval_dd(const fx_eval_params &prm, cudaStream_t st);  // out[npts][K][hi, lo]
cudaError_t fx_launch_rescue_real(const fx_integrate_params &prm, int nsectors, cudaStream_t st);
size_t fx_rescue_smem_bytes(const fx_integrate_params &prm);
// deterministic cubature (fx_kernels_cubature.cu; R21): Genz-Malik degree-7 rule with embedded degree 5
#define FX_GM_REC 36  // per-box record: I7[16], |I7-I5|[16], split axis, non-finite node values, sum of the 16 errors, pad
struct fx_gm_tables {
  double l2, l3, l5, ratio;  // node radii in units of the half-widths; (l2/l3)^2
  double w7[5], w5[5];       // weights of the node classes: centre, l2 axis, l3 axis, l3 pairs, corners
};
fx_gm_tables fx_gm_make_tables(int n);
int fx_gm_nodes_per_box(int n);
// boxes[nboxes][2][n] (centre, half-widths) -> x[nboxes][NN][n]
cudaError_t fx_launch_gm_nodes(const double *boxes, uint64_t nboxes, int n, double *x, cudaStream_t st);
// vals[nboxes][NN][ncomp] -> rec[nboxes][FX_GM_REC]; optional i5_out[nboxes][ncomp], d_out[nboxes][n]
cudaError_t fx_launch_gm_reduce(const double *vals, const double *boxes, uint64_t nboxes, int n, int ncomp, double *rec,
                                double *i5_out, double *d_out, cudaStream_t st);
cudaError_t fx_launch_fp64_peak(double *sink_dev, int iters, int blocks, cudaStream_t st);

#endif
