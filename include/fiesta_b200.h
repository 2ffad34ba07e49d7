/* fiesta_b200.h -- C ABI of the B200-native integration hot path of FIESTA 4 (arXiv:1511.03614).
 *
 * What the library does (citations: PAPER.md:<line> of the paper text, or DESIGN.md R<n> for a
 * reading taken where the paper is silent):
 *
 *   fiesta_compile    turns the integrand expressions of each sector, one text per epsilon order in
 *                     the integration worker's grammar, into a straight-line
 *                     FP64 instruction program ("a sequence of quadripples (operator, first
 *                     operand, second operand, result)") and uploads it to the GPU.
 *   fiesta_integrate  evaluates every program at quasi-/pseudo-Monte-Carlo points generated on the
 *                     device and reduces per sector and per order to (value, error)
 *                     (PAPER.md:110, :118-124 for the evaluation; PAPER.md:316 for value +- error).
 *
 * Conventions
 *   - every function returns 0 on success or a negative FIESTA_E_* code; no exception crosses
 *     the ABI.  fiesta_last_error(ctx) gives a ctx-owned NUL-terminated message, valid until the
 *     next call on that ctx.
 *   - pointers named *_host are HOST memory, caller-allocated, borrowed for the call only.
 *     pointers named *_dev are DEVICE memory on the ctx's device.
 *   - calls are synchronous unless the name ends in _async: on return the stream has been
 *     synchronised and host outputs are filled.
 *   - there is no CPU fallback: without an sm_100 device fiesta_create fails with FIESTA_E_CUDA.
 *   - all arithmetic is IEEE FP64 on the device.
 */
#ifndef FIESTA_B200_H
#define FIESTA_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  FIESTA_OK = 0,
  FIESTA_E_PARSE = -1,     /* text does not follow the grammar; message has sector/order/column   */
  FIESTA_E_DIM = -2,       /* x[i] with i > dim, dim out of range, inconsistent nvars             */
  FIESTA_E_NOTPOLY = -3,   /* deformation F is not a polynomial in x                              */
  FIESTA_E_RULE = -4,      /* bad rule parameters (lattice size not 2^m, bins out of range, ...)  */
  FIESTA_E_CUDA = -5,      /* CUDA runtime error or no suitable device                            */
  FIESTA_E_NONFINITE = -6, /* some integrand value was NaN/Inf; results filled, n_nonfinite > 0   */
  FIESTA_E_ARG = -7,       /* NULL pointer, bad index, size out of range                          */
  FIESTA_E_TOOBIG = -8     /* a program exceeds the per-block shared-memory budget                */
};

#define FIESTA_MAX_DIM 12     /* integration variables per sector                                 */
#define FIESTA_MAX_ORDERS 8   /* epsilon orders (outputs) per sector                              */
#define FIESTA_MAX_BINS 128   /* Vegas bins per dimension                                         */

typedef struct fiesta_ctx fiesta_ctx;         /* opaque; owns device scratch; bound to one device+stream */
typedef struct fiesta_program fiesta_program; /* opaque; immutable after compile; free with _program_free */

/* Create a context on CUDA device `cuda_device`.  `cuda_stream` is a cudaStream_t (may be 0 for
 * the default stream); every launch and copy of this ctx goes to it. */
int fiesta_create(fiesta_ctx **out, int cuda_device, void *cuda_stream);
void fiesta_destroy(fiesta_ctx *ctx);
const char *fiesta_last_error(const fiesta_ctx *ctx);

/* One sector = K expression texts (one per epsilon order), each
 *   "<nvars>;\n<nfunc>;\n<f1>;\n...\n<final>;\n|"
 * with tokens: floats, x[i], f[i], + - * / ( ), p[expr,exponent], l[expr], P, G and the seven
 * hard-coded PolyGamma[n,m].  The K texts of one sector may share f-lines; common
 * subexpressions are evaluated once per point (R7).  An "evaluation" in the metric is
 * still one (point, sector, order). */
typedef struct {
  int32_t sector_id;         /* caller's label; enters the random streams (R3)           */
  int32_t n_orders;          /* K, 1..FIESTA_MAX_ORDERS                                            */
  const char *const *expr;   /* K NUL-terminated texts                                             */
  int32_t is_complex;        /* 0 real, 1 complex arithmetic                        */
  int32_t deform_f_index;    /* >=1: f[deform_f_index] of text 0 is the polynomial F whose gradient
                                drives the contour deformation (R11);
                                0: no deformation.  Implies complex.                               */
  double lambda;             /* deformation size; ignored if deform_f_index == 0                   */
} fiesta_sector_desc;

typedef struct {
  int32_t n_ir_ops;          /* instructions of the main program                                   */
  int32_t n_fp64_ops;        /* of which FP64 arithmetic (fma/mul/add/div/log/exp ...)             */
  int32_t n_fma;             /* fused multiply-adds                                                */
  int32_t n_log, n_exp, n_div;
  int32_t n_reg_temps;       /* register temporaries S[] used (the ISA has FX_NS = 1)              */
  int32_t n_mem_slots;       /* shared-memory spill slots per point (compiler-directed; 0 is best) */
  int32_t n_deform_ops;      /* instructions of the gradient/Hessian program (0 if none)           */
  double flops;              /* FP64 flops per point counted as fma=2, mul/add=1, div=~15, log/exp~40 (nominal) */
} fiesta_compile_info;

/* Parse, optimise, register-allocate and upload.  `info` may be NULL, else [nsectors].
 *
 * Two forms of the same instruction program exist ("transforms to an internal form"):
 *   (1) the fx_ins sequence, uploaded to the device arena and walked by the interpreter kernels.
 *       It is complete when fiesta_compile returns: the program can be integrated at once.
 *   (2) that same sequence lowered instruction by instruction to PTX, spliced into the evaluation
 *       kernel and assembled for sm_100a in process: one native kernel per (sector, mode), mode =
 *       a FIESTA_RULE_* or FIESTA_MODE_EVAL (real and complex sectors).  The program's own
 *       background threads assemble them (~0.1-0.2 s of one host core per kernel), from the first
 *       call on that can use them: a call asks for the kernels of its rule for those of its
 *       sectors whose work per pass (points x instructions) is large enough for a launch of their
 *       own to pay (FIESTA_NATIVE_MIN_WORK, default 2e7); smaller sectors stay on the interpreter,
 *       which takes all of them in one launch.
 * fiesta_integrate serves every such sector with its native kernel if that is ready and with the
 * interpreter otherwise; both forms perform the same operations in the same order with the same
 * roundings, so a sector's sums are bit-identical whichever served it.
 * Environment (read at each fiesta_compile): FIESTA_JIT=0 no native tier; FIESTA_JIT=eager queue the
 * lattice kernels of all sectors at once; FIESTA_JIT=sync the same and return only when they are
 * ready; FIESTA_CACHE_DIR=<dir> keep assembled kernels on disk, keyed by the program (a process-wide
 * in-memory cache always exists). */
int fiesta_compile(fiesta_ctx *ctx, const fiesta_sector_desc *sectors, int32_t nsectors, int32_t dim,
                   fiesta_program **out, fiesta_compile_info *info);
void fiesta_program_free(fiesta_program *prog);

enum { FIESTA_RULE_LATTICE = 0, FIESTA_RULE_MC = 1, FIESTA_RULE_VEGAS = 2 };
/* modes of the native kernels: the three rules, and the parity hook fiesta_eval_points */
enum { FIESTA_MODE_EVAL = 3, FIESTA_N_MODES = 4 };
/* tier arguments: whichever form is ready / interpreter only / native only (waits for the assembly) */
enum { FIESTA_TIER_ANY = -1, FIESTA_TIER_INTERPRETER = 0, FIESTA_TIER_NATIVE = 1 };

/* Sampling rule (R1-R4, R8; the paper names only "Vegas").
 *   LATTICE: npoints = n_shifts * N_L, N_L = 2^m; rank-1 lattice with generating vector genvec
 *            (or Korobov g_k = korobov_a^k mod N_L), n_shifts random shifts from Philox,
 *            Korobov periodising transform of weight periodize_r (0..6).
 *   MC:      npoints Philox points, x = u.
 *   VEGAS:   vegas_iters iterations of npoints Philox points through a vegas_bins-bin grid per
 *            dimension, refined between iterations with damping vegas_alpha. */
typedef struct {
  int32_t kind;
  int32_t n_shifts;
  uint64_t korobov_a;
  const uint64_t *genvec;   /* optional HOST [dim]; NULL -> Korobov form */
  int32_t periodize_r;
  int32_t vegas_bins;
  int32_t vegas_iters;
  double vegas_alpha;
} fiesta_rule;

/* Per (sector, order).  Real sectors: im = im_err = 0.  chi2: Vegas only (else 0). */
typedef struct {
  double re, re_err, im, im_err, chi2;
  uint64_t neval, n_nonfinite;
} fiesta_result;

/* Integrate sectors[0..nsectors) (indices into the program; NULL = 0..nsectors-1) and write
 * out_host[nsectors][K] row-major.  All sectors of one call use the same rule and seed. */
int fiesta_integrate(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsectors,
                     int32_t dim, uint64_t npoints, const fiesta_rule *rule, uint64_t seed,
                     fiesta_result *out_host);

/* Same work, but nothing is copied back and the stream is not synchronised; results stay in a
 * ctx-owned device buffer that fiesta_fetch_results copies out.  For device-side timing. */
int fiesta_integrate_async(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsectors,
                           int32_t dim, uint64_t npoints, const fiesta_rule *rule, uint64_t seed);
int fiesta_fetch_results(fiesta_ctx *ctx, int32_t nsectors, int32_t K, fiesta_result *out_host);

/* fiesta_integrate with the tier fixed (FIESTA_TIER_*).  out_host may be NULL (as _async). */
int fiesta_integrate_tier(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsectors,
                          int32_t dim, uint64_t npoints, const fiesta_rule *rule, uint64_t seed, int32_t tier,
                          fiesta_result *out_host);

/* Device time (ms, CUDA events on the ctx stream) that the evaluation kernels of the last
 * fiesta_integrate[_async] took (chunk reductions between batches included), and how many kernels
 * the call launched.  Synchronises. */
int fiesta_last_timing(fiesta_ctx *ctx, double *eval_kernel_ms, int32_t *n_launches);

/* How many (sector, pass) units of the last integrate-family call ran on a native kernel and how
 * many on the interpreter. */
int fiesta_last_tiers(fiesta_ctx *ctx, int32_t *n_native, int32_t *n_interpreter);

/* ---- parity hooks: the same device code paths, exposed piecewise -------------------------- */

/* Integrand values at caller-given points (PAPER.md:414 `justEvaluate`; PAPER.md:531 `Debug`).
 * x_host[npts][dim]; out_host[npts][K][2] = (re, im) of o_k(x) -- for deformed sectors
 * o_k(z(x)) * det J(x) -- WITHOUT the rule's weight.  The native tier runs the sector's generated
 * program body -- the text the integration kernels are assembled from -- in an eval kernel;
 * fiesta_eval_points takes it when ready, _tier fixes the tier (FIESTA_TIER_NATIVE waits). */
int fiesta_eval_points(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, const double *x_host,
                       uint64_t npts, double *out_host);
int fiesta_eval_points_tier(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, int32_t tier,
                            const double *x_host, uint64_t npts, double *out_host);

/* ---- few, huge sectors: the shifts of the lattice rule split over ranks ----------
 *
 * fiesta_partial_sums_shifts: fiesta_partial_sums for the shifts shift_first .. shift_first +
 * shift_count - 1 of the rule's n_shifts only (lattice rule; npoints is still the rule's total,
 * n_shifts x N_L).  sums_host[nsel][shift_count][K][C][2].  A shift's sums do not depend on which
 * other shifts a call computes: the rows are, bit for bit, those of the full call.
 * fiesta_last_nonfinite: the per-sector counts of NaN / Inf values of the last integrate-family call.
 * fiesta_estimate_from_sums: the estimator (R5) on the device from per-shift sums in the
 * layout of fiesta_partial_sums ([nsel][n_shifts][K][C][2]; all sectors with the same K), e.g. the
 * rows the ranks have exchanged; nonfinite_host[nsel] may be NULL (zeros).  out[nsel][K]. */
int fiesta_partial_sums_shifts(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsel,
                               int32_t dim, uint64_t npoints, const fiesta_rule *rule, uint64_t seed, int32_t tier,
                               int32_t shift_first, int32_t shift_count, double *sums_host);
int fiesta_last_nonfinite(fiesta_ctx *ctx, int32_t nsel, uint64_t *counts_host);
int fiesta_estimate_from_sums(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsel,
                              int32_t n_shifts, uint64_t n_per_shift, const double *sums_host,
                              const uint64_t *nonfinite_host, fiesta_result *out);

/* ---- no device allocation (for callers that cannot call cudaMalloc) ----------------------------
 *
 * The per-shift sums of fiesta_partial_sums for ONE real sector under the lattice or the plain-MC
 * rule, computed without cudaMalloc, cudaFree or any allocating library routine: the partial records
 * live in a file-scope device array of fixed size that every GPU holds from the moment it loads
 * the library until the process exits (1 MiB + 256 B: 4096 records).  Limit: n_shifts x chunks <=
 * 4096 -- a chunk is at most 2^17 points, so up to 2^29 points per call; beyond it the call fails
 * with FIESTA_E_TOOBIG before anything is launched.  Vegas: FIESTA_E_RULE; complex sector:
 * FIESTA_E_ARG.  The evaluation runs on the interpreter kernel in plain FP64 (fiesta_set_mixed is
 * ignored), with the chunking and the order of additions of fiesta_partial_sums: the same bits.
 *
 * sums_dev: DEVICE memory of the caller, [n_shifts][K][2] doubles (S1, S2; n_shifts = 1 for MC);
 * nonfinite_dev: DEVICE memory, one uint64 (count of NaN / Inf values), or NULL.  The work is queued
 * on the context's stream and the call returns without waiting (_async): synchronise that stream
 * before reading.  The first call on a device resolves the array's address, which may load this
 * part of the library's device code: make one warm-up call before a region that must not allocate.
 * All calls on a device share the array: calls that overlap on the GPU (other streams or contexts)
 * race -- serialise them. */
int fiesta_partial_sums_noalloc_async(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, int32_t dim,
                                      uint64_t npoints, const fiesta_rule *rule, uint64_t seed, double *sums_dev,
                                      uint64_t *nonfinite_dev);

/* ---- deterministic integrator (PAPER.md:412 `CurrentIntegrator -> cuhreCuba`) ------
 *
 * A Cuhre-like globally adaptive cubature on the same evaluator (R21): the degree-7 rule of
 * Genz and Malik with its embedded degree-5 rule on boxes of the unit cube (1 + 4n + 2n(n-1) + 2^n
 * nodes per box; the error of a box is |I7 - I5| per component).  Rounds: the boxes that carry the
 * worst half of the summed error are halved along the axis of their largest fourth difference, until
 * for every order and component  sum err <= max(epsabs, epsrel |sum I7|)  or another round would pass
 * maxeval integrand evaluations.  No random numbers: a call is reproducible bit by bit.
 *
 * sectors[nsel] (NULL: 0..nsel-1), all with the same number of orders K; dim >= 2 (FIESTA_E_DIM);
 * tier as for fiesta_eval_points_tier.  out[nsel][K]: re / im = the estimates, re_err / im_err = the
 * summed box errors, chi2 = 0, neval = integrand evaluations spent on the sector; nboxes_out[nsel]
 * (may be NULL): boxes at the end.  A NaN or Inf at a node ends the sector's rounds; the call then
 * returns FIESTA_E_NONFINITE after filling out (n_nonfinite > 0). */
int fiesta_integrate_cubature(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsel,
                              double epsrel, double epsabs, uint64_t maxeval, int32_t tier, fiesta_result *out,
                              uint64_t *nboxes_out);

/* Parity hook: the rule on caller-given boxes.  boxes_host[nboxes][2][dim] = centre, half-widths (inside
 * the unit cube, else FIESTA_E_ARG); i7_host, i5_host [nboxes][K][2] (re, im), fourth_host[nboxes][dim]
 * (fourth differences summed over the components), axis_host[nboxes]; any output may be NULL. */
int fiesta_cubature_rule(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, int32_t tier,
                         const double *boxes_host, uint64_t nboxes, double *i7_host, double *i5_host,
                         double *fourth_host, int32_t *axis_host);

/* ---- mixed precision ("MPFR, Native and Mixed (default variant)") ---
 *
 * fiesta_set_mixed: from now on the lattice, plain-MC and Vegas rules of this context evaluate every point
 * with min_k x_k < small_x (the paper's SmallX knob) in double-double
 * arithmetic (two doubles, ~106 bits: this library's stand-in for MPFR) and all other points in
 * double, as before (R20).  The points, their weights and the order of the sums do not
 * change; with no point below small_x the results are bit-identical to small_x = 0.  small_x = 0
 * (the default) switches the mode off; small_x > 1 sends every point through the double-double
 * walk ("-mpfr: evaluate all integration points with the use of MPFR").  Under the
 * Vegas rule the decision is taken on the mapped point and the rescued points enter the histogram.
 * Real sectors only: with the mode on, a call that selects a complex sector fails with
 * FIESTA_E_RULE, and so does FIESTA_TIER_NATIVE (the first phase runs on the interpreter kernels;
 * the default tier choice follows).  Constants enter the double-double walk as the doubles the compiler
 * stored.  small_x < 0 or NaN: FIESTA_E_ARG. */
int fiesta_set_mixed(fiesta_ctx *ctx, double small_x);

/* Parity hook of the double-double walk: out_host[npts][K][2] = (hi, lo) with o_k(x) = hi + lo
 * (|lo| <= ulp(hi)/2) for the real sector `sector` at x_host[npts][dim].  Complex sector:
 * FIESTA_E_ARG. */
int fiesta_eval_points_dd(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, const double *x_host,
                          uint64_t npts, double *out_host);

/* The 64-bit integers t[j][k] (R2/R3) behind points j = first..first+count-1 of shift
 * (lattice) or iteration (MC/Vegas) `shift_or_iter` of the sector labelled sector_id.
 * n_lattice is used by the lattice rule only.  t_host[count][dim]. */
int fiesta_generate_points(fiesta_ctx *ctx, const fiesta_rule *rule, uint64_t seed, int32_t sector_id,
                           int32_t shift_or_iter, uint64_t n_lattice, uint64_t first, uint64_t count,
                           int32_t dim, uint64_t *t_host);

/* The unit-cube point and weight the rule makes from those integers (lattice: after the
 * periodising transform; MC: x = u, w = 1).  x_host[count][dim], xbar_host[count][dim] (= 1 - x,
 * computed without cancellation), w_host[count]. */
int fiesta_transform_points(fiesta_ctx *ctx, const fiesta_rule *rule, const uint64_t *t_host, uint64_t count,
                            int32_t dim, double *x_host, double *xbar_host, double *w_host);

/* Lattice / MC: per-shift sums S1 = sum_j g, S2 = sum_j g^2, g = W * o_k component, before the
 * estimator.  sums_host[nsectors][R][K][C][2], C = 1 (real) or 2 (complex: Re, Im). */
int fiesta_partial_sums(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsectors,
                        int32_t dim, uint64_t npoints, const fiesta_rule *rule, uint64_t seed,
                        double *sums_host);
int fiesta_partial_sums_tier(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsectors,
                             int32_t dim, uint64_t npoints, const fiesta_rule *rule, uint64_t seed, int32_t tier,
                             double *sums_host);

/* The first level of the two-level reduction: the partial record of every block.  A block sums the
 * points j = c * chunk_points .. min((c+1) * chunk_points, N_L) - 1 of one (sector, shift), c <
 * nchunks.  sums_host[nsectors][R][nchunks][K][C][2]; with sums_host == NULL only the geometry is
 * returned.  For sampled checks of a full-size launch: the chunking is that of fiesta_integrate for
 * the same rule and npoints.  nsectors must fit one batch (FIESTA_E_ARG otherwise). */
int fiesta_chunk_sums(fiesta_ctx *ctx, const fiesta_program *prog, const int32_t *sectors, int32_t nsectors,
                      int32_t dim, uint64_t npoints, const fiesta_rule *rule, uint64_t seed, int32_t tier,
                      uint64_t *chunk_points, int32_t *nchunks, double *sums_host);

/* One Vegas iteration of one sector on a caller-given grid (R8):
 * grid_host[dim][NB+1] in; sums_host[K][C][2] (S1, S2) and hist_host[dim][NB] out. */
int fiesta_vegas_iteration(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, int32_t dim,
                           uint64_t npoints, const fiesta_rule *rule, uint64_t seed, int32_t iteration,
                           const double *grid_host, double *sums_host, double *hist_host);
int fiesta_vegas_iteration_tier(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, int32_t dim,
                                uint64_t npoints, const fiesta_rule *rule, uint64_t seed, int32_t iteration,
                                int32_t tier, const double *grid_host, double *sums_host, double *hist_host);

/* The grid refinement step alone: ngrids independent (grid[NB+1], hist[NB]) pairs. */
int fiesta_vegas_refine(fiesta_ctx *ctx, int32_t ngrids, int32_t nbins, double alpha, const double *grid_host,
                        const double *hist_host, double *grid_out_host);

/* Grid and last histogram of sector index `sector` after the last VEGAS fiesta_integrate.
 * grid_host[dim][NB+1], hist_host[dim][NB] (either may be NULL). */
int fiesta_vegas_grid(fiesta_ctx *ctx, int32_t sector, int32_t dim, int32_t nbins, double *grid_host,
                      double *hist_host);

/* ---- contour deformation: -testF and the choice of lambda ---------------- */

/* What the F(z) of a deformed sector does at sampled points. */
typedef struct {
  uint64_t n_points;  /* points looked at                                                            */
  uint64_t n_bad;     /* of which Im F(z) >= 0 (or NaN): the deformation is on the wrong side there  */
  double max_im_f;    /* max Im F(z) over the points (< 0 when n_bad == 0)                           */
  double min_abs_f;   /* min |F(z)|: how close the contour comes to a zero of F                      */
  double lambda;      /* the lambda this was evaluated with                                          */
} fiesta_testf_result;

/* "-testF: instead of the integration, the code checks whether the sign of the imaginary part of F is
 * negative".  Evaluates F(z(x)) -- F = f[deform_f_index] of the sector -- at the points
 * of `rule` (lattice or MC; npoints, seed as in fiesta_integrate), deformed with `lambda` (< 0: the
 * sector's own), on the device.  FIESTA_E_ARG if the sector has no deformation. */
int fiesta_test_f(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, int32_t dim, uint64_t npoints,
                  const fiesta_rule *rule, uint64_t seed, double lambda, fiesta_testf_result *out_host);

/* The deformation size "is tuned automatically in the interval from zero to MaxComplexShift" with
 * LambdaSplit candidates and LambdaIterations sampling points; ConservativeComplexShift halves the
 * result.  The paper does not give the search (it defers to the FIESTA 3 paper);
 * DESIGN.md R19: candidates lambda_max * i / lambda_split, i = 1..lambda_split, each tested with
 * fiesta_test_f on the same `npoints` Philox points; admissible = no point with Im F(z) >= 0; the
 * admissible candidate with the largest min |F(z)| wins (the contour that stays furthest from the
 * zeros of F), halved if `conservative`.  scan_host (may be NULL) receives the lambda_split test
 * results.  FIESTA_E_RULE (lambda 0) if no candidate is admissible.  The choice is returned, not
 * applied: fiesta_program_set_lambda does that. */
int fiesta_select_lambda(fiesta_ctx *ctx, const fiesta_program *prog, int32_t sector, int32_t dim, uint64_t npoints,
                         uint64_t seed, double lambda_max, int32_t lambda_split, int32_t conservative,
                         double *lambda_host, fiesta_testf_result *scan_host);

/* Change the deformation size of one sector of a compiled program (lambda is a run-time parameter of
 * both tiers' kernels: nothing is recompiled).  Synchronises the ctx stream. */
int fiesta_program_set_lambda(fiesta_ctx *ctx, fiesta_program *prog, int32_t sector, double lambda);

/* Sum over sectors with errors combined in mean square.  Host arithmetic on
 * nsectors*K numbers; total_host[K]. */
int fiesta_combine(const fiesta_result *per_sector_host, int32_t nsectors, int32_t K, fiesta_result *total_host);

/* 1 if the native kernel of (`sector`, `mode`) is ready, else 0; <0 on bad arguments.  info_host (may
 * be NULL) receives, when ready, the assembler's resource report ("Used N registers, ... bytes spill
 * stores ..."), else why not ("" = never requested or the native tier is off, "being assembled",
 * or the assembler's error). */
int fiesta_program_native(const fiesta_program *prog, int32_t sector, int32_t mode, char *info_host, uint64_t buflen);

/* Request the `mode` kernels of all sectors and wait (timeout_s < 0: for ever) until none is queued or
 * being assembled.  Returns how many are ready, or <0. */
int fiesta_program_wait_native(fiesta_program *prog, int32_t mode, double timeout_s);

/* Background assembly so far: kernels assembled, kernels taken from the cache, host-core seconds
 * spent (summed over the program's threads), number of threads.  Any pointer may be NULL. */
int fiesta_program_native_stats(const fiesta_program *prog, int32_t *n_assembled, int32_t *n_cache_hits,
                                double *assemble_cpu_seconds, int32_t *n_threads);

/* Host only (no context, no GPU): compile one sector and run the native tier's lowering and assembly
 * on it for `mode`.  Writes the generated PTX (the .const array of the program's FP64 immediates, then
 * the program body or bodies; NUL-terminated, truncated to buflen) to ptx_body_host (may be NULL), the
 * size of the assembled sm_100a cubin to cubin_bytes (may be NULL) and the assembler's resource report
 * to info_host (may be NULL).  FIESTA_E_PARSE etc. as fiesta_compile; FIESTA_E_CUDA if the PTX
 * assembler rejects the module (message in ptx_body_host). */
int fiesta_native_assemble(const fiesta_sector_desc *sector, int32_t dim, int32_t mode, char *ptx_body_host,
                           uint64_t buflen, uint64_t *cubin_bytes, char *info_host, uint64_t infolen);

/* Disassembly of a compiled sector (main program, then the deformation program) into buf. */
int fiesta_program_dump(const fiesta_program *prog, int32_t sector, char *buf_host, uint64_t buflen);

/* FP64 pipe micro-benchmark: independent DFMA chains on every SM for about `ms_target`
 * milliseconds; writes achieved TFLOP/s (2 flops per DFMA).  The roofline denominator. */
int fiesta_fp64_peak(fiesta_ctx *ctx, double ms_target, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* FIESTA_B200_H */
