// fx_interp.cuh -- the program walk ("the code runs a cycle
// through all the operations evaluating the function").
//
// One thread evaluates P points at once (ILP: P independent FP64 chains per handler), the walk
// is warp-uniform (every thread of a block runs the same program), and every operand register
// is named by the opcode, so the handlers are plain DFMA/DMUL/DADD on physical registers: no
// indexed register file, no per-point temporaries in memory (contrast PAPER.md:126).
//
// Two levels:
//   fast path  fx_fast<T,NX,P>::run  -- generated inline PTX (gen_interp_ptx.py): fetch, brx.idx
//              dispatch and the arithmetic handlers; runs until it meets an opcode
//              it does not implement and hands that instruction back;
//   slow path  the switch below, in C++: outputs (FX_OUT), FX_END and the rare library-backed
//              operations (log, exp; complex division, square root).  A few per point.
#ifndef FX_INTERP_CUH
#define FX_INTERP_CUH

#include "fx_isa.h"
#include "fx_math.cuh"

template <typename T>
struct fx_mem;  // shared-memory spill slots, one column per thread
template <>
struct fx_mem<double> {
  double *base;  // &M[0][tid]
  int stride;    // threads per block
  __device__ __forceinline__ double ld(int slot, int p, int P) const { return base[(slot * P + p) * stride]; }
  __device__ __forceinline__ void st(int slot, int p, int P, double v) const { base[(slot * P + p) * stride] = v; }
};
template <>
struct fx_mem<cplx> {
  double *base;
  int stride;
  __device__ __forceinline__ cplx ld(int slot, int p, int P) const {
    return cplx{base[((2 * slot) * P + p) * stride], base[((2 * slot + 1) * P + p) * stride]};
  }
  __device__ __forceinline__ void st(int slot, int p, int P, cplx v) const {
    base[((2 * slot) * P + p) * stride] = v.re;
    base[((2 * slot + 1) * P + p) * stride] = v.im;
  }
};

#define FX_PLOOP _Pragma("unroll") for (int p = 0; p < P; ++p)

template <typename T, int NX, int P>
struct fx_fast;  // specialised by the generated file for the variants FX_WANT selects

#ifndef FX_WANT
#error "define FX_WANT(is_cplx, nx, p) before including fx_interp.cuh"
#endif
#include "fx_interp_gen.inc"

// Library-backed operations, out of line (one copy per kernel: instruction-cache footprint, see
// fx_device_common.cuh) and over all P points of the thread at once, so that the P dependency
// chains of a log or exp overlap instead of running one after the other.
template <typename T, int P>
struct fx_vec {
  T v[P];
};
#ifndef FX_SLOW_ATTR  // a translation unit may ask for inline copies (see fx_kernels_cplx.cu)
#define FX_SLOW_ATTR __noinline__
#endif
#define FX_SLOW_UNARY(name, fn)                                                  \
  template <typename T, int P>                                                   \
  static __device__ FX_SLOW_ATTR fx_vec<T, P> name(fx_vec<T, P> a) {             \
    _Pragma("unroll") for (int p = 0; p < P; ++p) a.v[p] = fn(a.v[p]);           \
    return a;                                                                    \
  }
FX_SLOW_UNARY(fx_slow_log, t_log)
FX_SLOW_UNARY(fx_slow_exp, t_exp)
FX_SLOW_UNARY(fx_slow_sqrt, t_sqrt)
template <typename T, int P>
static __device__ FX_SLOW_ATTR fx_vec<T, P> fx_slow_div(fx_vec<T, P> a, fx_vec<T, P> b) {
#pragma unroll
  for (int p = 0; p < P; ++p) a.v[p] = t_div(a.v[p], b.v[p]);
  return a;
}
template <typename T, int P>
__device__ __forceinline__ fx_vec<T, P> fx_pack(const T (&A)[P]) {
  fx_vec<T, P> r;
#pragma unroll
  for (int p = 0; p < P; ++p) r.v[p] = A[p];
  return r;
}
template <typename T, int P>
__device__ __forceinline__ void fx_unpack(T (&A)[P], const fx_vec<T, P> &r) {
#pragma unroll
  for (int p = 0; p < P; ++p) A[p] = r.v[p];
}

// R[r] for a run-time r: only the slow path uses it (complex division by a register)
template <typename T, int NX, int P>
__device__ __forceinline__ void fx_reg_dyn(int r, const T (&X)[NX][P], const T (&S)[FX_NS][P], T (&out)[P]) {
#pragma unroll
  for (int k = 0; k < NX; ++k)
    if (r == k) FX_PLOOP { out[p] = X[k][p]; }
#pragma unroll
  for (int j = 0; j < FX_NS; ++j)
    if (r == FX_NXMAX + j) FX_PLOOP { out[p] = S[j][p]; }
}

// Walk `prog` (shared memory) for the P points whose variables are in X.  `sink(k, A)` receives
// output k (FX_OUT).  M are this thread's spill slots (stride must be FX_THREADS).
template <typename T, int NX, int P, class Sink>
__device__ __forceinline__ void fx_run(const fx_ins *prog, T (&X)[NX][P], const fx_mem<T> M, Sink &sink) {
  T AL[FX_L][P];  // accumulator levels; the slow path only ever touches level 0
  T S[FX_NS][P];
#pragma unroll
  for (int d = 0; d < FX_L; ++d) FX_PLOOP { AL[d][p] = t_from_real(0.0, T{}); }
#pragma unroll
  for (int j = 0; j < FX_NS; ++j) FX_PLOOP { S[j][p] = t_from_real(0.0, T{}); }
  T(&A)[P] = AL[0];
  uint32_t pc = (uint32_t)__cvta_generic_to_shared(prog);
  const uint32_t mem = (uint32_t)__cvta_generic_to_shared(M.base);
  for (;;) {
    uint32_t w0, w2, w3;
    fx_fast<T, NX, P>::run(AL, X, S, pc, mem, w0, w2, w3);
    const int op = w0 & 0xffff;
    const int aux = w0 >> 16;
    const double imm = __hiloint2double((int)w3, (int)w2);
    if (op == FX_OUT) {
      sink(aux, A);
    } else if (op == FX_LOG) {
      fx_unpack(A, fx_slow_log(fx_pack<T, P>(A)));
    } else if (op == FX_EXP) {
      fx_unpack(A, fx_slow_exp(fx_pack<T, P>(A)));
    } else if (op == FX_SQRT) {
      fx_unpack(A, fx_slow_sqrt(fx_pack<T, P>(A)));
    } else if (op == FX_RDIVC) {
      FX_PLOOP { A[p] = t_rdivc(imm, A[p]); }
    } else if (op == FX_DIVM) {
      T R[P];
      FX_PLOOP { R[p] = M.ld(aux, p, P); }
      fx_unpack(A, fx_slow_div(fx_pack<T, P>(A), fx_pack<T, P>(R)));
    } else if (op == FX_RDIVM) {
      T R[P];
      FX_PLOOP { R[p] = M.ld(aux, p, P); }
      fx_unpack(A, fx_slow_div(fx_pack<T, P>(R), fx_pack<T, P>(A)));
    } else if (op >= FX_DIV_R && op < FX_DIV_R + FX_NR) {
      T R[P];
      FX_PLOOP { R[p] = A[p]; }
      fx_reg_dyn<T, NX, P>(op - FX_DIV_R, X, S, R);
      fx_unpack(A, fx_slow_div(fx_pack<T, P>(A), fx_pack<T, P>(R)));
    } else if (op >= FX_RDIV_R && op < FX_RDIV_R + FX_NR) {
      T R[P];
      FX_PLOOP { R[p] = A[p]; }
      fx_reg_dyn<T, NX, P>(op - FX_RDIV_R, X, S, R);
      fx_unpack(A, fx_slow_div(fx_pack<T, P>(R), fx_pack<T, P>(A)));
    } else if (op == FX_END) {
      return;
    } else {
      __trap();  // an opcode this kernel has no handler for (compiler / interpreter mismatch, or a variable
                 // index >= NX): fail loudly (the launch reports an error) instead of dropping outputs
    }
  }
}

#endif
