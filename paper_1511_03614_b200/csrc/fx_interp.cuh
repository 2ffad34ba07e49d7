// fx_interp.cuh -- the program walk ("the code runs a cycle
// through all the operations evaluating the function").
//
// One thread evaluates P points at once (ILP: P independent FP64 chains per handler), the walk
// is warp-uniform (every thread of a block runs the same program), and every operand register
// is named by the opcode, so the handlers are plain DFMA/DMUL/DADD on physical registers: no
// indexed register file, no per-point temporaries in memory (contrast PAPER.md:126).
#ifndef FX_INTERP_CUH
#define FX_INTERP_CUH

#include "fx_isa.h"
#include "fx_math.cuh"

template <int r, typename T, int NX, int P>
__device__ __forceinline__ T (&fx_reg(T (&X)[NX][P], T (&S)[FX_NS][P]))[P] {
  if constexpr (r < FX_NXMAX) return X[r < NX ? r : 0];
  else return S[r - FX_NXMAX];
}

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

#define FX_REP8(M, ...) M(0, __VA_ARGS__) M(1, __VA_ARGS__) M(2, __VA_ARGS__) M(3, __VA_ARGS__) \
  M(4, __VA_ARGS__) M(5, __VA_ARGS__) M(6, __VA_ARGS__) M(7, __VA_ARGS__)
#define FX_REP20(M, ...) M(0, __VA_ARGS__) M(1, __VA_ARGS__) M(2, __VA_ARGS__) M(3, __VA_ARGS__) \
  M(4, __VA_ARGS__) M(5, __VA_ARGS__) M(6, __VA_ARGS__) M(7, __VA_ARGS__) M(8, __VA_ARGS__) \
  M(9, __VA_ARGS__) M(10, __VA_ARGS__) M(11, __VA_ARGS__) M(12, __VA_ARGS__) M(13, __VA_ARGS__) \
  M(14, __VA_ARGS__) M(15, __VA_ARGS__) M(16, __VA_ARGS__) M(17, __VA_ARGS__) M(18, __VA_ARGS__) \
  M(19, __VA_ARGS__)

// one handler of a register family: Rr names R[r] statically
#define FX_CASE_R(r, base, stmt)                       \
  case (base) + (r): {                                 \
    if constexpr ((r) >= FX_NXMAX || (r) < NX) {       \
      T(&Rr)[P] = fx_reg<(r), T, NX, P>(X, S);         \
      FX_PLOOP { stmt; }                               \
    }                                                  \
    break;                                             \
  }
// A = A*R[r] + S[j]
#define FX_CASE_RS_J(j, r)                                              \
  case FX_FMA_AR_S + (r) * FX_NS + (j): {                               \
    if constexpr ((r) >= FX_NXMAX || (r) < NX) {                        \
      T(&Rr)[P] = fx_reg<(r), T, NX, P>(X, S);                          \
      FX_PLOOP { A[p] = t_fma(A[p], Rr[p], S[j][p]); }                  \
    }                                                                   \
    break;                                                              \
  }
#define FX_CASE_RS(r, unused) FX_REP8(FX_CASE_RS_J, r)
#define FX_CASE_ST(j, unused) \
  case FX_ST_S + (j): {       \
    FX_PLOOP { S[j][p] = A[p]; } \
    break;                    \
  }

// Walk `prog` (shared memory) for the P points whose variables are in X.  `sink(k, A)` receives
// output k (FX_OUT).  M are this thread's spill slots.
template <typename T, int NX, int P, class Sink>
__device__ __forceinline__ void fx_run(const fx_ins *prog, T (&X)[NX][P], const fx_mem<T> M, Sink &sink) {
  T A[P];
  T S[FX_NS][P];
  FX_PLOOP { A[p] = t_from_real(0.0, T{}); }
#pragma unroll
  for (int j = 0; j < FX_NS; ++j) FX_PLOOP { S[j][p] = t_from_real(0.0, T{}); }
  const uint4 *pc = reinterpret_cast<const uint4 *>(prog);
  uint4 w = *pc;
  for (;;) {
    const uint4 cur = w;
    ++pc;
    w = *pc;  // prefetch the next instruction (programs end with FX_END followed by padding)
    const int op = cur.x & 0xffff;
    const int aux = cur.x >> 16;
    const double imm = __hiloint2double((int)cur.w, (int)cur.z);
    switch (op) {
      FX_REP20(FX_CASE_R, FX_FMA_AR_C, A[p] = t_fma_c(A[p], Rr[p], imm))
      FX_REP20(FX_CASE_R, FX_FMA_RC_A, A[p] = t_fma_rc(Rr[p], imm, A[p]))
      FX_REP20(FX_CASE_R, FX_MUL_R, A[p] = t_mul(A[p], Rr[p]))
      FX_REP20(FX_CASE_R, FX_ADD_R, A[p] = t_add(A[p], Rr[p]))
      FX_REP20(FX_CASE_R, FX_SUB_R, A[p] = t_sub(A[p], Rr[p]))
      FX_REP20(FX_CASE_R, FX_RSUB_R, A[p] = t_sub(Rr[p], A[p]))
      FX_REP20(FX_CASE_R, FX_LD_R, A[p] = Rr[p])
      FX_REP20(FX_CASE_R, FX_MULC_R, A[p] = t_mulc(Rr[p], imm))
      FX_REP20(FX_CASE_R, FX_DIV_R, A[p] = t_div(A[p], Rr[p]))
      FX_REP20(FX_CASE_R, FX_RDIV_R, A[p] = t_div(Rr[p], A[p]))
      FX_REP20(FX_CASE_R, FX_FMA_AR_M, A[p] = t_fma(A[p], Rr[p], M.ld(aux, p, P)))
      FX_REP20(FX_CASE_RS, 0)
      FX_REP8(FX_CASE_ST, 0)
      case FX_LDC: FX_PLOOP { A[p] = t_from_real(imm, T{}); } break;
      case FX_ADDC: FX_PLOOP { A[p] = t_addc(A[p], imm); } break;
      case FX_MULC: FX_PLOOP { A[p] = t_mulc(A[p], imm); } break;
      case FX_RSUBC: FX_PLOOP { A[p] = t_rsubc(imm, A[p]); } break;
      case FX_DIVC: FX_PLOOP { A[p] = t_divc(A[p], imm); } break;
      case FX_RDIVC: FX_PLOOP { A[p] = t_rdivc(imm, A[p]); } break;
      case FX_LDM: FX_PLOOP { A[p] = M.ld(aux, p, P); } break;
      case FX_STM: FX_PLOOP { M.st(aux, p, P, A[p]); } break;
      case FX_ADDM: FX_PLOOP { A[p] = t_add(A[p], M.ld(aux, p, P)); } break;
      case FX_SUBM: FX_PLOOP { A[p] = t_sub(A[p], M.ld(aux, p, P)); } break;
      case FX_RSUBM: FX_PLOOP { A[p] = t_sub(M.ld(aux, p, P), A[p]); } break;
      case FX_MULM: FX_PLOOP { A[p] = t_mul(A[p], M.ld(aux, p, P)); } break;
      case FX_DIVM: FX_PLOOP { A[p] = t_div(A[p], M.ld(aux, p, P)); } break;
      case FX_RDIVM: FX_PLOOP { A[p] = t_div(M.ld(aux, p, P), A[p]); } break;
      case FX_FMA_AM_C: FX_PLOOP { A[p] = t_fma_c(A[p], M.ld(aux, p, P), imm); } break;
      case FX_FMA_MC_A: FX_PLOOP { A[p] = t_fma_rc(M.ld(aux, p, P), imm, A[p]); } break;
      case FX_NEG: FX_PLOOP { A[p] = t_neg(A[p]); } break;
      case FX_SQR: FX_PLOOP { A[p] = t_mul(A[p], A[p]); } break;
      case FX_LOG: FX_PLOOP { A[p] = t_log(A[p]); } break;
      case FX_EXP: FX_PLOOP { A[p] = t_exp(A[p]); } break;
      case FX_SQRT: FX_PLOOP { A[p] = t_sqrt(A[p]); } break;
      case FX_OUT: sink(aux, A); break;
      default: return;  // FX_END
    }
  }
}

#endif
