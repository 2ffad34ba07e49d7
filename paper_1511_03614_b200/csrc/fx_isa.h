// fx_isa.h -- the device instruction set the host compiler emits and the sm_100a interpreter walks.
//
// PAPER.md:108 describes the reference's internal form as "a sequence of quadripples (operator,
// first operand, second operand, result)" walked by "a cycle through all the operations".  That
// three-address form needs an indexable per-point register file, which on a GPU means local or
// shared memory traffic for every operand (PAPER.md:126 keeps the temporaries in GPU memory).
// This ISA names every operand STATICALLY in the opcode, so each handler is straight FP64 code on
// physical registers:
//
//   A[0..L)  a small stack of accumulators ("levels").  Nested Horner evaluation of a sparse
//            polynomial p = q*v + r puts r in A[d], q in A[d+1] and folds with one FMA_UP; no
//            store/reload instructions are spent on temporaries.  Level 0 is "the" accumulator
//            of every non-polynomial operation.
//   R[0..11] = X[i], the integration variables (real x, or complex z after deformation)
//   R[12..]  = S[j], FX_NS register temporaries for values used more than once
//   M[slot]  compiler-directed slots in shared memory (dynamic index; overflow of S)
//   imm      one FP64 immediate carried in the instruction (always real)
//
// P points per thread share one instruction fetch and dispatch.  An instruction is 16 bytes so
// one LDS.128 fetches opcode and immediate together.
#ifndef FX_ISA_H
#define FX_ISA_H

#include <stdint.h>

#define FX_NXMAX 12
#define FX_NS 1
#define FX_NR (FX_NXMAX + FX_NS)
#define FX_L 3  // accumulator levels
#define FX_REG_S(j) (FX_NXMAX + (j))
#define FX_LR (FX_L * FX_NR)  // opcodes of one (level, register) family

struct fx_ins {
  uint16_t op;
  uint16_t aux;  // memory slot, or output index
  uint32_t pad;
  double imm;
};

// (level, register) families: opcode = base + d*FX_NR + r
// level families:             opcode = base + d
// level-0 register families:  opcode = base + r
enum fx_op : uint16_t {
  FX_MULC_R = 0,                      // A[d] = imm*R[r]
  FX_MUL_R = FX_MULC_R + FX_LR,       // A[d] = A[d]*R[r]
  FX_FMA_AR_C = FX_MUL_R + FX_LR,     // A[d] = A[d]*R[r] + imm
  FX_FMA_RC_A = FX_FMA_AR_C + FX_LR,  // A[d] = R[r]*imm + A[d]
  FX_FMA_UP = FX_FMA_RC_A + FX_LR,    // A[d] = A[d+1]*R[r] + A[d]        (d < L-1)
  FX_ADD_R = FX_FMA_UP + FX_LR,       // A[d] = A[d] + R[r]
  FX_LD_R = FX_ADD_R + FX_LR,         // A[d] = R[r]
  FX_FMA_AR_M = FX_LD_R + FX_LR,      // A[d] = A[d]*R[r] + M[aux]
  // level families
  FX_LDC = FX_FMA_AR_M + FX_LR,       // A[d] = imm
  FX_ADDC = FX_LDC + FX_L,            // A[d] = A[d] + imm
  FX_MULC = FX_ADDC + FX_L,           // A[d] = A[d]*imm
  FX_ADD_UP = FX_MULC + FX_L,         // A[d] = A[d] + A[d+1]
  FX_MUL_UP = FX_ADD_UP + FX_L,       // A[d] = A[d]*A[d+1]
  FX_LDM = FX_MUL_UP + FX_L,          // A[d] = M[aux]
  FX_STM = FX_LDM + FX_L,             // M[aux] = A[d]
  FX_ADDM = FX_STM + FX_L,            // A[d] = A[d] + M[aux]
  FX_MULM = FX_ADDM + FX_L,           // A[d] = A[d]*M[aux]
  FX_FMA_MC_A = FX_MULM + FX_L,       // A[d] = M[aux]*imm + A[d]
  FX_FMA_AM_C = FX_FMA_MC_A + FX_L,   // A[d] = A[d]*M[aux] + imm
  FX_FMA_UPC = FX_FMA_AM_C + FX_L,    // A[d] = A[d+1]*imm + A[d]         (d < L-1)
  // level-0 register families
  FX_SUB_R = FX_FMA_UPC + FX_L,       // A = A - R[r]
  FX_RSUB_R = FX_SUB_R + FX_NR,       // A = R[r] - A
  FX_DIV_R = FX_RSUB_R + FX_NR,       // A = A / R[r]
  FX_RDIV_R = FX_DIV_R + FX_NR,       // A = R[r] / A
  FX_ST_S = FX_RDIV_R + FX_NR,        // opcode = base + j : S[j] = A
  // level-0 singles
  FX_RSUBC = FX_ST_S + FX_NS,         // A = imm - A
  FX_DIVC,                            // A = A / imm
  FX_RDIVC,                           // A = imm / A
  FX_SUBM,                            // A = A - M
  FX_RSUBM,                           // A = M - A
  FX_DIVM,                            // A = A / M
  FX_RDIVM,                           // A = M / A
  FX_NEG,                             // A = -A
  FX_SQR,                             // A = A*A
  FX_LOG,                             // A = log A   (natural; complex: principal branch)
  FX_EXP,                             // A = exp A
  FX_SQRT,                            // A = sqrt A  (complex: principal branch)
  FX_OUT,                             // output aux (epsilon order index) = A
  FX_END,
  FX_NOPS
};

#endif
