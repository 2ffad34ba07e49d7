// fx_isa.h -- the device instruction set the host compiler emits and the sm_100a interpreter walks.
//
// PAPER.md:108 describes the reference's internal form as "a sequence of quadripples (operator,
// first operand, second operand, result)" walked by "a cycle through all the operations".  That
// three-address form needs an indexable per-point register file, which on a GPU means local or
// shared memory traffic for every operand (PAPER.md:126 keeps the temporaries in GPU memory).
// This ISA is an accumulator machine instead: every operand is named STATICALLY by the opcode, so
// each handler is straight FP64 code on real registers:
//
//   A        accumulator                       (P points per thread, all in registers)
//   R[0..11] = X[i], the integration variables (real x, or complex z after deformation)
//   R[12..19]= S[j], eight register temporaries
//   M[slot]  compiler-directed spill slots in shared memory (dynamic index, rarely used)
//   imm      one FP64 immediate carried in the instruction (always real)
//
// An instruction is 16 bytes so one LDS.128 fetches opcode and immediate together.
#ifndef FX_ISA_H
#define FX_ISA_H

#include <stdint.h>

#define FX_NXMAX 12
#define FX_NS 8
#define FX_NR 20  // FX_NXMAX + FX_NS
#define FX_REG_S(j) (FX_NXMAX + (j))

struct fx_ins {
  uint16_t op;
  uint16_t aux;  // memory slot, or output index
  uint32_t pad;
  double imm;
};

enum fx_op : uint16_t {
  // register families: opcode = base + r, r in [0, FX_NR)
  FX_FMA_AR_C = 0,    // A = A*R[r] + imm
  FX_FMA_RC_A = 20,   // A = R[r]*imm + A
  FX_MUL_R = 40,      // A = A*R[r]
  FX_ADD_R = 60,      // A = A + R[r]
  FX_SUB_R = 80,      // A = A - R[r]
  FX_RSUB_R = 100,    // A = R[r] - A
  FX_LD_R = 120,      // A = R[r]
  FX_MULC_R = 140,    // A = imm*R[r]
  FX_DIV_R = 160,     // A = A / R[r]
  FX_RDIV_R = 180,    // A = R[r] / A
  FX_FMA_AR_M = 200,  // A = A*R[r] + M[aux]
  FX_FMA_AR_S = 220,  // opcode = base + r*8 + j :  A = A*R[r] + S[j]
  FX_ST_S = 380,      // opcode = base + j       :  S[j] = A
  // singles
  FX_LDC = 388,       // A = imm
  FX_ADDC,            // A = A + imm
  FX_MULC,            // A = A * imm
  FX_RSUBC,           // A = imm - A
  FX_DIVC,            // A = A / imm
  FX_RDIVC,           // A = imm / A
  FX_LDM,             // A = M[aux]
  FX_STM,             // M[aux] = A
  FX_ADDM,            // A = A + M
  FX_SUBM,            // A = A - M
  FX_RSUBM,           // A = M - A
  FX_MULM,            // A = A * M
  FX_DIVM,            // A = A / M
  FX_RDIVM,           // A = M / A
  FX_FMA_AM_C,        // A = A*M + imm
  FX_FMA_MC_A,        // A = M*imm + A
  FX_NEG,             // A = -A
  FX_SQR,             // A = A*A
  FX_LOG,             // A = log A   (natural; complex: principal branch)
  FX_EXP,             // A = exp A
  FX_SQRT,            // A = sqrt A  (complex: principal branch)
  FX_OUT,             // output aux (epsilon order index) = A
  FX_END,
  FX_NOPS
};

#endif
