// fx_compiler.hpp -- host compiler: expression text -> fx_ins program.
#ifndef FX_COMPILER_HPP
#define FX_COMPILER_HPP

#include <string>
#include <vector>

#include "../../include/fiesta_b200.h"
#include "fx_isa.h"

namespace fx {

struct CompileError {
  int code;
  std::string msg;
};

struct CompiledSector {
  std::vector<fx_ins> main;    // K outputs through FX_OUT, ends with FX_END
  std::vector<fx_ins> deform;  // gradient/Hessian of F through FX_STM, ends with FX_END; empty if none
  std::vector<fx_ins> testf;   // deformed sectors: complex program with the single output F(z) (PAPER.md:474 -testF)
  int K = 0;
  int dim = 0;
  int sector_id = 0;
  bool is_complex = false;
  bool deform_on = false;
  double lambda = 0.0;
  int n_mem_main = 0;    // M slots (scalars of the program's arithmetic type) of the main program
  int n_mem_deform = 0;  // M slots (doubles) of the deformation program, outputs included
  int n_mem_testf = 0;   // M slots (complex) of the F(z) program
  fiesta_compile_info info{};
};

// Throws CompileError.
CompiledSector compile_sector(const char *const *texts, int K, int dim, bool is_complex, int deform_f_index,
                              double lambda);

std::string disassemble(const std::vector<fx_ins> &prog);

}  // namespace fx
#endif
