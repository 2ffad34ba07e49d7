// fx_jit.hpp -- native tier of fiesta_compile: fx_ins program -> straight-line PTX spliced into an
// evaluation-kernel template (fx_jit_template*.cu) -> sm_100a cubin (in-process PTX assembler) ->
// one kernel per (sector, mode).  See fx_jit_template.cu for the design.
#ifndef FX_JIT_HPP
#define FX_JIT_HPP

#include <string>
#include <vector>

#include "fx_compiler.hpp"
#include "fx_isa.h"
#include "fx_kernels.h"

namespace fx {

// A sector has up to four native kernels, assembled on demand: one per sampling rule (the FIESTA_RULE_*
// numbers) and one that evaluates the same program body at caller-given points (fiesta_eval_points).
enum JitMode { JIT_LATTICE = 0, JIT_MC = 1, JIT_VEGAS = 2, JIT_EVAL = 3, JIT_NMODES = 4 };

// True when sectors of this kind can run on the native tier (real: dim <= 12; complex: dim <= 8).
bool jit_supported(bool is_complex, int dim);

// Lower the sector's program(s) for `mode` and assemble.  Thread-safe.  Returns false and fills `err`
// on failure (the caller keeps the sector on the interpreter and keeps err).
bool jit_assemble(const CompiledSector &cs, int mode, std::string &cubin, std::string &err);

// The generated PTX alone (tests, disassembly): the .const array of immediates, then the body that
// replaces the FXJIT_BODY marker (for deformed sectors preceded by the gradient/Hessian body).
std::string jit_generated_ptx(const CompiledSector &cs, int mode);

struct JitKernel {
  void *module = nullptr;    // CUmodule
  void *function = nullptr;  // CUfunction
};

// Driver-API side (libcuda is opened with dlopen: the library must load on a box without a GPU).
// The CUDA context of the program's device must be current on the calling thread.
bool jit_load(const std::string &cubin, int mode, size_t max_dynamic_smem, JitKernel &out, std::string &err);
void jit_unload(JitKernel &k);
// grid blocks of FX_THREADS threads; prm by value (the kernel's single parameter, prm_bytes long)
bool jit_launch(const JitKernel &k, unsigned grid, size_t smem, cudaStream_t st, const void *prm, std::string &err);

}  // namespace fx
#endif
