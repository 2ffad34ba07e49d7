// fx_jit.hpp -- native tier of fiesta_compile: fx_ins program -> straight-line PTX spliced into the
// evaluation-kernel template (fx_jit_template.cu) -> sm_100a cubin (in-process PTX assembler) ->
// one kernel per sector.  See fx_jit_template.cu for the design.
#ifndef FX_JIT_HPP
#define FX_JIT_HPP

#include <string>
#include <vector>

#include "fx_isa.h"
#include "fx_kernels.h"

namespace fx {

// True when this program can run on the native tier (real arithmetic, dim <= 12).
bool jit_supported(bool is_complex, int dim);

// Lower `prog` (main program of a real sector, K outputs) and assemble.  Thread-safe.
// Returns false and fills `err` on failure (the caller falls back to the interpreter and keeps err).
bool jit_assemble(const std::vector<fx_ins> &prog, int dim, int K, std::string &cubin, std::string &err);

// The PTX text of the program body alone (tests, disassembly).
std::string jit_body_ptx(const std::vector<fx_ins> &prog, int K, const std::vector<std::string> &operands,
                         std::string *const_decl = nullptr);

struct JitKernel {
  void *module = nullptr;    // CUmodule
  void *function = nullptr;  // CUfunction
};

// Driver-API side (libcuda is opened with dlopen: the library must load on a box without a GPU).
bool jit_load(const std::string &cubin, size_t max_dynamic_smem, JitKernel &out, std::string &err);
void jit_unload(JitKernel &k);
// grid blocks of FX_THREADS threads, prm by value (the kernel's single parameter)
bool jit_launch(const JitKernel &k, unsigned grid, size_t smem, cudaStream_t st, const fx_integrate_params &prm,
                std::string &err);

}  // namespace fx
#endif
