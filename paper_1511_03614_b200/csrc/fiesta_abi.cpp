// fiesta_abi.cpp -- the C ABI of include/fiesta_b200.h: argument checking, launch planning and
// device-buffer management.  All arithmetic of the hot path is in the kernels; this file only
// marshals.  No CPU fallback exists: every entry point that computes needs the sm_100 device.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <mutex>
#include <thread>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/fiesta_b200.h"
#include "fx_compiler.hpp"
#include "fx_jit.hpp"
#include "fx_kernels.h"

cudaError_t fx_launch_integrate_real(const fx_integrate_params &prm, cudaStream_t st);
cudaError_t fx_launch_integrate_cplx(const fx_integrate_params &prm, cudaStream_t st);
cudaError_t fx_launch_eval_real(const fx_eval_params &prm, cudaStream_t st);
cudaError_t fx_launch_eval_cplx(const fx_eval_params &prm, cudaStream_t st);
size_t fx_eval_cplx_smem_bytes(const fx_eval_params &prm);

namespace {

template <typename T>
struct DevBuf {  // grow-only device scratch
  T *p = nullptr;
  size_t cap = 0;
  cudaError_t reserve(size_t n) {
    if (n <= cap) return cudaSuccess;
    if (p) cudaFree(p);
    p = nullptr;
    cap = 0;
    cudaError_t e = cudaMalloc((void **)&p, std::max<size_t>(n, 1) * sizeof(T));
    if (e == cudaSuccess) cap = n;
    return e;
  }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
    cap = 0;
  }
};

}  // namespace

struct fiesta_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  std::string err;
  int sm_count = 148;
  size_t smem_optin = 0;
  DevBuf<int32_t> sel;
  DevBuf<double> partials, sums, grid, hist, iter_stats, scratch_d, scratch_d2;
  DevBuf<uint64_t> scratch_u;
  DevBuf<unsigned long long> nonfinite;
  DevBuf<fx_result_dev> results;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  // native per-sector kernels are spread over a few side streams, so that the blocks of the next
  // sector's kernel fill the SMs while the last blocks of the previous one drain
  static constexpr int NAUX = 4;
  cudaStream_t aux[NAUX] = {};
  cudaEvent_t aux_done[NAUX] = {};
  cudaEvent_t fork = nullptr;
  bool timed = false;
  int n_launches = 0;
  int last_nsel = 0, last_dim = 0, last_nbins = 0;
};

struct fiesta_program {
  int device = 0;
  int dim = 0;
  std::vector<fx::CompiledSector> host;
  std::vector<fx_sector_dev> sec_host;
  fx_ins *arena = nullptr;
  fx_sector_dev *sectors = nullptr;
  size_t arena_len = 0;
  // native tier (fx_jit): one assembled kernel per real sector; function == nullptr -> interpreter
  std::vector<fx::JitKernel> jit;
  std::vector<std::string> jit_err;  // why a sector has no native kernel ("" if it has one or JIT is off)
};

namespace {

int fail(fiesta_ctx *ctx, int code, const std::string &msg) {
  if (ctx) ctx->err = msg;
  return code;
}
int cuda_fail(fiesta_ctx *ctx, cudaError_t e, const char *what) {
  return fail(ctx, FIESTA_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define FX_CUDA(ctx, call)                                      \
  do {                                                          \
    cudaError_t e_ = (call);                                    \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);    \
  } while (0)

fx_transform_host make_transform(int r) {
  fx_transform_host tf{};
  tf.r = r;
  auto fact = [](int n) {
    double f = 1.0;
    for (int i = 2; i <= n; ++i) f *= i;
    return f;
  };
  const double c = fact(2 * r + 1) / (fact(r) * fact(r));  // exact in FP64 for r <= 6
  tf.cw = c;
  for (int i = 0; i <= r && i < 7; ++i) {
    double binom = fact(r) / (fact(i) * fact(r - i));
    tf.coef[i] = c * binom * ((i & 1) ? -1.0 : 1.0) / (double)(r + 1 + i);
  }
  return tf;
}

struct Plan {
  fx_integrate_params prm{};
  const fiesta_program *pg = nullptr;
  std::vector<int32_t> selv;  // selected sector indices (host copy)
  bool native = false;        // every selected sector is real and has a native kernel, rule = lattice
  bool any_real = false, any_cplx = false;
  int Kmax = 0;
  size_t smem = 0;
};

int ilog2_exact(uint64_t n) {
  if (n == 0 || (n & (n - 1))) return -1;
  int m = 0;
  while ((1ull << m) < n) ++m;
  return m;
}

}  // namespace

size_t fx_integrate_smem_bytes(const fx_integrate_params &prm);

extern "C" {

int fiesta_create(fiesta_ctx **out, int cuda_device, void *cuda_stream) {
  if (!out) return FIESTA_E_ARG;
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return FIESTA_E_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return FIESTA_E_CUDA;
  if (prop.major != 10) return FIESTA_E_CUDA;  // kernels are built for sm_100a only; no fallback
  if (cudaSetDevice(cuda_device) != cudaSuccess) return FIESTA_E_CUDA;
  fiesta_ctx *c = new fiesta_ctx;
  c->device = cuda_device;
  c->stream = (cudaStream_t)cuda_stream;
  c->sm_count = prop.multiProcessorCount;
  c->smem_optin = prop.sharedMemPerBlockOptin;
  bool aux_ok = cudaEventCreateWithFlags(&c->fork, cudaEventDisableTiming) == cudaSuccess;
  for (int i = 0; i < fiesta_ctx::NAUX && aux_ok; ++i)
    aux_ok = cudaStreamCreateWithFlags(&c->aux[i], cudaStreamNonBlocking) == cudaSuccess &&
             cudaEventCreateWithFlags(&c->aux_done[i], cudaEventDisableTiming) == cudaSuccess;
  if (!aux_ok || cudaEventCreate(&c->ev0) != cudaSuccess || cudaEventCreate(&c->ev1) != cudaSuccess) {
    delete c;
    return FIESTA_E_CUDA;
  }
  *out = c;
  return FIESTA_OK;
}

void fiesta_destroy(fiesta_ctx *c) {
  if (!c) return;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  c->sel.release();
  c->partials.release();
  c->sums.release();
  c->grid.release();
  c->hist.release();
  c->iter_stats.release();
  c->scratch_d.release();
  c->scratch_d2.release();
  c->scratch_u.release();
  c->nonfinite.release();
  c->results.release();
  if (c->fork) cudaEventDestroy(c->fork);
  for (int i = 0; i < fiesta_ctx::NAUX; ++i) {
    if (c->aux_done[i]) cudaEventDestroy(c->aux_done[i]);
    if (c->aux[i]) cudaStreamDestroy(c->aux[i]);
  }
  if (c->ev0) cudaEventDestroy(c->ev0);
  if (c->ev1) cudaEventDestroy(c->ev1);
  delete c;
}

const char *fiesta_last_error(const fiesta_ctx *c) { return c ? c->err.c_str() : "null context"; }

int fiesta_compile(fiesta_ctx *ctx, const fiesta_sector_desc *sectors, int32_t nsectors, int32_t dim,
                   fiesta_program **out, fiesta_compile_info *info) {
  if (!ctx || !out) return FIESTA_E_ARG;
  *out = nullptr;
  if (!sectors || nsectors < 1) return fail(ctx, FIESTA_E_ARG, "need at least one sector");
  fiesta_program *pg = new fiesta_program;
  pg->device = ctx->device;
  pg->dim = dim;
  std::vector<fx_ins> arena;
  // sectors are independent: parse/optimise them on the host cores in parallel, then lay the
  // programs out in the arena in sector order
  std::vector<fx::CompiledSector> compiled(nsectors);
  // FIESTA_JIT=0 keeps every sector on the interpreter (tests compare the two tiers)
  const char *jit_env = std::getenv("FIESTA_JIT");
  const bool jit_on = !(jit_env && jit_env[0] == '0');
  std::vector<std::string> cubins(nsectors);
  pg->jit.resize(nsectors);
  pg->jit_err.assign(nsectors, "");
  {
    std::atomic<int> next{0};
    std::mutex err_mu;
    int err_sector = nsectors;
    fx::CompileError err{0, ""};
    auto worker = [&]() {
      for (;;) {
        const int s = next.fetch_add(1);
        if (s >= nsectors) return;
        const fiesta_sector_desc &d = sectors[s];
        try {
          if (!d.expr || d.n_orders < 1 || d.n_orders > FIESTA_MAX_ORDERS)
            throw fx::CompileError{FIESTA_E_ARG, "n_orders must be in 1..8 and expr non-NULL"};
          compiled[s] = fx::compile_sector(d.expr, d.n_orders, dim, d.is_complex != 0, d.deform_f_index, d.lambda);
          compiled[s].sector_id = d.sector_id;
          const fx::CompiledSector &cs = compiled[s];
          if (jit_on && fx::jit_supported(cs.is_complex || cs.deform_on, dim))
            if (!fx::jit_assemble(cs.main, dim, cs.K, cubins[s], pg->jit_err[s])) cubins[s].clear();
        } catch (fx::CompileError &e) {
          std::lock_guard<std::mutex> g(err_mu);
          if (s < err_sector) {
            err_sector = s;
            err = e;
            err.msg = "sector " + std::to_string(s) + " (id " + std::to_string(d.sector_id) + "), " + e.msg;
          }
        } catch (std::exception &e) {
          std::lock_guard<std::mutex> g(err_mu);
          if (s < err_sector) {
            err_sector = s;
            err = fx::CompileError{FIESTA_E_ARG, std::string("sector ") + std::to_string(s) + ": " + e.what()};
          }
        }
      }
    };
    unsigned nthr = std::min<unsigned>(std::max(1u, std::thread::hardware_concurrency()), 32u);
    nthr = std::min<unsigned>(nthr, (unsigned)(jit_on ? nsectors : (nsectors + 7) / 8));
    if (nthr <= 1) {
      worker();
    } else {
      std::vector<std::thread> pool;
      for (unsigned t = 0; t < nthr; ++t) pool.emplace_back(worker);
      for (auto &t : pool) t.join();
    }
    if (err_sector < nsectors) {
      delete pg;
      return fail(ctx, err.code, err.msg);
    }
  }
  for (int s = 0; s < nsectors; ++s) {
    fx::CompiledSector &cs = compiled[s];
    fx_sector_dev sd{};
    fx_ins pad{};
    pad.op = FX_END;
    sd.main_off = (uint32_t)arena.size();
    arena.insert(arena.end(), cs.main.begin(), cs.main.end());
    arena.push_back(pad);
    sd.main_len = (uint32_t)cs.main.size() + 1;
    if (!cs.deform.empty()) {
      sd.deform_off = (uint32_t)arena.size();
      arena.insert(arena.end(), cs.deform.begin(), cs.deform.end());
      arena.push_back(pad);
      sd.deform_len = (uint32_t)cs.deform.size() + 1;
    }
    sd.K = cs.K;
    sd.is_complex = cs.is_complex ? 1 : 0;
    sd.sector_id = cs.sector_id;
    sd.n_mem_main = cs.n_mem_main;
    sd.n_mem_deform = cs.n_mem_deform;
    sd.lambda = cs.lambda;
    if (info) info[s] = cs.info;
    pg->sec_host.push_back(sd);
    pg->host.push_back(std::move(cs));
  }
  cudaSetDevice(ctx->device);
  pg->arena_len = arena.size();
  cudaError_t e = cudaMalloc((void **)&pg->arena, arena.size() * sizeof(fx_ins));
  if (e == cudaSuccess) e = cudaMalloc((void **)&pg->sectors, pg->sec_host.size() * sizeof(fx_sector_dev));
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(pg->arena, arena.data(), arena.size() * sizeof(fx_ins), cudaMemcpyHostToDevice, ctx->stream);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(pg->sectors, pg->sec_host.data(), pg->sec_host.size() * sizeof(fx_sector_dev),
                        cudaMemcpyHostToDevice, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) {
    fiesta_program_free(pg);
    return cuda_fail(ctx, e, "program upload");
  }
  {
    const size_t smem = fx_integrate_smem_bytes_native(dim);
    for (int s = 0; s < nsectors; ++s)
      if (!cubins[s].empty() && !fx::jit_load(cubins[s], smem, pg->jit[s], pg->jit_err[s])) pg->jit[s] = fx::JitKernel{};
  }
  *out = pg;
  return FIESTA_OK;
}

void fiesta_program_free(fiesta_program *pg) {
  if (!pg) return;
  cudaSetDevice(pg->device);
  if (pg->arena) cudaFree(pg->arena);
  if (pg->sectors) cudaFree(pg->sectors);
  for (fx::JitKernel &k : pg->jit) fx::jit_unload(k);
  delete pg;
}

int fiesta_native_assemble(const fiesta_sector_desc *d, int32_t dim, char *ptx, uint64_t buflen, uint64_t *cubin_bytes) {
  if (!d || !d->expr || d->n_orders < 1 || d->n_orders > FIESTA_MAX_ORDERS) return FIESTA_E_ARG;
  if (d->is_complex || d->deform_f_index > 0 || !fx::jit_supported(false, dim)) return FIESTA_E_ARG;
  try {
    const fx::CompiledSector cs = fx::compile_sector(d->expr, d->n_orders, dim, false, 0, 0.0);
    std::vector<std::string> operands = {"%nonfinite", "%valid", "%acc"};
    for (int p = 0; p < FXJ_P; ++p) operands.push_back("%W" + std::to_string(p));
    const int nx = dim <= 4 ? 4 : dim <= 8 ? 8 : 12;
    for (int k = 0; k < nx; ++k)
      for (int p = 0; p < FXJ_P; ++p) operands.push_back("%x" + std::to_string(k) + "_" + std::to_string(p));
    if (ptx && buflen) {
      std::string decl;
      const std::string body = fx::jit_body_ptx(cs.main, cs.K, operands, &decl);
      std::snprintf(ptx, buflen, "%s%s", decl.c_str(), body.c_str());  // the immediates' .const array, then the body
    }
    std::string cubin, err;
    if (!fx::jit_assemble(cs.main, dim, cs.K, cubin, err)) {
      if (ptx && buflen) std::snprintf(ptx, buflen, "%s", err.c_str());
      return FIESTA_E_CUDA;
    }
    if (cubin_bytes) *cubin_bytes = cubin.size();
    return FIESTA_OK;
  } catch (fx::CompileError &e) {
    if (ptx && buflen) std::snprintf(ptx, buflen, "%s", e.msg.c_str());
    return e.code;
  }
}

int fiesta_program_native(const fiesta_program *pg, int32_t sector, char *why, uint64_t buflen) {
  if (!pg || sector < 0 || sector >= (int)pg->host.size()) return FIESTA_E_ARG;
  if (why && buflen) std::snprintf(why, buflen, "%s", pg->jit_err[sector].c_str());
  return pg->jit[sector].function ? 1 : 0;
}

int fiesta_program_dump(const fiesta_program *pg, int32_t sector, char *buf, uint64_t buflen) {
  if (!pg || !buf || buflen == 0 || sector < 0 || sector >= (int)pg->host.size()) return FIESTA_E_ARG;
  std::string s = "main:\n" + fx::disassemble(pg->host[sector].main);
  if (!pg->host[sector].deform.empty()) s += "deform:\n" + fx::disassemble(pg->host[sector].deform);
  std::snprintf(buf, buflen, "%s", s.c_str());
  return FIESTA_OK;
}

int fiesta_combine(const fiesta_result *per_sector, int32_t nsectors, int32_t K, fiesta_result *total) {
  if (!per_sector || !total || nsectors < 0 || K < 1) return FIESTA_E_ARG;
  for (int k = 0; k < K; ++k) {
    fiesta_result t{};
    double vr = 0.0, vi = 0.0;
    for (int s = 0; s < nsectors; ++s) {
      const fiesta_result &r = per_sector[(size_t)s * K + k];
      t.re += r.re;
      t.im += r.im;
      vr += r.re_err * r.re_err;
      vi += r.im_err * r.im_err;
      t.chi2 += r.chi2;
      t.neval += r.neval;
      t.n_nonfinite += r.n_nonfinite;
    }
    t.re_err = std::sqrt(vr);
    t.im_err = std::sqrt(vi);
    total[k] = t;
  }
  return FIESTA_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// planning and the integrate family (second half of this file)
// ------------------------------------------------------------------------------------------------
#include "fiesta_abi_integrate.inc"

// ------------------------------------------------------------------------------------------------
// dispatch of the complex kernels, one translation unit per dimension (fx_kernels_cplx.cu -DFX_N=n)
// ------------------------------------------------------------------------------------------------
#define FX_DECL_CPLX(n)                                                                                         \
  cudaError_t fx_launch_integrate_cplx_n##n(const fx_integrate_params &prm, size_t smem, cudaStream_t st);     \
  cudaError_t fx_launch_eval_cplx_n##n(const fx_eval_params &prm, size_t smem, cudaStream_t st);
FX_DECL_CPLX(1) FX_DECL_CPLX(2) FX_DECL_CPLX(3) FX_DECL_CPLX(4) FX_DECL_CPLX(5) FX_DECL_CPLX(6) FX_DECL_CPLX(7) FX_DECL_CPLX(8)

size_t fx_eval_cplx_smem_bytes(const fx_eval_params &prm) {
  return (size_t)prm.prog_ins_max * 16 + (size_t)prm.mem_doubles * 8;
}

cudaError_t fx_launch_integrate_cplx(const fx_integrate_params &prm, cudaStream_t st) {
  const size_t smem = fx_integrate_smem_bytes(prm);
  switch (prm.dim) {
#define FX_CASE(n) case n: return fx_launch_integrate_cplx_n##n(prm, smem, st);
    FX_CASE(1) FX_CASE(2) FX_CASE(3) FX_CASE(4) FX_CASE(5) FX_CASE(6) FX_CASE(7) FX_CASE(8)
#undef FX_CASE
  }
  return cudaErrorInvalidValue;
}

cudaError_t fx_launch_eval_cplx(const fx_eval_params &prm, cudaStream_t st) {
  const size_t smem = fx_eval_cplx_smem_bytes(prm);
  switch (prm.dim) {
#define FX_CASE(n) case n: return fx_launch_eval_cplx_n##n(prm, smem, st);
    FX_CASE(1) FX_CASE(2) FX_CASE(3) FX_CASE(4) FX_CASE(5) FX_CASE(6) FX_CASE(7) FX_CASE(8)
#undef FX_CASE
  }
  return cudaErrorInvalidValue;
}
