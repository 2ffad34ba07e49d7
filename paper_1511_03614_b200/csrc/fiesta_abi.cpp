// fiesta_abi.cpp -- the C ABI of include/fiesta_b200.h: argument checking, launch planning and
// device-buffer management.  All arithmetic of the hot path is in the kernels; this file only
// marshals.  No CPU fallback exists: every entry point that computes needs the sm_100 device.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cmath>
#include <condition_variable>
#include <deque>
#include <memory>
#include <mutex>
#include <thread>
#include <unordered_map>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/fiesta_b200.h"
#include "fx_compiler.hpp"
#include "fx_jit.hpp"
#include "fx_kernels.h"

cudaError_t fx_launch_integrate_real(const fx_integrate_params &prm, int nsectors, cudaStream_t st);
cudaError_t fx_launch_integrate_cplx(const fx_integrate_params &prm, int nsectors, cudaStream_t st);
cudaError_t fx_launch_eval_real(const fx_eval_params &prm, cudaStream_t st);
cudaError_t fx_launch_eval_cplx(const fx_eval_params &prm, cudaStream_t st);
size_t fx_eval_cplx_smem_bytes(const fx_eval_params &prm);
cudaError_t fx_launch_testf_cplx(const fx_integrate_params &prm, int nsectors, cudaStream_t st);

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
  DevBuf<int32_t> sel, maps;
  DevBuf<double> partials, hist_part, sums, grid, hist, iter_stats, scratch_d, scratch_d2;
  DevBuf<uint64_t> scratch_u;
  DevBuf<double> cub_boxes, cub_rec, cub_aux;  // fiesta_integrate_cubature
  DevBuf<unsigned long long> nonfinite;
  DevBuf<fx_result_dev> results;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  // the evaluation kernels of a pass are spread over a few side streams, so that the blocks of the
  // next sector's kernel fill the SMs while the last blocks of the previous one drain
  static constexpr int NAUX = 16;  // run_pass uses 4 for large kernels, more when a sector's grid is small
  cudaStream_t aux[NAUX] = {};
  cudaEvent_t aux_done[NAUX] = {};
  cudaEvent_t fork = nullptr;
  cudaEvent_t reduced[2] = {};  // the chunk reduction of the last batch that used partials buffer 0 / 1
  bool timed = false;
  int n_launches = 0;
  int n_native_sectors = 0, n_interp_sectors = 0;  // of the last call, summed over passes
  int last_nsel = 0, last_dim = 0, last_nbins = 0;
  // geometry of the last single-batch pass (fiesta_chunk_sums)
  int last_nchunks = 0, last_R = 0;
  uint64_t last_chunk = 0;
  double small_x = 0.0;  // fiesta_set_mixed
};

// One native kernel of a sector: assembled by a background thread of the program, used by
// fiesta_integrate once it is READY (until then the sector runs on the interpreter: same sums).
struct NativeSlot {
  enum { NONE = 0, QUEUED = 1, ASSEMBLING = 2, READY = 3, FAILED = 4 };
  std::atomic<int> state{NONE};
  fx::JitKernel k;
  std::string info;  // READY: the assembler's resource report; FAILED: why
};

struct fiesta_program {
  int device = 0;
  int dim = 0;
  std::vector<fx::CompiledSector> host;
  std::vector<fx_sector_dev> sec_host;
  fx_ins *arena = nullptr;
  fx_sector_dev *sectors = nullptr;
  size_t arena_len = 0;
  // native tier (fx_jit): per (sector, mode) one kernel, assembled on demand in the background
  bool jit_on = true;
  size_t smem_optin = 0;
  std::unique_ptr<NativeSlot[]> slots;  // [nsectors][JIT_NMODES]
  NativeSlot &slot(int sector, int mode) const { return slots[(size_t)sector * fx::JIT_NMODES + mode]; }
  std::mutex mu;
  std::condition_variable cv_work, cv_done;
  std::deque<std::pair<int, int>> queue;  // (sector, mode); workers pop from the front
  std::vector<std::thread> workers;
  int pending = 0;  // queued + being assembled
  bool stop = false;
  double assemble_seconds = 0.0;  // summed over worker threads
  int n_assembled = 0, n_cache_hits = 0;
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
  int mode = 0;               // fx::JitMode of the rule
  int batch = 1;              // sectors per batch (run_pass)
  bool allow_native = true;
  bool force_native = false;  // FIESTA_TIER_NATIVE: also for sectors below the work threshold
  double min_work = 0.0;      // points x instructions per sector and pass from which a native launch pays
  bool uniform_K = true;
  bool any_real = false, any_cplx = false;
  int Kmax = 0;
  size_t smem = 0;
  int mem_dd = 0;             // mixed precision: spill doubles per block of the double-double walk
  bool no_mixed = false;      // a caller that never runs phase 2 (fiesta_test_f)
  int shift_first = 0, shift_count = 0;  // lattice: only shifts [first, first + count) of the rule's R (0: all)
};

int ilog2_exact(uint64_t n) {
  if (n == 0 || (n & (n - 1))) return -1;
  int m = 0;
  while ((1ull << m) < n) ++m;
  return m;
}

}  // namespace

size_t fx_integrate_smem_bytes(const fx_integrate_params &prm);

// ------------------------------------------------------------------------------------------------
// native tier: cubin cache and the program's background assembly threads
// ------------------------------------------------------------------------------------------------
namespace {

// Assembled kernels keyed by everything the machine code depends on (the fx_ins programs, K, dim,
// arithmetic type, mode, assembler level) -- NOT by sector id or lambda, which are run-time
// parameters.  Process-wide; with FIESTA_CACHE_DIR set also kept on disk (one file per kernel, the
// full key stored inside and compared on a hit).
struct CubinCache {
  std::mutex mu;
  std::unordered_map<std::string, std::shared_ptr<const std::pair<std::string, std::string>>> map;  // key -> (cubin, info)
};
CubinCache &cubin_cache() {
  static CubinCache c;
  return c;
}

std::string cache_key(const fx::CompiledSector &cs, int mode) {
  std::string k;
  auto put = [&](const void *p, size_t n) { k.append((const char *)p, n); };
  const int32_t hdr[6] = {mode, cs.dim, cs.K, cs.is_complex, cs.deform_on, (int32_t)cs.main.size()};
  put(hdr, sizeof hdr);
  const char *opt = std::getenv("FIESTA_JIT_OPT");
  k.push_back(opt ? opt[0] : '3');
  put(cs.main.data(), cs.main.size() * sizeof(fx_ins));
  put(cs.deform.data(), cs.deform.size() * sizeof(fx_ins));
  return k;
}

std::string cache_file(const std::string &key) {
  const char *dir = std::getenv("FIESTA_CACHE_DIR");
  if (!dir || !dir[0]) return "";
  uint64_t h1 = 1469598103934665603ull, h2 = 0x9E3779B97F4A7C15ull;  // two FNV-1a style hashes -> 128-bit name
  for (unsigned char c : key) {
    h1 = (h1 ^ c) * 1099511628211ull;
    h2 = (h2 + c) * 0xD6E8FEB86659FD93ull;
    h2 ^= h2 >> 29;
  }
  char name[64];
  std::snprintf(name, sizeof name, "/fxj_%016llx%016llx.cubin", (unsigned long long)h1, (unsigned long long)h2);
  return std::string(dir) + name;
}

bool assemble_cached(const fx::CompiledSector &cs, int mode, std::string &cubin, std::string &info, bool &hit) {
  const std::string key = cache_key(cs, mode);
  CubinCache &cc = cubin_cache();
  hit = false;
  {
    std::lock_guard<std::mutex> g(cc.mu);
    auto it = cc.map.find(key);
    if (it != cc.map.end()) {
      cubin = it->second->first;
      info = it->second->second;
      hit = true;
      return true;
    }
  }
  const std::string file = cache_file(key);
  if (!file.empty()) {
    if (FILE *f = std::fopen(file.c_str(), "rb")) {
      uint64_t n[3] = {0, 0, 0};
      std::string k2, inf, cb;
      bool ok = std::fread(n, 8, 3, f) == 3 && n[0] == key.size() && n[1] < (1u << 20) && n[2] < (1u << 28);
      if (ok) {
        k2.resize(n[0]);
        inf.resize(n[1]);
        cb.resize(n[2]);
        ok = std::fread(&k2[0], 1, n[0], f) == n[0] && std::fread(&inf[0], 1, n[1], f) == n[1] &&
             std::fread(&cb[0], 1, n[2], f) == n[2] && k2 == key;
      }
      std::fclose(f);
      if (ok) {
        cubin = cb;
        info = inf;
        hit = true;
      }
    }
  }
  if (!hit) {
    std::string err;
    if (!fx::jit_assemble(cs, mode, cubin, err)) {
      info = err;
      return false;
    }
    info = err;  // on success: the assembler's resource report
    if (!file.empty()) {
      const std::string tmp = file + ".tmp" + std::to_string((unsigned long long)(uintptr_t)&cubin);
      if (FILE *f = std::fopen(tmp.c_str(), "wb")) {
        const uint64_t n[3] = {key.size(), info.size(), cubin.size()};
        std::fwrite(n, 8, 3, f);
        std::fwrite(key.data(), 1, key.size(), f);
        std::fwrite(info.data(), 1, info.size(), f);
        std::fwrite(cubin.data(), 1, cubin.size(), f);
        std::fclose(f);
        std::rename(tmp.c_str(), file.c_str());
      }
    }
  }
  {
    std::lock_guard<std::mutex> g(cc.mu);
    cc.map.emplace(key, std::make_shared<const std::pair<std::string, std::string>>(cubin, info));
  }
  return true;
}

size_t native_smem_max(const fiesta_program *pg, const fx::CompiledSector &cs, int mode) {
  const bool vegas = mode == fx::JIT_VEGAS;
  const size_t want = fxj_layout(cs.dim, FIESTA_MAX_BINS, vegas, fxj_acc_slots(vegas, cs.is_complex, cs.K)).total;
  return mode == fx::JIT_EVAL ? 0 : std::min(want, pg->smem_optin);
}

void native_worker(fiesta_program *pg) {
  cudaSetDevice(pg->device);  // binds the device's primary context: cuModuleLoadData needs one
  cudaFree(nullptr);
  for (;;) {
    std::pair<int, int> job;
    {
      std::unique_lock<std::mutex> lk(pg->mu);
      pg->cv_work.wait(lk, [&] { return pg->stop || !pg->queue.empty(); });
      if (pg->stop) return;
      job = pg->queue.front();
      pg->queue.pop_front();
    }
    NativeSlot &sl = pg->slot(job.first, job.second);
    sl.state.store(NativeSlot::ASSEMBLING);
    const auto t0 = std::chrono::steady_clock::now();
    std::string cubin, info;
    bool hit = false;
    bool ok = assemble_cached(pg->host[job.first], job.second, cubin, info, hit);
    if (ok) {
      std::string err;
      ok = fx::jit_load(cubin, job.second, native_smem_max(pg, pg->host[job.first], job.second), sl.k, err);
      if (!ok) info = err;
    }
    sl.info = info;
    const double dt = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    {
      std::lock_guard<std::mutex> g(pg->mu);
      sl.state.store(ok ? NativeSlot::READY : NativeSlot::FAILED);
      pg->pending--;
      pg->assemble_seconds += dt;
      pg->n_assembled += hit ? 0 : 1;
      pg->n_cache_hits += hit ? 1 : 0;
    }
    pg->cv_done.notify_all();
  }
}

// Queue the kernels of `mode` for the given sectors (those not requested before).  `urgent` puts them
// ahead of everything queued.  The LAST sector of the list is assembled first: fiesta_integrate
// walks its sectors front to back on the interpreter while the kernels arrive from the back.
void native_request(fiesta_program *pg, const int32_t *sectors, int n, int mode, bool urgent) {
  if (!pg->jit_on || pg->workers.empty()) return;
  int added = 0;
  {
    std::lock_guard<std::mutex> g(pg->mu);
    std::vector<std::pair<int, int>> fresh;
    for (int i = 0; i < n; ++i) {
      const int s = sectors ? sectors[i] : i;
      NativeSlot &sl = pg->slot(s, mode);
      if (sl.state.load() != NativeSlot::NONE) continue;
      if (!fx::jit_supported(pg->host[s].is_complex, pg->dim)) {
        sl.info = "";
        sl.state.store(NativeSlot::FAILED);
        continue;
      }
      sl.state.store(NativeSlot::QUEUED);
      fresh.push_back({s, mode});
    }
    added = (int)fresh.size();
    pg->pending += added;
    if (urgent) {
      for (auto &j : fresh) pg->queue.push_front(j);  // the list's last sector ends up first
    } else {
      for (auto it = fresh.rbegin(); it != fresh.rend(); ++it) pg->queue.push_back(*it);
    }
  }
  if (added) pg->cv_work.notify_all();
}

// wait until none of the sectors' `mode` kernels is queued or being assembled; returns how many are READY
int native_wait(fiesta_program *pg, const int32_t *sectors, int n, int mode, double timeout_s) {
  auto settled = [&] {
    for (int i = 0; i < n; ++i) {
      const int st = pg->slot(sectors ? sectors[i] : i, mode).state.load();
      if (st == NativeSlot::QUEUED || st == NativeSlot::ASSEMBLING) return false;
    }
    return true;
  };
  std::unique_lock<std::mutex> lk(pg->mu);
  if (timeout_s < 0) pg->cv_done.wait(lk, settled);
  else pg->cv_done.wait_for(lk, std::chrono::duration<double>(timeout_s), settled);
  int ready = 0;
  for (int i = 0; i < n; ++i) ready += pg->slot(sectors ? sectors[i] : i, mode).state.load() == NativeSlot::READY;
  return ready;
}

}  // namespace

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
  for (int i = 0; i < 2 && aux_ok; ++i) aux_ok = cudaEventCreateWithFlags(&c->reduced[i], cudaEventDisableTiming) == cudaSuccess;
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
  c->maps.release();
  c->partials.release();
  c->hist_part.release();
  c->sums.release();
  c->grid.release();
  c->hist.release();
  c->iter_stats.release();
  c->scratch_d.release();
  c->scratch_d2.release();
  c->scratch_u.release();
  c->cub_boxes.release();
  c->cub_rec.release();
  c->cub_aux.release();
  c->nonfinite.release();
  c->results.release();
  if (c->fork) cudaEventDestroy(c->fork);
  for (int i = 0; i < 2; ++i)
    if (c->reduced[i]) cudaEventDestroy(c->reduced[i]);
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
  pg->smem_optin = ctx->smem_optin;
  std::vector<fx_ins> arena;
  // sectors are independent: parse/optimise them on the host cores in parallel, then lay the
  // programs out in the arena in sector order
  std::vector<fx::CompiledSector> compiled(nsectors);
  // FIESTA_JIT: "0" no native tier; "eager" the lattice kernels of all sectors are queued for assembly
  // here; "sync" the same, and fiesta_compile returns only when they are ready; default: kernels are
  // requested by the first call that can use them (it knows the rule and the number of points)
  const char *jit_env = std::getenv("FIESTA_JIT");
  pg->jit_on = !(jit_env && jit_env[0] == '0');
  const bool jit_sync = jit_env && std::strcmp(jit_env, "sync") == 0;
  const bool jit_eager = jit_sync || (jit_env && std::strcmp(jit_env, "eager") == 0);
  const unsigned ncpu = std::min<unsigned>(std::max(1u, std::thread::hardware_concurrency()), 32u);
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
    const unsigned nthr = std::min<unsigned>(ncpu, (unsigned)((nsectors + 7) / 8));
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
    if (!cs.testf.empty()) {
      sd.testf_off = (uint32_t)arena.size();
      arena.insert(arena.end(), cs.testf.begin(), cs.testf.end());
      arena.push_back(pad);
      sd.testf_len = (uint32_t)cs.testf.size() + 1;
    }
    sd.n_mem_testf = cs.n_mem_testf;
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
  // The interpreter form is ready: the program can be integrated from here on.  Native kernels are
  // assembled by the program's own threads when a call first asks for them (or, FIESTA_JIT=eager,
  // the lattice rule's from now on).
  pg->slots.reset(new NativeSlot[(size_t)nsectors * fx::JIT_NMODES]);
  if (pg->jit_on) {
    const unsigned nw = std::min<unsigned>(ncpu, (unsigned)nsectors);
    for (unsigned t = 0; t < nw; ++t) pg->workers.emplace_back(native_worker, pg);
    if (jit_eager) native_request(pg, nullptr, nsectors, fx::JIT_LATTICE, false);
    if (jit_sync) native_wait(pg, nullptr, nsectors, fx::JIT_LATTICE, -1.0);
  }
  *out = pg;
  return FIESTA_OK;
}

void fiesta_program_free(fiesta_program *pg) {
  if (!pg) return;
  {
    std::lock_guard<std::mutex> g(pg->mu);
    pg->stop = true;
  }
  pg->cv_work.notify_all();
  for (auto &t : pg->workers) t.join();
  cudaSetDevice(pg->device);
  if (pg->arena) cudaFree(pg->arena);
  if (pg->sectors) cudaFree(pg->sectors);
  if (pg->slots)
    for (size_t i = 0; i < pg->host.size() * fx::JIT_NMODES; ++i) fx::jit_unload(pg->slots[i].k);
  delete pg;
}

int fiesta_native_assemble(const fiesta_sector_desc *d, int32_t dim, int32_t mode, char *ptx, uint64_t buflen,
                           uint64_t *cubin_bytes, char *info, uint64_t infolen) {
  if (!d || !d->expr || d->n_orders < 1 || d->n_orders > FIESTA_MAX_ORDERS) return FIESTA_E_ARG;
  if (mode < 0 || mode >= fx::JIT_NMODES) return FIESTA_E_ARG;
  try {
    fx::CompiledSector cs = fx::compile_sector(d->expr, d->n_orders, dim, d->is_complex != 0, d->deform_f_index, d->lambda);
    if (!fx::jit_supported(cs.is_complex, dim)) return FIESTA_E_ARG;
    if (ptx && buflen) std::snprintf(ptx, buflen, "%s", fx::jit_generated_ptx(cs, mode).c_str());
    std::string cubin, err;
    if (!fx::jit_assemble(cs, mode, cubin, err)) {
      if (ptx && buflen) std::snprintf(ptx, buflen, "%s", err.c_str());
      return FIESTA_E_CUDA;
    }
    if (cubin_bytes) *cubin_bytes = cubin.size();
    if (info && infolen) std::snprintf(info, infolen, "%s", err.c_str());
    return FIESTA_OK;
  } catch (fx::CompileError &e) {
    if (ptx && buflen) std::snprintf(ptx, buflen, "%s", e.msg.c_str());
    return e.code;
  }
}

int fiesta_program_native(const fiesta_program *pg, int32_t sector, int32_t mode, char *why, uint64_t buflen) {
  if (!pg || sector < 0 || sector >= (int)pg->host.size() || mode < 0 || mode >= fx::JIT_NMODES) return FIESTA_E_ARG;
  const NativeSlot &sl = pg->slot(sector, mode);
  const int st = sl.state.load();
  if (why && buflen)
    std::snprintf(why, buflen, "%s",
                  st == NativeSlot::READY || st == NativeSlot::FAILED ? sl.info.c_str()
                  : st == NativeSlot::NONE                            ? ""
                                                                      : "being assembled");
  return st == NativeSlot::READY ? 1 : 0;
}

int fiesta_program_wait_native(fiesta_program *pg, int32_t mode, double timeout_s) {
  if (!pg || mode < 0 || mode >= fx::JIT_NMODES) return FIESTA_E_ARG;
  if (!pg->jit_on) return 0;
  native_request(pg, nullptr, (int)pg->host.size(), mode, true);
  return native_wait(pg, nullptr, (int)pg->host.size(), mode, timeout_s);
}

int fiesta_program_native_stats(const fiesta_program *pg, int32_t *n_assembled, int32_t *n_cache_hits,
                                double *assemble_cpu_seconds, int32_t *n_threads) {
  if (!pg) return FIESTA_E_ARG;
  fiesta_program *p = const_cast<fiesta_program *>(pg);
  std::lock_guard<std::mutex> g(p->mu);
  if (n_assembled) *n_assembled = p->n_assembled;
  if (n_cache_hits) *n_cache_hits = p->n_cache_hits;
  if (assemble_cpu_seconds) *assemble_cpu_seconds = p->assemble_seconds;
  if (n_threads) *n_threads = (int)p->workers.size();
  return FIESTA_OK;
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
#include "fiesta_abi_cubature.inc"
#include "fiesta_abi_noalloc.inc"

// ------------------------------------------------------------------------------------------------
// dispatch of the complex kernels, one translation unit per dimension (fx_kernels_cplx.cu -DFX_N=n)
// ------------------------------------------------------------------------------------------------
#define FX_DECL_CPLX(n)                                                                                         \
  cudaError_t fx_launch_testf_cplx_n##n(const fx_integrate_params &prm, int nsectors, size_t smem, cudaStream_t st); \
  cudaError_t fx_launch_integrate_cplx_n##n(const fx_integrate_params &prm, int nsectors, size_t smem, cudaStream_t st); \
  cudaError_t fx_launch_eval_cplx_n##n(const fx_eval_params &prm, size_t smem, cudaStream_t st);
FX_DECL_CPLX(1) FX_DECL_CPLX(2) FX_DECL_CPLX(3) FX_DECL_CPLX(4) FX_DECL_CPLX(5) FX_DECL_CPLX(6) FX_DECL_CPLX(7) FX_DECL_CPLX(8)

size_t fx_eval_cplx_smem_bytes(const fx_eval_params &prm) {
  return (size_t)prm.prog_ins_max * 16 + (size_t)prm.mem_doubles * 8;
}

cudaError_t fx_launch_integrate_cplx(const fx_integrate_params &prm, int nsectors, cudaStream_t st) {
  const size_t smem = fx_integrate_cplx_smem_bytes(prm);
  switch (prm.dim) {
#define FX_CASE(n) case n: return fx_launch_integrate_cplx_n##n(prm, nsectors, smem, st);
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

cudaError_t fx_launch_testf_cplx(const fx_integrate_params &prm, int nsectors, cudaStream_t st) {
  const size_t smem = fx_integrate_smem_bytes(prm);
  switch (prm.dim) {
#define FX_CASE(n) case n: return fx_launch_testf_cplx_n##n(prm, nsectors, smem, st);
    FX_CASE(1) FX_CASE(2) FX_CASE(3) FX_CASE(4) FX_CASE(5) FX_CASE(6) FX_CASE(7) FX_CASE(8)
#undef FX_CASE
  }
  return cudaErrorInvalidValue;
}
