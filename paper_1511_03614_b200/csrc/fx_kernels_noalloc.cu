// fx_kernels_noalloc.cu -- per-shift sums of one real sector WITHOUT any device allocation.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
// harnesses that forbid it).  The integrate family keeps its per-block partial records, the
// selection and the non-finite counter in scratch buffers that the context grows with cudaMalloc
// on demand (fiesta_abi.cpp, DevBuf).  Here the same scratch is ONE file-scope device array of a
// fixed size, which every GPU that loads the library holds until the process exits:
//
//     FX_NOALLOC_MAX_BLOCKS = 4096 partial records of 32 doubles + a 256-byte header = 1 MiB + 256 B.
//
// A call covers one real sector under the lattice or the plain-MC rule with at most 4096 blocks
// (= shifts x chunks; a chunk is at most 2^17 points, so up to 2^29 points per call).  The
// evaluation kernel is the interpreter's (fx_launch_integrate_real), given the ADDRESS of the
// array; the second level of the reduction is a variant of k_reduce_chunks (fx_kernels_small.cu)
// that names the array directly and writes to the caller's device buffers.  Same chunking, same
// order of additions: the sums are the bits fiesta_partial_sums returns.
//
// In host code `fx_noalloc_scratch` is a host-side stand-in for the symbol, not a device address: a
// kernel given it would fault (or, where the GPU can reach host memory, silently use the wrong
// memory).  The address comes from cudaGetSymbolAddress, once per device with that device current
// (fx_noalloc_address below); device code in this file names the array directly.
//
// Every call shares the array, and the array keeps the last call's contents.  Nothing in it has to
// start at zero except the non-finite counter, which k_noalloc_prepare clears (every block writes all
// 32 slots of its record, and the reduction reads only the records of this call).  Two calls that
// overlap on the GPU (different streams, different contexts on one device) RACE on it: callers
// serialise them.
#include <mutex>

#include "../../include/fiesta_b200.h"
#include "fx_kernels.h"

cudaError_t fx_launch_integrate_real(const fx_integrate_params &prm, int nsectors, cudaStream_t st);

#define FX_NOALLOC_MAX_BLOCKS 4096
#define FX_NOALLOC_HEADER 32  // doubles behind the records: [0] non-finite counter, [1] the selected sector index

static __device__ __align__(256) double fx_noalloc_scratch[(size_t)FX_NOALLOC_MAX_BLOCKS * FX_ACC_SLOTS + FX_NOALLOC_HEADER];

namespace {

constexpr size_t kRecords = (size_t)FX_NOALLOC_MAX_BLOCKS * FX_ACC_SLOTS;

// what must not be stale: the counter the evaluation kernel adds to, and which sector it works on
__global__ void k_noalloc_prepare(int32_t sector) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    *reinterpret_cast<unsigned long long *>(fx_noalloc_scratch + kRecords) = 0ull;
    *reinterpret_cast<int32_t *>(fx_noalloc_scratch + kRecords + 1) = sector;
  }
}

// k_reduce_chunks on the static records: sums_out[row][slot < nslots] = sum over the row's chunks, in chunk order
__global__ void k_noalloc_reduce(int nrows, int nchunks, int nslots, double *sums_out, unsigned long long *nonfinite_out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;  // row*nslots + slot
  if (i == 0 && nonfinite_out) *nonfinite_out = *reinterpret_cast<const unsigned long long *>(fx_noalloc_scratch + kRecords);
  if (i >= nrows * nslots) return;
  const int row = i / nslots, slot = i % nslots;
  double s = 0.0;
  for (int c = 0; c < nchunks; ++c) s += fx_noalloc_scratch[((size_t)row * nchunks + c) * FX_ACC_SLOTS + slot];
  sums_out[i] = s;
}

constexpr int kMaxDevices = 64;
std::mutex g_mu;
double *g_address[kMaxDevices] = {};

}  // namespace

int fx_noalloc_max_blocks() { return FX_NOALLOC_MAX_BLOCKS; }

// The device address of the scratch array on `device` (which must be current): resolved once per device.
cudaError_t fx_noalloc_address(int device, double **out) {
  if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> g(g_mu);
  if (!g_address[device]) {
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, fx_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_address[device] = static_cast<double *>(p);
  }
  *out = g_address[device];
  return cudaSuccess;
}

// prm: a planned pass (fiesta_abi_integrate.inc make_plan) over ONE real sector; its partials / sel / nonfinite /
// launch_map fields are set here.  sums_dev[n_shifts][2K], nonfinite_dev (may be NULL): the caller's device memory.
cudaError_t fx_noalloc_partial_sums(fx_integrate_params prm, int device, int32_t sector, int K, double *sums_dev,
                                    unsigned long long *nonfinite_dev, cudaStream_t st) {
  double *scratch = nullptr;
  cudaError_t e = fx_noalloc_address(device, &scratch);
  if (e != cudaSuccess) return e;
  prm.partials = scratch;
  prm.nonfinite = reinterpret_cast<unsigned long long *>(scratch + kRecords);
  prm.sel = reinterpret_cast<const int32_t *>(scratch + kRecords + 1);
  prm.nsel = 1;
  prm.launch_map = nullptr;
  prm.sel_base = 0;
  prm.batch_base = 0;
  prm.hist_part = nullptr;
  prm.grid = nullptr;
  prm.testf_out = nullptr;
  prm.lambda_override = -1.0;
  k_noalloc_prepare<<<1, 32, 0, st>>>(sector);
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  if ((e = fx_launch_integrate_real(prm, 1, st)) != cudaSuccess) return e;
  const int nslots = 2 * K, total = prm.n_shifts * nslots;
  k_noalloc_reduce<<<(total + 127) / 128, 128, 0, st>>>(prm.n_shifts, prm.nchunks, nslots, sums_dev, nonfinite_dev);
  return cudaGetLastError();
}
