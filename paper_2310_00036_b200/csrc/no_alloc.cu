// cb_permutation_static: the PPO minibatch permutation (A17, cleanba.h) for callers that may not allocate -- code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc.  cb_permutation allocates its Fisher-Yates draw buffer per call
// (cudaMallocAsync) and cb_permutation_ws takes it from the caller; here the buffer is a file-scope device array, so the call
// allocates nothing and the caller passes only the output.
//
// Cost and limits: CB_PERM_STATIC_MAX draws = 256 KiB of device memory held, until exit, by every GPU that loads the library.
// Every call on a device shares the one array: calls that overlap on the GPU (different streams, or graphs replayed concurrently)
// race on it; calls ordered on one stream do not.  Nothing has to start at zero: the kernel writes every draw jb[q], q < N - 1,
// before its swap loop reads it (rl.cu, permutation_kernel), so what the last call left behind is never read.
#include "common.cuh"

#include <mutex>

namespace cb {

static __device__ __align__(256) uint32_t g_perm_draws[CB_PERM_STATIC_MAX];

// In host code `g_perm_draws` is the host-side stand-in of the symbol, not a device address: the address a kernel may be given
// comes from cudaGetSymbolAddress, resolved once per device with that device current.
static int perm_draws_address(uint32_t** out) {
  constexpr int MAX_DEV = 64;
  static std::mutex mu; static uint32_t* addr[MAX_DEV];
  int dev = 0; CB_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEV) { set_error("cb_permutation_static: device ordinal %d out of range", dev); return CB_EINVAL; }
  std::lock_guard<std::mutex> lk(mu);
  if (!addr[dev]) {
    uint32_t* p = nullptr;
    CB_CUDA(cudaGetSymbolAddress((void**)&p, g_perm_draws));
    addr[dev] = p;
  }
  *out = addr[dev];
  return CB_OK;
}

}  // namespace cb

using namespace cb;

extern "C" int cb_permutation_static(uint64_t seed, uint32_t epoch, int N, int32_t* perm, void* stream) {
  if (N < 0 || (!perm && N > 0)) { set_error("bad argument"); return CB_EINVAL; }
  if (N > CB_PERM_STATIC_MAX) {
    set_error("cb_permutation_static: N = %d exceeds the static scratch (CB_PERM_STATIC_MAX = %d); use cb_permutation_ws", N, CB_PERM_STATIC_MAX);
    return CB_EINVAL;
  }
  if (N == 0) return CB_OK;
  uint32_t* draws = nullptr;
  { int rc = perm_draws_address(&draws); if (rc) return rc; }
  return launch_permutation(seed, epoch, 1, N, perm, draws, (cudaStream_t)stream);
}
