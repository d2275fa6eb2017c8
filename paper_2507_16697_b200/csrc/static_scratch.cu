// static_scratch.cu -- ringx_attn_fwd_static (include/ringx.h): the chunked forward for callers that cannot hand the
// library a device workspace.  The running fp32 accumulator (o_acc, lse_acc) that the chunk kernel's fold epilogue reads and
// rewrites between KV-chunk passes (Eq. 5 folded left to right) -- and, when a pass is split over the
// keys, the splits' partials -- live in ONE fixed array that is part of the library's device image instead of in memory the
// caller allocated.  Nothing here (and nothing it calls) allocates or frees device memory.
//
// The array below is device memory.  In HOST code its name is only a handle for the runtime: it is not a device address and
// must never be given to a kernel.  The device address is looked up with cudaGetSymbolAddress, once per device, with that
// device current, and that pointer is what the kernels get.
#include <mutex>

#include "kernels.cuh"

namespace {

constexpr size_t kStaticScratchBytes = RINGX_STATIC_SCRATCH_BYTES;

// Every GPU that loads libringx holds these bytes from the moment the module is loaded on it until the process exits.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

std::mutex g_mu;
void* g_scratch_ptr[ringx::kMaxDevices];   // device address of g_static_scratch on device i; nullptr = not looked up yet

// Device address of the array on the CURRENT device (looked up on the first call per device, cached afterwards).
int static_scratch_of_current_device(void** out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return RINGX_ERR_CUDA;
  }
  const bool cacheable = dev >= 0 && dev < ringx::kMaxDevices;
  std::lock_guard<std::mutex> g(g_mu);
  if (cacheable && g_scratch_ptr[dev]) {
    *out = g_scratch_ptr[dev];
    return RINGX_OK;
  }
  void* p = nullptr;
  const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
  if (e != cudaSuccess || !p) {
    cudaGetLastError();
    return RINGX_ERR_CUDA;
  }
  if (cacheable) g_scratch_ptr[dev] = p;
  *out = p;
  return RINGX_OK;
}

}  // namespace

extern "C" {

int ringx_attn_fwd_static(const void* q, const void* k, const void* v, void* o, float* lse, int B, int H, int N, int d,
                          int kv_chunk, float scale, int dtype, void* stream) {
  if (!q || !k || !v || !o || !lse) return RINGX_ERR_NULL_PTR;
  // 0 for a shape outside ringx_attn_fwd's domain (which then rejects it below, before anything is enqueued) and for a
  // single pass that needs no scratch at all: neither touches the array
  const size_t need = ringx_attn_fwd_workspace_bytes(B, H, N, d, kv_chunk, dtype);
  if (need > kStaticScratchBytes) return RINGX_ERR_WORKSPACE_TOO_SMALL;
  void* scratch = nullptr;
  if (need) {
    const int st = static_scratch_of_current_device(&scratch);
    if (st != RINGX_OK) return st;
  }
  // Nothing in the forward's scratch has to start at zero: the first pass overwrites the accumulator rows it later folds
  // into, and every split partial is written before the merge reads it -- what an earlier call left behind is never read.
  return ringx_attn_fwd(q, k, v, o, lse, B, H, N, d, kv_chunk, scale, dtype, scratch, need ? kStaticScratchBytes : 0, stream);
}

}  // extern "C"
