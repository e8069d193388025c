// static_scratch.cu -- strata_na3d_fwd_static (include/strata_na3d.h): the forward for callers that cannot allocate.
//
// Who this is for: code that sits inside somebody else's process and owns no device memory -- a plug-in under a host
// whose memory pool has taken the whole GPU, a step inside a loop where the device-wide synchronisation of
// cudaMalloc / cudaFree is not tolerable, a component that is only called after the host has declared "no more
// allocations".  Such a caller has its inputs and outputs (somebody gave them to it) but nothing it could pass as
// `workspace`.  Here the scratch is an array in the library image instead, so that this file calls no cudaMalloc,
// no cudaFree and no allocating library routine; the price is STRATA_STATIC_SCRATCH_BYTES (1 MiB) of every GPU the
// library is loaded on, held until the process exits, and a bound on the problems it serves.
//
// What runs is strata_na3d_fwd itself (strata_na3d.cu), handed the array's device address as its workspace: the same
// kernels and the same results.  The kernels only see a pointer; they do not know where it came from.
#include "../../include/strata_na3d.h"

#include <cuda_runtime.h>

#include <mutex>

// The scratch.  `g_static_scratch` in HOST code is only a handle for the runtime (its value is not a device
// address, and a kernel given it would fault or scribble over host memory): host code has to ask
// cudaGetSymbolAddress for the address on the current device, which scratch_on_current_device() does once per device.
// Contents: whatever the last call left (rotated Q / K copies of the fp32 and tile paths, or the list of rows for
// the fix-up kernel, see common.cuh) -- per device, shared by every call on that device.
static __device__ __align__(256) unsigned char g_static_scratch[STRATA_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
void* g_scratch_addr[kMaxDevices] = {};      // device address of g_static_scratch, by device ordinal (nullptr: not looked up yet)
std::mutex g_scratch_mu;

// Device address of the array on the CURRENT device.  The look-up happens on the first call per device; it does not
// allocate (the array came with the module), but it is a set-up step that belongs before any stream capture.
strata_status_t scratch_on_current_device(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return STRATA_ERR_CUDA; }
  if (dev < 0 || dev >= kMaxDevices) return STRATA_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (!g_scratch_addr[dev]) {
    unsigned char* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
    if (e != cudaSuccess || !ptr) { (void)cudaGetLastError(); return STRATA_ERR_CUDA; }
    g_scratch_addr[dev] = ptr;
  }
  *out = g_scratch_addr[dev];
  return STRATA_OK;
}

}  // namespace

extern "C" strata_status_t strata_na3d_fwd_static(const strata_na3d_desc_t* desc, const void* q, const void* k,
                                                  const void* v, const float* coords, const float* freqs, void* o,
                                                  float* lse, void* stream) {
  // Order: everything that can be decided on the host first (so a bad call costs no CUDA call and enqueues nothing),
  // then the address, then the kernels.
  const size_t need = strata_na3d_workspace_bytes(desc, 0);
  if (need == 0)                                   // invalid or unsupported descriptor: let the forward name the reason
    return strata_na3d_fwd(desc, q, k, v, coords, freqs, o, lse, nullptr, 0, stream);
  if (need > (size_t)STRATA_STATIC_SCRATCH_BYTES) return STRATA_ERR_STATIC_SCRATCH;
  if (!q || !k || !v || !o || !lse) return STRATA_ERR_INVALID_ARG;
  void* scratch = nullptr;
  const strata_status_t s = scratch_on_current_device(&scratch);
  if (s != STRATA_OK) return s;
  // The array still holds what the previous call wrote.  The one part a call needs at zero is the 16-byte header of
  // the fix-up list (row count, take-all flag) at its start: cleared here, on `stream`, ahead of the kernels
  // (cudaMemsetAsync enqueues a fill, it does not allocate), so a list left by the previous call is never read.  The
  // rotated copies of the fp32 / tile paths are written in full by the rotation kernel before anything reads them.
  if (cudaMemsetAsync(scratch, 0, 16, reinterpret_cast<cudaStream_t>(stream)) != cudaSuccess) {
    (void)cudaGetLastError();
    return STRATA_ERR_CUDA;
  }
  return strata_na3d_fwd(desc, q, k, v, coords, freqs, o, lse, scratch, (size_t)STRATA_STATIC_SCRATCH_BYTES, stream);
}
