// static_scratch.cu -- bm_simulate_static (include/bm.h): bm_simulate for callers that cannot allocate device memory.
//
// Who this is for.  bm_simulate needs a few KB to a few MB of device scratch (one 64-byte partial sum per thread block,
// read back by the grid pass of the ensemble reduction) and leaves it to the caller to provide it.  Some callers have no
// way to do that: a plug-in running inside a host application that owns the whole GPU heap and hands out no allocator; a
// real-time or latency-bound loop in which cudaMalloc is forbidden because it may synchronise the device and takes an
// unbounded time; a process that runs with the device memory already fully committed to other buffers.  For them the
// scratch lives here, in a fixed array in the library's device image.  It is reserved on every GPU that loads libbm.so,
// from the moment the module is loaded until the process exits, whether or not this entry point is ever called -- which
// is why its size is a stated, small constant (BM_STATIC_SCRATCH_BYTES) rather than something that grows on demand.
//
// What it does not do: no cudaMalloc / cudaMallocAsync / cudaFree, no memory pool, no library routine that allocates.
// The only CUDA calls are cudaGetDevice, cudaGetSymbolAddress (first call on a device) and what bm_simulate itself
// does (cudaFuncSetAttribute for the shared-memory opt-in, the kernel launches).
#include <mutex>

#include "common.cuh"

namespace {

// The scratch itself.  In host code the name `static_scratch` is only a handle the runtime uses to look the array up; it
// is NOT a device address, and a kernel given `static_scratch` (or &static_scratch[0]) from the host would fault or, on
// a system where the GPU can reach host memory, quietly scribble over the wrong bytes.  Host code must go through
// cudaGetSymbolAddress, once per device, with that device current (every device has its own copy of the array).
static __device__ __align__(256) unsigned char static_scratch[BM_STATIC_SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;

// Device address of the array on the CURRENT device; nullptr (with *err set) if the runtime cannot give it.  The table
// is filled lazily: the first call on a device does the look-up, later calls only read the table.
void *static_scratch_on_current_device(cudaError_t *err) {
  static void *address[MAX_DEVICES] = {};
  static std::mutex guard;  // the entry point may be called from several host threads
  int dev = -1;
  *err = cudaGetDevice(&dev);
  if (*err != cudaSuccess) return nullptr;
  if (dev < 0 || dev >= MAX_DEVICES) { *err = cudaErrorInvalidDevice; return nullptr; }
  std::lock_guard<std::mutex> lock(guard);
  if (!address[dev]) {
    void *ptr = nullptr;
    *err = cudaGetSymbolAddress(&ptr, static_scratch);
    if (*err != cudaSuccess || !ptr) {
      if (*err == cudaSuccess) *err = cudaErrorInvalidSymbol;
      return nullptr;
    }
    address[dev] = ptr;
  }
  return address[dev];
}

}  // namespace

// Device code may name the array directly.  This kernel is never launched; it pins the array into the device image (an
// array that no device code refers to could be dropped from it, and the look-up above would then fail).  Not exported
// (the library is built with hidden visibility).
__global__ void bm_static_scratch_anchor(unsigned char *out) {
  if (out) *out = static_scratch[0];
}

extern "C" {

BM_API bm_status bm_simulate_static(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                                    int64_t n_steps, double dt, uint64_t seed, bm_stats *out_stats, double *out_paths,
                                    double *out_trace, void *stream) {
  // size check first: it needs no device and gives the caller the clearest answer
  const size_t need = bm_workspace_bytes(cfg, n_points, n_paths);
  if (need == 0) return BM_ERR_INVALID_ARG;                    // bad cfg / counts (bm_simulate would say the same)
  if (need > (size_t)BM_STATIC_SCRATCH_BYTES) return BM_ERR_WORKSPACE;  // more thread blocks than the array has slots for
  cudaError_t err = cudaSuccess;
  void *scratch = static_scratch_on_current_device(&err);
  if (!scratch) {
    cudaGetLastError();
    return BM_ERR_CUDA;
  }
  // Nothing in the array has to start at zero: the path kernel writes the whole 64-byte slot of every block of this
  // call before the grid pass reads exactly those slots, so what an earlier call left behind is never looked at.
  return bm_simulate(cfg, params, n_points, n_paths, n_steps, dt, seed, out_stats, out_paths, out_trace, scratch,
                     (size_t)BM_STATIC_SCRATCH_BYTES, stream);
}

}  // extern "C"
