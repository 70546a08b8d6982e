// noalloc.cu -- gwc_los_allsky_static: the all-sky prior of the denominator for callers that cannot
// let the library allocate device memory.
//
// Every other entry point of gwc.h needs a gwc_ctx, and gwc_create / the grow-only scratch of the context call
// cudaMalloc.  Some programs cannot afford that call:
//   * a process that has handed all of the device's memory to its own pool or arena (a framework's caching allocator,
//     a job with a fixed memory budget): a cudaMalloc from inside a library then fails, or takes memory the owner
//     believes it has;
//   * a serving or sampling loop with work in flight on other streams: cudaMalloc and cudaFree take a device-wide
//     lock and may wait for the device, which stalls every stream, not only the caller's;
//   * code that is simply not allowed to create a context (no gwc_create) because of the two rules above.
// For them the two-kernel all-sky mean runs here with its partial sums in a fixed array that is part of the library
// image itself: nothing is allocated, at the price of a size limit and of one shared buffer per GPU.
//
// The arithmetic is that of gwc_los_allsky: the same two kernels (reduce.cu: allsky_partial_kernel, allsky_final_kernel)
// in the same order, so the result is bit-identical.
#include <cstdio>
#include <mutex>

#include "gwc_internal.h"

namespace {

// The scratch: one partial sum per (block of 512 rows, redshift node).  File scope, so it lives in the module's global
// segment: EVERY GPU that loads libgwc.so holds these 4 MiB from the moment the module is loaded until the process
// exits, whether or not this entry point is ever called.
static __device__ __align__(256) double g_allsky_static_scratch[GWC_ALLSKY_STATIC_MAX_DOUBLES];

// In host code the name above is only a handle for the runtime, NOT a device address (passing it to a kernel would
// fault, or on a system where the GPU can read host memory silently use the wrong bytes).  The device address differs
// per GPU and is asked for once per device, with that device current.
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
double* g_scratch_addr[MAX_DEVICES] = {};

thread_local char t_err[320] = "";

gwc_status fail(gwc_status st, const char* msg) {
  snprintf(t_err, sizeof(t_err), "%s", msg);
  return st;
}

// set-up on first use: the address of the scratch array on the calling thread's current device
gwc_status scratch_on_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    snprintf(t_err, sizeof(t_err), "gwc_los_allsky_static: cudaGetDevice: %s", cudaGetErrorString(e));
    return GWC_ERR_CUDA;
  }
  if (dev < 0 || dev >= MAX_DEVICES) return fail(GWC_ERR_INVALID_ARG, "gwc_los_allsky_static: device index above 63");
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_allsky_static_scratch);
    if (e != cudaSuccess || !p) {
      snprintf(t_err, sizeof(t_err), "gwc_los_allsky_static: cudaGetSymbolAddress on device %d: %s", dev,
               cudaGetErrorString(e));
      cudaGetLastError();
      return GWC_ERR_CUDA;
    }
    g_scratch_addr[dev] = (double*)p;
  }
  *out = g_scratch_addr[dev];
  return GWC_OK;
}

}  // namespace

extern "C" {

gwc_status gwc_los_allsky_static(const gwc_los* los, double* d_allsky, void* cuda_stream) {
  t_err[0] = 0;
  // the argument rules of gwc_los_allsky
  if (!los) return fail(GWC_ERR_INVALID_ARG, "gwc_los_allsky_static: los is NULL");
  if (los->n_z < 2 || los->n_z > 65536) return fail(GWC_ERR_SHAPE, "gwc_los_allsky_static: los->n_z out of range");
  if (!(los->z_max > 0.0)) return fail(GWC_ERR_INVALID_ARG, "gwc_los_allsky_static: los->z_max must be positive");
  if (los->prec != GWC_F64 && los->prec != GWC_F32) return fail(GWC_ERR_INVALID_ARG, "gwc_los_allsky_static: los->prec");
  if (!los->table || los->n_rows < 1 || los->n_rows > 0x7fffffffLL)
    return fail(GWC_ERR_INVALID_ARG, "gwc_los_allsky_static: los->table is NULL or n_rows out of range");
  if (!d_allsky) return fail(GWC_ERR_INVALID_ARG, "gwc_los_allsky_static: d_allsky is NULL");
  // the size limit of the fixed scratch: refused before anything is enqueued, d_allsky untouched
  const size_t need = gwc::allsky_scratch_doubles(los->n_rows, los->n_z);
  if (need > (size_t)GWC_ALLSKY_STATIC_MAX_DOUBLES) {
    snprintf(t_err, sizeof(t_err),
             "gwc_los_allsky_static: table too large for the fixed scratch: ceil(n_rows / %d) * n_z = %zu partial sums, "
             "the limit is %d (use gwc_los_allsky, which allocates)",
             GWC_ALLSKY_STATIC_ROWS_PER_PART, need, GWC_ALLSKY_STATIC_MAX_DOUBLES);
    return GWC_ERR_SHAPE;
  }
  double* scratch = nullptr;
  const gwc_status st = scratch_on_current_device(&scratch);
  if (st != GWC_OK) return st;
  // Nothing in the scratch has to start at zero: the first kernel writes every one of the `need` partial sums before
  // the second kernel reads exactly those, so what an earlier call left behind is never read.
  if (gwc::launch_allsky(los->table, los->prec, los->n_rows, los->n_z, scratch, d_allsky, (cudaStream_t)cuda_stream) < 0) {
    return fail(GWC_ERR_CUDA, "gwc_los_allsky_static: a kernel launch failed (invalid stream, or the device is in an error state)");
  }
  return GWC_OK;
}

const char* gwc_los_allsky_static_error(void) { return t_err; }

}  // extern "C"
