// relocate_static.cu — satsplat_relocate_static: the relocation of dead surfels (relocate.cu) for callers that
// have no device memory of their own to hand over as scratch.
//
// Who that is: a training process whose framework has already taken the whole device for its caching pool (nothing is left
// for a cudaMalloc, and the pool's own allocator is not reachable from C), a job running inside a fixed memory quota, or a
// loop that must not pay the device-wide stall a cudaMalloc / cudaFree causes in the middle of an iteration.  satsplat_relocate
// asks such a caller for satsplat_relocate_scratch_bytes(N) bytes of working memory; this variant takes them from an array
// that is part of the library image instead, so the only device memory the caller supplies is its own inputs and outputs.
//
// The price: the array has a fixed size (enough for SATSPLAT_RELOCATE_STATIC_MAX_SURFELS surfels, about 3.5 MB), every GPU
// that has loaded the library keeps it until the process exits whether or not this call is ever made, and all calls on one
// GPU use the same bytes.
#include <stdio.h>

#include <mutex>

#include "internal.cuh"

using namespace satsplat;

namespace {

// 28 bytes per surfel (cumulative weights, new scales, counts, sources, new logits) + the scan's block partials + slack;
// relocate_scratch_bytes(N) is checked against this at run time, so a change of the layout cannot overrun it silently.
constexpr size_t kStaticBytes = (size_t)SATSPLAT_RELOCATE_STATIC_MAX_SURFELS * 28 + 4096;
static __device__ __align__(256) unsigned char g_relocate_scratch[kStaticBytes];

// In host code `g_relocate_scratch` is only a handle for the runtime, not an address a kernel can use: the device address
// is looked up once per device with cudaGetSymbolAddress (that device current) and remembered here.
constexpr int kMaxDevices = 64;
void* g_scratch_addr[kMaxDevices] = {};
std::mutex g_scratch_mutex;

cudaError_t scratch_for_current_device(void** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_relocate_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" int satsplat_relocate_static(int64_t N, float* means, float* quats, float* scales, float* opacity_logits, float* rgb,
                                        float* adam_m, float* adam_v, const float* u, float o_min, int32_t n_max,
                                        int32_t* src_out, satsplat_stream stream) {
  auto fail = [&](int code, const char* what, const char* detail) {
    char msg[256];
    snprintf(msg, sizeof(msg), "satsplat_relocate_static: %s%s", what, detail);
    set_thread_error(msg);                               // read back with satsplat_last_error(NULL)
    return code;
  };
  if (N < 0 || !(o_min > 0.f && o_min < 1.f) || n_max < 1 || (adam_m == nullptr) != (adam_v == nullptr))
    return fail(SATSPLAT_E_INVALID, "bad argument", "");
  if (N > (int64_t)SATSPLAT_RELOCATE_STATIC_MAX_SURFELS || (size_t)relocate_scratch_bytes(N) > kStaticBytes) {
    char detail[160];
    snprintf(detail, sizeof(detail), "N = %lld, the built-in scratch holds at most %d surfels; use satsplat_relocate", (long long)N,
             (int)SATSPLAT_RELOCATE_STATIC_MAX_SURFELS);
    return fail(SATSPLAT_E_INVALID, "too many surfels: ", detail);
  }
  if (N > 0 && (!means || !quats || !scales || !opacity_logits || !rgb || !u)) return fail(SATSPLAT_E_INVALID, "NULL pointer", "");
  if (N == 0) return SATSPLAT_OK;
  void* scratch = nullptr;
  cudaError_t e = scratch_for_current_device(&scratch);
  if (e != cudaSuccess) return fail(SATSPLAT_E_CUDA, "looking up the built-in scratch: ", cudaGetErrorString(e));
  // Nothing in the array has to be zero on entry: the first kernel of the sequence writes the weight, count and source of
  // every surfel below N, the scan writes every partial it later reads, and nothing above those is read.  What an earlier
  // call left behind is therefore overwritten before use.
  e = launch_relocate(N, means, quats, scales, opacity_logits, rgb, adam_m, adam_v, u, o_min, (int)n_max, scratch, src_out,
                      (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(SATSPLAT_E_CUDA, "", cudaGetErrorString(e));
  return SATSPLAT_OK;
}
