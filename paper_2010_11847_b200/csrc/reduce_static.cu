// reduce_static.cu -- fpm_reduce_static: the pyramid REDUCE (Alg. 2; R14) for
// callers that must not allocate device memory.
//
// Who that is.  fpm_reduce needs a context (fpm_create cudaMallocs its plan tables) and a caller-allocated
// workspace for the two intermediates of each level's three axis passes.  Some hosts of this library can do
// neither: a plug-in living inside a process whose device memory has all been handed to another owner (a
// framework's caching pool, a fixed MIG/MPS memory budget) where a fresh cudaMalloc fails or forces that owner to
// release and re-grow its pool; and a steady-state loop that cannot take the device-wide synchronisation
// cudaMalloc/cudaFree imply while other streams are in flight.  For them the intermediates live in the
// file-scope device array below, which is part of the loaded library image: it exists on every GPU that loads
// libfpm's kernels from the moment the module is loaded until the process exits, whether or not this entry point
// is ever called.  That is why its size is a fixed, modest maximum (8 MiB: meshes up to 128^3).
//
// The array's name means two different things.  In device code it is the array.  In host code it is only a
// host-side handle for the symbol -- not a device address; handing `reduce_scratch` itself to a kernel would make
// the kernel fault (or, where the GPU can dereference host addresses, scribble over unrelated host memory).  The
// device address is obtained once per device with cudaGetSymbolAddress, with that device current, in THIS
// translation unit (a static __device__ symbol is not visible from any other), and that pointer is what the axis
// passes receive.
#include <cstdio>
#include <mutex>

#include "fpm_internal.h"

namespace {

constexpr int kMaxNg = 128;                                   // FPM_REDUCE_STATIC_MAX_NG in fpm.h
constexpr int64_t kScratchFloats = (int64_t)kMaxNg * kMaxNg * kMaxNg;
static_assert(kMaxNg == FPM_REDUCE_STATIC_MAX_NG, "fpm.h and reduce_static.cu disagree on the maximum mesh");

// All levels of one call fit in ng^3 floats: level l of an n^3 mesh uses 3/4 n^3 (the z- and y-reduced
// intermediates) + n^3/8 (its output, the next level's input), and n^3 (7/8)(1 + 1/8 + 1/64 + ...) = n^3.
static __device__ __align__(256) float reduce_scratch[kScratchFloats];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
float* g_scratch_ptr[kMaxDevices] = {};                       // device address of reduce_scratch, per device

int report(char* err, size_t err_len, int rc, const char* what, const char* detail = "") {
  if (err && err_len) std::snprintf(err, err_len, "fpm_reduce_static: %s%s", what, detail);
  return rc;
}

// Device address of the scratch array on the CURRENT device; looked up on the first call there, cached after.
cudaError_t scratch_on_current_device(float** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_ptr[dev]) {
    float* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), reduce_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_ptr[dev] = p;
  }
  *out = g_scratch_ptr[dev];
  return cudaSuccess;
}

inline int64_t cube(int64_t n) { return n * n * n; }

}  // namespace

extern "C" int fpm_reduce_static(const float* in, int ng, int levels, float* out, void* cuda_stream, char* err,
                                 size_t err_len) {
  if (err && err_len) err[0] = '\0';
  if (!in || !out || in == out) return report(err, err_len, FPM_EINVAL, "in and out must be two distinct device arrays");
  if (ng < 8 || (ng & (ng - 1))) return report(err, err_len, FPM_EINVAL, "ng must be a power of two >= 8");
  if (ng > kMaxNg) {
    char detail[96];
    std::snprintf(detail, sizeof detail, "ng = %d exceeds the built-in scratch (meshes up to %d^3); use fpm_reduce", ng, kMaxNg);
    return report(err, err_len, FPM_EINVAL, detail);
  }
  if (levels < 0 || levels >= 8 || (ng >> levels) < 8)
    return report(err, err_len, FPM_EINVAL, "levels out of range (ng >> levels >= 8)");
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  if (levels == 0) {                                           // a copy, as in fpm_reduce; no scratch involved
    cudaError_t e = cudaMemcpyAsync(out, in, sizeof(float) * cube(ng), cudaMemcpyDeviceToDevice, s);
    return e == cudaSuccess ? FPM_OK : report(err, err_len, FPM_ECUDA, "cudaMemcpyAsync: ", cudaGetErrorString(e));
  }
  float* scratch = nullptr;
  cudaError_t e = scratch_on_current_device(&scratch);
  if (e != cudaSuccess) return report(err, err_len, FPM_ECUDA, "cudaGetSymbolAddress: ", cudaGetErrorString(e));
  // Same level plan as fpm_reduce (api.cu pyr_reduce).  Every scratch element a pass reads was written by the
  // pass before it in this same call, so nothing left over from an earlier call is ever read: no clearing needed.
  const float* cur = in;
  int n = ng;
  for (int l = 0; l < levels; ++l) {
    float* tmp = scratch;
    float* dst = (l == levels - 1) ? out : scratch + 3 * cube(n) / 4;
    e = fpm::pyramid_reduce_level(cur, n, tmp, dst, s);
    if (e != cudaSuccess) return report(err, err_len, FPM_ECUDA, "kernel launch: ", cudaGetErrorString(e));
    scratch += 3 * cube(n) / 4 + cube(n / 2);
    cur = dst;
    n /= 2;
  }
  return FPM_OK;
}
