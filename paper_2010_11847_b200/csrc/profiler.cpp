// profiler.cpp -- per-kernel CUDA-event timing on the context's stream (used by bench.py for the
// live roofline numbers) and the launch counter behind fpm_launch_count().
#include <cstdlib>
#include <map>
#include <string>
#include <mutex>
#include <utility>

#include "fpm_internal.h"

namespace fpm {

// the driver entry point, without linking libcuda
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    cudaGetLastError();
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// (kernel, device) pairs whose MaxDynamicSharedMemorySize attribute is already raised to >= bytes
cudaError_t ensure_dynamic_smem_impl(const void* kernel, size_t bytes) {
  static std::mutex mu;
  static std::map<std::pair<const void*, int>, size_t> done;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  size_t& have = done[std::make_pair(kernel, dev)];
  if (have >= bytes) return cudaSuccess;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e == cudaSuccess) have = bytes;
  return e;
}

const char* kernel_name(int kid) {
  static const char* names[K_COUNT] = {
      "paint", "fft_z_r2c", "fft_cols_y", "fft_cols_x", "fft_z_c2r", "apply_force_kernel", "readout",
      "readout_kick_drift", "kick", "drift", "readout_grad", "lpt_elementwise", "fft_x_force",
      "fft_y_inv3", "memset", "fft_z_c2r3"};
  return (kid >= 0 && kid < K_COUNT) ? names[kid] : "?";
}

void Profiler::begin(int kid) {
  if (!enabled) return;
  if (open.size() >= 8192) flush();
  Rec r;
  r.kid = kid;
  if (pool.size() >= 2) {
    r.a = pool.back(); pool.pop_back();
    r.b = pool.back(); pool.pop_back();
  } else {
    if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) {
      enabled = false;
      return;
    }
  }
  cudaEventRecord(r.a, stream);
  open.push_back(r);
}

void Profiler::end() {
  if (!enabled || open.empty()) return;
  cudaEventRecord(open.back().b, stream);
}

void Profiler::flush() {
  for (Rec& r : open) {
    float t = 0.f;
    if (cudaEventSynchronize(r.b) == cudaSuccess && cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) {
      ms[r.kid] += t;
      count[r.kid] += 1;
    }
    pool.push_back(r.a);
    pool.push_back(r.b);
  }
  open.clear();
}

void Profiler::reset() {
  flush();
  for (int k = 0; k < K_COUNT; ++k) { ms[k] = 0.0; count[k] = 0; }
  launches = 0;
}

void Profiler::destroy() {
  flush();
  for (cudaEvent_t e : pool) cudaEventDestroy(e);
  pool.clear();
}

}  // namespace fpm
