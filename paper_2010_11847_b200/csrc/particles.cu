// particles.cu -- kick and drift (Eq. 1-2) as streaming passes (the fused
// readout + kick + drift pass of the whole-run driver lives in mesh_ops.cu).
#include "fpm_internal.h"

namespace fpm {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ float wrap_box(float x, float ng, float inv_ng) {
  x -= ng * floorf(x * inv_ng);
  if (x >= ng) x -= ng;
  if (x < 0.f) x += ng;
  return x >= ng ? 0.f : x;
}

__global__ void __launch_bounds__(kThreads)
kick_kernel(float* __restrict__ mom, const float* __restrict__ force, int64_t n, float fac) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  const int64_t n4 = n / 4;
  float4* m4 = reinterpret_cast<float4*>(mom);
  const float4* f4 = reinterpret_cast<const float4*>(force);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
    float4 m = m4[i];
    const float4 f = __ldcs(f4 + i);
    m.x = fmaf(f.x, fac, m.x);
    m.y = fmaf(f.y, fac, m.y);
    m.z = fmaf(f.z, fac, m.z);
    m.w = fmaf(f.w, fac, m.w);
    m4[i] = m;
  }
  for (int64_t i = n4 * 4 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
    mom[i] = fmaf(force[i], fac, mom[i]);
}

__global__ void __launch_bounds__(kThreads)
drift_kernel(float* __restrict__ pos, const float* __restrict__ mom, int64_t n, float fac, float ng,
             float inv_ng) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  const int64_t n4 = n / 4;
  float4* x4 = reinterpret_cast<float4*>(pos);
  const float4* p4 = reinterpret_cast<const float4*>(mom);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
    float4 x = x4[i];
    const float4 p = __ldcs(p4 + i);
    x.x = wrap_box(fmaf(p.x, fac, x.x), ng, inv_ng);
    x.y = wrap_box(fmaf(p.y, fac, x.y), ng, inv_ng);
    x.z = wrap_box(fmaf(p.z, fac, x.z), ng, inv_ng);
    x.w = wrap_box(fmaf(p.w, fac, x.w), ng, inv_ng);
    x4[i] = x;
  }
  for (int64_t i = n4 * 4 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
    pos[i] = wrap_box(fmaf(mom[i], fac, pos[i]), ng, inv_ng);
}

// Scalar fallbacks for unaligned pointers.
__global__ void __launch_bounds__(kThreads)
kick_scalar_kernel(float* __restrict__ mom, const float* __restrict__ force, int64_t n, float fac) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x)
    mom[i] = fmaf(force[i], fac, mom[i]);
}
__global__ void __launch_bounds__(kThreads)
drift_scalar_kernel(float* __restrict__ pos, const float* __restrict__ mom, int64_t n, float fac,
                    float ng, float inv_ng) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x)
    pos[i] = wrap_box(fmaf(mom[i], fac, pos[i]), ng, inv_ng);
}

inline unsigned grid_for(int64_t n) {
  int64_t b = (n + kThreads - 1) / kThreads;
  const int64_t cap = 148LL * 64;
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (unsigned)b;
}

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

}  // namespace

cudaError_t kick(float* mom, const float* force, int64_t n3, float fac, cudaStream_t s) {
  if (n3 == 0) return cudaSuccess;
  if (aligned16(mom) && aligned16(force))
    kick_kernel<<<grid_for(n3 / 4 + 1), kThreads, 0, s>>>(mom, force, n3, fac);
  else
    kick_scalar_kernel<<<grid_for(n3), kThreads, 0, s>>>(mom, force, n3, fac);
  return cudaGetLastError();
}

cudaError_t drift(float* pos, const float* mom, int64_t n3, float fac, int ng, cudaStream_t s) {
  if (n3 == 0) return cudaSuccess;
  if (aligned16(pos) && aligned16(mom))
    drift_kernel<<<grid_for(n3 / 4 + 1), kThreads, 0, s>>>(pos, mom, n3, fac, (float)ng, 1.f / ng);
  else
    drift_scalar_kernel<<<grid_for(n3), kThreads, 0, s>>>(pos, mom, n3, fac, (float)ng, 1.f / ng);
  return cudaGetLastError();
}

}  // namespace fpm
