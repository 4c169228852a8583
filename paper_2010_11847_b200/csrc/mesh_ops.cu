// mesh_ops.cu -- cloud-in-cell paint (scatter), readout (gather) and their position gradients.
// PAPER.md:47 "linear window of unit size corresponding to the cloud-in-cell (CIC) interpolation
// scheme"; PAPER.md:51 readout "with the same kernel"; adjoints per SURVEY.md 8(c) R11.
#include "fpm_internal.h"

namespace fpm {

namespace {

struct Cic {
  int i0[3], i1[3];
  float t[3];
};

__device__ __forceinline__ Cic cic_of(float x, float y, float z, int mask) {
  Cic c;
  const float p[3] = {x, y, z};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const float fl = floorf(p[d]);
    c.t[d] = p[d] - fl;
    const int i = (int)fl;
    c.i0[d] = i & mask;
    c.i1[d] = (i + 1) & mask;
  }
  return c;
}

__device__ __forceinline__ float ld_stream(const float* p) {
  float v;
  asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}

constexpr int kThreads = 256;

// Baseline scatter: one thread per particle, 8 fp32 reductions (RED.ADD.F32) into L2.
__global__ void __launch_bounds__(kThreads)
paint_kernel(const float* __restrict__ pos, const float* __restrict__ mass, float mass_const,
             int64_t n, int ng, float* __restrict__ mesh) {
  const int mask = ng - 1;
  const int64_t g = ng;
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n;
       p += (int64_t)gridDim.x * blockDim.x) {
    const Cic c = cic_of(ld_stream(pos + p), ld_stream(pos + n + p), ld_stream(pos + 2 * n + p), mask);
    const float m = mass ? ld_stream(mass + p) : mass_const;
    const float wx[2] = {m * (1.f - c.t[0]), m * c.t[0]};
    const float wy[2] = {1.f - c.t[1], c.t[1]};
    const float wz[2] = {1.f - c.t[2], c.t[2]};
    const int ix[2] = {c.i0[0], c.i1[0]}, iy[2] = {c.i0[1], c.i1[1]}, iz[2] = {c.i0[2], c.i1[2]};
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        float* row = mesh + ((int64_t)ix[a] * g + iy[b]) * g;
        const float w = wx[a] * wy[b];
        atomicAdd(row + iz[0], w * wz[0]);
        atomicAdd(row + iz[1], w * wz[1]);
      }
  }
}

template <int NMESH>
__global__ void __launch_bounds__(kThreads)
readout_kernel(const float* __restrict__ m0, const float* __restrict__ m1,
               const float* __restrict__ m2, const float* __restrict__ pos, int64_t n, int ng,
               float* __restrict__ out) {
  const int mask = ng - 1;
  const int64_t g = ng;
  const float* mesh[3] = {m0, m1, m2};
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n;
       p += (int64_t)gridDim.x * blockDim.x) {
    const Cic c = cic_of(ld_stream(pos + p), ld_stream(pos + n + p), ld_stream(pos + 2 * n + p), mask);
    const float wx[2] = {1.f - c.t[0], c.t[0]};
    const float wy[2] = {1.f - c.t[1], c.t[1]};
    const float wz[2] = {1.f - c.t[2], c.t[2]};
    const int ix[2] = {c.i0[0], c.i1[0]}, iy[2] = {c.i0[1], c.i1[1]}, iz[2] = {c.i0[2], c.i1[2]};
    float acc[NMESH];
#pragma unroll
    for (int k = 0; k < NMESH; ++k) acc[k] = 0.f;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        const int64_t row = ((int64_t)ix[a] * g + iy[b]) * g;
        const float w = wx[a] * wy[b];
#pragma unroll
        for (int k = 0; k < NMESH; ++k) {
          acc[k] = fmaf(__ldg(mesh[k] + row + iz[0]), w * wz[0], acc[k]);
          acc[k] = fmaf(__ldg(mesh[k] + row + iz[1]), w * wz[1], acc[k]);
        }
      }
#pragma unroll
    for (int k = 0; k < NMESH; ++k) out[k * n + p] = acc[k];
  }
}

// out3[d][p] = s_p * sum_c mesh[c] dW/dx_d ; optional out_value[p] = sum_c mesh[c] W
__global__ void __launch_bounds__(kThreads)
readout_grad_kernel(const float* __restrict__ mesh, const float* __restrict__ pos,
                    const float* __restrict__ scale, float scale_const, int64_t n, int ng,
                    float* __restrict__ out3, float* __restrict__ out_value) {
  const int mask = ng - 1;
  const int64_t g = ng;
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n;
       p += (int64_t)gridDim.x * blockDim.x) {
    const Cic c = cic_of(ld_stream(pos + p), ld_stream(pos + n + p), ld_stream(pos + 2 * n + p), mask);
    const float wx[2] = {1.f - c.t[0], c.t[0]};
    const float wy[2] = {1.f - c.t[1], c.t[1]};
    const float wz[2] = {1.f - c.t[2], c.t[2]};
    const float sg[2] = {-1.f, 1.f};
    const int ix[2] = {c.i0[0], c.i1[0]}, iy[2] = {c.i0[1], c.i1[1]}, iz[2] = {c.i0[2], c.i1[2]};
    float gx = 0.f, gy = 0.f, gz = 0.f, val = 0.f;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        const int64_t row = ((int64_t)ix[a] * g + iy[b]) * g;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const float v = __ldg(mesh + row + iz[e]);
          gx = fmaf(v, sg[a] * wy[b] * wz[e], gx);
          gy = fmaf(v, wx[a] * sg[b] * wz[e], gy);
          gz = fmaf(v, wx[a] * wy[b] * sg[e], gz);
          val = fmaf(v, wx[a] * wy[b] * wz[e], val);
        }
      }
    const float s = scale ? ld_stream(scale + p) : scale_const;
    out3[p] = s * gx;
    out3[n + p] = s * gy;
    out3[2 * n + p] = s * gz;
    if (out_value) out_value[p] = val;
  }
}

inline unsigned grid_for(int64_t n) {
  int64_t b = (n + kThreads - 1) / kThreads;
  const int64_t cap = 148LL * 64;   // grid-stride beyond 64 waves of CTAs per SM
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (unsigned)b;
}

}  // namespace

cudaError_t paint(const float* pos, const float* mass, float mass_const, int64_t n, int ng,
                  float* mesh, bool zero_first, cudaStream_t s) {
  if (zero_first) {
    cudaError_t e = cudaMemsetAsync(mesh, 0, sizeof(float) * (size_t)ng * ng * ng, s);
    if (e != cudaSuccess) return e;
  }
  if (n == 0) return cudaSuccess;
  paint_kernel<<<grid_for(n), kThreads, 0, s>>>(pos, mass, mass_const, n, ng, mesh);
  return cudaGetLastError();
}

cudaError_t readout(const float* mesh, const float* pos, int64_t n, int ng, float* out,
                    cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  readout_kernel<1><<<grid_for(n), kThreads, 0, s>>>(mesh, nullptr, nullptr, pos, n, ng, out);
  return cudaGetLastError();
}

cudaError_t readout3(const float* fx, const float* fy, const float* fz, const float* pos, int64_t n,
                     int ng, float* out3, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  readout_kernel<3><<<grid_for(n), kThreads, 0, s>>>(fx, fy, fz, pos, n, ng, out3);
  return cudaGetLastError();
}

cudaError_t readout_grad(const float* mesh, const float* pos, const float* scale, float scale_const,
                         int64_t n, int ng, float* out3, float* out_value, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  readout_grad_kernel<<<grid_for(n), kThreads, 0, s>>>(mesh, pos, scale, scale_const, n, ng, out3,
                                                       out_value);
  return cudaGetLastError();
}

}  // namespace fpm
