// recon.cu -- element-wise kernels of the MAP reconstruction loop (PAPER.md:407-418
// Eq. 12 and Listing 7.1): the likelihood residual, the Gaussian prior in k-space and
// the Adam update.  The forward model and its reverse are the PM kernels of the rest of the library.
#include "fpm_internal.h"

namespace fpm {

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ void block_add(double v, double* acc) {
  __shared__ double part[kThreads / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    double t = threadIdx.x < kThreads / 32 ? part[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (threadIdx.x == 0) atomicAdd(acc, t);
  }
}

// gbar = (rho - data) / sigma^2 ;  *acc += sum (rho - data)^2   (float64 accumulation)
__global__ void __launch_bounds__(kThreads)
residual_kernel(const float* __restrict__ rho, const float* __restrict__ data, float inv_s2, int64_t n,
                float* __restrict__ gbar, double* __restrict__ acc) {
  double sum = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const float r = rho[i] - data[i];
    gbar[i] = r * inv_s2;
    sum += (double)r * (double)r;
  }
  block_add(sum, acc);
}

// gk = inv_power * sk * n3 (so that c2r, which divides by n3, returns the gradient of the prior);
// *acc += sum over the FULL k-space of inv_power |sk|^2 (half-space weights 2 for 0 < kz < n/2)
__global__ void __launch_bounds__(kThreads)
prior_rows_kernel(const float2* __restrict__ sk, const float* __restrict__ inv_power, int n, float n3,
                  float2* __restrict__ gk, double* __restrict__ acc) {
  const int nzh = n / 2 + 1;
  const int64_t row = (int64_t)blockIdx.x * nzh;
  double sum = 0.0;
  for (int z = threadIdx.x; z < nzh; z += blockDim.x) {
    const float2 v = sk[row + z];
    const float ip = inv_power[row + z];
    const double wt = (z == 0 || 2 * z == n) ? 1.0 : 2.0;
    sum += wt * (double)ip * ((double)v.x * v.x + (double)v.y * v.y);
    const float f = ip * n3;
    gk[row + z] = make_float2(v.x * f, v.y * f);
  }
  block_add(sum, acc);
}

// Adam with bias correction c1 = 1 - b1^t, c2 = 1 - b2^t; omb = 1 - beta (all from the host, float64)
__global__ void __launch_bounds__(kThreads)
adam_kernel(float* __restrict__ x, const float* __restrict__ g, float* __restrict__ m,
            float* __restrict__ v, int64_t n, float lr, float b1, float b2, float omb1, float omb2,
            float eps, float inv_c1, float inv_c2) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const float gi = g[i];
    const float mi = b1 * m[i] + omb1 * gi;
    const float vi = b2 * v[i] + omb2 * gi * gi;
    m[i] = mi;
    v[i] = vi;
    x[i] -= lr * (mi * inv_c1) / (sqrtf(vi * inv_c2) + eps);
  }
}

inline unsigned grid_for(int64_t n) {
  int64_t b = (n + kThreads - 1) / kThreads;
  if (b > 148LL * 16) b = 148LL * 16;
  return (unsigned)(b < 1 ? 1 : b);
}

}  // namespace

cudaError_t recon_residual(const float* rho, const float* data, float inv_s2, int64_t n, float* gbar,
                           double* acc, cudaStream_t s) {
  residual_kernel<<<grid_for(n), kThreads, 0, s>>>(rho, data, inv_s2, n, gbar, acc);
  return cudaGetLastError();
}

cudaError_t recon_prior(const float2* sk, const float* inv_power, int n, float2* gk, double* acc,
                        cudaStream_t s) {
  prior_rows_kernel<<<(unsigned)(n * n), kThreads, 0, s>>>(sk, inv_power, n, (float)((double)n * n * n), gk, acc);
  return cudaGetLastError();
}

// 1 - beta is formed in float64 on the host: 1.f - 0.999f is off by 1.7e-5 relative
cudaError_t adam_update(float* x, const float* g, float* m, float* v, int64_t n, double lr, double b1,
                        double b2, double eps, double inv_c1, double inv_c2, cudaStream_t s) {
  adam_kernel<<<grid_for(n), kThreads, 0, s>>>(x, g, m, v, n, (float)lr, (float)b1, (float)b2,
                                               (float)(1.0 - b1), (float)(1.0 - b2), (float)eps,
                                               (float)inv_c1, (float)inv_c2);
  return cudaGetLastError();
}

}  // namespace fpm
