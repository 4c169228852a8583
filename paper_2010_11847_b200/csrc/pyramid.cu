// pyramid.cu -- REDUCE / EXPAND of the multi-grid pyramid (Eq. 6-9,
// Alg. 2) and the combination step of Alg. 3 Force.
//
// DESIGN.md reading R14: BSpline(6) = the two-scale mask of the order-6 cardinal B-spline,
// h = [1, 6, 15, 20, 15, 6, 1] / 64 per axis (offsets -3..3), K = h (x) h (x) h; Conv3D with stride 2 and
// periodic wrap; TransposedConv3D with 8 K.  The paper runs them as TensorFlow 3-D convolutions; K is
// separable, so here one level is three axis passes of 7 (reduce) or 3-4 (expand) taps each -- 21 instead of
// 343 multiply-adds per coarse cell -- streaming each intermediate once.  On one GPU the pyramid is strictly
// more work than the single-mesh force: these kernels serve the accuracy study, not the hot path.
#include "fpm_internal.h"

namespace fpm {

namespace {

constexpr int kThreads = 256;

// view of a contiguous array as (outer, n, inner): element (o, i, k) at (o n + i) inner + k
// out(o, X, k) = sum_j h[j] in(o, (2 X + j) mod n, k),  X < n / 2
__global__ void __launch_bounds__(kThreads)
reduce_axis_kernel(const float* __restrict__ in, float* __restrict__ out, int64_t total, int n, int64_t inner) {
  const int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (t >= total) return;
  const int m = n >> 1;
  const int64_t k = t % inner, r = t / inner;
  const int X = (int)(r % m);
  const int64_t o = r / m;
  const float* line = in + o * n * inner + k;
  const int mask = n - 1, c = 2 * X;
  const float a0 = line[(int64_t)c * inner];
  const float a1 = line[(int64_t)((c + 1) & mask) * inner] + line[(int64_t)((c - 1) & mask) * inner];
  const float a2 = line[(int64_t)((c + 2) & mask) * inner] + line[(int64_t)((c - 2) & mask) * inner];
  const float a3 = line[(int64_t)((c + 3) & mask) * inner] + line[(int64_t)((c - 3) & mask) * inner];
  out[t] = (20.f * a0 + 15.f * a1 + 6.f * a2 + a3) * (1.f / 64.f);
}

// out(o, x, k) = sum_X 2 h[x - 2 X] in(o, X, k),  x < 2 m  (one axis' share of the factor 8)
//   x = 2 q     : (6 in[q+1] + 20 in[q] + 6 in[q-1]) / 32
//   x = 2 q + 1 : (in[q+2] + 15 in[q+1] + 15 in[q] + in[q-1]) / 32
__global__ void __launch_bounds__(kThreads)
expand_axis_kernel(const float* __restrict__ in, float* __restrict__ out, int64_t total, int m, int64_t inner) {
  const int64_t t = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (t >= total) return;
  const int n = 2 * m, mask = m - 1;
  const int64_t k = t % inner, r = t / inner;
  const int x = (int)(r % n);
  const int64_t o = r / n;
  const float* line = in + o * m * inner + k;
  const int q = x >> 1;
  const float c0 = line[(int64_t)q * inner], cp = line[(int64_t)((q + 1) & mask) * inner],
              cm = line[(int64_t)((q - 1) & mask) * inner];
  float v;
  if (x & 1) v = (line[(int64_t)((q + 2) & mask) * inner] + 15.f * (cp + c0) + cm) * (1.f / 32.f);
  else v = (6.f * (cp + cm) + 20.f * c0) * (1.f / 32.f);
  out[t] = v;
}

// Alg. 3: F_i <= F_iL + (F_iS - F_il)
__global__ void __launch_bounds__(kThreads)
pyramid_combine_kernel(float* __restrict__ fs, const float* __restrict__ up, const float* __restrict__ lowup, int64_t n) {
  const int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (i < n) fs[i] = up[i] + (fs[i] - lowup[i]);
}

inline unsigned blocks_for(int64_t n) { return (unsigned)((n + kThreads - 1) / kThreads); }

}  // namespace

// One REDUCE level n^3 -> (n/2)^3: z, y, x passes.  tmp holds n^2 (n/2) + n (n/2)^2 floats; out may not alias in.
cudaError_t pyramid_reduce_level(const float* in, int n, float* tmp, float* out, cudaStream_t s) {
  const int64_t g = n, m = n / 2;
  float* t1 = tmp;                    // (n, n, m)
  float* t2 = tmp + g * g * m;        // (n, m, m)
  reduce_axis_kernel<<<blocks_for(g * g * m), kThreads, 0, s>>>(in, t1, g * g * m, n, 1);
  reduce_axis_kernel<<<blocks_for(g * m * m), kThreads, 0, s>>>(t1, t2, g * m * m, n, m);
  reduce_axis_kernel<<<blocks_for(m * m * m), kThreads, 0, s>>>(t2, out, m * m * m, n, m * m);
  return cudaGetLastError();
}

// One EXPAND level m^3 -> (2m)^3: x, y, z passes.  tmp holds 2 m^3 + 4 m^3 floats.
cudaError_t pyramid_expand_level(const float* in, int m_, float* tmp, float* out, cudaStream_t s) {
  const int64_t m = m_, g = 2 * m;
  float* t1 = tmp;                    // (2m, m, m)
  float* t2 = tmp + g * m * m;        // (2m, 2m, m)
  expand_axis_kernel<<<blocks_for(g * m * m), kThreads, 0, s>>>(in, t1, g * m * m, m_, m * m);
  expand_axis_kernel<<<blocks_for(g * g * m), kThreads, 0, s>>>(t1, t2, g * g * m, m_, m);
  expand_axis_kernel<<<blocks_for(g * g * g), kThreads, 0, s>>>(t2, out, g * g * g, m_, 1);
  return cudaGetLastError();
}

cudaError_t pyramid_combine(float* fs, const float* up, const float* lowup, int64_t n, cudaStream_t s) {
  pyramid_combine_kernel<<<blocks_for(n), kThreads, 0, s>>>(fs, up, lowup, n);
  return cudaGetLastError();
}

}  // namespace fpm
