// green.cu -- the transfer function grad laplace^-1 in k-space (Eq. 3-5) as a
// stand-alone element-wise kernel (the fused variants ride on the FFT x passes, fft.cu), and the
// spectral element-wise kernels of the LPT initial conditions (Alg. 4).
#include <cmath>
#include <vector>

#include "fpm_internal.h"

namespace fpm {

namespace {

const double kPi = 3.14159265358979323846264338327950288;
constexpr int kThreads = 128;

// One block per (x, y) row of the half-complex mesh, threads over kz.
__global__ void __launch_bounds__(kThreads)
force_kernel_rows(const float2* __restrict__ dk, int n, const float* __restrict__ lap,
                  const float* __restrict__ grad, float scale, float2* __restrict__ fkx,
                  float2* __restrict__ fky, float2* __restrict__ fkz) {
  const int nzh = n / 2 + 1;
  const int x = blockIdx.x / n, y = blockIdx.x % n;
  const float lxy = __ldg(lap + x) + __ldg(lap + y);
  const float gx = __ldg(grad + x), gy = __ldg(grad + y);
  const int64_t row = (int64_t)blockIdx.x * nzh;
  for (int z = threadIdx.x; z < nzh; z += blockDim.x) {
    const float k2 = lxy + __ldg(lap + z);
    const float inv = (blockIdx.x == 0 && z == 0) ? 0.f : scale / k2;
    const float2 d = dk[row + z];
    // i g d / K^2 : (re, im) -> (-im, re) * g * inv
    const float2 id = make_float2(-d.y * inv, d.x * inv);
    const float gz = __ldg(grad + z);
    fkx[row + z] = make_float2(id.x * gx, id.y * gx);
    fky[row + z] = make_float2(id.x * gy, id.y * gy);
    fkz[row + z] = make_float2(id.x * gz, id.y * gz);
  }
}

// out = sign * mult(k) * (-1/k^2) * in ; mult = -k_a^2 (a == b), (i k_a)(i k_b) (a != b, b >= 0),
// i k_a (b < 0); i k_d uses the Nyquist-zeroed table, -k_a^2 the full one.
__global__ void __launch_bounds__(kThreads)
lpt_spectral_rows(const float2* __restrict__ in, float2* __restrict__ out, int n,
                  const float* __restrict__ kv, const float* __restrict__ kv0, int a, int b,
                  float sign, int accumulate) {
  const int nzh = n / 2 + 1;
  const int x = blockIdx.x / n, y = blockIdx.x % n;
  const int64_t row = (int64_t)blockIdx.x * nzh;
  const float kx = __ldg(kv + x), ky = __ldg(kv + y);
  for (int z = threadIdx.x; z < nzh; z += blockDim.x) {
    const int idx[3] = {x, y, z};
    const float kz = __ldg(kv + z);
    const float k2 = kx * kx + ky * ky + kz * kz;
    const float inv = (blockIdx.x == 0 && z == 0) ? 0.f : -sign / k2;
    const float2 v = in[row + z];
    float2 r;
    if (a == b) {
      const float ka = __ldg(kv + idx[a]);
      const float m = -ka * ka * inv;
      r = make_float2(v.x * m, v.y * m);
    } else if (b >= 0) {
      const float m = -__ldg(kv0 + idx[a]) * __ldg(kv0 + idx[b]) * inv;   // (i ka)(i kb) = -ka kb
      r = make_float2(v.x * m, v.y * m);
    } else {
      const float m = __ldg(kv0 + idx[a]) * inv;                          // i ka
      r = make_float2(-v.y * m, v.x * m);
    }
    if (accumulate) { const float2 o = out[row + z]; r.x += o.x; r.y += o.y; }
    out[row + z] = r;
  }
}

// Transpose of force_kernel_rows: the mesh-to-mesh operator
// M_d = c2r o (i s g_d / K^2) o r2c is a real convolution with an odd kernel, so M_d^T = -M_d and
// rho_bar_k = - sum_d (i s g_d / K^2) Fbar_d,k.
__global__ void __launch_bounds__(kThreads)
force_kernel_transpose_rows(const float2* __restrict__ f0, const float2* __restrict__ f1,
                            const float2* __restrict__ f2, int n, const float* __restrict__ lap,
                            const float* __restrict__ grad, float scale, float2* __restrict__ out) {
  const int nzh = n / 2 + 1;
  const int x = blockIdx.x / n, y = blockIdx.x % n;
  const float lxy = __ldg(lap + x) + __ldg(lap + y);
  const float gx = __ldg(grad + x), gy = __ldg(grad + y);
  const int64_t row = (int64_t)blockIdx.x * nzh;
  for (int z = threadIdx.x; z < nzh; z += blockDim.x) {
    const float k2 = lxy + __ldg(lap + z);
    const float inv = (blockIdx.x == 0 && z == 0) ? 0.f : -scale / k2;
    const float gz = __ldg(grad + z);
    const float2 a = f0[row + z], b = f1[row + z], c = f2[row + z];
    const float re = gx * a.x + gy * b.x + gz * c.x, im = gx * a.y + gy * b.y + gz * c.y;
    out[row + z] = make_float2(-im * inv, re * inv);    // i (re + i im) inv
  }
}

__global__ void __launch_bounds__(256)
lpt_displace_kernel(const float* __restrict__ psi, int np, int bfac, int axis, float dcoef,
                    float vcoef, int first, float* __restrict__ pos_d, float* __restrict__ mom_d) {
  const int64_t n3 = (int64_t)np * np * np;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n3;
       i += (int64_t)gridDim.x * blockDim.x) {
    const float s = psi[i] * (float)bfac;
    if (first) {
      const int64_t q = axis == 0 ? i / ((int64_t)np * np) : (axis == 1 ? (i / np) % np : i % np);
      pos_d[i] = (float)(q * bfac) + dcoef * s;
      mom_d[i] = vcoef * s;
    } else {
      pos_d[i] += dcoef * s;
      mom_d[i] += vcoef * s;
    }
  }
}

__global__ void __launch_bounds__(256)
lpt_wrap_kernel(float* __restrict__ pos, int64_t n, float ng, float inv_ng) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x) {
    float x = pos[i];
    x -= ng * floorf(x * inv_ng);
    if (x >= ng) x -= ng;
    if (x < 0.f) x += ng;
    pos[i] = x >= ng ? 0.f : x;
  }
}

__global__ void __launch_bounds__(256)
lpt_source_kernel(float* __restrict__ s, const float* __restrict__ a, const float* __restrict__ b,
                  const float* __restrict__ c, int64_t n, int mode) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x) {
    if (mode == 0) s[i] = a[i] * b[i];
    else if (mode == 1) s[i] += (a[i] + b[i]) * c[i];
    else s[i] -= a[i] * a[i];
  }
}

// g[c] = sum_d (D_d f_d)[c],  (D f)[i] = (-f[i+2] + 8 f[i+1] - 8 f[i-1] + f[i-2]) / 12 along axis d, periodic.
// D has the symbol i g(w) of PAPER.md Eq. 5, so r2c(g) = sum_d i g_d r2c(f_d): the backward pass forms
// this sum in real space and runs ONE potential solve instead of three forward transforms (R12).
// A block owns a 64 (z) x 4 (y) tile and walks kStencilXC planes along x, so the x-difference needs one
// new load per cell and plane (five-deep register ring) and the y / z neighbours come from L1.
constexpr int kStencilXC = 32;
__global__ void __launch_bounds__(256)
stencil_divergence_kernel(const float* __restrict__ f0, const float* __restrict__ f1,
                          const float* __restrict__ f2, int n, float* __restrict__ g) {
  const int mask = n - 1;
  const int z = blockIdx.x * 64 + (threadIdx.x & 63);
  const int y = blockIdx.y * 4 + (threadIdx.x >> 6);
  if (z >= n || y >= n) return;
  const int x0 = blockIdx.z * kStencilXC;
  const int xc = n - x0 < kStencilXC ? n - x0 : kStencilXC;
  const int64_t nn = (int64_t)n * n;
  const int64_t yz = (int64_t)y * n + z;
  const int zm2 = (z - 2) & mask, zm1 = (z - 1) & mask, zp1 = (z + 1) & mask, zp2 = (z + 2) & mask;
  const int64_t ym2 = (int64_t)((y - 2) & mask) * n + z, ym1 = (int64_t)((y - 1) & mask) * n + z,
                yp1 = (int64_t)((y + 1) & mask) * n + z, yp2 = (int64_t)((y + 2) & mask) * n + z;
  float am2 = __ldg(f0 + (int64_t)((x0 - 2) & mask) * nn + yz), am1 = __ldg(f0 + (int64_t)((x0 - 1) & mask) * nn + yz);
  float a0 = __ldg(f0 + (int64_t)x0 * nn + yz), ap1 = __ldg(f0 + (int64_t)((x0 + 1) & mask) * nn + yz);
  for (int i = 0; i < xc; ++i) {
    const int x = x0 + i;
    const int64_t pl = (int64_t)x * nn;
    const float ap2 = __ldg(f0 + (int64_t)((x + 2) & mask) * nn + yz);
    const float dx = -ap2 + 8.f * ap1 - 8.f * am1 + am2;
    const float dy = -__ldg(f1 + pl + yp2) + 8.f * __ldg(f1 + pl + yp1) - 8.f * __ldg(f1 + pl + ym1) + __ldg(f1 + pl + ym2);
    const int64_t row = pl + (int64_t)y * n;
    const float dz = -__ldg(f2 + row + zp2) + 8.f * __ldg(f2 + row + zp1) - 8.f * __ldg(f2 + row + zm1) + __ldg(f2 + row + zm2);
    g[pl + yz] = (dx + dy + dz) * (1.f / 12.f);
    am2 = am1; am1 = a0; a0 = ap1; ap1 = ap2;
  }
}

// y += a x
__global__ void __launch_bounds__(256)
axpy_kernel(float* __restrict__ y, const float* __restrict__ x, float a, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    y[i] = fmaf(a, x[i], y[i]);
}

// out = ca a + cb b
__global__ void __launch_bounds__(256)
lincomb2_kernel(float* __restrict__ out, const float* __restrict__ a, float ca,
                const float* __restrict__ b, float cb, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = ca * a[i] + cb * b[i];
}

// cotangent of a second-derivative field of the 2LPT source S (product rule):
// diagonal: out = sbar (pa + pb) ;  off-diagonal (pb == nullptr): out = -2 sbar pa
__global__ void __launch_bounds__(256)
lpt_phibar_kernel(float* __restrict__ out, const float* __restrict__ sbar, const float* __restrict__ pa,
                  const float* __restrict__ pb, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = pb ? sbar[i] * (pa[i] + pb[i]) : -2.f * sbar[i] * pa[i];
}

inline unsigned grid_for(int64_t n) {
  int64_t b = (n + 255) / 256;
  if (b > 148LL * 32) b = 148LL * 32;
  return (unsigned)(b < 1 ? 1 : b);
}

}  // namespace

cudaError_t kernel_tables_create(int n, int kernel_mode, KernelTables* out) {
  std::vector<float> host(4 * (size_t)n);
  for (int i = 0; i < n; ++i) {
    const int f = i <= n / 2 ? i : i - n;       // integer frequency in (-n/2, n/2]
    const double w = 2.0 * kPi * f / n;
    const bool nyq = (2 * f == n);
    double lap, grad;
    if (kernel_mode == FPM_KERNEL_PAPER) {
      const double s = 2.0 * std::sin(0.5 * w);
      lap = s * s;                                                // Eq. 4, (w sinc(w/2))^2
    } else {
      lap = w * w;
    }
    if (kernel_mode == FPM_KERNEL_NAIVE) grad = w;
    else grad = (8.0 * std::sin(w) - std::sin(2.0 * w)) / 6.0;    // Eq. 5
    if (nyq) grad = 0.0;
    host[i] = (float)lap;
    host[n + i] = (float)grad;
    host[2 * n + i] = (float)w;
    host[3 * n + i] = nyq ? 0.f : (float)w;
  }
  float* dev = nullptr;
  cudaError_t e = cudaMalloc(&dev, host.size() * sizeof(float));
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(dev, host.data(), host.size() * sizeof(float), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaFree(dev); return e; }
  out->n = n;
  out->dev = dev;
  out->lap = dev;
  out->grad = dev + n;
  out->kvec = dev + 2 * n;
  out->kvec0 = dev + 3 * n;
  return cudaSuccess;
}

void kernel_tables_destroy(KernelTables* t) {
  if (t->dev) cudaFree(t->dev);
  *t = KernelTables{};
}

cudaError_t apply_force_kernel(const KernelTables& kt, const float2* dk, float scale, float2* fkx,
                               float2* fky, float2* fkz, cudaStream_t s) {
  force_kernel_rows<<<(unsigned)(kt.n * kt.n), kThreads, 0, s>>>(dk, kt.n, kt.lap, kt.grad, scale,
                                                                fkx, fky, fkz);
  return cudaGetLastError();
}

cudaError_t lpt_spectral(const KernelTables& kt, const float2* in, float2* out, int a, int b,
                         float sign, cudaStream_t s, bool accumulate) {
  lpt_spectral_rows<<<(unsigned)(kt.n * kt.n), kThreads, 0, s>>>(in, out, kt.n, kt.kvec, kt.kvec0, a,
                                                                b, sign, accumulate ? 1 : 0);
  return cudaGetLastError();
}

cudaError_t apply_force_kernel_transpose(const KernelTables& kt, const float2* f0, const float2* f1,
                                         const float2* f2, float scale, float2* out, cudaStream_t s) {
  force_kernel_transpose_rows<<<(unsigned)(kt.n * kt.n), kThreads, 0, s>>>(f0, f1, f2, kt.n, kt.lap,
                                                                          kt.grad, scale, out);
  return cudaGetLastError();
}

cudaError_t stencil_divergence(const float* f0, const float* f1, const float* f2, int n, float* g, cudaStream_t s) {
  dim3 grid((n + 63) / 64, (n + 3) / 4, (n + kStencilXC - 1) / kStencilXC);
  stencil_divergence_kernel<<<grid, 256, 0, s>>>(f0, f1, f2, n, g);
  return cudaGetLastError();
}

cudaError_t axpy(float* y, const float* x, float a, int64_t n, cudaStream_t s) {
  axpy_kernel<<<grid_for(n), 256, 0, s>>>(y, x, a, n);
  return cudaGetLastError();
}

cudaError_t lincomb2(float* out, const float* a, float ca, const float* b, float cb, int64_t n,
                     cudaStream_t s) {
  lincomb2_kernel<<<grid_for(n), 256, 0, s>>>(out, a, ca, b, cb, n);
  return cudaGetLastError();
}

cudaError_t lpt_phibar(float* out, const float* sbar, const float* pa, const float* pb, int64_t n,
                       cudaStream_t s) {
  lpt_phibar_kernel<<<grid_for(n), 256, 0, s>>>(out, sbar, pa, pb, n);
  return cudaGetLastError();
}

cudaError_t lpt_displace(const float* psi, int np, int bfac, int axis, float dcoef, float vcoef,
                         bool first, float* pos_d, float* mom_d, cudaStream_t s) {
  const int64_t n3 = (int64_t)np * np * np;
  lpt_displace_kernel<<<grid_for(n3), 256, 0, s>>>(psi, np, bfac, axis, dcoef, vcoef, first ? 1 : 0,
                                                   pos_d, mom_d);
  return cudaGetLastError();
}

cudaError_t lpt_wrap(float* pos, int64_t n3, int ng, cudaStream_t s) {
  lpt_wrap_kernel<<<grid_for(n3), 256, 0, s>>>(pos, n3, (float)ng, 1.f / ng);
  return cudaGetLastError();
}

cudaError_t lpt_source(float* s, const float* a, const float* b, const float* c, int64_t n, int mode,
                       cudaStream_t st) {
  lpt_source_kernel<<<grid_for(n), 256, 0, st>>>(s, a, b, c, n, mode);
  return cudaGetLastError();
}

}  // namespace fpm
