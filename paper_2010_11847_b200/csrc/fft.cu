// fft.cu -- plan tables and launchers of the 3-D r2c / c2r transforms.
// Forward order z (r2c) -> y -> x; inverse x -> y -> z (c2r).  The y and x passes are in place
// on the half-complex buffer.  No cuFFT anywhere in this library.
#include <cmath>
#include <vector>

#include "fft_kernels.cuh"
#include "fpm_internal.h"

namespace fpm {

namespace {

const double kPi = 3.14159265358979323846264338327950288;

PlanInfo plan_info(int n) {
  switch (n) {
    case 4: return Plan<4>::info();
    case 8: return Plan<8>::info();
    case 16: return Plan<16>::info();
    case 32: return Plan<32>::info();
    case 64: return Plan<64>::info();
    case 128: return Plan<128>::info();
    case 256: return Plan<256>::info();
    case 512: return Plan<512>::info();
    case 1024: return Plan<1024>::info();
    default: return PlanInfo{0, 0, 0, {0, 0, 0}};
  }
}

// stage s >= 1: table[(t-1) NS + k] = exp(-2 pi i t k / (NS R_s)), t = 1..R_s-1, k < NS
PlanInfo plan_info_x(int n) {      // plan of the fused x round trip (fft_x_force_kernel)
  if (n == 512) return Plan<512, 1>::info();
  if (n == 1024) return Plan<1024, 1>::info();
  return plan_info(n);
}

void build_stage_table(const PlanInfo& pi, std::vector<float2>& out) {
  int ns = pi.r[0];
  for (int s = 1; s < pi.nst; ++s) {
    const int r = pi.r[s];
    for (int t = 1; t < r; ++t)
      for (int k = 0; k < ns; ++k) {
        const double ang = -2.0 * kPi * (double)t * k / ((double)ns * r);
        out.push_back(make_float2((float)std::cos(ang), (float)std::sin(ang)));
      }
    ns *= r;
  }
}

template <class K>
cudaError_t set_smem(K kernel, size_t bytes) { return ensure_dynamic_smem(kernel, bytes); }

template <int N, bool INV>
cudaError_t launch_cols(const float2* in, float2* out, int batches, int64_t batch_stride, int ncols,
                        int64_t line_stride, const float2* tw, cudaStream_t s) {
  constexpr int T = col_tile<N>();
  constexpr int threads = T * Plan<N>::P;
  const size_t smem = Plan<N>::NST > 1 ? sizeof(float2) * N * T : 0;
  auto kern = fft_cols_kernel<N, INV, OpNone, OpNone>;
  cudaError_t e = set_smem(kern, smem);
  if (e != cudaSuccess) return e;
  dim3 grid((ncols + T - 1) / T, batches);
  kern<<<grid, threads, smem, s>>>(in, out, batch_stride, ncols, line_stride, tw, OpNone{}, OpNone{});
  return cudaGetLastError();
}

template <int N>
cudaError_t r2c_impl(const FftTables& t, const float* real, float2* cplx, cudaStream_t s,
                     Profiler* prof) {
  constexpr int M = N / 2, nzh = M + 1, G = z_rows<N>();
  const int64_t nrows = (int64_t)N * N;
  {
    ProfScope sc(prof, K_FFT_Z_R2C);
    constexpr int threads = G * Plan<M>::P;
    const size_t smem = sizeof(float2) * G * row_pitch(M);
    auto kern = fft_z_r2c_kernel<N>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)((nrows + G - 1) / G), threads, smem, s>>>(real, cplx, nrows, t.stage_m, t.full, nzh);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  // y: one batch per x slab, columns kz, lines y (stride nzh)
  cudaError_t e;
  {
    ProfScope sc(prof, K_FFT_Y);
    e = launch_cols<N, false>(cplx, cplx, N, (int64_t)N * nzh, nzh, nzh, t.stage_n, s);
  }
  if (e != cudaSuccess) return e;
  // x: columns (y, kz) flattened, lines x (stride N nzh)
  ProfScope sc(prof, K_FFT_X);
  return launch_cols<N, false>(cplx, cplx, 1, 0, N * nzh, (int64_t)N * nzh, t.stage_n, s);
}

template <int N>
cudaError_t launch_z_c2r(const FftTables& t, const float2* cplx, float* real, const float* gz,
                         cudaStream_t s, Profiler* prof, int pitch = N / 2 + 1, int batch = 1) {
  constexpr int M = N / 2, G = z_rows<N>();
  const int64_t nrows = (int64_t)N * N * batch;
  ProfScope sc(prof, K_FFT_Z_C2R);
  constexpr int threads = G * Plan<M>::P;
  const float scale = (float)(1.0 / ((double)N * N * N));
  const unsigned grid = (unsigned)((nrows + G - 1) / G);
  // bulk row loads need whole blocks of an even number of rows (16-byte aligned runs)
  const bool tma = G % 2 == 0 && nrows % G == 0 && (reinterpret_cast<uintptr_t>(cplx) & 15) == 0;
  cudaError_t e;
  if (tma) {
    auto kern = fft_z_c2r_kernel<N, true>;
    e = set_smem(kern, zc_smem_bytes<N>());
    if (e != cudaSuccess) return e;
    kern<<<grid, threads, zc_smem_bytes<N>(), s>>>(cplx, real, nrows, t.stage_m, t.full, scale, gz, pitch);
  } else {
    const size_t smem = Plan<M>::NST > 1 ? sizeof(float2) * G * row_pitch(M) : 0;
    auto kern = fft_z_c2r_kernel<N, false>;
    e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, threads, smem, s>>>(cplx, real, nrows, t.stage_m, t.full, scale, gz, pitch);
  }
  return cudaGetLastError();
}

template <int N>
cudaError_t c2r_impl(const FftTables& t, float2* cplx, float* real, cudaStream_t s, Profiler* prof) {
  constexpr int nzh = N / 2 + 1;
  cudaError_t e;
  {
    ProfScope sc(prof, K_FFT_X);
    e = launch_cols<N, true>(cplx, cplx, 1, 0, N * nzh, (int64_t)N * nzh, t.stage_n, s);
  }
  if (e != cudaSuccess) return e;
  {
    ProfScope sc(prof, K_FFT_Y);
    e = launch_cols<N, true>(cplx, cplx, N, (int64_t)N * nzh, nzh, nzh, t.stage_n, s);
  }
  if (e != cudaSuccess) return e;
  return launch_z_c2r<N>(t, cplx, real, nullptr, s, prof);
}

// Fused force meshes: r2c z, y forward, x round trip with the transfer
// function (one forward, two inverse transforms per column), 3 inverse y passes in one launch, then
// either 3 planar c2r z passes into F[0..2] or, when F4 is given, one launch writing the interleaved
// (F_x, F_y, F_z, 0) mesh (g(w_z) fused into the z pass of the third component either way).
// wa, wb, wc: three half-complex scratch buffers; dk is both input scratch and Fy scratch.  All four are
// internal, with the padded row pitch PZ = padded_pitch(N) (128-byte aligned rows and 16-column tiles).
template <int N>
cudaError_t launch_x_round_trip(const FftTables& t, const KernelTables& kt, const float2* in, float2* out_a,
                                float2* out_bx, float scale, bool poisson, cudaStream_t s, int batch = 1,
                                const CUtensorMap* m_in = nullptr, const CUtensorMap* m_a = nullptr,
                                const CUtensorMap* m_bx = nullptr) {
  constexpr int nzh = N / 2 + 1, PZ = padded_pitch(N), TX = xf_tile<N>();
  const dim3 grid((nzh + TX - 1) / TX, N, batch);
  const unsigned threads = TX * Plan<N, xf_variant<N>()>::P;
  cudaError_t e;
  // (at N = 1024 the three-buffer tile is 192 KB, one block per SM, and the ld.global version with its two
  //  64 KB buffers is faster: 6.1 vs 6.7 ms at C5)
  if (m_in && m_a && (poisson || m_bx) && N <= 512) {     // TMA tile movers
    const size_t smem = xf_tma_smem_bytes<N>();
    if (poisson) {
      auto kern = fft_x_force_tma_kernel<N, true>;
      e = set_smem(kern, smem);
      if (e != cudaSuccess) return e;
      kern<<<grid, threads, smem, s>>>(*m_in, *m_a, *m_a, t.stage_x, kt.lap, kt.grad, scale);
    } else {
      auto kern = fft_x_force_pair_tma_kernel<N>;
      e = set_smem(kern, smem);
      if (e != cudaSuccess) return e;
      kern<<<grid, threads, smem, s>>>(*m_in, *m_a, *m_bx, t.stage_x, kt.lap, kt.grad, scale);
    }
    return cudaGetLastError();
  }
  auto go = [&](auto kern) -> cudaError_t {
    e = set_smem(kern, xf_smem_bytes<N>());
    if (e != cudaSuccess) return e;
    kern<<<grid, threads, xf_smem_bytes<N>(), s>>>(in, out_a, poisson ? nullptr : out_bx, nzh, PZ, t.stage_x, kt.lap,
                                                   kt.grad, scale);
    return cudaGetLastError();
  };
  return poisson ? go(fft_x_force_kernel<N, true, false>) : go(fft_x_force_kernel<N, false, false>);
}

template <int N>
cudaError_t launch_z_r2c_padded(const FftTables& t, const float* real, float2* cplx, cudaStream_t s, int batch = 1) {
  constexpr int M = N / 2, G = z_rows<N>(), PZ = padded_pitch(N);
  const int64_t nrows = (int64_t)N * N * batch;      // rows of consecutive meshes are consecutive
  constexpr int threads = G * Plan<M>::P;
  const size_t smem = sizeof(float2) * G * row_pitch(M);
  auto kern = fft_z_r2c_kernel<N>;
  cudaError_t e = set_smem(kern, smem);
  if (e != cudaSuccess) return e;
  kern<<<(unsigned)((nrows + G - 1) / G), threads, smem, s>>>(real, cplx, nrows, t.stage_m, t.full, PZ);
  return cudaGetLastError();
}

template <int N>
cudaError_t force_fused_impl(const FftTables& t, const KernelTables& kt, const float* rho, float2* dk,
                             float2* wa, float2* wb, float2* wc, float* const* F, float* F4, float scale,
                             cudaStream_t s, Profiler* prof, int batch, const TileMaps* maps) {
  constexpr int nzh = N / 2 + 1, PZ = padded_pitch(N);
  const bool tma = maps && maps->ok;
  // a batch of meshes back to back: its z rows and its x slabs are just more rows / slabs; only the x
  // round trip, whose lines stride across a whole mesh, takes the mesh index as a grid dimension
  if (batch < 1 || (batch > 1 && !F4) || (int64_t)N * batch > 65535) return cudaErrorInvalidValue;
  const int64_t nrows = (int64_t)N * N * batch;
  const int slabs = N * batch;
  cudaError_t e;
  {
    ProfScope sc(prof, K_FFT_Z_R2C);
    e = launch_z_r2c_padded<N>(t, rho, dk, s, batch);
    if (e != cudaSuccess) return e;
  }
  {
    ProfScope sc(prof, K_FFT_Y);
    if (tma) {
      constexpr int TY = yi_tile<N>();
      const size_t ysmem = sizeof(float2) * N * TY + 16;
      dim3 grid((nzh + TY - 1) / TY, slabs);
      auto go = [&](auto kern) {
        e = set_smem(kern, ysmem);
        if (e != cudaSuccess) return;
        kern<<<grid, yi_threads<N>(), ysmem, s>>>(maps->y[0], maps->y[0], maps->y[0], maps->y[0],
                                                  yi_variant<N>() ? t.stage_x : t.stage_n, kt.grad, 0);
        e = cudaGetLastError();
      };
      go(fft_y_inv3_tma_kernel<N, false, (N == 512 ? 6 : 1)>);
    } else {
      e = launch_cols<N, false>(dk, dk, slabs, (int64_t)N * PZ, nzh, PZ, t.stage_n, s);
    }
    if (e != cudaSuccess) return e;
  }
  {
    ProfScope sc(prof, K_FFT_X_FORCE);
    e = launch_x_round_trip<N>(t, kt, dk, wa, wb, scale, false, s, batch, tma ? &maps->x[0] : nullptr,
                               tma ? &maps->x[1] : nullptr, tma ? &maps->x[2] : nullptr);
    if (e != cudaSuccess) return e;
  }
  {
    ProfScope sc(prof, K_FFT_Y_INV3);
    using YPL = Plan<N, yi_variant<N>()>;
    // Fx: wb in place; Fy: g_y A -> dk (free now); Fz: A -> wc
    if (tma) {
      constexpr int TY = yi_tile<N>();
      const size_t ysmem = sizeof(float2) * N * TY + 16;
      dim3 grid(3 * ((nzh + TY - 1) / TY), slabs);
      auto go = [&](auto kern) {
        e = set_smem(kern, ysmem);
        if (e != cudaSuccess) return;
        kern<<<grid, yi_threads<N>(), ysmem, s>>>(maps->y[2], maps->y[1], maps->y[0], maps->y[3],
                                                  yi_variant<N>() ? t.stage_x : t.stage_n, kt.grad, 0);
      };
      go(fft_y_inv3_tma_kernel<N, true, (N == 512 ? 6 : 1)>);
      if (e != cudaSuccess) return e;
    } else {                    // no tensor maps: the ld.global column-pair pass
      constexpr int TY = yi_tile<N>();
      const size_t ysmem = YPL::NST > 1 ? sizeof(float2) * N * TY : 0;
      auto kern = fft_y_inv3_pair_kernel<N>;
      e = set_smem(kern, ysmem);
      if (e != cudaSuccess) return e;
      dim3 grid(3 * ((nzh + TY - 1) / TY), slabs);
      kern<<<grid, yi_threads<N>(), ysmem, s>>>(wb, wa, wb, dk, wc, (int64_t)N * PZ, nzh, PZ,
                                                yi_variant<N>() ? t.stage_x : t.stage_n, kt.grad);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  if (F4) {   // interleaved (F_x, F_y, F_z, -) per cell for the fused readout
    ProfScope sc(prof, K_FFT_Z_C2R3);
    constexpr int GC = z3_rows<N>();
    const size_t zsmem = z3_smem_bytes<N>();
    auto go = [&](auto kern) -> cudaError_t {
      e = set_smem(kern, zsmem);
      if (e != cudaSuccess) return e;
      kern<<<(unsigned)((nrows + GC - 1) / GC), z3_threads<N>(), zsmem, s>>>(
          wb, dk, wc, reinterpret_cast<float4*>(F4), nrows, t.stage_m, t.full,
          (float)(1.0 / ((double)N * N * N)), kt.grad);
      return cudaGetLastError();
    };
    return go(fft_z_c2r3_kernel<N, true>);
  }
  e = launch_z_c2r<N>(t, wb, F[0], nullptr, s, prof, PZ);
  if (e != cudaSuccess) return e;
  e = launch_z_c2r<N>(t, dk, F[1], nullptr, s, prof, PZ);
  if (e != cudaSuccess) return e;
  return launch_z_c2r<N>(t, wc, F[2], kt.grad, s, prof, PZ);
}

// real mesh -> real mesh:  out = c2r[ (scale / K^2) r2c[src] ]  (K^2 of the context's kernel mode, 0 at k = 0),
// with the multiplier fused into the x round trip; work: one half-complex scratch buffer (padded pitch).
template <int N>
cudaError_t poisson_impl(const FftTables& t, const KernelTables& kt, const float* src, float2* work, float* out,
                         float scale, cudaStream_t s, Profiler* prof, const CUtensorMap* work_map_x) {
  constexpr int nzh = N / 2 + 1, PZ = padded_pitch(N);
  cudaError_t e;
  {
    ProfScope sc(prof, K_FFT_Z_R2C);
    e = launch_z_r2c_padded<N>(t, src, work, s);
    if (e != cudaSuccess) return e;
  }
  {
    ProfScope sc(prof, K_FFT_Y);
    e = launch_cols<N, false>(work, work, N, (int64_t)N * PZ, nzh, PZ, t.stage_n, s);
    if (e != cudaSuccess) return e;
  }
  {
    ProfScope sc(prof, K_FFT_X_FORCE);
    e = launch_x_round_trip<N>(t, kt, work, work, nullptr, scale, true, s, 1, work_map_x, work_map_x, nullptr);
    if (e != cudaSuccess) return e;
  }
  {
    ProfScope sc(prof, K_FFT_Y);
    e = launch_cols<N, true>(work, work, N, (int64_t)N * PZ, nzh, PZ, t.stage_n, s);
    if (e != cudaSuccess) return e;
  }
  return launch_z_c2r<N>(t, work, out, nullptr, s, prof, PZ);
}

}  // namespace

namespace {
template <int N>
cudaError_t make_maps_impl(int batch, float2* const bufs[4], TileMaps* out) {
  EncodeTiledFn enc = encode_tiled_fn();
  out->ok = false;
  if (!enc) return cudaSuccess;
  constexpr int nzh = N / 2 + 1, PZ = padded_pitch(N), BOXR = tma_box_rows<N>();
  // a mesh as a 3-D tensor of 8-byte elements: (kz < nzh, pitch PZ) x (y < N) x (x slab < N batch)
  const cuuint64_t dims[3] = {(cuuint64_t)nzh, (cuuint64_t)N, (cuuint64_t)N * batch};
  const cuuint64_t strides[2] = {sizeof(float2) * (cuuint64_t)PZ, sizeof(float2) * (cuuint64_t)PZ * N};
  const cuuint32_t ones[3] = {1, 1, 1};
  const cuuint32_t box_y[3] = {(cuuint32_t)yi_tile<N>(), (cuuint32_t)BOXR, 1};
  const cuuint32_t box_x[3] = {(cuuint32_t)xf_tile<N>(), 1, (cuuint32_t)BOXR};
  for (int i = 0; i < 4; ++i) {
    if (enc(&out->y[i], CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, bufs[i], dims, strides, box_y, ones,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaSuccess;
    if (enc(&out->x[i], CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, bufs[i], dims, strides, box_x, ones,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaSuccess;
  }
  out->ok = true;
  return cudaSuccess;
}
}  // namespace

cudaError_t fft_make_tile_maps(int n, int batch, float2* const bufs[4], TileMaps* out) {
  switch (n) {
    case 8: return make_maps_impl<8>(batch, bufs, out);
    case 16: return make_maps_impl<16>(batch, bufs, out);
    case 32: return make_maps_impl<32>(batch, bufs, out);
    case 64: return make_maps_impl<64>(batch, bufs, out);
    case 128: return make_maps_impl<128>(batch, bufs, out);
    case 256: return make_maps_impl<256>(batch, bufs, out);
    case 512: return make_maps_impl<512>(batch, bufs, out);
    case 1024: return make_maps_impl<1024>(batch, bufs, out);
    default: return cudaErrorInvalidValue;
  }
}

bool fft_size_supported(int n) { return n >= 8 && n <= 1024 && (n & (n - 1)) == 0; }

cudaError_t fft_tables_create(int n, FftTables* out) {
  std::vector<float2> host;
  build_stage_table(plan_info(n), host);
  const size_t off_m = host.size();
  build_stage_table(plan_info(n / 2), host);
  const size_t off_x = host.size();
  build_stage_table(plan_info_x(n), host);
  const size_t off_f = host.size();
  for (int k = 0; k < n / 2; ++k) {
    const double ang = -2.0 * kPi * k / n;
    host.push_back(make_float2((float)std::cos(ang), (float)std::sin(ang)));
  }
  float2* dev = nullptr;
  cudaError_t e = cudaMalloc(&dev, host.size() * sizeof(float2));
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(dev, host.data(), host.size() * sizeof(float2), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaFree(dev); return e; }
  out->n = n;
  out->dev = dev;
  out->stage_n = dev;
  out->stage_m = dev + off_m;
  out->stage_x = dev + off_x;
  out->full = dev + off_f;
  return cudaSuccess;
}

void fft_tables_destroy(FftTables* t) {
  if (t->dev) cudaFree(t->dev);
  *t = FftTables{};
}

#define FPM_FFT_DISPATCH(fn, ...)                        \
  switch (t.n) {                                         \
    case 8: return fn<8>(__VA_ARGS__);                   \
    case 16: return fn<16>(__VA_ARGS__);                 \
    case 32: return fn<32>(__VA_ARGS__);                 \
    case 64: return fn<64>(__VA_ARGS__);                 \
    case 128: return fn<128>(__VA_ARGS__);               \
    case 256: return fn<256>(__VA_ARGS__);               \
    case 512: return fn<512>(__VA_ARGS__);               \
    case 1024: return fn<1024>(__VA_ARGS__);             \
    default: return cudaErrorInvalidValue;               \
  }

cudaError_t fft_r2c(const FftTables& t, const float* real, float2* cplx, cudaStream_t s,
                    Profiler* prof) {
  FPM_FFT_DISPATCH(r2c_impl, t, real, cplx, s, prof)
}
cudaError_t fft_c2r(const FftTables& t, float2* cplx, float* real, cudaStream_t s, Profiler* prof) {
  FPM_FFT_DISPATCH(c2r_impl, t, cplx, real, s, prof)
}

cudaError_t fft_poisson(const FftTables& t, const KernelTables& kt, const float* src, float2* work, float* out,
                        float scale, cudaStream_t s, Profiler* prof, const CUtensorMap* work_map_x) {
  if (kt.n != t.n) return cudaErrorInvalidValue;
  FPM_FFT_DISPATCH(poisson_impl, t, kt, src, work, out, scale, s, prof, work_map_x)
}

cudaError_t fft_force_fused(const FftTables& t, const KernelTables& kt, const float* rho, float2* dk,
                            float2* wa, float2* wb, float2* wc, float* const* F, float* F4, float scale,
                            cudaStream_t s, Profiler* prof, int batch, const TileMaps* maps) {
  if (kt.n != t.n) return cudaErrorInvalidValue;
  FPM_FFT_DISPATCH(force_fused_impl, t, kt, rho, dk, wa, wb, wc, F, F4, scale, s, prof, batch, maps)
}

}  // namespace fpm
