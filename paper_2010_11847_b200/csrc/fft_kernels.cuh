// fft_kernels.cuh -- the three pass kernels of the 3-D transform (see fft.cuh for the design).
//   fft_z_r2c_kernel : contiguous axis, real -> half-complex, N/2-point complex FFT + split
//   fft_cols_kernel  : strided axes (y then x forward; x then y inverse), in place, tile of T columns,
//                      with optional element-wise LoadOp/StoreOp (the fused Green's function,
//                      PAPER.md:49-59, rides on the x pass)
//   fft_z_c2r_kernel : contiguous axis, half-complex -> real, merge + N/2-point inverse FFT
#pragma once
#include <cuda.h>

#include "fft.cuh"

namespace fpm {

struct OpNone {
  // v: value, line: index along the transformed axis, col: column index inside the batch
  __device__ __forceinline__ float2 load(float2 v, int, int64_t, int) const { return v; }
  __device__ __forceinline__ float2 store(float2 v, int, int64_t, int) const { return v; }
};

// ---- TMA bulk copy + mbarrier (sm_90+/sm_100a) ------------------------------------------------------------
// One elected thread arms the barrier with the byte count and issues cp.async.bulk; the copy engine writes
// shared memory directly (no LSU data-pipe wavefronts, no registers) and completes the transaction count.
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MBAR_DONE;\n"
      "bra MBAR_WAIT;\n"
      "MBAR_DONE:\n"
      "}\n" ::"r"(a), "r"(parity) : "memory");
}
// global -> shared, bytes a multiple of 16, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, unsigned bytes, uint64_t* bar) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst), b = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(d), "l"(gsrc), "r"(bytes), "r"(b) : "memory");
}

// 3-D tiled tensor copies (cp.async.bulk.tensor): one instruction moves a box of up to 256 lines x 128 bytes
// between a half-complex mesh (dims kz, y, x-slab; padded pitch) and a dense shared-memory tile.  Columns
// beyond n/2 + 1 are out of bounds for the tensor map: zero-filled on load, dropped on store.
__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2,
                                            uint64_t* bar) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst), b = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(d), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(b) : "memory");
}
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, int c0, int c1, int c2, const void* smem_src) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_src);
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.tile.bulk_group [%0, {%2, %3, %4}], [%1];"
               ::"l"(reinterpret_cast<uint64_t>(map)), "r"(sa), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// generic-proxy writes to shared memory -> visible to the async proxy (before a TMA store reads them)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int N> __host__ __device__ constexpr int tma_box_rows() { return N < 256 ? N : 256; }

template <int N> __host__ __device__ constexpr int col_tile() { return N >= 64 ? 16 : 32; }
// resident blocks per SM the column kernels are compiled for: at N = 512 the 64 KB tile allows three,
// which needs <= 85 registers (the compiler otherwise settles just above and only two fit)
template <int N> __host__ __device__ constexpr int cols_min_blocks() { return N == 512 ? 3 : 1; }
template <int N> __host__ __device__ constexpr int z_rows() {          // lines per block on the z pass
  constexpr int P = Plan<N / 2>::P;
  return P >= 256 ? 1 : 256 / P;
}

// in/out may alias (in place): each block reads its whole tile before writing it.
// grid = (ceil(ncols / T), batches); element (line i, column c) of batch b at
//   b * batch_stride + i * line_stride + c.
template <int N, bool INV, class LOADOP, class STOREOP>
__global__ void __launch_bounds__(col_tile<N>() * Plan<N>::P, cols_min_blocks<N>())
fft_cols_kernel(const float2* in, float2* out, int64_t batch_stride, int ncols,
                int64_t line_stride, const float2* __restrict__ tw, LOADOP lop, STOREOP sop) {
  extern __shared__ float2 smem[];
  using PL = Plan<N>;
  constexpr int T = col_tile<N>(), E = PL::E, P = PL::P;
  const int c = threadIdx.x % T, p = threadIdx.x / T;
  const int64_t col = (int64_t)blockIdx.x * T + c;
  const bool ok = col < ncols;
  const int64_t off = (int64_t)blockIdx.y * batch_stride + col;
  float2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = p + P * e;
    float2 x = make_float2(0.f, 0.f);
    if (ok) x = lop.load(in[off + (int64_t)i * line_stride], i, col, blockIdx.y);
    v[e] = INV ? cswap(x) : x;
  }
  ColSmem<T> sm{smem, c};
  fft_line<N>(v, p, sm, tw);
  if (ok) {
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int i = p + P * e;
      const float2 x = INV ? cswap(v[e]) : v[e];
      out[off + (int64_t)i * line_stride] = sop.store(x, i, col, blockIdx.y);
    }
  }
}

// Fused transfer function (Eq. 3-5) on the x axis: forward x transform of the
// y-transformed density, times  i s / K^2  ("A")  and  i s g(w_x) / K^2  ("Bx"), and the two inverse x
// transforms, all inside one block -- delta_k, and the three force spectra of the unfused path, never
// reach HBM.  Since g(w_y) and g(w_z) are constant along x, F_y and F_z follow from A by a
// multiplication in the y and z passes.  The spectrum A is parked in a second shared-memory tile
// while its inverse runs, so the forward transform is done once (1 forward + 2 inverse per column).
// columns = flattened (y, kz), lines = x with stride line_stride; no normalisation here.
// Tile of TX columns; shared memory = [exchange N*TX | parked spectrum N*TX] float2.
#ifndef FPM_XF_TILE_1024
#define FPM_XF_TILE_1024 8
#endif
#ifndef FPM_YI_TILE_1024
#define FPM_YI_TILE_1024 8
#endif
template <int N> __host__ __device__ constexpr int xf_tile() { return N >= 1024 ? FPM_XF_TILE_1024 : (N >= 512 ? 8 : col_tile<N>()); }
// plan variant of the x round trip: three transforms per tile make it compute-latency bound, so at
// N = 512 it runs the 8-points-per-thread plan (32 instead of 12 resident warps per SM)
template <int N> __host__ __device__ constexpr int xf_variant() { return N >= 512 ? 1 : 0; }
template <int N> __host__ __device__ constexpr size_t xf_smem_bytes() {
  return sizeof(float2) * 2 * (size_t)N * xf_tile<N>();
}

// POISSON: only  out_a = inverse_x[ (scale / K^2) forward_x[in] ]  (real multiplier, no gradient variant;
// out_a may alias in) -- the x round trip of the backward pass's single potential solve.
// grid = (ceil(nzh / T), N, batch): block (bx, y, b) owns the T columns kz = bx T .. of row y of mesh b;
// element (x, y, kz) of a mesh at (x N + y) pitch + kz.
template <int N, bool POISSON = false, bool SWZ = false>
__global__ void __launch_bounds__(xf_tile<N>() * Plan<N, xf_variant<N>()>::P, N == 512 ? 2 : 1)
fft_x_force_kernel(const float2* in, float2* out_a,
                   float2* __restrict__ out_bx, int nzh, int pitch,
                   const float2* __restrict__ tw, const float* __restrict__ lap,
                   const float* __restrict__ grad, float scale) {
  extern __shared__ float2 smem[];
  using PL = Plan<N, xf_variant<N>()>;
  constexpr int T = xf_tile<N>(), E = PL::E, P = PL::P;
  const int c = threadIdx.x % T, p = threadIdx.x / T;
  const int y = blockIdx.y, kz = blockIdx.x * T + c;
  const bool ok = kz < nzh;
  // blockIdx.z: mesh of a batch (meshes back to back)
  const int64_t line_stride = (int64_t)N * pitch, col = (int64_t)blockIdx.z * N * line_stride + (int64_t)y * pitch + kz;
  float2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e)
    v[e] = ok ? in[col + (int64_t)(p + P * e) * line_stride] : make_float2(0.f, 0.f);
  ColSmem<T, SWZ> sm{smem, c};
  fft_line_plan<PL>(v, p, sm, tw);
  const float lyz = __ldg(lap + y) + __ldg(lap + (ok ? kz : 0));
  float2* park = smem + N * T + threadIdx.x;          // element e of this thread at park[e * T * P]
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = p + P * e;
    const float k2 = __ldg(lap + i) + lyz;
    const float f = ((y | kz | i) == 0) ? 0.f : scale / k2;
    if constexpr (POISSON) {
      v[e] = make_float2(v[e].y * f, v[e].x * f);        // f v, (im, re)-swapped
    } else {
      // i f v = (-im, re) f ; kept (im, re)-swapped for the inverse transform
      v[e] = make_float2(v[e].x * f, -v[e].y * f);
      park[e * (T * P)] = v[e];
    }
  }
  if constexpr (PL::NST > 1) __syncthreads();
  fft_line_plan<PL>(v, p, sm, tw);
  if (ok) {
#pragma unroll
    for (int e = 0; e < E; ++e) out_a[col + (int64_t)(p + P * e) * line_stride] = cswap(v[e]);
  }
  if constexpr (POISSON) return;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const float g = __ldg(grad + p + P * e);
    const float2 a = park[e * (T * P)];
    v[e] = make_float2(a.x * g, a.y * g);
  }
  if constexpr (PL::NST > 1) __syncthreads();
  fft_line_plan<PL>(v, p, sm, tw);
  if (ok) {
#pragma unroll
    for (int e = 0; e < E; ++e) out_bx[col + (int64_t)(p + P * e) * line_stride] = cswap(v[e]);
  }
}

// The three inverse y passes of the fused force path in one launch.  Block b: tile b / 3 of x slab
// blockIdx.y, variant b % 3:  0: Bx -> Fx (in place),  1: g(w_y) A -> Fy,  2: A -> Fz (g(w_z) is applied
// by the z pass).  in0/out0 may alias; A is read by variants 1 and 2 and written by neither.
// A thread transforms a PAIR of adjacent columns (cpair): every global and shared access is 16 bytes per
// lane, a tile line is 16 columns = one 128-byte line (the meshes have the padded pitch, a multiple of 16).
// At N >= 512 it runs the 8/16-points-per-thread plan variant and 8-column tiles (64-byte lines; 32 / 64 KB).
template <int N> __host__ __device__ constexpr int yi_tile() { return N >= 512 ? 8 : 16; }
template <int N> __host__ __device__ constexpr int yi_variant() { return N >= 512 ? 1 : 0; }
template <int N> __host__ __device__ constexpr int yi_threads() { return (yi_tile<N>() / 2) * Plan<N, yi_variant<N>()>::P; }

template <int N>
__global__ void __launch_bounds__(yi_threads<N>())
fft_y_inv3_pair_kernel(const float2* in_bx, const float2* __restrict__ in_a, float2* out_x,
                  float2* __restrict__ out_y, float2* __restrict__ out_z, int64_t batch_stride,
                  int ncols, int64_t line_stride, const float2* __restrict__ tw,
                  const float* __restrict__ grad) {
  extern __shared__ float2 smem[];
  using PL = Plan<N, yi_variant<N>()>;
  constexpr int T = yi_tile<N>(), E = PL::E, P = PL::P;
  const int c2 = threadIdx.x % (T / 2), p = threadIdx.x / (T / 2);
  const int variant = blockIdx.x % 3;
  const int col = (blockIdx.x / 3) * T + 2 * c2;        // first column of the pair (the pitch is even)
  const bool ok = col < ncols;                          // a pair may hold one pad column: computed, never used
  const int64_t off = (int64_t)blockIdx.y * batch_stride + col;
  const float2* in = variant == 0 ? in_bx : in_a;
  float2* out = variant == 0 ? out_x : (variant == 1 ? out_y : out_z);
  cpair v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = p + P * e;
    float4 q = make_float4(0.f, 0.f, 0.f, 0.f);
    if (ok) q = *reinterpret_cast<const float4*>(in + off + (int64_t)i * line_stride);
    if (variant == 1) { const float g = __ldg(grad + i); q.x *= g; q.y *= g; q.z *= g; q.w *= g; }
    v[e] = cpair{make_float2(q.y, q.x), make_float2(q.w, q.z)};     // (im, re)-swapped: inverse transform
  }
  ColSmem2<T> sm{reinterpret_cast<float4*>(smem), c2};
  fft_line_plan<PL>(v, p, sm, tw);
  if (ok) {
#pragma unroll
    for (int e = 0; e < E; ++e)
      *reinterpret_cast<float4*>(out + off + (int64_t)(p + P * e) * line_stride) =
          make_float4(v[e].a.y, v[e].a.x, v[e].b.y, v[e].b.x);
  }
}

// real rows of N floats -> rows of N/2+1 complex.  twn[k] = exp(-2 pi i k / N), k < N/2.
template <int N>
__global__ void __launch_bounds__(z_rows<N>() * Plan<N / 2>::P)
fft_z_r2c_kernel(const float* __restrict__ in, float2* __restrict__ out, int64_t nrows,
                 const float2* __restrict__ tw, const float2* __restrict__ twn, int out_pitch) {
  extern __shared__ float2 smem[];
  constexpr int M = N / 2;
  using PL = Plan<M>;
  constexpr int E = PL::E, P = PL::P, G = z_rows<N>();
  const int p = threadIdx.x % P, g = threadIdx.x / P;
  const int64_t row = (int64_t)blockIdx.x * G + g;
  const bool ok = row < nrows;
  const float2* src = reinterpret_cast<const float2*>(in) + row * M;
  float2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) v[e] = ok ? src[p + P * e] : make_float2(0.f, 0.f);
  RowSmem sm{smem + g * row_pitch(M)};
  fft_line<M>(v, p, sm, tw);
  if constexpr (PL::NST > 1) __syncthreads();
#pragma unroll
  for (int e = 0; e < E; ++e) sm.st(p + P * e, v[e]);
  __syncthreads();
  if (!ok) return;
  float2* dst = out + row * out_pitch;
  float2 wn[E];
  twiddle_ladder<2 * E>(__ldg(twn + p), wn, std::make_integer_sequence<int, E>{});
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int k = p + P * e;
    const float2 zk = v[e];
    if (k == 0) {
      dst[0] = make_float2(zk.x + zk.y, 0.f);
      dst[M] = make_float2(zk.x - zk.y, 0.f);
    } else {
      const float2 zm = sm.ld(M - k);
      // Xe = (Z[k] + conj Z[M-k])/2, Xo = (Z[k] - conj Z[M-k])/(2i), X[k] = Xe + W_N^k Xo
      const float2 xe = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
      const float2 d = make_float2(0.5f * (zk.x - zm.x), 0.5f * (zk.y + zm.y));
      const float2 xo = make_float2(d.y, -d.x);
      dst[k] = cadd(xe, cmul(wn[e], xo));
    }
  }
}

// rows of N/2+1 complex -> real rows of N floats, times `scale`.
// TMA: the block's G rows are one contiguous, 16-byte aligned run at any even G (dense or padded pitch), so
// they arrive by one bulk copy and the Hermitian merge reads X[k], X[M-k] from shared memory (see
// fft_z_c2r3_kernel); the caller uses it when nrows is a multiple of G.
template <int N> __host__ __device__ constexpr int zc_row_pitch() {
  return row_pitch(N / 2) > padded_pitch(N) ? row_pitch(N / 2) : padded_pitch(N);
}
template <int N> __host__ __device__ constexpr size_t zc_smem_bytes() {
  return sizeof(float2) * (size_t)z_rows<N>() * zc_row_pitch<N>() + 16;
}

template <int N, bool TMA = false>
__global__ void __launch_bounds__(z_rows<N>() * Plan<N / 2>::P)
fft_z_c2r_kernel(const float2* __restrict__ in, float* __restrict__ out, int64_t nrows,
                 const float2* __restrict__ tw, const float2* __restrict__ twn, float scale,
                 const float* __restrict__ gz, int in_pitch) {
  extern __shared__ __align__(128) float2 smem[];
  constexpr int M = N / 2;
  using PL = Plan<M>;
  constexpr int E = PL::E, P = PL::P, G = z_rows<N>();
  const int p = threadIdx.x % P, g = threadIdx.x / P;
  const int64_t row0 = (int64_t)blockIdx.x * G, row = row0 + g;
  const bool ok = row < nrows;
  const float2* src = in + row * in_pitch;
  if (TMA) {
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + G * zc_row_pitch<N>());
    if (threadIdx.x == 0) mbar_init(bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
      const unsigned bytes = (unsigned)(sizeof(float2) * G * in_pitch);
      mbar_expect_tx(bar, bytes);
      bulk_load(smem, in + row0 * in_pitch, bytes, bar);
    }
    mbar_wait(bar, 0);
    src = smem + g * in_pitch;
  }
  float2 v[E], wn[E];
  twiddle_ladder<2 * E>(__ldg(twn + p), wn, std::make_integer_sequence<int, E>{});
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int k = p + P * e;
    float2 z = make_float2(0.f, 0.f);
    if (ok) {
      float2 xk = src[k], xm = src[M - k];
      if (gz) {   // fused gradient along z: g(w_z) with g(0) = g(Nyquist) = 0
        const float gk = __ldg(gz + k), gm = __ldg(gz + M - k);
        xk.x *= gk; xk.y *= gk; xm.x *= gm; xm.y *= gm;
      }
      if (k == 0) {
        z = make_float2(xk.x + xm.x, xk.x - xm.x);
      } else {
        // A = X[k] + conj X[M-k], B = (X[k] - conj X[M-k]) exp(+2 pi i k/N), Z = A + i B
        const float2 a = make_float2(xk.x + xm.x, xk.y - xm.y);
        const float2 d = make_float2(xk.x - xm.x, xk.y + xm.y);
        const float2 w = wn[e];
        const float2 b = cmul(d, make_float2(w.x, -w.y));
        z = make_float2(a.x - b.y, a.y + b.x);
      }
    }
    v[e] = cswap(z);
  }
  if (TMA) __syncthreads();            // the staged rows are in registers: the buffer becomes the exchange buffer
  RowSmem sm{smem + g * row_pitch(M)};
  fft_line<M>(v, p, sm, tw);
  if (!ok) return;
  float2* dst = reinterpret_cast<float2*>(out) + row * M;
#pragma unroll
  for (int e = 0; e < E; ++e) dst[p + P * e] = make_float2(v[e].y * scale, v[e].x * scale);
}


// The three inverse y passes (see fft_y_inv3_pair_kernel) with the tiles moved by TMA: the whole 16-column
// tile (N lines x 128 bytes) lands in shared memory with N / 256 tensor copies issued by one thread, the
// transform runs register-resident out of it, the exchange reuses the same tile, and the result leaves by
// TMA stores.  No global load or store goes through the LSU data pipe, which bounded the ld.global version
// (profiles/r01_E: L1 data-pipe 85 %, 56 % of it global accesses).
// INV3 = false: the plain forward y pass of the same meshes (in place through m_bx), one variant.
// OCC: resident blocks per SM the kernel is compiled for (3 x 64 KB tiles fit at N = 512 with <= 42 registers).
template <int N, bool INV3 = true, int OCC = 1>
__global__ void __launch_bounds__(yi_threads<N>(), OCC)
fft_y_inv3_tma_kernel(const __grid_constant__ CUtensorMap m_bx, const __grid_constant__ CUtensorMap m_a,
                      const __grid_constant__ CUtensorMap m_y, const __grid_constant__ CUtensorMap m_z,
                      const float2* __restrict__ tw, const float* __restrict__ grad, int slab0) {
  extern __shared__ __align__(128) float2 smem[];
  using PL = Plan<N, yi_variant<N>()>;
  constexpr int T = yi_tile<N>(), E = PL::E, P = PL::P, BOXR = tma_box_rows<N>(), NBOX = N / BOXR;
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + N * T);
  const int c2 = threadIdx.x % (T / 2), p = threadIdx.x / (T / 2);
  const int variant = INV3 ? blockIdx.x % 3 : 0, col0 = (INV3 ? blockIdx.x / 3 : blockIdx.x) * T,
            slab = slab0 + blockIdx.y;
  const CUtensorMap* in = variant == 0 ? &m_bx : &m_a;
  const CUtensorMap* out = variant == 0 ? &m_bx : (variant == 1 ? &m_y : &m_z);
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) {
    mbar_expect_tx(bar, (unsigned)(sizeof(float2) * N * T));
#pragma unroll
    for (int b = 0; b < NBOX; ++b) tma_load_3d(smem + b * BOXR * T, in, col0, b * BOXR, slab, bar);
  }
  mbar_wait(bar, 0);
  float4* tile4 = reinterpret_cast<float4*>(smem);
  cpair v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = p + P * e;
    float4 q = tile4[i * (T / 2) + c2];
    if (INV3 && variant == 1) { const float g = __ldg(grad + i); q.x *= g; q.y *= g; q.z *= g; q.w *= g; }
    // inverse: (im, re)-swapped data through the forward butterflies
    v[e] = INV3 ? cpair{make_float2(q.y, q.x), make_float2(q.w, q.z)} : cpair{make_float2(q.x, q.y), make_float2(q.z, q.w)};
  }
  if constexpr (PL::NST > 1) __syncthreads();       // the landed tile is in registers: it becomes the exchange buffer
  ColSmem2<T> sm{tile4, c2};
  fft_line_plan<PL>(v, p, sm, tw);
  if constexpr (PL::NST > 1) __syncthreads();       // last exchange read: the tile becomes the output stage
#pragma unroll
  for (int e = 0; e < E; ++e)
    tile4[(p + P * e) * (T / 2) + c2] = INV3 ? make_float4(v[e].a.y, v[e].a.x, v[e].b.y, v[e].b.x)
                                             : make_float4(v[e].a.x, v[e].a.y, v[e].b.x, v[e].b.y);
  fence_proxy_async();
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int b = 0; b < NBOX; ++b) tma_store_3d(out, col0, b * BOXR, slab, smem + b * BOXR * T);
    tma_store_commit();
    tma_store_wait_read();
  }
}

// The fused x round trip (see fft_x_force_kernel) with TMA tiles: input tile -> stage buffer; A leaves from the
// stage buffer and Bx from the park buffer while the next transform runs, so no store is waited for before
// the end.  Shared memory = [exchange | park | stage] (3 N T complex) + the barrier.
template <int N> __host__ __device__ constexpr size_t xf_tma_smem_bytes() {
  return sizeof(float2) * 3 * (size_t)N * xf_tile<N>() + 16;
}

// VAR: plan variant.  (The 32-points-per-thread, one-exchange plan Plan<512, 0> halves the shared-memory
// traffic but leaves 8 warps per SM: 0.617 vs 0.522 ms.)
template <int N, bool POISSON = false, int VAR = xf_variant<N>()>
__global__ void __launch_bounds__(xf_tile<N>() * Plan<N, VAR>::P, N == 512 ? 2 : 1)
fft_x_force_tma_kernel(const __grid_constant__ CUtensorMap m_in, const __grid_constant__ CUtensorMap m_a,
                       const __grid_constant__ CUtensorMap m_bx, const float2* __restrict__ tw,
                       const float* __restrict__ lap, const float* __restrict__ grad, float scale) {
  extern __shared__ __align__(128) float2 smem[];
  using PL = Plan<N, VAR>;
  constexpr int T = xf_tile<N>(), E = PL::E, P = PL::P, BOXR = tma_box_rows<N>(), NBOX = N / BOXR;
  float2* xch = smem;
  float2* park_tile = smem + N * T;
  float2* stage = smem + 2 * N * T;
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + 3 * N * T);
  const int c = threadIdx.x % T, p = threadIdx.x / T;
  const int y = blockIdx.y, col0 = blockIdx.x * T, kz = col0 + c, x0 = blockIdx.z * N;
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) {
    mbar_expect_tx(bar, (unsigned)(sizeof(float2) * N * T));
#pragma unroll
    for (int b = 0; b < NBOX; ++b) tma_load_3d(stage + b * BOXR * T, &m_in, col0, y, x0 + b * BOXR, bar);
  }
  mbar_wait(bar, 0);
  float2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) v[e] = stage[(p + P * e) * T + c];
  ColSmem<T> sm{xch, c};
  fft_line_plan<PL>(v, p, sm, tw);
  const float lyz = __ldg(lap + y) + __ldg(lap + (kz <= N / 2 ? kz : 0));
  float2* park = park_tile + threadIdx.x;              // element e of this thread at park[e * T * P]
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = p + P * e;
    const float k2 = __ldg(lap + i) + lyz;
    const float f = ((y | kz | i) == 0) ? 0.f : scale / k2;
    if constexpr (POISSON) {
      v[e] = make_float2(v[e].y * f, v[e].x * f);        // f v, (im, re)-swapped
    } else {
      v[e] = make_float2(v[e].x * f, -v[e].y * f);       // i f v, (im, re)-swapped
      park[e * (T * P)] = v[e];
    }
  }
  if constexpr (PL::NST > 1) __syncthreads();
  fft_line_plan<PL>(v, p, sm, tw);
  // every thread read its part of the stage buffer before the first transform's barriers: reuse it for A
#pragma unroll
  for (int e = 0; e < E; ++e) stage[(p + P * e) * T + c] = cswap(v[e]);
  fence_proxy_async();
  if constexpr (!POISSON) {
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const float g = __ldg(grad + p + P * e);
      const float2 a = park[e * (T * P)];
      v[e] = make_float2(a.x * g, a.y * g);
    }
  }
  __syncthreads();                                      // A staged (and the park slots read) by every thread
  if (threadIdx.x == 0) {
#pragma unroll
    for (int b = 0; b < NBOX; ++b) tma_store_3d(&m_a, col0, y, x0 + b * BOXR, stage + b * BOXR * T);
    tma_store_commit();
  }
  if constexpr (!POISSON) {
    fft_line_plan<PL>(v, p, sm, tw);
#pragma unroll
    for (int e = 0; e < E; ++e) park_tile[(p + P * e) * T + c] = cswap(v[e]);
    fence_proxy_async();
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
      for (int b = 0; b < NBOX; ++b) tma_store_3d(&m_bx, col0, y, x0 + b * BOXR, park_tile + b * BOXR * T);
      tma_store_commit();
    }
  }
  if (threadIdx.x == 0) tma_store_wait_read();
}

// The same round trip with the two inverse transforms run TOGETHER as one transform of pairs
// (A, g(w_x) A): the pair lives in registers, so the spectrum is never parked in shared memory, the two
// inverses share their barriers, and the pair exchange moves 16 bytes per element in 128-byte tile lines
// (conflict-free, unlike the 64-byte lines of the 8-column complex tile).  15 instead of 17 passes over the
// tile through the L1 data pipe, which bounds this kernel (profiles/r02_final_C4.md: 79 %).
// Shared memory = [pair exchange 2 N T | stage N T] complex + the barrier (the same 96 KB at N = 512).
template <int N>
__global__ void __launch_bounds__(xf_tile<N>() * Plan<N, xf_variant<N>()>::P, N == 512 ? 2 : 1)
fft_x_force_pair_tma_kernel(const __grid_constant__ CUtensorMap m_in, const __grid_constant__ CUtensorMap m_a,
                            const __grid_constant__ CUtensorMap m_bx, const float2* __restrict__ tw,
                            const float* __restrict__ lap, const float* __restrict__ grad, float scale) {
  extern __shared__ __align__(128) float2 smem[];
  using PL = Plan<N, xf_variant<N>()>;
  constexpr int T = xf_tile<N>(), E = PL::E, P = PL::P, BOXR = tma_box_rows<N>(), NBOX = N / BOXR;
  float2* xch = smem;                                   // 2 N T complex: forward exchange, pair exchange, B_x stage
  float2* stage = smem + 2 * N * T;                     // N T complex: input tile, then A stage
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + 3 * N * T);
  const int c = threadIdx.x % T, p = threadIdx.x / T;
  const int y = blockIdx.y, col0 = blockIdx.x * T, kz = col0 + c, x0 = blockIdx.z * N;
  if (threadIdx.x == 0) mbar_init(bar, 1);
  __syncthreads();
  if (threadIdx.x == 0) {
    mbar_expect_tx(bar, (unsigned)(sizeof(float2) * N * T));
#pragma unroll
    for (int b = 0; b < NBOX; ++b) tma_load_3d(stage + b * BOXR * T, &m_in, col0, y, x0 + b * BOXR, bar);
  }
  mbar_wait(bar, 0);
  cpair w[E];
  {
    float2 v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = stage[(p + P * e) * T + c];
    ColSmemB<T, T == 8 ? ilog2_c(PL::R0) : 0> sm{xch, c};   // 64-byte lines: swizzled
    fft_line_plan<PL>(v, p, sm, tw);
    const float lyz = __ldg(lap + y) + __ldg(lap + (kz <= N / 2 ? kz : 0));
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int i = p + P * e;
      const float k2 = __ldg(lap + i) + lyz;
      const float f = ((y | kz | i) == 0) ? 0.f : scale / k2;
      const float g = __ldg(grad + i);
      const float2 a = make_float2(v[e].x * f, -v[e].y * f);       // i f v, (im, re)-swapped
      w[e] = cpair{a, make_float2(a.x * g, a.y * g)};
    }
  }
  if constexpr (PL::NST > 1) __syncthreads();           // the forward exchange is read: reuse it for the pairs
  ColSmemQ<T> smq{reinterpret_cast<float4*>(xch), c};
  fft_line_plan<PL>(w, p, smq, tw);
  if constexpr (PL::NST > 1) __syncthreads();           // the last pair exchange is read: B_x is staged over it
#pragma unroll
  for (int e = 0; e < E; ++e) {
    stage[(p + P * e) * T + c] = cswap(w[e].a);
    xch[(p + P * e) * T + c] = cswap(w[e].b);
  }
  fence_proxy_async();
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int b = 0; b < NBOX; ++b) tma_store_3d(&m_a, col0, y, x0 + b * BOXR, stage + b * BOXR * T);
#pragma unroll
    for (int b = 0; b < NBOX; ++b) tma_store_3d(&m_bx, col0, y, x0 + b * BOXR, xch + b * BOXR * T);
    tma_store_commit();
    tma_store_wait_read();
  }
}

// The three c2r z passes of the fused force path in one launch, writing the force mesh interleaved
// per cell as float4 (F_x, F_y, F_z, 0): the readout then needs one 16-byte gather per CIC corner
// instead of three 4-byte ones (round-1 ncu capture: the gather was request- and latency-bound).
// A block owns GC rows; its three thread groups (GC*P threads each, whole warps) invert the rows of
// component 0, 1, 2 concurrently, each with its own exchange buffer, park the real rows there, and
// the block then writes its GC*N cells as fully coalesced float4.
// The input rows (padded pitch: the GC rows of a component are one contiguous, 16-byte aligned run) arrive
// by ONE TMA bulk copy per component into the exchange buffers: the Hermitian merge reads X[k] and X[M-k],
// which as global loads fetched every element twice through L1 (profiles/r01_E: L1 data pipe 69 %, 60 % of
// it global-load wavefronts).
// g(w_z) of Eq. 5 is applied on load to component 2 (see fft_z_c2r_kernel).
template <int N> __host__ __device__ constexpr int z3_rows() {
  constexpr int g = z_rows<N>() / 8;   // swept 2 / 4 / 8 at N = 512: 0.92 / 0.87 / 0.84 ms
  return g < 2 ? 2 : g;                // even, so a block's rows are a 16-byte multiple at any pitch
}
template <int N> __host__ __device__ constexpr int z3_threads() { return 3 * z3_rows<N>() * Plan<N / 2>::P; }
template <int N> __host__ __device__ constexpr int z3_row_pitch() {
  return row_pitch(N / 2) > padded_pitch(N) ? row_pitch(N / 2) : padded_pitch(N);
}
template <int N> __host__ __device__ constexpr size_t z3_smem_bytes() {
  return sizeof(float2) * 3 * (size_t)z3_rows<N>() * z3_row_pitch<N>() + 16;
}

template <int N, bool TMA = true>
__global__ void __launch_bounds__(z3_threads<N>())
fft_z_c2r3_kernel(const float2* __restrict__ in0, const float2* __restrict__ in1,
                  const float2* __restrict__ in2, float4* __restrict__ out4, int64_t nrows,
                  const float2* __restrict__ tw, const float2* __restrict__ twn, float scale,
                  const float* __restrict__ gz) {
  extern __shared__ __align__(128) float2 smem[];
  constexpr int M = N / 2, PZ = padded_pitch(N);
  using PL = Plan<M>;
  constexpr int E = PL::E, P = PL::P, GC = z3_rows<N>(), TG = GC * P, R = GC * z3_row_pitch<N>();
  static_assert(TG % 32 == 0 || TG * 3 <= 32, "component groups are whole warps");
  static_assert((GC * PZ) % 2 == 0 && (R % 2) == 0, "bulk copies move 16-byte multiples to 16-byte aligned regions");
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + 3 * R);
  const int comp = threadIdx.x / TG, t = threadIdx.x % TG;
  const int p = t % P, g = t / P;
  const int64_t row0 = (int64_t)blockIdx.x * GC, row = row0 + g;   // nrows = N^2 is a multiple of GC
  float2* region = smem + comp * R;
  if (TMA) {
    if (threadIdx.x == 0) mbar_init(bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
      constexpr unsigned bytes = sizeof(float2) * GC * PZ;
      mbar_expect_tx(bar, 3 * bytes);
      bulk_load(smem, in0 + row0 * PZ, bytes, bar);
      bulk_load(smem + R, in1 + row0 * PZ, bytes, bar);
      bulk_load(smem + 2 * R, in2 + row0 * PZ, bytes, bar);
    }
    mbar_wait(bar, 0);
  }
  const float2* src = TMA ? region + g * PZ : (comp == 0 ? in0 : (comp == 1 ? in1 : in2)) + row * PZ;
  float2 v[E], wn[E];
  twiddle_ladder<2 * E>(__ldg(twn + p), wn, std::make_integer_sequence<int, E>{});
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int k = p + P * e;
    float2 xk = src[k], xm = src[M - k];
    if (comp == 2) {
      const float gk = __ldg(gz + k), gm = __ldg(gz + M - k);
      xk.x *= gk; xk.y *= gk; xm.x *= gm; xm.y *= gm;
    }
    float2 z;
    if (k == 0) {
      z = make_float2(xk.x + xm.x, xk.x - xm.x);
    } else {
      const float2 a = make_float2(xk.x + xm.x, xk.y - xm.y);
      const float2 d = make_float2(xk.x - xm.x, xk.y + xm.y);
      const float2 w = wn[e];
      const float2 b = cmul(d, make_float2(w.x, -w.y));
      z = make_float2(a.x - b.y, a.y + b.x);
    }
    v[e] = cswap(z);
  }
  if (TMA) __syncthreads();                       // every input row is in registers: the regions become exchange buffers
  RowSmem sm{region + g * row_pitch(M)};
  fft_line<M>(v, p, sm, tw);
  if constexpr (PL::NST > 1) __syncthreads();   // exchange buffers free: park the real rows in them
  // cells (2k, 2k+1) of row g = (im, re) of the swapped result
#pragma unroll
  for (int e = 0; e < E; ++e) region[g * M + p + P * e] = make_float2(v[e].y * scale, v[e].x * scale);
  __syncthreads();
  const float* b0 = reinterpret_cast<const float*>(smem);
  const float* b1 = reinterpret_cast<const float*>(smem + R);
  const float* b2 = reinterpret_cast<const float*>(smem + 2 * R);
  const int64_t left = nrows - row0;
  const int cells = (int)(left < GC ? left : GC) * N;
  float4* dst = out4 + row0 * N;
  for (int i = threadIdx.x; i < cells; i += 3 * TG) dst[i] = make_float4(b0[i], b1[i], b2[i], 0.f);
}

}  // namespace fpm
