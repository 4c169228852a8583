// fft.cuh -- hand-written batched 1-D FFT passes for the 3-D r2c / c2r transforms of the PM step
// ("one forward 3D FFT ... three inverse FFTs"; Alg. 3 FFT3D / iFFT3D,
// PAPER.md:283-290).  sm_100a design notes:
//   * the transform is HBM-bound (2.8 flop/B), so each axis is exactly one read + one write of
//     the mesh; a thread keeps E = 8..32 complex points in registers, which gives every SM
//     >100 KB of loads in flight with few resident warps;
//   * Stockham autosort stages of radix <= 32 in registers; stages exchange through shared
//     memory once (N <= 1024 needs at most 2 stages); first-stage loads and last-stage stores
//     go straight between HBM and registers;
//   * strided axes (y, x) are processed as tiles of T contiguous columns so that every global
//     access is a >=128-byte segment and shared memory is conflict-free by construction;
//   * inverse transforms run the forward butterflies on (im, re)-swapped data;
//   * inter-stage twiddles come from small per-stage tables laid out [t][k] (coalesced, L1
//     resident, correctly rounded from float64) -- no sincosf in the loop.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <utility>

namespace fpm {

// ------------------------------------------------------------------------------------------
// complex helpers
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cswap(float2 a) { return make_float2(a.y, a.x); }

// The same line position of two ADJACENT columns, transformed together by one thread: a column pass that
// moves 16 bytes per lane touches half as many 128-byte lines per request as one that moves 8 (the L1 data
// pipe, not DRAM, bounded the 8-byte column passes: profiles/r01_E_C4.md), and the two independent
// butterflies give the scheduler twice the instruction-level parallelism.
struct cpair { float2 a, b; };
__device__ __forceinline__ cpair cadd(cpair x, cpair y) { return cpair{cadd(x.a, y.a), cadd(x.b, y.b)}; }
__device__ __forceinline__ cpair csub(cpair x, cpair y) { return cpair{csub(x.a, y.a), csub(x.b, y.b)}; }
__device__ __forceinline__ cpair cmul(cpair x, float2 w) { return cpair{cmul(x.a, w), cmul(x.b, w)}; }
__device__ __forceinline__ cpair cswap(cpair x) { return cpair{cswap(x.a), cswap(x.b)}; }

// cos(2 pi k / 64), k = 0..16 (correctly rounded)
__host__ __device__ constexpr float cos64_table(int k) {
  constexpr float c[17] = {1.0f,
                           0.995184726672196886245f,
                           0.980785280403230449126f,
                           0.956940335732208864936f,
                           0.923879532511286756128f,
                           0.881921264348355029713f,
                           0.831469612302545237079f,
                           0.773010453362736960811f,
                           0.707106781186547524401f,
                           0.634393284163645498215f,
                           0.555570233019602224743f,
                           0.471396736825997648556f,
                           0.382683432365089771728f,
                           0.290284677254462367636f,
                           0.195090322016128267848f,
                           0.0980171403295606019942f,
                           0.0f};
  return c[k];
}
__host__ __device__ constexpr float cos64(int k) {
  k = ((k % 64) + 64) % 64;
  if (k > 32) k = 64 - k;
  return k > 16 ? -cos64_table(32 - k) : cos64_table(k);
}
__host__ __device__ constexpr float sin64(int k) { return cos64(k - 16); }

// x * exp(-2 pi i I / R), resolved at compile time (R a power of two <= 64)
template <int R, int I>
__device__ __forceinline__ float2 mul_twiddle(float2 x);
template <int R, int I>
__device__ __forceinline__ cpair mul_twiddle(cpair x) { return cpair{mul_twiddle<R, I>(x.a), mul_twiddle<R, I>(x.b)}; }
template <int R, int I>
__device__ __forceinline__ float2 mul_twiddle(float2 x) {
  constexpr int k = (I * (64 / R)) % 64;
  if constexpr (k == 0) return x;
  else if constexpr (k == 16) return make_float2(x.y, -x.x);
  else if constexpr (k == 32) return make_float2(-x.x, -x.y);
  else if constexpr (k == 48) return make_float2(-x.y, x.x);
  else {
    constexpr float c = cos64(k), s = -sin64(k);
    return make_float2(x.x * c - x.y * s, x.x * s + x.y * c);
  }
}

// w[e] = w0 * exp(-2 pi i e / R), e < sizeof...(I): the twiddles W_N^(p + P e) of the real-transform split /
// merge from ONE table entry W_N^p (N = 2 E P, so W_N^(P e) = exp(-2 pi i e / (2 E)) is a compile-time constant);
// E - 1 table loads less per thread through the L1 data pipe that bounds the z passes.
template <int R, int... I>
__device__ __forceinline__ void twiddle_ladder(float2 w0, float2 (&w)[sizeof...(I)], std::integer_sequence<int, I...>) {
  ((w[I] = mul_twiddle<R, I>(w0)), ...);
}

// In-register forward DFT of R points (decimation in frequency), natural-order output.
// (C = float2, or cpair: two columns at once)
template <int R>
struct Dft {
  template <class C, int... I>
  static __device__ __forceinline__ void run(C (&v)[R], std::integer_sequence<int, I...>) {
    C e[R / 2], o[R / 2];
    ((e[I] = cadd(v[I], v[I + R / 2]), o[I] = mul_twiddle<R, I>(csub(v[I], v[I + R / 2]))), ...);
    Dft<R / 2>::apply(e);
    Dft<R / 2>::apply(o);
    ((v[2 * I] = e[I], v[2 * I + 1] = o[I]), ...);
  }
  template <class C>
  static __device__ __forceinline__ void apply(C (&v)[R]) {
    run(v, std::make_integer_sequence<int, R / 2>{});
  }
};
template <>
struct Dft<1> {
  template <class C>
  static __device__ __forceinline__ void apply(C (&)[1]) {}
};
template <>
struct Dft<2> {
  template <class C>
  static __device__ __forceinline__ void apply(C (&v)[2]) {
    const C a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
  }
};

// ------------------------------------------------------------------------------------------
// Plans: N = R0 * R1 * R2, every radix <= E (points held per thread), P = N / E threads per line.
// ------------------------------------------------------------------------------------------
struct PlanInfo {
  int n, e, nst, r[3];
};

// V = 0: the default plan of a size; V = 1: an alternative with fewer points per thread (more resident
// warps, one more shared-memory exchange) for kernels that run several transforms per tile.
template <int N, int V = 0> struct Plan;
#define FPM_PLAN(N_, E_, NST_, R0_, R1_, R2_) FPM_PLAN_V(N_, 0, E_, NST_, R0_, R1_, R2_)
#define FPM_PLAN_V(N_, V_, E_, NST_, R0_, R1_, R2_)                                  \
  template <> struct Plan<N_, V_> {                                                      \
    static constexpr int E = E_, NST = NST_, R0 = R0_, R1 = R1_, R2 = R2_;           \
    static constexpr int P = N_ / E_;                                                \
    __host__ __device__ static constexpr int radix(int s) { return s == 0 ? R0_ : (s == 1 ? R1_ : R2_); } \
    /* number of lines already combined before stage s */                            \
    __host__ __device__ static constexpr int ns(int s) { return s == 0 ? 1 : (s == 1 ? R0_ : R0_ * R1_); } \
    /* offset of stage s (>= 1) in the twiddle table */                              \
    __host__ __device__ static constexpr int toff(int s) { return s <= 1 ? 0 : (R1_ - 1) * R0_; } \
    static constexpr int table_len = (NST_ > 1 ? (R1_ - 1) * R0_ : 0) + (NST_ > 2 ? (R2_ - 1) * R0_ * R1_ : 0); \
    static constexpr PlanInfo info() { return PlanInfo{N_, E_, NST_, {R0_, R1_, R2_}}; } \
  };
FPM_PLAN(4, 4, 1, 4, 1, 1)
FPM_PLAN(8, 8, 1, 8, 1, 1)
FPM_PLAN(16, 16, 1, 16, 1, 1)
FPM_PLAN(32, 8, 2, 8, 4, 1)
FPM_PLAN(64, 8, 2, 8, 8, 1)
FPM_PLAN(128, 16, 2, 16, 8, 1)
FPM_PLAN(256, 16, 2, 16, 16, 1)
FPM_PLAN(512, 32, 2, 32, 16, 1)
FPM_PLAN(1024, 32, 2, 32, 32, 1)
FPM_PLAN_V(512, 1, 8, 3, 8, 8, 8)
FPM_PLAN_V(1024, 1, 16, 3, 16, 8, 8)
#undef FPM_PLAN
#undef FPM_PLAN_V

#ifndef FPM_TW_POW
#define FPM_TW_POW 1
#endif
constexpr bool kTwiddlePowers = FPM_TW_POW != 0;

// shared-memory accessors -----------------------------------------------------------------
// column tile: element i of column c at i*T + c.  With T = 16 a line of the tile is 128 bytes, all 32 banks:
// conflict-free by construction.  With T = 8 a line is 64 bytes, half the banks, and the two lines a
// half-warp touches must fall in different halves; the line index is therefore XOR-swizzled with the parity
// of its upper bits, which separates any two lines whose indices differ in exactly one bit (every access
// pattern of the Stockham stages: consecutive lines, or lines a power-of-two stride apart).
template <int T, bool SWZ = false>
struct ColSmem {
  float2* base;
  int c;
  __device__ __forceinline__ static int line(int i) { return (T == 8 && SWZ) ? (i ^ (__popc(i >> 1) & 1)) : i; }
  __device__ __forceinline__ void st(int i, float2 x) const { base[line(i) * T + c] = x; }
  __device__ __forceinline__ float2 ld(int i) const { return base[line(i) * T + c]; }
};
// a tile whose elements are pairs (two spectra of the SAME column, 16 bytes): element i of column c at
// i*T + c; with T = 8 a line is 128 bytes, all 32 banks
template <int T>
struct ColSmemQ {
  float4* base;
  int c;
  __device__ __forceinline__ void st(int i, cpair x) const { base[i * T + c] = make_float4(x.a.x, x.a.y, x.b.x, x.b.y); }
  __device__ __forceinline__ cpair ld(int i) const {
    const float4 q = base[i * T + c];
    return cpair{make_float2(q.x, q.y), make_float2(q.z, q.w)};
  }
};
// Exchange-buffer swizzle for tiles whose lines are 64 bytes (half the banks): line i sits at i ^ bit B of i.
// Two lines a quarter-/half-warp touches together are either neighbours (i, i + 1: they keep opposite halves,
// both flipped or neither) or R0 apart in the first stage's stores (lines R0 p + t of threads p, p + 1: with
// B = log2 R0 exactly one of them flips).  Enumerated over every exchange access of the plans in use: 1.25-1.5
// wavefronts per ideal one without it, 1.0 with it.  Used by the forward exchange of the x round trip
// (fft_x_force 0.467 -> 0.456 ms).
template <int B>
__device__ __forceinline__ int swz_line(int i) { return B > 0 ? (i ^ ((i >> B) & 1)) : i; }
__host__ __device__ constexpr int ilog2_c(int v) { return v <= 1 ? 0 : 1 + ilog2_c(v / 2); }
// a column tile of single elements with the bit swizzle (T = 8: 64-byte lines)
template <int T, int B>
struct ColSmemB {
  float2* base;
  int c;
  __device__ __forceinline__ void st(int i, float2 x) const { base[swz_line<B>(i) * T + c] = x; }
  __device__ __forceinline__ float2 ld(int i) const { return base[swz_line<B>(i) * T + c]; }
};
// the same tile accessed as column pairs: pair c2 of line i is one 16-byte word (T = 16: a line is 128 bytes)
// (with T = 8 the bit swizzle removes the 1.33 x STS.128 conflicts of fft_y_inv3 as well, but its address
// arithmetic does not fit the 40 registers of 6 blocks/SM: 0.461 ms at 5 blocks/SM against 0.452 without)
template <int T>
struct ColSmem2 {
  float4* base;
  int c2;
  __device__ __forceinline__ void st(int i, cpair x) const { base[i * (T / 2) + c2] = make_float4(x.a.x, x.a.y, x.b.x, x.b.y); }
  __device__ __forceinline__ cpair ld(int i) const {
    const float4 q = base[i * (T / 2) + c2];
    return cpair{make_float2(q.x, q.y), make_float2(q.z, q.w)};
  }
};
// contiguous line: lanes run over the butterfly index; one pad slot per 16 breaks stride-R conflicts
struct RowSmem {
  float2* row;
  __device__ __forceinline__ void st(int i, float2 x) const { row[i + (i >> 4)] = x; }
  __device__ __forceinline__ float2 ld(int i) const { return row[i + (i >> 4)]; }
};
__host__ __device__ constexpr int row_pitch(int m) { return m + (m >> 4) + 1; }

// ------------------------------------------------------------------------------------------
// One Stockham stage and the recursive driver.  Thread p of a line holds v[e] = x[p + P e].
// Stage with radix R, NS lines already combined: butterfly j reads x[j + t N/R], multiplies by
// exp(-2 pi i t k/(NS R)), k = j mod NS, and writes y[(j-k) R + k + t NS].
// ------------------------------------------------------------------------------------------
template <class PL, int S, class SM, class C>
__device__ __forceinline__ void fft_stage(C (&v)[PL::E], const int p, const SM& sm,
                                          const float2* __restrict__ tw) {
  constexpr int E = PL::E, P = PL::P, R = PL::radix(S), NS = PL::ns(S), M = E / R;
  constexpr bool last = (S == PL::NST - 1);
#pragma unroll
  for (int u = 0; u < M; ++u) {
    const int j = p + u * P;
    const int k = j & (NS - 1);
    C a[R];
#pragma unroll
    for (int t = 0; t < R; ++t) a[t] = v[u + t * M];
    if constexpr (NS > 1) {
      const float2* __restrict__ tws = tw + PL::toff(S) + k;
      if constexpr (kTwiddlePowers && R >= 4) {
        // only w^1, w^2, w^4, ... are loaded (correctly rounded table entries); w^t for the other t is one
        // complex product of two entries already at hand: the loads go through the same L1 data pipe as the
        // shared-memory exchanges that bound these kernels, the products through the idle FMA pipe
        float2 w[R];
#pragma unroll
        for (int t = 1; t < R; ++t) {
          if ((t & (t - 1)) == 0) w[t] = __ldg(tws + (t - 1) * NS);
          else w[t] = cmul(w[t & (t - 1)], w[t & -t]);
        }
#pragma unroll
        for (int t = 1; t < R; ++t) a[t] = cmul(a[t], w[t]);
      } else {
#pragma unroll
        for (int t = 1; t < R; ++t) a[t] = cmul(a[t], __ldg(tws + (t - 1) * NS));
      }
    }
    Dft<R>::apply(a);
    if constexpr (last) {
#pragma unroll
      for (int t = 0; t < R; ++t) v[u + t * M] = a[t];
    } else {
      const int base = (j - k) * R + k;
#pragma unroll
      for (int t = 0; t < R; ++t) sm.st(base + t * NS, a[t]);
    }
  }
  if constexpr (!last) {
    __syncthreads();
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = sm.ld(p + P * e);
    if constexpr (S + 1 < PL::NST - 1) __syncthreads();
    fft_stage<PL, S + 1, SM, C>(v, p, sm, tw);
  }
}

// forward DFT of one line: in v[e] = x[p + P e], out v[e] = X[p + P e]
template <int N, class SM>
__device__ __forceinline__ void fft_line(float2 (&v)[Plan<N>::E], const int p, const SM& sm,
                                         const float2* __restrict__ tw) {
  fft_stage<Plan<N>, 0, SM, float2>(v, p, sm, tw);
}
// the same with an explicit plan (tw must be that plan's stage table)
template <class PL, class SM, class C>
__device__ __forceinline__ void fft_line_plan(C (&v)[PL::E], const int p, const SM& sm,
                                              const float2* __restrict__ tw) {
  fft_stage<PL, 0, SM, C>(v, p, sm, tw);
}

// row pitch (in complex elements) of the library's INTERNAL half-complex meshes: n/2 + 1 rounded up to 16
// elements = 128 bytes, so every row and every 16-column tile starts on a 128-byte line and column pairs are
// 16-byte aligned.  Buffers that cross the C-ABI keep the dense pitch n/2 + 1 (the cuFFT r2c layout).
__host__ __device__ constexpr int padded_pitch(int n) { return (n / 2 + 1 + 15) & ~15; }

}  // namespace fpm
