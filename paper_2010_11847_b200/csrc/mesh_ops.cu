// mesh_ops.cu -- cloud-in-cell paint (scatter), readout (gather) and their position gradients.
// PAPER.md:47 "linear window of unit size corresponding to the cloud-in-cell (CIC) interpolation
// scheme"; PAPER.md:51 readout "with the same kernel"; adjoints per SURVEY.md 8(c) R11.
//
// sm_100a design:
//   * Particles of a run are stored in Lagrangian (lattice) order and move a few cells at most, so a
//     brick of 8 x 16 x 32 lattice neighbours stays a compact Eulerian cloud.  One CTA owns one
//     brick (or half of one).  Readout: the brick's gathers hit the same few mesh rows, which therefore
//     stay in that SM's L1; bricks are scheduled in memory order so the mesh streams through L2 exactly
//     once; the streamed per-particle operands arrive through a cp.async ring (rkd_pipelined_kernel,
//     brick_gather_kernel) and the force components are interleaved per cell (one 16-byte gather).
//   * Paint: global fp32 reductions are bounded by the L2 atomic units (measured ~0.6 T RED/s, 8 per
//     particle), so the brick accumulates into a shared-memory window placed at its mean
//     displacement and flushes the window with one 16-byte vector reduction per 4 cells
//     (RED.E.ADD.F32x4); the few particles outside the window fall back to direct reductions.
//     Shared memory has no native fp32 add (ATOMS.CAST.SPIN loop), so the window accumulates in
//     32-bit fixed point with a per-brick scale that cannot overflow (native ATOMS.ADD).
#include <cstdlib>
#include <type_traits>

#include "fpm_internal.h"

namespace fpm {

namespace {

struct Cic {
  int i0[3], i1[3];
  float t[3];
};

// floor / round-to-nearest without the conversion (XU) pipe: adding 1.5 * 2^23 leaves the integer in
// the low mantissa bits.  Exact for |x| < 2^22, far beyond any position in mesh cells (ng <= 1024);
// FRND/F2I issue at a quarter of the FMA rate and dominated the paint kernel in the first round-1 capture.
constexpr float kMagic = 12582912.f;
constexpr int kMagicBits = 0x4B400000;
__device__ __forceinline__ float fast_rint(float x, int& i) {
  const float t = x + kMagic;
  i = __float_as_int(t) - kMagicBits;
  return t - kMagic;
}
__device__ __forceinline__ float fast_floor(float x, int& i) {
  float r = fast_rint(x, i);
  if (r > x) { r -= 1.f; i -= 1; }
  return r;
}
// round(a * b) with one rounding: the product is formed inside the FMA that adds the magic constant
__device__ __forceinline__ int fast_round_mul_to_int(float a, float b) {
  return __float_as_int(fmaf(a, b, kMagic)) - kMagicBits;
}
__device__ __forceinline__ Cic cic_of(float x, float y, float z, int mask) {
  Cic c;
  const float p[3] = {x, y, z};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    int i;
    const float fl = fast_floor(p[d], i);
    c.t[d] = p[d] - fl;
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

// same, for arrays the kernel updates in place (no .nc; ordered against the later stores)
__device__ __forceinline__ float ld_stream_rw(const float* p) {
  float v;
  asm volatile("ld.global.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
  return v;
}

constexpr int kThreads = 256;

// ---- Lagrangian bricks ------------------------------------------------------------------------
// Brick = BX x BY x BZ neighbouring lattice sites (z fastest, one warp = one 128-byte z run).
constexpr int BX = 8, BY = 16, BZ = 32;
constexpr int kBrick = BX * BY * BZ;          // 4096 particles
constexpr int kBrickThreads = 512;
constexpr int kPerThread = kBrick / kBrickThreads;

struct BrickMap {
  int np, nbz, nby, lg_np;
  __device__ __forceinline__ void origin(int64_t bid, int& qx0, int& qy0, int& qz0) const {
    const int bz = (int)(bid % nbz);
    const int64_t r = bid / nbz;
    qz0 = bz * BZ;
    qy0 = (int)(r % nby) * BY;
    qx0 = (int)(r / nby) * BX;
  }
  // particle index of slot s (0 .. kBrick-1) of the brick with lattice origin (qx0, qy0, qz0)
  __device__ __forceinline__ int64_t index(int qx0, int qy0, int qz0, int s) const {
    const int lz = s & (BZ - 1), ly = (s >> 5) & (BY - 1), lx = s >> 9;
    return ((int64_t)(qx0 + lx) * np + (qy0 + ly)) * np + (qz0 + lz);
  }
};

inline bool brick_ok(int64_t n, int np) {
  return np >= 32 && np % 32 == 0 && n == (int64_t)np * np * np;
}

// ---- paint: direct reductions --------------------------------------------------------------------
__device__ __forceinline__ void deposit_global(float* __restrict__ mesh, int g, const Cic& c,
                                               float m) {
  const float wx[2] = {m * (1.f - c.t[0]), m * c.t[0]};
  const float wy[2] = {1.f - c.t[1], c.t[1]};
  const float wz[2] = {1.f - c.t[2], c.t[2]};
  const unsigned ix[2] = {(unsigned)c.i0[0], (unsigned)c.i1[0]}, iy[2] = {(unsigned)c.i0[1], (unsigned)c.i1[1]};
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      float* row = mesh + (ix[a] * (unsigned)g + iy[b]) * (unsigned)g;   // ng^3 <= 2^30
      const float w = wx[a] * wy[b];
      atomicAdd(row + c.i0[2], w * wz[0]);
      atomicAdd(row + c.i1[2], w * wz[1]);
    }
}

// One thread per particle in memory order, 8 fp32 reductions (RED.ADD.F32) into L2.  Blocks are
// contiguous chunks so the touched mesh rows form a sliding window that stays in L2.
__global__ void __launch_bounds__(kThreads)
paint_direct_kernel(const float* __restrict__ pos, const float* __restrict__ mass, float mass_const,
                    int64_t n, int ng, float* __restrict__ mesh) {
  const int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (p >= n) return;
  const Cic c = cic_of(ld_stream(pos + p), ld_stream(pos + n + p), ld_stream(pos + 2 * n + p), ng - 1);
  deposit_global(mesh, ng, c, mass ? ld_stream(mass + p) : mass_const);
}

// ---- paint: brick window in shared memory ----------------------------------------------------------
// Window of the brick (resolution factor 1): brick extent + kHalo cells either side + 1 (CIC reaches
// the next cell); z is padded so the origin can be rounded down to a multiple of 4 cells.
// Halo swept at C4 over the whole 40-step schedule (paint ms/step): 4 -> 1.034, 3 -> 1.001, 2 -> 0.986,
// 1 -> 1.016 (more particles take the slow path); late steps (a > 0.9): 1.137 / - / 1.117 / 1.190.
constexpr int kHalo = 2;
constexpr int WX = BX + 2 * kHalo + 1, WY = BY + 2 * kHalo + 1;
constexpr int WZ = (BZ + 2 * kHalo + 1 + 3 + 3) & ~3;
constexpr int kWinCells = WX * WY * WZ;       // 13 x 21 x 40 = 10920 cells, 43.7 KB

// floor without the conversion pipe: a round-down add of 1.5 * 2^23 leaves floor(x) in the low mantissa
// bits (exact for |x| < 2^22).  Returns floor(x) as a float; bits = kMagicBits + floor(x).
__device__ __forceinline__ float floor_magic(float x, int& bits) {
  const float t = __fadd_rd(x, kMagic);
  bits = __float_as_int(t);
  return t - kMagic;
}

// shared-memory reductions at [addr + OFF] with the offset folded into the instruction (ATOMS.ADD with an
// immediate): one base register serves the 8 corners of a particle
template <int OFF>
__device__ __forceinline__ void red_shared(unsigned addr, int v) {
  asm volatile("red.shared.add.u32 [%0+%2], %1;" ::"r"(addr), "r"(v), "n"(OFF) : "memory");
}
template <int OFF>
__device__ __forceinline__ void red_shared(unsigned addr, float v) {
  asm volatile("red.shared.add.f32 [%0+%2], %1;" ::"r"(addr), "f"(v), "n"(OFF) : "memory");
}
// the four cells (y, y+1) x (z, z+1) of one x plane of the window
template <int OFF, class V>
__device__ __forceinline__ void red_plane(unsigned addr, const V (&v)[4]) {
  red_shared<OFF>(addr, v[0]);
  red_shared<OFF + 4>(addr, v[1]);
  red_shared<OFF + 4 * WZ>(addr, v[2]);
  red_shared<OFF + 4 * WZ + 4>(addr, v[3]);
}

// RES = ng / np (1 or 2): the lattice spacing in cells.  The CTA's sub-brick of (8 x 16 x 32) / RES lattice
// sites always spans 8 x 16 x 32 cells, so the window is the same; with RES = 2 a thread owns one particle.
//
// FIXED: the window accumulates round(m w s) as 32-bit integers (native ATOMS.ADD), s a per-brick power of
// two:  s = 2^floor(log2 min(2^30 / sum_p |m_p|, 2^21 / max_p |m_p|))  (2^31 when every mass is the same
// positive constant: all deposits are >= 0 and the window is read back as unsigned).  No cell can overflow:
// a particle gives a cell at most its whole mass, so |cell| <= s sum|m| + particles/2 < 2^31 (resp. 2^32);
// the magic-number rounding needs |m w s| < 2^22.  Error per deposit <= 1/(2 s): 2^-20 m for the density
// paint of a run, <= max(2^-19 mean|m|, 2^-22 max|m|) with per-particle masses.  A brick whose masses are
// badly conditioned for that (max|m| > 64 mean|m|) or not finite is deposited with plain fp32 reductions
// instead, so an outlier or a NaN/Inf behaves as it would in the direct kernel.
// XMERGE (RES = 1): a thread's 8 particles are neighbours along x; when particle k+1 falls in the next x
// plane of the same (y, z) cell column, its lower-plane deposits are added in registers to the upper-plane
// deposits of particle k and go out as 4 reductions instead of 8.
template <bool FIXED, bool HAS_MASS, int RES = 1, bool XMERGE = false, int OCC = 2>
__global__ void __launch_bounds__(kBrickThreads, OCC)
paint_brick_kernel(const float* __restrict__ pos, const float* __restrict__ mass, float mass_const,
                   int64_t n, BrickMap bm, int ng, float* __restrict__ mesh) {
  constexpr int SX = BX / RES, SY = BY / RES, SZ = BZ / RES;          // lattice sites of the sub-brick
  constexpr int kPerThread = SX * SY * SZ / kBrickThreads;
  constexpr int kPerCta = SX * SY * SZ;
  static_assert(kPerThread >= 1 && SX % kPerThread == 0, "sub-brick shape");
  static_assert(!XMERGE || (RES == 1 && FIXED), "x-merge is implemented for the fixed-point lattice walk");
  using V = typename std::conditional<FIXED, int, float>::type;
  extern __shared__ __align__(16) float win_f[];
  __shared__ int red_i[3][kBrickThreads / 32];
  __shared__ float red_f[2][kBrickThreads / 32];
  // blockIdx.y: simulation of a batch ([batch][3][n] particles, [batch][ng^3] meshes)
  pos += (int64_t)blockIdx.y * 3 * n;
  mesh += (int64_t)blockIdx.y * ng * ng * ng;
  if (HAS_MASS) mass += (int64_t)blockIdx.y * n;
  const int mask = ng - 1;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // sub-brick origin (lattice sites): np is a power of two, so the brick coordinates are bit fields
  const int lg_nbz = bm.lg_np - (RES == 1 ? 5 : 4), lg_nby = bm.lg_np - (RES == 1 ? 4 : 3);
  const unsigned bid = blockIdx.x;
  const int qz0 = (int)(bid & ((1u << lg_nbz) - 1)) * SZ, qy0 = (int)((bid >> lg_nbz) & ((1u << lg_nby) - 1)) * SY,
            qx0 = (int)(bid >> (lg_nbz + lg_nby)) * SX;
  const int lz = tid % SZ, ly = (tid / SZ) % SY, lx0 = tid / (SZ * SY);
  constexpr int kDx = kBrickThreads / (SZ * SY);     // lattice planes advanced per k

  float x[kPerThread], y[kPerThread], z[kPerThread], m[HAS_MASS ? kPerThread : 1];
  const int64_t plane = (int64_t)bm.np * bm.np;
  const int64_t p0 = ((int64_t)(qx0 + lx0) * bm.np + (qy0 + ly)) * bm.np + (qz0 + lz);
  const float *px = pos + p0, *py = px + n, *pz = py + n;
#pragma unroll
  for (int k = 0; k < kPerThread; ++k) {
    const int64_t o = (int64_t)(k * kDx) * plane;
    x[k] = ld_stream(px + o);
    y[k] = ld_stream(py + o);
    z[k] = ld_stream(pz + o);
    if (HAS_MASS) m[k] = ld_stream(mass + p0 + o);
  }
  for (int i = tid; i < kWinCells / 4; i += kBrickThreads)
    reinterpret_cast<float4*>(win_f)[i] = make_float4(0.f, 0.f, 0.f, 0.f);

  // Window placement: mean cell displacement floor(x) - site (wrapped to [-ng/2, ng/2)) over a sample of the
  // brick's x planes, in integers (order-independent, so every thread gets the same origin).  The position
  // only decides how many particles take the slow path, never the result.
  constexpr int kMeanPlanes = kPerThread >= 2 ? 2 : 1, kMeanStep = kPerThread / kMeanPlanes;
  constexpr int kLgCnt = (RES == 1 ? 10 : 9);        // log2(kBrickThreads * kMeanPlanes)
  static_assert((1 << kLgCnt) == kBrickThreads * kMeanPlanes, "mean sample count");
  int sx = 0, sy = 0, sz = 0;
  const int half = ng >> 1;
#pragma unroll
  for (int k = 0; k < kPerThread; k += kMeanStep) {
    int bx, by, bz;
    floor_magic(x[k], bx); floor_magic(y[k], by); floor_magic(z[k], bz);
    sx += ((bx - kMagicBits - (qx0 + lx0 + k * kDx) * RES + half) & mask) - half;
    sy += ((by - kMagicBits - (qy0 + ly) * RES + half) & mask) - half;
    sz += ((bz - kMagicBits - (qz0 + lz) * RES + half) & mask) - half;
  }
  sx = __reduce_add_sync(0xffffffffu, sx);
  sy = __reduce_add_sync(0xffffffffu, sy);
  sz = __reduce_add_sync(0xffffffffu, sz);
  float sumabs = 0.f;
  unsigned mmax_bits = 0;
  if (HAS_MASS) {
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
      sumabs += fabsf(m[k]);
      mmax_bits = max(mmax_bits, (unsigned)__float_as_int(fabsf(m[k])));   // |m| as bits: NaN > Inf > finite
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sumabs += __shfl_xor_sync(0xffffffffu, sumabs, o);
    mmax_bits = __reduce_max_sync(0xffffffffu, mmax_bits);
  }
  if (lane == 0) {
    red_i[0][warp] = sx; red_i[1][warp] = sy; red_i[2][warp] = sz;
    if (HAS_MASS) { red_f[0][warp] = sumabs; red_f[1][warp] = __uint_as_float(mmax_bits); }
  }
  __syncthreads();   // also orders the window zeroing before the deposits
  constexpr int kWarps = kBrickThreads / 32;
  sx = __reduce_add_sync(0xffffffffu, lane < kWarps ? red_i[0][lane] : 0);
  sy = __reduce_add_sync(0xffffffffu, lane < kWarps ? red_i[1][lane] : 0);
  sz = __reduce_add_sync(0xffffffffu, lane < kWarps ? red_i[2][lane] : 0);
  // mean displacement = mean(floor) + 1/2 on average; the window is centred on floor(mean)
  const int ox = qx0 * RES + ((sx + (1 << (kLgCnt - 1))) >> kLgCnt) - kHalo;
  const int oy = qy0 * RES + ((sy + (1 << (kLgCnt - 1))) >> kLgCnt) - kHalo;
  const int oz = (qz0 * RES + ((sz + (1 << (kLgCnt - 1))) >> kLgCnt) - kHalo) & ~3;
  float mmax = fabsf(mass_const);
  sumabs = (float)kPerCta * mmax;
  bool use_window = true;
  if (HAS_MASS) {
    sumabs = lane < kWarps ? red_f[0][lane] : 0.f;
    mmax_bits = lane < kWarps ? (unsigned)__float_as_int(red_f[1][lane]) : 0u;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sumabs += __shfl_xor_sync(0xffffffffu, sumabs, o);
    mmax_bits = __reduce_max_sync(0xffffffffu, mmax_bits);
    mmax = __uint_as_float(mmax_bits);
    // fixed point only for a finite, reasonably conditioned brick (see the kernel comment)
    if (FIXED) use_window = mmax_bits < 0x7F800000u && sumabs < 3.0e38f && mmax * (float)kPerCta <= 64.f * sumabs;
  }
  const bool nonneg = !HAS_MASS && mass_const > 0.f;
  float scale = 1.f;
  if (FIXED) {
    const float cap = fminf((nonneg ? 2147483648.f : 1073741824.f) / sumabs, 2097152.f / mmax);
    scale = (mmax > 0.f && use_window) ? __int_as_float(__float_as_int(cap) & 0x7F800000) : 0.f;
  }
  const unsigned win_s = (unsigned)__cvta_generic_to_shared(win_f);
  const int cx = -kMagicBits - ox, cy = -kMagicBits - oy, cz = -kMagicBits - oz;

  unsigned pend = 0xffffffffu;     // XMERGE: window address of the deposits waiting in pv
  V pv[4] = {};
#pragma unroll
  for (int k = 0; k < kPerThread; ++k) {
    int bx, by, bz;
    const float tx = x[k] - floor_magic(x[k], bx), ty = y[k] - floor_magic(y[k], by),
                tz = z[k] - floor_magic(z[k], bz);
    const unsigned rx = (bx + cx) & mask, ry = (by + cy) & mask, rz = (bz + cz) & mask;
    const float mk = HAS_MASS ? m[k] : mass_const;
    if (rx < WX - 1 && ry < WY - 1 && rz < WZ - 1 && use_window) {
      const float mm = mk * scale;
      const float m0 = mm - mm * tx, m1 = mm * tx;                 // mass in x planes ix, ix + 1
      const float w00 = m0 - m0 * ty, w01 = m0 * ty, w10 = m1 - m1 * ty, w11 = m1 * ty;
      const float wz0 = 1.f - tz;
      const unsigned addr = win_s + 4u * ((rx * WY + ry) * WZ + rz);
      V lo[4], hi[4];
      if (FIXED) {
        lo[0] = fast_round_mul_to_int(w00, wz0); lo[1] = fast_round_mul_to_int(w00, tz);
        lo[2] = fast_round_mul_to_int(w01, wz0); lo[3] = fast_round_mul_to_int(w01, tz);
        hi[0] = fast_round_mul_to_int(w10, wz0); hi[1] = fast_round_mul_to_int(w10, tz);
        hi[2] = fast_round_mul_to_int(w11, wz0); hi[3] = fast_round_mul_to_int(w11, tz);
      } else {
        lo[0] = w00 * wz0; lo[1] = w00 * tz; lo[2] = w01 * wz0; lo[3] = w01 * tz;
        hi[0] = w10 * wz0; hi[1] = w10 * tz; hi[2] = w11 * wz0; hi[3] = w11 * tz;
      }
      if (XMERGE) {
        if (addr == pend) {
#pragma unroll
          for (int j = 0; j < 4; ++j) lo[j] += pv[j];
        } else if (pend != 0xffffffffu) {
          red_plane<0>(pend, pv);
        }
        red_plane<0>(addr, lo);
        pend = addr + 4u * WY * WZ;
#pragma unroll
        for (int j = 0; j < 4; ++j) pv[j] = hi[j];
      } else {
        red_plane<0>(addr, lo);
        red_plane<4 * WY * WZ>(addr, hi);
      }
    } else {
      Cic c;
      c.t[0] = tx; c.t[1] = ty; c.t[2] = tz;
      const int ix = bx - kMagicBits, iy = by - kMagicBits, iz = bz - kMagicBits;
      c.i0[0] = ix & mask; c.i1[0] = (ix + 1) & mask;
      c.i0[1] = iy & mask; c.i1[1] = (iy + 1) & mask;
      c.i0[2] = iz & mask; c.i1[2] = (iz + 1) & mask;
      deposit_global(mesh, ng, c, mk);
    }
  }
  if (XMERGE && pend != 0xffffffffu) red_plane<0>(pend, pv);
  __syncthreads();

  // flush: one 16-byte vector reduction per 4 z-cells (oz and ng are multiples of 4)
  const float inv_scale = FIXED ? (scale > 0.f ? 1.f / scale : 0.f) : 1.f;
  constexpr int WZ4 = WZ / 4;
  // (kx, ky, kz) of group gidx advance incrementally: no division in the loop
  constexpr int dKz = kBrickThreads % WZ4, dRow = kBrickThreads / WZ4, dKy = dRow % WY, dKx = dRow / WY;
  static_assert(dKy + 1 < WY, "one carry per step");
  int kz = tid % WZ4, ky = (tid / WZ4) % WY, kx = (tid / WZ4) / WY;
  const int* win_i = reinterpret_cast<const int*>(win_f);
  for (int gidx = tid; gidx < kWinCells / 4; gidx += kBrickThreads) {
    const int4 q = reinterpret_cast<const int4*>(win_i)[gidx];
    // (an all-zero group holds no deposit, in fixed point and -- as +0.0f bit patterns or -0.0f -- in fp32)
    if (((q.x | q.y | q.z | q.w) & (FIXED ? -1 : 0x7fffffff)) != 0) {
      float4 v;
      if (!FIXED)
        v = make_float4(__int_as_float(q.x), __int_as_float(q.y), __int_as_float(q.z), __int_as_float(q.w));
      else if (nonneg)
        v = make_float4(__uint2float_rn((unsigned)q.x) * inv_scale, __uint2float_rn((unsigned)q.y) * inv_scale,
                        __uint2float_rn((unsigned)q.z) * inv_scale, __uint2float_rn((unsigned)q.w) * inv_scale);
      else
        v = make_float4(q.x * inv_scale, q.y * inv_scale, q.z * inv_scale, q.w * inv_scale);
      const unsigned gx = (ox + kx) & mask, gy = (oy + ky) & mask, gz = (oz + 4 * kz) & mask;
      atomicAdd(reinterpret_cast<float4*>(mesh + ((gx * (unsigned)ng + gy) * (unsigned)ng + gz)), v);
    }
    kz += dKz; ky += dKy; kx += dKx;
    if (kz >= WZ4) { kz -= WZ4; ky += 1; }
    if (ky >= WY) { ky -= WY; kx += 1; }
  }
}

// ---- readout -----------------------------------------------------------------------------------
// 32-bit cell indices (ng <= 1024: ng^3 <= 2^30), so every gather address is one IMAD.WIDE.U32; the
// 64-bit row arithmetic was most of the instruction count of the readout kernels in a round-1 capture.
template <int NMESH>
__device__ __forceinline__ void gather(const float* const* mesh, const Cic& c, unsigned g,
                                       float (&acc)[NMESH]) {
  const float wx[2] = {1.f - c.t[0], c.t[0]};
  const float wy[2] = {1.f - c.t[1], c.t[1]};
  const float wz[2] = {1.f - c.t[2], c.t[2]};
  const unsigned ix[2] = {(unsigned)c.i0[0] * g, (unsigned)c.i1[0] * g};
  const unsigned iy[2] = {(unsigned)c.i0[1], (unsigned)c.i1[1]};
  const unsigned z0 = (unsigned)c.i0[2], z1 = (unsigned)c.i1[2];
#pragma unroll
  for (int k = 0; k < NMESH; ++k) acc[k] = 0.f;
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const unsigned row = (ix[a] + iy[b]) * g;
      const float w = wx[a] * wy[b];
      const float w0 = w * wz[0], w1 = w * wz[1];
#pragma unroll
      for (int k = 0; k < NMESH; ++k) {
        acc[k] = fmaf(__ldg(mesh[k] + (row + z0)), w0, acc[k]);
        acc[k] = fmaf(__ldg(mesh[k] + (row + z1)), w1, acc[k]);
      }
    }
}

// The three force components interleaved per cell (x, y, z, unused): one 16-byte load per corner.
__device__ __forceinline__ void gather4(const float4* __restrict__ mesh, const Cic& c, unsigned g,
                                        float (&acc)[3]) {
  const float wx[2] = {1.f - c.t[0], c.t[0]};
  const float wy[2] = {1.f - c.t[1], c.t[1]};
  const float wz[2] = {1.f - c.t[2], c.t[2]};
  const unsigned ix[2] = {(unsigned)c.i0[0] * g, (unsigned)c.i1[0] * g};
  const unsigned iy[2] = {(unsigned)c.i0[1], (unsigned)c.i1[1]};
  const unsigned z0 = (unsigned)c.i0[2], z1 = (unsigned)c.i1[2];
  acc[0] = acc[1] = acc[2] = 0.f;
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const unsigned row = (ix[a] + iy[b]) * g;
      const float w = wx[a] * wy[b];
      const float w0 = w * wz[0], w1 = w * wz[1];
      const float4 v0 = __ldg(mesh + (row + z0)), v1 = __ldg(mesh + (row + z1));
      acc[0] = fmaf(v0.x, w0, acc[0]); acc[1] = fmaf(v0.y, w0, acc[1]); acc[2] = fmaf(v0.z, w0, acc[2]);
      acc[0] = fmaf(v1.x, w1, acc[0]); acc[1] = fmaf(v1.y, w1, acc[1]); acc[2] = fmaf(v1.z, w1, acc[2]);
    }
}

// particle handled by (block, thread, k): brick order when bm.np > 0, memory order otherwise
template <int NMESH, bool BRICK>
__global__ void __launch_bounds__(BRICK ? kBrickThreads : kThreads)
readout_kernel(const float* __restrict__ m0, const float* __restrict__ m1,
               const float* __restrict__ m2, const float* __restrict__ pos, int64_t n, int ng,
               BrickMap bm, float* __restrict__ out) {
  const float* const mesh3[3] = {m0, m1, m2};
  const float* meshn[NMESH];
#pragma unroll
  for (int j = 0; j < NMESH; ++j) meshn[j] = mesh3[j];
  int qx0 = 0, qy0 = 0, qz0 = 0;
  if (BRICK) bm.origin(blockIdx.x, qx0, qy0, qz0);
  constexpr int K = BRICK ? kPerThread : 1;
#pragma unroll 2
  for (int k = 0; k < K; ++k) {
    int64_t p;
    if (BRICK) p = bm.index(qx0, qy0, qz0, threadIdx.x + k * kBrickThreads);
    else { p = (int64_t)blockIdx.x * kThreads + threadIdx.x; if (p >= n) return; }
    const Cic c = cic_of(ld_stream(pos + p), ld_stream(pos + n + p), ld_stream(pos + 2 * n + p), ng - 1);
    float acc[NMESH];
    gather<NMESH>(meshn, c, ng, acc);
#pragma unroll
    for (int j = 0; j < NMESH; ++j) out[j * n + p] = acc[j];
  }
}

__device__ __forceinline__ float wrap_box(float x, float ng, float inv_ng) {
  int unused;
  x -= ng * fast_floor(x * inv_ng, unused);
  if (x >= ng) x -= ng;
  if (x < 0.f) x += ng;
  return x >= ng ? 0.f : x;
}

// One pass over the particles: gather the three force components at x (CIC),
// p += f * kfac (Eq. 2), x = wrap(x + p * dfac) (Eq. 1).  Generic variant: one thread per particle in
// memory order, for particle sets that are not a full lattice (the brick variant follows).
// F4: fx is the interleaved (F_x, F_y, F_z, -) mesh written by fft_z_c2r3_kernel.
template <bool F4>
__global__ void __launch_bounds__(kThreads, 4)
readout_kick_drift_kernel(const float* __restrict__ fx, const float* __restrict__ fy,
                          const float* __restrict__ fz, float* __restrict__ pos,
                          float* __restrict__ mom, int64_t n, int ngi, float kfac, float dfac) {
  const float ng = (float)ngi, inv_ng = 1.f / ng;
  const float* const mesh[3] = {fx, fy, fz};
  const int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (p >= n) return;
  float x[3], m[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    x[d] = ld_stream_rw(pos + d * n + p);
    m[d] = ld_stream_rw(mom + d * n + p);
  }
  const Cic c = cic_of(x[0], x[1], x[2], ngi - 1);
  float acc[3];
  if (F4) gather4(reinterpret_cast<const float4*>(fx), c, ngi, acc);
  else gather<3>(mesh, c, ngi, acc);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const float mn = fmaf(acc[d], kfac, m[d]);
    __stcs(mom + d * n + p, mn);
    __stcs(pos + d * n + p, wrap_box(fmaf(mn, dfac, x[d]), ng, inv_ng));
  }
}

// ---- pipelined brick variant ----------------------------------------------------------------
// The streaming operands (x, p of the next planes) are fetched with cp.async into a small
// shared-memory ring while the current planes are gathered, so the DRAM latency of the 48 B/particle
// stream is never on a warp's critical path.  Each warp copies exactly the 32 particles it will
// process (12 runs of 128 B per batch = 96 16-byte copies, 3 per lane), so the ring needs only
// warp-level synchronisation.  .cg copies bypass L1, which stays reserved for the mesh gathers.
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int STAGES, int KB, int MINB, bool F4 = false>
__global__ void __launch_bounds__(kThreads, MINB)
rkd_pipelined_kernel(const float* __restrict__ fx, const float* __restrict__ fy,
                     const float* __restrict__ fz, float* __restrict__ pos, float* __restrict__ mom,
                     int64_t n, int ngi, BrickMap bm, float kfac, float dfac) {
  static_assert(BX % KB == 0, "batch shape");
  constexpr int NB = BX / KB;             // batches (groups of KB x-planes) per half-brick
  constexpr int DIST = STAGES - 1;        // prefetch distance
  constexpr int NCP = KB * 6 * 8;         // 16-byte copies per warp and batch
  constexpr int CPL = (NCP + 31) / 32;
  __shared__ __align__(16) float ring[STAGES][KB][6][kThreads];
  const float ng = (float)ngi, inv_ng = 1.f / ng;
  // blockIdx.y: simulation of a batch (interleaved force mesh only: [batch][ng^3] float4)
  pos += (int64_t)blockIdx.y * 3 * n;
  mom += (int64_t)blockIdx.y * 3 * n;
  if (F4) fx += (int64_t)blockIdx.y * 4 * ngi * ngi * ngi;
  const float* const mesh[3] = {fx, fy, fz};
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int qx0, qy0, qz0;
  static_assert(kThreads == (BY / 2) * BZ, "a CTA walks half a brick: 8 of its 16 y rows, all x planes");
  bm.origin(blockIdx.x >> 1, qx0, qy0, qz0);
  const int64_t plane = (int64_t)bm.np * bm.np;
  // lattice row of this warp in plane 0 of the brick: lane 0's particle index
  const int64_t row0 = ((int64_t)qx0 * bm.np + (qy0 + (BY / 2) * (blockIdx.x & 1) + warp)) * bm.np + qz0;

  auto issue = [&](int batch) {
    const int st = batch % STAGES;
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
      const int t = lane + 32 * i, r = t >> 3, c = t & 7;
      if (NCP % 32 != 0 && t >= NCP) break;
      const int j = r / 6, a = r - 6 * j;
      const float* src = (a < 3 ? pos + a * n : mom + (a - 3) * n) + row0 + (int64_t)(batch * KB + j) * plane + 4 * c;
      cp_async16(&ring[st][j][a][warp * 32 + 4 * c], src);
    }
  };
#pragma unroll
  for (int b = 0; b < DIST; ++b) { if (b < NB) issue(b); cp_async_commit(); }
#pragma unroll 1
  for (int b = 0; b < NB; ++b) {
    if (b + DIST < NB) issue(b + DIST);
    cp_async_commit();
    cp_async_wait<DIST>();
    __syncwarp();
    const int st = b % STAGES;
#pragma unroll
    for (int j = 0; j < KB; ++j) {
      const int64_t p = row0 + lane + (int64_t)(b * KB + j) * plane;
      float x[3], m[3];
#pragma unroll
      for (int d = 0; d < 3; ++d) { x[d] = ring[st][j][d][tid]; m[d] = ring[st][j][3 + d][tid]; }
      const Cic c = cic_of(x[0], x[1], x[2], ngi - 1);
      float acc[3];
      if (F4) gather4(reinterpret_cast<const float4*>(fx), c, ngi, acc);
      else gather<3>(mesh, c, ngi, acc);
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const float mn = fmaf(acc[d], kfac, m[d]);
        __stcs(mom + d * n + p, mn);
        __stcs(pos + d * n + p, wrap_box(fmaf(mn, dfac, x[d]), ng, inv_ng));
      }
    }
    __syncwarp();   // the stage is refilled by the issue of the next iteration
  }
}

// out3[d][p] = s_p * sum_c mesh[c] dW/dx_d ; optional out_value[p] = sum_c mesh[c] W
__global__ void __launch_bounds__(kThreads)
readout_grad_kernel(const float* __restrict__ mesh, const float* __restrict__ pos,
                    const float* __restrict__ scale, float scale_const, int64_t n, int ng,
                    float* __restrict__ out3, float* __restrict__ out_value, int accumulate) {
  const int64_t g = ng;
  const int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (p >= n) return;
  const Cic c = cic_of(ld_stream(pos + p), ld_stream(pos + n + p), ld_stream(pos + 2 * n + p), ng - 1);
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
  if (accumulate) {
    out3[p] = fmaf(s, gx, out3[p]);
    out3[n + p] = fmaf(s, gy, out3[n + p]);
    out3[2 * n + p] = fmaf(s, gz, out3[2 * n + p]);
  } else {
    out3[p] = s * gx;
    out3[n + p] = s * gy;
    out3[2 * n + p] = s * gz;
  }
  if (out_value) out_value[p] = val;
}

// Direct term of the force VJP: the force f_d = readout(F_d, x) depends on x
// through the CIC weights;  gx[e][p] += coef * sum_d v[d][p] * sum_c F_d[c] dW/dx_e.
__global__ void __launch_bounds__(kThreads)
readout3_grad_accum_kernel(const float* __restrict__ f0, const float* __restrict__ f1,
                           const float* __restrict__ f2, const float* __restrict__ pos,
                           const float* __restrict__ v, float coef, int64_t n, int ng,
                           float* __restrict__ gx) {
  const int64_t p = (int64_t)blockIdx.x * kThreads + threadIdx.x;
  if (p >= n) return;
  const unsigned g = ng;
  const Cic c = cic_of(ld_stream(pos + p), ld_stream(pos + n + p), ld_stream(pos + 2 * n + p), ng - 1);
  const float v0 = ld_stream(v + p), v1 = ld_stream(v + n + p), v2 = ld_stream(v + 2 * n + p);
  const float wx[2] = {1.f - c.t[0], c.t[0]};
  const float wy[2] = {1.f - c.t[1], c.t[1]};
  const float wz[2] = {1.f - c.t[2], c.t[2]};
  const float sg[2] = {-1.f, 1.f};
  const unsigned ix[2] = {(unsigned)c.i0[0], (unsigned)c.i1[0]}, iy[2] = {(unsigned)c.i0[1], (unsigned)c.i1[1]},
                 iz[2] = {(unsigned)c.i0[2], (unsigned)c.i1[2]};
  float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const unsigned row = (ix[a] * g + iy[b]) * g;
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const unsigned i = row + iz[e];
        const float f = v0 * __ldg(f0 + i) + v1 * __ldg(f1 + i) + v2 * __ldg(f2 + i);
        ax = fmaf(f, sg[a] * wy[b] * wz[e], ax);
        ay = fmaf(f, wx[a] * sg[b] * wz[e], ay);
        az = fmaf(f, wx[a] * wy[b] * sg[e], az);
      }
    }
  gx[p] = fmaf(coef, ax, gx[p]);
  gx[n + p] = fmaf(coef, ay, gx[n + p]);
  gx[2 * n + p] = fmaf(coef, az, gx[2 * n + p]);
}

// ---- generic pipelined brick walker (backward-pass gathers) ------------------------------------------
// Same ring as rkd_pipelined_kernel, for NPL streamed planes and a per-particle functor:
// op(vals[NPL], out[NOUT]) computes NOUT results that are stored to the planes dst[0..NOUT-1].
template <int NPL>
struct Planes { const float* src[NPL]; };
template <int NOUT>
struct OutPlanes { float* dst[NOUT]; };

template <int STAGES, int NPL, int NOUT, class OP>
__global__ void __launch_bounds__(kThreads, 4)
brick_gather_kernel(Planes<NPL> in, OutPlanes<NOUT> out, BrickMap bm, OP op) {
  constexpr int DIST = STAGES - 1, NCP = NPL * 8, CPL = (NCP + 31) / 32;
  __shared__ __align__(16) float ring[STAGES][NPL][kThreads];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int qx0, qy0, qz0;
  bm.origin(blockIdx.x >> 1, qx0, qy0, qz0);
  const int64_t plane = (int64_t)bm.np * bm.np;
  const int64_t row0 = ((int64_t)qx0 * bm.np + (qy0 + (BY / 2) * (blockIdx.x & 1) + warp)) * bm.np + qz0;
  auto issue = [&](int b) {
    const int st = b % STAGES;
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
      const int t = lane + 32 * i, a = t >> 3, c = t & 7;
      if (NCP % 32 != 0 && t >= NCP) break;
      cp_async16(&ring[st][a][warp * 32 + 4 * c], in.src[a] + row0 + (int64_t)b * plane + 4 * c);
    }
  };
#pragma unroll
  for (int b = 0; b < DIST; ++b) { if (b < BX) issue(b); cp_async_commit(); }
#pragma unroll 1
  for (int b = 0; b < BX; ++b) {
    if (b + DIST < BX) issue(b + DIST);
    cp_async_commit();
    cp_async_wait<DIST>();
    __syncwarp();
    const int st = b % STAGES;
    float vals[NPL], res[NOUT];
#pragma unroll
    for (int a = 0; a < NPL; ++a) vals[a] = ring[st][a][tid];
    op(vals, res);
    const int64_t p = row0 + lane + (int64_t)b * plane;
#pragma unroll
    for (int a = 0; a < NOUT; ++a) __stcs(out.dst[a] + p, res[a]);
    __syncwarp();
  }
}

// planes: x y z | v0 v1 v2 | gx gy gz ; result: g + coef * sum_d v_d sum_c F_d[c] dW/dx  (interleaved F)
struct ForceVjpDirectOp {
  const float4* mesh;
  unsigned g;
  float coef;
  __device__ __forceinline__ void operator()(const float (&v)[9], float (&r)[3]) const {
    const Cic c = cic_of(v[0], v[1], v[2], (int)g - 1);
    const float wx[2] = {1.f - c.t[0], c.t[0]}, wy[2] = {1.f - c.t[1], c.t[1]}, wz[2] = {1.f - c.t[2], c.t[2]};
    const float sg[2] = {-1.f, 1.f};
    const unsigned ix[2] = {(unsigned)c.i0[0] * g, (unsigned)c.i1[0] * g};
    const unsigned iy[2] = {(unsigned)c.i0[1], (unsigned)c.i1[1]}, iz[2] = {(unsigned)c.i0[2], (unsigned)c.i1[2]};
    float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        const unsigned row = (ix[a] + iy[b]) * g;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const float4 F = __ldg(mesh + (row + iz[e]));
          const float f = v[3] * F.x + v[4] * F.y + v[5] * F.z;
          ax = fmaf(f, sg[a] * wy[b] * wz[e], ax);
          ay = fmaf(f, wx[a] * sg[b] * wz[e], ay);
          az = fmaf(f, wx[a] * wy[b] * sg[e], az);
        }
      }
    r[0] = fmaf(coef, ax, v[6]);
    r[1] = fmaf(coef, ay, v[7]);
    r[2] = fmaf(coef, az, v[8]);
  }
};

// planes: x y z | gx gy gz ; result: g + scale * sum_c mesh[c] dW/dx
struct GradAccumOp {
  const float* mesh;
  unsigned g;
  float scale;
  __device__ __forceinline__ void operator()(const float (&v)[6], float (&r)[3]) const {
    const Cic c = cic_of(v[0], v[1], v[2], (int)g - 1);
    const float wx[2] = {1.f - c.t[0], c.t[0]}, wy[2] = {1.f - c.t[1], c.t[1]}, wz[2] = {1.f - c.t[2], c.t[2]};
    const float sg[2] = {-1.f, 1.f};
    const unsigned ix[2] = {(unsigned)c.i0[0] * g, (unsigned)c.i1[0] * g};
    const unsigned iy[2] = {(unsigned)c.i0[1], (unsigned)c.i1[1]}, iz[2] = {(unsigned)c.i0[2], (unsigned)c.i1[2]};
    float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b) {
        const unsigned row = (ix[a] + iy[b]) * g;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const float f = __ldg(mesh + (row + iz[e]));
          ax = fmaf(f, sg[a] * wy[b] * wz[e], ax);
          ay = fmaf(f, wx[a] * sg[b] * wz[e], ay);
          az = fmaf(f, wx[a] * wy[b] * sg[e], az);
        }
      }
    r[0] = fmaf(scale, ax, v[3]);
    r[1] = fmaf(scale, ay, v[4]);
    r[2] = fmaf(scale, az, v[5]);
  }
};

inline bool aligned16(const void* a, const void* b = nullptr, const void* c = nullptr) {
  return ((reinterpret_cast<uintptr_t>(a) | reinterpret_cast<uintptr_t>(b) | reinterpret_cast<uintptr_t>(c)) & 15) == 0;
}

inline unsigned blocks_for(int64_t n) { return (unsigned)((n + kThreads - 1) / kThreads); }

inline int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
inline BrickMap brick_map(int np) { return BrickMap{np, np / BZ, np / BY, ilog2(np)}; }

}  // namespace

cudaError_t paint(const float* pos, const float* mass, float mass_const, int64_t n, int ng,
                  float* mesh, bool zero_first, const ParticleOrder& ord, cudaStream_t s, int batch) {
  const size_t g3 = (size_t)ng * ng * ng;
  if (zero_first) {
    cudaError_t e = cudaMemsetAsync(mesh, 0, sizeof(float) * g3 * batch, s);
    if (e != cudaSuccess) return e;
  }
  if (n == 0) return cudaSuccess;
  int mode = ord.paint_mode;
  const int res = ord.np > 0 ? ng / ord.np : 0;
  const bool can_brick = brick_ok(n, ord.np) && (res == 1 || res == 2) && ng == res * ord.np && ng % 4 == 0 &&
                         (reinterpret_cast<uintptr_t>(mesh) & 15) == 0;
  if (mode == FPM_PAINT_AUTO) mode = can_brick ? FPM_PAINT_BRICK_FIXED : FPM_PAINT_DIRECT;
  if (mode != FPM_PAINT_DIRECT && !can_brick) mode = FPM_PAINT_DIRECT;
  if (mode == FPM_PAINT_DIRECT) {
    for (int b = 0; b < batch; ++b)
      paint_direct_kernel<<<blocks_for(n), kThreads, 0, s>>>(pos + (size_t)b * 3 * n, mass ? mass + (size_t)b * n : nullptr,
                                                             mass_const, n, ng, mesh + b * g3);
    return cudaGetLastError();
  }
  const size_t smem = sizeof(float) * (size_t)kWinCells;
  const dim3 grid((unsigned)(n / (kBrick / (res * res * res))), (unsigned)batch);
  const BrickMap bm = brick_map(ord.np);
  auto go = [&](auto kern) -> cudaError_t {
    cudaError_t e = ensure_dynamic_smem(kern, smem);
    if (e != cudaSuccess) return e;
    kern<<<grid, kBrickThreads, smem, s>>>(pos, mass, mass_const, n, bm, ng, mesh);
    return cudaGetLastError();
  };
  if (res == 2) {
    if (mode == FPM_PAINT_BRICK_FIXED)
      return mass ? go(paint_brick_kernel<true, true, 2>) : go(paint_brick_kernel<true, false, 2>);
    return mass ? go(paint_brick_kernel<false, true, 2>) : go(paint_brick_kernel<false, false, 2>);
  }
  if (mode == FPM_PAINT_BRICK_FIXED) {
    return mass ? go(paint_brick_kernel<true, true, 1, true>) : go(paint_brick_kernel<true, false, 1, true, 3>);
  }
  return mass ? go(paint_brick_kernel<false, true>) : go(paint_brick_kernel<false, false>);
}

cudaError_t readout(const float* mesh, const float* pos, int64_t n, int ng, float* out,
                    const ParticleOrder& ord, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  if (brick_ok(n, ord.np))
    readout_kernel<1, true><<<(unsigned)(n / kBrick), kBrickThreads, 0, s>>>(mesh, nullptr, nullptr, pos, n, ng,
                                                                           brick_map(ord.np), out);
  else
    readout_kernel<1, false><<<blocks_for(n), kThreads, 0, s>>>(mesh, nullptr, nullptr, pos, n, ng,
                                                               BrickMap{0, 1, 1, 0}, out);
  return cudaGetLastError();
}

cudaError_t readout3(const float* fx, const float* fy, const float* fz, const float* pos, int64_t n,
                     int ng, float* out3, const ParticleOrder& ord, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  if (brick_ok(n, ord.np))
    readout_kernel<3, true><<<(unsigned)(n / kBrick), kBrickThreads, 0, s>>>(fx, fy, fz, pos, n, ng,
                                                                           brick_map(ord.np), out3);
  else
    readout_kernel<3, false><<<blocks_for(n), kThreads, 0, s>>>(fx, fy, fz, pos, n, ng, BrickMap{0, 1, 1, 0}, out3);
  return cudaGetLastError();
}

cudaError_t readout_kick_drift(const float* fx, const float* fy, const float* fz, float* pos,
                               float* mom, int64_t n, int ng, float kfac, float dfac,
                               const ParticleOrder& ord, cudaStream_t s, int batch) {
  if (n == 0) return cudaSuccess;
  const bool f4 = (fy == nullptr);   // interleaved force mesh
  if (batch > 1 && !f4) return cudaErrorInvalidValue;      // batches run the fused path only
  const bool aligned = ((reinterpret_cast<uintptr_t>(pos) | reinterpret_cast<uintptr_t>(mom)) & 15) == 0;
  if (brick_ok(n, ord.np) && aligned) {
    const dim3 grid((unsigned)(2 * (n / kBrick)), (unsigned)batch);
    const BrickMap bm = brick_map(ord.np);
    if (f4)
      rkd_pipelined_kernel<3, 1, 4, true><<<grid, kThreads, 0, s>>>(fx, fy, fz, pos, mom, n, ng, bm, kfac, dfac);
    else
      rkd_pipelined_kernel<3, 1, 4, false><<<grid, kThreads, 0, s>>>(fx, fy, fz, pos, mom, n, ng, bm, kfac, dfac);
    return cudaGetLastError();
  }
  if (f4) {
    for (int b = 0; b < batch; ++b)
      readout_kick_drift_kernel<true><<<blocks_for(n), kThreads, 0, s>>>(
          fx + (size_t)b * 4 * ng * ng * ng, fy, fz, pos + (size_t)b * 3 * n, mom + (size_t)b * 3 * n, n, ng, kfac, dfac);
  } else {
    readout_kick_drift_kernel<false><<<blocks_for(n), kThreads, 0, s>>>(fx, fy, fz, pos, mom, n, ng, kfac, dfac);
  }
  return cudaGetLastError();
}

cudaError_t readout_grad(const float* mesh, const float* pos, const float* scale, float scale_const,
                         int64_t n, int ng, float* out3, float* out_value, cudaStream_t s,
                         bool accumulate) {
  if (n == 0) return cudaSuccess;
  readout_grad_kernel<<<blocks_for(n), kThreads, 0, s>>>(mesh, pos, scale, scale_const, n, ng, out3,
                                                         out_value, accumulate ? 1 : 0);
  return cudaGetLastError();
}

cudaError_t readout3_grad_accum(const float* f0, const float* f1, const float* f2, const float* pos,
                                const float* v, float coef, int64_t n, int ng, float* gx,
                                cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  readout3_grad_accum_kernel<<<blocks_for(n), kThreads, 0, s>>>(f0, f1, f2, pos, v, coef, n, ng, gx);
  return cudaGetLastError();
}

bool brick_walk_ok(int64_t n, const ParticleOrder& ord, const void* a, const void* b, const void* c) {
  return brick_ok(n, ord.np) && aligned16(a, b, c);
}

cudaError_t force_vjp_direct_brick(const float* f4, const float* pos, const float* v, float coef,
                                   int64_t n, int ng, float* gx, const ParticleOrder& ord, cudaStream_t s) {
  if (!brick_walk_ok(n, ord, pos, v, gx)) return cudaErrorInvalidValue;
  Planes<9> in{{pos, pos + n, pos + 2 * n, v, v + n, v + 2 * n, gx, gx + n, gx + 2 * n}};
  OutPlanes<3> out{{gx, gx + n, gx + 2 * n}};
  ForceVjpDirectOp op{reinterpret_cast<const float4*>(f4), (unsigned)ng, coef};
  brick_gather_kernel<3, 9, 3, ForceVjpDirectOp><<<(unsigned)(2 * (n / kBrick)), kThreads, 0, s>>>(in, out, brick_map(ord.np), op);
  return cudaGetLastError();
}

cudaError_t grad_accum_brick(const float* mesh, const float* pos, float scale, int64_t n, int ng,
                             float* gx, const ParticleOrder& ord, cudaStream_t s) {
  if (!brick_walk_ok(n, ord, pos, gx, nullptr)) return cudaErrorInvalidValue;
  Planes<6> in{{pos, pos + n, pos + 2 * n, gx, gx + n, gx + 2 * n}};
  OutPlanes<3> out{{gx, gx + n, gx + 2 * n}};
  GradAccumOp op{mesh, (unsigned)ng, scale};
  brick_gather_kernel<3, 6, 3, GradAccumOp><<<(unsigned)(2 * (n / kBrick)), kThreads, 0, s>>>(in, out, brick_map(ord.np), op);
  return cudaGetLastError();
}

}  // namespace fpm
