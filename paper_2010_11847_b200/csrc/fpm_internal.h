// fpm_internal.h -- context and internal launch interfaces of libfpm (not part of the C-ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/fpm.h"

namespace fpm {

// ---- per-kernel accounting: launch counter (always) + CUDA-event timing (when enabled) --------
enum KernelId {
  K_PAINT = 0, K_FFT_Z_R2C, K_FFT_Y, K_FFT_X, K_FFT_Z_C2R, K_GREEN, K_READOUT, K_READOUT_KICK_DRIFT,
  K_KICK, K_DRIFT, K_READOUT_GRAD, K_LPT, K_FFT_X_FORCE, K_FFT_Y_INV3, K_MEMSET, K_FFT_Z_C2R3, K_COUNT
};
const char* kernel_name(int kid);

struct Profiler {
  bool enabled = false;
  cudaStream_t stream = nullptr;
  struct Rec { int kid; cudaEvent_t a, b; };
  std::vector<cudaEvent_t> pool;
  std::vector<Rec> open;
  double ms[K_COUNT] = {0};
  long long count[K_COUNT] = {0};
  long long launches = 0;          // kernels of this library launched since the last reset
  void begin(int kid);
  void end();
  void flush();                    // synchronises the recorded events and accumulates ms[]
  void reset();
  void destroy();
};

struct ProfScope {
  Profiler* p;
  ProfScope(Profiler* prof, int kid, int nlaunch = 1) : p(prof) {
    if (p) { p->launches += nlaunch; p->begin(kid); }
  }
  ~ProfScope() { if (p) p->end(); }
};

// Opt a kernel in to more than 48 KB of dynamic shared memory, once per kernel and device (the attribute
// is per device; calling cudaFuncSetAttribute before every launch showed up on the small configurations).
cudaError_t ensure_dynamic_smem_impl(const void* kernel, size_t bytes);     // profiler.cpp
template <class K>
inline cudaError_t ensure_dynamic_smem(K kernel, size_t bytes) {
  if (bytes <= 48 * 1024) return cudaSuccess;
  return ensure_dynamic_smem_impl(reinterpret_cast<const void*>(kernel), bytes);
}

// cuTensorMapEncodeTiled through cudaGetDriverEntryPoint (no libcuda link); nullptr when unavailable (profiler.cpp)
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn();

// ---- FFT (fft.cu) ---------------------------------------------------------------------------
struct FftTables {
  int n = 0;
  float2* dev = nullptr;       // one allocation: [stage table N][stage table N/2][stage table x plan][W_N^k, k < N/2]
  float2* stage_n = nullptr;
  float2* stage_m = nullptr;
  float2* stage_x = nullptr;   // stage table of the plan fft_x_force_kernel uses (may equal stage_n's)
  float2* full = nullptr;
};
cudaError_t fft_tables_create(int n, FftTables* out);
void fft_tables_destroy(FftTables* t);
bool fft_size_supported(int n);

// per-axis tables of the transfer function, fp32 rounded from float64 (green.cu)
struct KernelTables {
  int n = 0;
  float* dev = nullptr;
  float* lap = nullptr;    // K^2 contribution of one axis: (2 sin(w/2))^2 or w^2
  float* grad = nullptr;   // g(w) with the Nyquist entry zeroed
  float* kvec = nullptr;   // w = 2 pi f / n (Nyquist kept)           [LPT spectral kernels]
  float* kvec0 = nullptr;  // w with the Nyquist entry zeroed          [LPT spectral kernels]
};
cudaError_t kernel_tables_create(int n, int kernel_mode, KernelTables* out);
void kernel_tables_destroy(KernelTables* t);

// element-wise epilogue/prologue selectors for the fused x passes (fft.cu)
enum XOp { XOP_NONE = 0, XOP_INVLAP = 1, XOP_GRAD = 2 };

// TMA tensor maps of the four internal half-complex meshes of the fused paths (dk, wa, wb, wc; padded
// pitch): `y` moves 16-column x 256-line boxes of one x slab, `x` moves TX-column boxes of 256 x lines.
struct TileMaps {
  bool ok = false;
  CUtensorMap y[4];
  CUtensorMap x[4];
};
// bufs: dk, wa, wb, wc (each `batch` meshes back to back).  Leaves out->ok false (and returns cudaSuccess)
// when the driver has no tensor-map support: the callers then use the ld.global tile movers.
cudaError_t fft_make_tile_maps(int n, int batch, float2* const bufs[4], TileMaps* out);

cudaError_t fft_r2c(const FftTables& t, const float* real, float2* cplx, cudaStream_t s,
                    Profiler* prof = nullptr);
cudaError_t fft_c2r(const FftTables& t, float2* cplx, float* real, cudaStream_t s,
                    Profiler* prof = nullptr);

// paint'ed density -> the three force meshes F[0..2] with the transfer function fused into the
// transform passes (fft.cu); scale = 1.5 omega_m (or 1).  F4 != nullptr: the three components are
// written interleaved per cell as float4 (x, y, z, unused) into F4[4 ng^3] instead of F[0..2].
// batch > 1 (F4 only): every buffer holds `batch` meshes back to back and each pass covers them all
cudaError_t fft_force_fused(const FftTables& t, const KernelTables& kt, const float* rho, float2* dk,
                            float2* wa, float2* wb, float2* wc, float* const* F, float* F4, float scale,
                            cudaStream_t s, Profiler* prof = nullptr, int batch = 1, const TileMaps* maps = nullptr);

// out = c2r[(scale / K^2) r2c[src]] with the multiplier fused into the x round trip (backward pass)
cudaError_t fft_poisson(const FftTables& t, const KernelTables& kt, const float* src, float2* work, float* out,
                        float scale, cudaStream_t s, Profiler* prof = nullptr, const CUtensorMap* work_map_x = nullptr);

// ---- particle <-> mesh (mesh_ops.cu) ---------------------------------------------------------
// How the caller's particle arrays are ordered: np > 0 says "n == np^3 particles in lattice
// (Lagrangian) order", which lets the kernels walk them brick by brick; results never depend on it.
struct ParticleOrder {
  int np = 0;
  int paint_mode = FPM_PAINT_AUTO;
};
// batch > 1: [batch][3][n] positions, [batch][n] masses, [batch][ng^3] meshes in one launch (N2)
cudaError_t paint(const float* pos, const float* mass, float mass_const, int64_t n, int ng,
                  float* mesh, bool zero_first, const ParticleOrder& ord, cudaStream_t s, int batch = 1);
cudaError_t readout(const float* mesh, const float* pos, int64_t n, int ng, float* out,
                    const ParticleOrder& ord, cudaStream_t s);
cudaError_t readout3(const float* fx, const float* fy, const float* fz, const float* pos, int64_t n,
                     int ng, float* out3, const ParticleOrder& ord, cudaStream_t s);
// gradient of the CIC sum w.r.t. the position, times scale_p (mass[p] or vbar[p] or constant)
// accumulate: out3 += instead of out3 =
cudaError_t readout_grad(const float* mesh, const float* pos, const float* scale, float scale_const,
                         int64_t n, int ng, float* out3, float* out_value, cudaStream_t s,
                         bool accumulate = false);
// gx[e][p] += coef * sum_d v[d][p] * sum_c F_d[c] dW/dx_e  (direct term of the force VJP, R12)
cudaError_t readout3_grad_accum(const float* f0, const float* f1, const float* f2, const float* pos,
                                const float* v, float coef, int64_t n, int ng, float* gx,
                                cudaStream_t s);

// Lagrangian-brick, cp.async-pipelined versions of the two gathers of the force VJP (valid when
// brick_walk_ok: full lattice set, 16-byte aligned arrays).  f4: interleaved (F_x, F_y, F_z, -) mesh.
bool brick_walk_ok(int64_t n, const ParticleOrder& ord, const void* a, const void* b, const void* c);
cudaError_t force_vjp_direct_brick(const float* f4, const float* pos, const float* v, float coef,
                                   int64_t n, int ng, float* gx, const ParticleOrder& ord, cudaStream_t s);
cudaError_t grad_accum_brick(const float* mesh, const float* pos, float scale, int64_t n, int ng,
                             float* gx, const ParticleOrder& ord, cudaStream_t s);

// ---- particle updates (particles.cu) -----------------------------------------------------------
cudaError_t kick(float* mom, const float* force, int64_t n3, float fac, cudaStream_t s);
cudaError_t drift(float* pos, const float* mom, int64_t n3, float fac, int ng, cudaStream_t s);
// mom += force(pos) * kfac ; pos = wrap(pos + mom * dfac), gathering the three force meshes
// fy == fz == nullptr: fx is the interleaved float4 force mesh of fft_force_fused
cudaError_t readout_kick_drift(const float* fx, const float* fy, const float* fz, float* pos,
                               float* mom, int64_t n, int ng, float kfac, float dfac,
                               const ParticleOrder& ord, cudaStream_t s, int batch = 1);

// ---- transfer function and LPT element-wise kernels (green.cu) ---------------------------------
cudaError_t apply_force_kernel(const KernelTables& kt, const float2* dk, float scale, float2* fkx,
                               float2* fky, float2* fkz, cudaStream_t s);
// out = mult(k) in, mult = sign * (a == b ? -k_a^2 : (i k_a)(b >= 0 ? i k_b : 1)) * (-1/k^2)
// accumulate: out += instead of out =
cudaError_t lpt_spectral(const KernelTables& kt, const float2* in, float2* out, int a, int b,
                         float sign, cudaStream_t s, bool accumulate = false);
// backward pass: out_k = - sum_d (i scale g_d / K^2) f_d,k  (= sum_d M_d^T)
cudaError_t apply_force_kernel_transpose(const KernelTables& kt, const float2* f0, const float2* f1,
                                         const float2* f2, float scale, float2* out, cudaStream_t s);
// g = sum_d D_d f_d, D the periodic 4-point central difference whose symbol is i g(w) of Eq. 5
cudaError_t stencil_divergence(const float* f0, const float* f1, const float* f2, int n, float* g, cudaStream_t s);
cudaError_t axpy(float* y, const float* x, float a, int64_t n, cudaStream_t s);            // y += a x
cudaError_t lincomb2(float* out, const float* a, float ca, const float* b, float cb, int64_t n,
                     cudaStream_t s);                                                        // ca a + cb b
// out = sbar (pa + pb), or -2 sbar pa when pb == nullptr (2LPT product rule)
cudaError_t lpt_phibar(float* out, const float* sbar, const float* pa, const float* pb, int64_t n,
                       cudaStream_t s);
cudaError_t lpt_displace(const float* psi, int np, int bfac, int axis, float dcoef, float vcoef,
                         bool first, float* pos_d, float* mom_d, cudaStream_t s);
cudaError_t lpt_wrap(float* pos, int64_t n3, int ng, cudaStream_t s);
// s = a*b (mode 0), s += (a+b)*c (mode 1), s -= a*a (mode 2)
cudaError_t lpt_source(float* s, const float* a, const float* b, const float* c, int64_t n, int mode,
                       cudaStream_t st);

// ---- multi-grid pyramid (pyramid.cu, Alg. 2-3) --------------------------------
// one REDUCE level n^3 -> (n/2)^3; tmp: 3 n^3 / 4 floats
cudaError_t pyramid_reduce_level(const float* in, int n, float* tmp, float* out, cudaStream_t s);
// one EXPAND level m^3 -> (2m)^3; tmp: 6 m^3 floats
cudaError_t pyramid_expand_level(const float* in, int m, float* tmp, float* out, cudaStream_t s);
cudaError_t pyramid_combine(float* fs, const float* up, const float* lowup, int64_t n, cudaStream_t s);

// ---- MAP reconstruction element-wise kernels (recon.cu) ----------------------
cudaError_t recon_residual(const float* rho, const float* data, float inv_s2, int64_t n, float* gbar,
                           double* acc, cudaStream_t s);
cudaError_t recon_prior(const float2* sk, const float* inv_power, int n, float2* gk, double* acc,
                        cudaStream_t s);
cudaError_t adam_update(float* x, const float* g, float* m, float* v, int64_t n, double lr, double b1,
                        double b2, double eps, double inv_c1, double inv_c2, cudaStream_t s);

// ---- background cosmology on the host, float64 (cosmology.cpp) ---------------------------------
struct GrowthOut { double D1, f1, D2, f2, E, Gf, gf; };
GrowthOut growth(double omega_m, double a);
double drift_factor(double omega_m, double ai, double ac, double af, int factor_mode);
double kick_factor(double omega_m, double ai, double ac, double af, int factor_mode);

}  // namespace fpm

struct fpm_ctx {
  fpm_config cfg;
  int device = 0;                   // the CUDA device that was current in fpm_create; every call runs there
  cudaStream_t stream = nullptr;
  fpm::FftTables fft_g, fft_p;      // plans for ng and np (same object when equal)
  fpm::KernelTables kt_g, kt_p;     // transfer-function tables on ng; spectral tables on np
  void* ws = nullptr;
  size_t ws_bytes = 0;
  fpm::TileMaps maps;               // tensor maps of the workspace's half-complex meshes (fpm_set_workspace)
  int tile_movers = FPM_MOVERS_AUTO; // FPM_MOVERS_GLOBAL: maps.ok is kept false (fpm_set_tile_movers)
  int coarse_n = 0;                 // plans of the coarse mesh of the pyramid scheme (fpm_force_pyramid), made on demand
  fpm::FftTables fft_c;
  fpm::KernelTables kt_c;
  double* d_acc = nullptr;          // two float64 accumulators (loss terms of fpm_recon_loss_grad)
  bool sticky = false;
  std::string err;
  fpm::Profiler prof;
  // whole-run CUDA graphs of fpm_nbody (api.cu): captured on an internal stream, replayed on `stream`
  int graph_mode = FPM_GRAPH_AUTO;
  cudaStream_t capture_stream = nullptr;
  struct RunGraph {
    float *pos, *mom, *traj;
    std::vector<double> kf, dr;
    cudaGraphExec_t exec;
    long long launches;
  };
  std::vector<RunGraph> graphs;
  // the argument set of the last fpm_nbody call that missed the cache under FPM_GRAPH_AUTO: a run is captured
  // only when the same set comes back (a caller with fresh buffers every call never pays for a capture)
  struct { float *pos = nullptr, *mom = nullptr, *traj = nullptr; std::vector<double> kf, dr; bool valid = false; } seen;
};
