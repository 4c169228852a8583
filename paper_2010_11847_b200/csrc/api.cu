// api.cu -- the C-ABI of libfpm (include/fpm.h): validation, context, workspace carving and the
// step / run / initial-condition drivers.  Every numerical step runs in the kernels of this
// library (fft.cu, mesh_ops.cu, green.cu, particles.cu); there is no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "fpm_internal.h"

using namespace fpm;

namespace {

inline size_t align256(size_t b) { return (b + 255) & ~size_t(255); }
inline size_t real_bytes(int n) { return align256(sizeof(float) * (size_t)n * n * n); }
// half-complex scratch meshes are sized for the padded internal row pitch (n/2 + 1 rounded up to 16 elements;
// fft.cuh padded_pitch), which the dense cuFFT-layout uses of the same buffers fit inside
inline size_t cplx_bytes(int n) { return align256(sizeof(float2) * (size_t)n * n * (size_t)((n / 2 + 1 + 15) & ~15)); }

bool config_ok(const fpm_config* c) {
  if (!c) return false;
  if (!fft_size_supported(c->ng) || !fft_size_supported(c->np)) return false;
  if (c->np > c->ng || c->ng % c->np != 0) return false;
  if (!(c->omega_m > 0.0 && c->omega_m <= 1.0)) return false;
  if (c->kernel_mode < FPM_KERNEL_PAPER || c->kernel_mode > FPM_KERNEL_MIXED) return false;
  if (c->factor_mode < FPM_FACTORS_FASTPM || c->factor_mode > FPM_FACTORS_QUINN) return false;
  if (c->force_path < FPM_FORCE_UNFUSED || c->force_path > FPM_FORCE_FUSED) return false;
  if (c->paint_mode < FPM_PAINT_AUTO || c->paint_mode > FPM_PAINT_BRICK_FIXED) return false;
  if (c->batch < 0 || (int64_t)c->batch * c->ng > 65535) return false;
  // a batch runs the fused path over Lagrangian bricks only (fpm.h "Batches")
  if (c->batch > 1 && (c->force_path != FPM_FORCE_FUSED || c->np % 32 != 0)) return false;
  return true;
}

// bytes between consecutive half-complex buffers (a skew was measured to make no difference: DESIGN.md 15)
constexpr size_t kSkew = 0;

inline int batch_of(const fpm_config& c) { return c.batch > 1 ? c.batch : 1; }

// cached run graphs bake in the workspace pointers and the kernel selection: drop them when either changes
void drop_graphs(fpm_ctx* ctx) {
  for (auto& g : ctx->graphs) cudaGraphExecDestroy(g.exec);
  ctx->graphs.clear();
}

// carved views of the caller's workspace
struct Workspace {
  float* rho;
  float2* dk;
  float2* fk[3];
  float* F[3];
};

// every region holds `batch` meshes back to back; rho | F[0] | F[1] | F[2] stay contiguous (the interleaved
// force mesh of the fused path, [batch][ng^3] float4, overlays them)
Workspace carve(const fpm_ctx* ctx) {
  Workspace w;
  char* p = static_cast<char*>(ctx->ws);
  const int n = ctx->cfg.ng;
  const size_t b = (size_t)batch_of(ctx->cfg);
  w.rho = reinterpret_cast<float*>(p); p += b * real_bytes(n);
  for (int d = 0; d < 3; ++d) { w.F[d] = reinterpret_cast<float*>(p); p += b * real_bytes(n); }
  // (the four half-complex buffers are streamed concurrently at the same relative offset by the fused passes;
  //  a skew between them was measured to make no difference: DESIGN.md section 15)
  w.dk = reinterpret_cast<float2*>(p); p += b * cplx_bytes(n) + kSkew;
  for (int d = 0; d < 3; ++d) { w.fk[d] = reinterpret_cast<float2*>(p); p += b * cplx_bytes(n) + kSkew; }
  return w;
}

int fail(fpm_ctx* ctx, int code, const char* what) {
  if (ctx) {
    ctx->err = what;
    if (code == FPM_ECUDA) ctx->sticky = true;
  }
  return code;
}

int cuda_fail(fpm_ctx* ctx, cudaError_t e, const char* where) {
  char buf[256];
  std::snprintf(buf, sizeof buf, "%s: %s", where, cudaGetErrorString(e));
  return fail(ctx, FPM_ECUDA, buf);
}

// Every entry point runs on the device the context was created on, whatever device is current in the
// calling thread; the caller's current device is restored on return.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

#define FPM_ENTER(ctx)                                              \
  if (!(ctx)) return FPM_EINVAL;                                    \
  if ((ctx)->sticky) return FPM_ECUDA;                              \
  DeviceGuard device_guard__((ctx)->device);
#define FPM_CUDA(ctx, call)                                         \
  do {                                                              \
    cudaError_t e__ = (call);                                       \
    if (e__ != cudaSuccess) return cuda_fail((ctx), e__, #call);    \
  } while (0)
#define FPM_REQUIRE(ctx, cond, what)                                \
  if (!(cond)) return fail((ctx), FPM_EINVAL, what);
#define FPM_NO_BATCH(ctx, what)                                     \
  if (batch_of((ctx)->cfg) > 1) return fail((ctx), FPM_ENOTIMPL, what ": not available on a batched context");
#define FPM_NEED_WS(ctx)                                            \
  if (!(ctx)->ws || (ctx)->ws_bytes < fpm_workspace_bytes(&(ctx)->cfg)) \
    return fail((ctx), FPM_ENOMEM, "workspace missing or too small (fpm_set_workspace)");

inline ParticleOrder order_of(const fpm_ctx* ctx, int64_t n) {
  ParticleOrder o;
  const int64_t np = ctx->cfg.np;
  o.np = (n == np * np * np) ? (int)np : 0;
  o.paint_mode = ctx->cfg.paint_mode;
  return o;
}

inline float particle_mass(const fpm_ctx* ctx) {
  const float b = (float)(ctx->cfg.ng / ctx->cfg.np);
  return b * b * b;
}

// paint -> r2c -> transfer function -> 3x c2r : the three force meshes of Alg. 3 ForceGrids(local)
// interleaved: (fused path only) the components go to one float4-per-cell mesh that overlays
// rho | F[0] | F[1] | F[2] (16 ng^3 contiguous bytes; rho is dead once the z r2c pass has read it).
int force_meshes(fpm_ctx* ctx, const Workspace& w, const float* pos, int64_t n, bool interleaved = false) {
  const int ng = ctx->cfg.ng;
  cudaStream_t s = ctx->stream;
  Profiler* pr = &ctx->prof;
  const int batch = batch_of(ctx->cfg);
  { ProfScope sc(pr, K_PAINT);
    FPM_CUDA(ctx, paint(pos, nullptr, particle_mass(ctx), n, ng, w.rho, true, order_of(ctx, n), s, batch)); }
  if (ctx->cfg.force_path == FPM_FORCE_FUSED) {
    FPM_CUDA(ctx, fft_force_fused(ctx->fft_g, ctx->kt_g, w.rho, w.dk, w.fk[0], w.fk[1], w.fk[2], w.F,
                                  interleaved ? w.rho : nullptr, (float)(1.5 * ctx->cfg.omega_m), s, pr, batch,
                                  &ctx->maps));
    return FPM_OK;
  }
  FPM_CUDA(ctx, fft_r2c(ctx->fft_g, w.rho, w.dk, s, pr));
  {
    ProfScope sc(pr, K_GREEN);
    FPM_CUDA(ctx, apply_force_kernel(ctx->kt_g, w.dk, (float)(1.5 * ctx->cfg.omega_m), w.fk[0],
                                     w.fk[1], w.fk[2], s));
  }
  for (int d = 0; d < 3; ++d) FPM_CUDA(ctx, fft_c2r(ctx->fft_g, w.fk[d], w.F[d], s, pr));
  return FPM_OK;
}

// One PM step: force at the current positions, p += f K, x = wrap(x + p D).
int pm_step(fpm_ctx* ctx, const Workspace& w, float* pos, float* mom, int64_t n, double kfac,
            double dfac) {
  const bool f4 = ctx->cfg.force_path == FPM_FORCE_FUSED;
  const int rc = force_meshes(ctx, w, pos, n, f4);
  if (rc != FPM_OK) return rc;
  ProfScope sc(&ctx->prof, K_READOUT_KICK_DRIFT);
  if (f4)
    FPM_CUDA(ctx, readout_kick_drift(w.rho, nullptr, nullptr, pos, mom, n, ctx->cfg.ng, (float)kfac,
                                     (float)dfac, order_of(ctx, n), ctx->stream, batch_of(ctx->cfg)));
  else
    FPM_CUDA(ctx, readout_kick_drift(w.F[0], w.F[1], w.F[2], pos, mom, n, ctx->cfg.ng, (float)kfac,
                                     (float)dfac, order_of(ctx, n), ctx->stream));
  return FPM_OK;
}

// gx += coef * J_f(pos)^T v, f = the force evaluation of force_meshes + readout.
int force_vjp(fpm_ctx* ctx, const Workspace& w, const float* pos, int64_t n, const float* v, double coef,
              float* gx) {
  const int ng = ctx->cfg.ng;
  cudaStream_t s = ctx->stream;
  Profiler* pr = &ctx->prof;
  const ParticleOrder ord = order_of(ctx, n);
  const double sc = 1.5 * ctx->cfg.omega_m;
  // forward force meshes F_d at pos (recomputed, not stored); interleaved when the brick walker applies
  const bool brick = ctx->cfg.force_path == FPM_FORCE_FUSED && brick_walk_ok(n, ord, pos, v, gx);
  const int rc = force_meshes(ctx, w, pos, n, brick);
  if (rc != FPM_OK) return rc;
  // f_d = readout(F_d, pos): direct dW/dx term
  { ProfScope sc2(pr, K_READOUT_GRAD);
    if (brick) FPM_CUDA(ctx, force_vjp_direct_brick(w.rho, pos, v, (float)coef, n, ng, gx, ord, s));
    else FPM_CUDA(ctx, readout3_grad_accum(w.F[0], w.F[1], w.F[2], pos, v, (float)coef, n, ng, gx, s)); }
  // ... and the cotangent of the meshes: Fbar_d = paint(pos, mass = v_d);
  // rho_bar = sum_d M_d^T Fbar_d = -sum_d M_d Fbar_d  (M_d odd and imaginary in k-space)
  if (ctx->cfg.kernel_mode != FPM_KERNEL_NAIVE) {
    // Eq. 5's i g(w) is the symbol of the 4-point difference D, so sum_d i g_d Fbar_d,k is the transform of
    // the real-space stencil divergence: three paints, one stencil pass, ONE potential solve.
    for (int d = 0; d < 3; ++d) {
      ProfScope sc2(pr, K_PAINT);
      FPM_CUDA(ctx, paint(pos, v + d * n, 0.f, n, ng, w.F[d], true, ord, s));
    }
    { ProfScope sc2(pr, K_GREEN); FPM_CUDA(ctx, stencil_divergence(w.F[0], w.F[1], w.F[2], ng, w.rho, s)); }
    FPM_CUDA(ctx, fft_poisson(ctx->fft_g, ctx->kt_g, w.rho, w.dk, w.F[0], (float)(-coef * sc), s, pr,
                              ctx->maps.ok ? &ctx->maps.x[0] : nullptr));
  } else {
    for (int d = 0; d < 3; ++d) {
      { ProfScope sc2(pr, K_PAINT); FPM_CUDA(ctx, paint(pos, v + d * n, 0.f, n, ng, w.rho, true, ord, s)); }
      FPM_CUDA(ctx, fft_r2c(ctx->fft_g, w.rho, w.fk[d], s, pr));
    }
    { ProfScope sc2(pr, K_GREEN);
      FPM_CUDA(ctx, apply_force_kernel_transpose(ctx->kt_g, w.fk[0], w.fk[1], w.fk[2], (float)(coef * sc), w.dk, s)); }
    FPM_CUDA(ctx, fft_c2r(ctx->fft_g, w.dk, w.F[0], s, pr));
  }
  // rho = paint(pos, m): cotangent of pos = m sum_c rho_bar[c] dW/dx
  ProfScope sc2(pr, K_READOUT_GRAD);
  if (brick_walk_ok(n, ord, pos, gx, nullptr))
    FPM_CUDA(ctx, grad_accum_brick(w.F[0], pos, particle_mass(ctx), n, ng, gx, ord, s));
  else
    FPM_CUDA(ctx, readout_grad(w.F[0], pos, nullptr, particle_mass(ctx), n, ng, gx, nullptr, s, true));
  return FPM_OK;
}

// merged kick / drift factors of the n_steps + 1 PM steps of a run (R6); see fpm_step_factors in fpm.h
void step_factors(const fpm_ctx* ctx, const double* a, int n_steps, double* kf, double* dr) {
  const double om = ctx->cfg.omega_m;
  const int fm = ctx->cfg.factor_mode;
  double pending = 0.0;   // second half kick of the previous step, same force mesh
  for (int j = 0; j <= n_steps; ++j) {
    kf[j] = pending;
    dr[j] = 0.0;
    if (j < n_steps) {
      const double ai = a[j], af = a[j + 1], ah = std::sqrt(ai * af);
      kf[j] += kick_factor(om, ai, ai, ah, fm);
      dr[j] = drift_factor(om, ai, ah, af, fm);
      pending = kick_factor(om, ah, af, af, fm);
    }
  }
}

}  // namespace

extern "C" {

const char* fpm_version(void) { return "fpm-b200 0.1 (sm_100a)"; }

size_t fpm_workspace_bytes(const fpm_config* cfg) {
  if (!config_ok(cfg)) return 0;
  return (size_t)batch_of(*cfg) * (4 * real_bytes(cfg->ng) + 4 * cplx_bytes(cfg->ng)) + 4 * kSkew;
}

int fpm_create(const fpm_config* cfg, void* cuda_stream, fpm_ctx** out) {
  if (!out) return FPM_EINVAL;
  *out = nullptr;
  if (!config_ok(cfg)) return FPM_EINVAL;
  fpm_ctx* ctx = new (std::nothrow) fpm_ctx();
  if (!ctx) return FPM_ENOMEM;
  ctx->cfg = *cfg;
  if (cudaGetDevice(&ctx->device) != cudaSuccess) { delete ctx; return FPM_ECUDA; }
  ctx->stream = static_cast<cudaStream_t>(cuda_stream);
  ctx->prof.stream = ctx->stream;
  cudaError_t e = fft_tables_create(cfg->ng, &ctx->fft_g);
  if (e == cudaSuccess) e = fft_tables_create(cfg->np, &ctx->fft_p);
  if (e == cudaSuccess) e = kernel_tables_create(cfg->ng, cfg->kernel_mode, &ctx->kt_g);
  if (e == cudaSuccess) e = kernel_tables_create(cfg->np, FPM_KERNEL_NAIVE, &ctx->kt_p);
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_acc, 2 * sizeof(double));
  if (e != cudaSuccess) {
    fpm_destroy(ctx);
    return FPM_ECUDA;
  }
  *out = ctx;
  return FPM_OK;
}

int fpm_destroy(fpm_ctx* ctx) {
  if (!ctx) return FPM_EINVAL;
  DeviceGuard device_guard__(ctx->device);
  drop_graphs(ctx);
  if (ctx->capture_stream) cudaStreamDestroy(ctx->capture_stream);
  ctx->prof.destroy();
  if (ctx->d_acc) cudaFree(ctx->d_acc);
  fft_tables_destroy(&ctx->fft_g);
  fft_tables_destroy(&ctx->fft_p);
  fft_tables_destroy(&ctx->fft_c);
  kernel_tables_destroy(&ctx->kt_c);
  kernel_tables_destroy(&ctx->kt_g);
  kernel_tables_destroy(&ctx->kt_p);
  delete ctx;
  return FPM_OK;
}

const char* fpm_last_error(const fpm_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int fpm_set_workspace(fpm_ctx* ctx, void* ws, size_t bytes) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, ws != nullptr, "workspace is null");
  FPM_REQUIRE(ctx, (reinterpret_cast<uintptr_t>(ws) & 255) == 0, "workspace must be 256-byte aligned");
  if (bytes < fpm_workspace_bytes(&ctx->cfg)) return fail(ctx, FPM_ENOMEM, "workspace too small");
  drop_graphs(ctx);
  ctx->ws = ws;
  ctx->ws_bytes = bytes;
  const Workspace w = carve(ctx);
  float2* const bufs[4] = {w.dk, w.fk[0], w.fk[1], w.fk[2]};
  FPM_CUDA(ctx, fft_make_tile_maps(ctx->cfg.ng, batch_of(ctx->cfg), bufs, &ctx->maps));
  if (ctx->tile_movers == FPM_MOVERS_GLOBAL) ctx->maps.ok = false;
  return FPM_OK;
}

int fpm_set_tile_movers(fpm_ctx* ctx, int tile_movers) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, tile_movers == FPM_MOVERS_AUTO || tile_movers == FPM_MOVERS_GLOBAL, "unknown tile mover mode");
  drop_graphs(ctx);
  ctx->tile_movers = tile_movers;
  if (ctx->ws) {
    const Workspace w = carve(ctx);
    float2* const bufs[4] = {w.dk, w.fk[0], w.fk[1], w.fk[2]};
    FPM_CUDA(ctx, fft_make_tile_maps(ctx->cfg.ng, batch_of(ctx->cfg), bufs, &ctx->maps));
  }
  if (tile_movers == FPM_MOVERS_GLOBAL) ctx->maps.ok = false;
  return FPM_OK;
}

int fpm_tile_movers(const fpm_ctx* ctx) {
  if (!ctx) return FPM_EINVAL;
  return ctx->ws && ctx->maps.ok ? FPM_MOVERS_TENSOR_MAPS : FPM_MOVERS_GLOBAL;
}

int fpm_set_paint_mode(fpm_ctx* ctx, int paint_mode) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, paint_mode >= FPM_PAINT_AUTO && paint_mode <= FPM_PAINT_BRICK_FIXED, "unknown paint mode");
  drop_graphs(ctx);
  ctx->cfg.paint_mode = paint_mode;
  return FPM_OK;
}

int fpm_set_graph_mode(fpm_ctx* ctx, int graph_mode) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, graph_mode >= FPM_GRAPH_OFF && graph_mode <= FPM_GRAPH_ALWAYS, "unknown graph mode");
  ctx->graph_mode = graph_mode;
  return FPM_OK;
}

int fpm_growth(const fpm_ctx* ctx, double a, double* out) {
  if (!ctx || !out || !(a > 0.0)) return FPM_EINVAL;
  const GrowthOut g = growth(ctx->cfg.omega_m, a);
  out[0] = g.D1; out[1] = g.f1; out[2] = g.D2; out[3] = g.f2; out[4] = g.E; out[5] = g.Gf; out[6] = g.gf;
  return FPM_OK;
}

int fpm_drift_factor(const fpm_ctx* ctx, double ai, double ac, double af, double* out) {
  if (!ctx || !out || !(ai > 0.0 && ac > 0.0 && af > 0.0)) return FPM_EINVAL;
  *out = drift_factor(ctx->cfg.omega_m, ai, ac, af, ctx->cfg.factor_mode);
  return FPM_OK;
}

int fpm_kick_factor(const fpm_ctx* ctx, double ai, double ac, double af, double* out) {
  if (!ctx || !out || !(ai > 0.0 && ac > 0.0 && af > 0.0)) return FPM_EINVAL;
  *out = kick_factor(ctx->cfg.omega_m, ai, ac, af, ctx->cfg.factor_mode);
  return FPM_OK;
}

int fpm_step_factors(const fpm_ctx* ctx, const double* a_stages, int n_steps, double* kick_fac,
                     double* drift_fac) {
  if (!ctx || !a_stages || !kick_fac || !drift_fac || n_steps < 0) return FPM_EINVAL;
  for (int j = 0; j <= n_steps; ++j)
    if (!(a_stages[j] > 0.0)) return FPM_EINVAL;
  step_factors(ctx, a_stages, n_steps, kick_fac, drift_fac);
  return FPM_OK;
}

int fpm_paint(fpm_ctx* ctx, const float* pos, const float* mass, int64_t n, float* mesh) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, n >= 0 && mesh && (pos || n == 0), "fpm_paint: bad arguments");
  ProfScope sc(&ctx->prof, K_PAINT);
  FPM_CUDA(ctx, paint(pos, mass, particle_mass(ctx), n, ctx->cfg.ng, mesh, true, order_of(ctx, n), ctx->stream,
                      batch_of(ctx->cfg)));
  return FPM_OK;
}

int fpm_fft_r2c(fpm_ctx* ctx, const float* real, float* cplx) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_fft_r2c");
  FPM_REQUIRE(ctx, real && cplx, "fpm_fft_r2c: null pointer");
  FPM_REQUIRE(ctx, (reinterpret_cast<uintptr_t>(real) & 7) == 0 && (reinterpret_cast<uintptr_t>(cplx) & 7) == 0,
              "fpm_fft_r2c: pointers must be 8-byte aligned");
  FPM_CUDA(ctx, fft_r2c(ctx->fft_g, real, reinterpret_cast<float2*>(cplx), ctx->stream, &ctx->prof));
  return FPM_OK;
}

int fpm_fft_c2r(fpm_ctx* ctx, float* cplx, float* real) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_fft_c2r");
  FPM_REQUIRE(ctx, real && cplx, "fpm_fft_c2r: null pointer");
  FPM_REQUIRE(ctx, (reinterpret_cast<uintptr_t>(real) & 7) == 0 && (reinterpret_cast<uintptr_t>(cplx) & 7) == 0,
              "fpm_fft_c2r: pointers must be 8-byte aligned");
  FPM_CUDA(ctx, fft_c2r(ctx->fft_g, reinterpret_cast<float2*>(cplx), real, ctx->stream, &ctx->prof));
  return FPM_OK;
}

int fpm_apply_force_kernel(fpm_ctx* ctx, const float* delta_k, float scale, float* fkx, float* fky,
                           float* fkz) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_apply_force_kernel");
  FPM_REQUIRE(ctx, delta_k && fkx && fky && fkz, "fpm_apply_force_kernel: null pointer");
  FPM_REQUIRE(ctx, delta_k != fkx && delta_k != fky && delta_k != fkz,
              "fpm_apply_force_kernel: outputs must not alias the input");
  ProfScope sc(&ctx->prof, K_GREEN);
  FPM_CUDA(ctx, apply_force_kernel(ctx->kt_g, reinterpret_cast<const float2*>(delta_k), scale,
                                   reinterpret_cast<float2*>(fkx), reinterpret_cast<float2*>(fky),
                                   reinterpret_cast<float2*>(fkz), ctx->stream));
  return FPM_OK;
}

int fpm_readout(fpm_ctx* ctx, const float* mesh, const float* pos, int64_t n, float* out) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_readout");
  FPM_REQUIRE(ctx, n >= 0 && mesh && ((pos && out) || n == 0), "fpm_readout: bad arguments");
  ProfScope sc(&ctx->prof, K_READOUT);
  FPM_CUDA(ctx, readout(mesh, pos, n, ctx->cfg.ng, out, order_of(ctx, n), ctx->stream));
  return FPM_OK;
}

int fpm_force(fpm_ctx* ctx, const float* pos, int64_t n, float* force) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_force");
  FPM_REQUIRE(ctx, n >= 0 && ((pos && force) || n == 0), "fpm_force: bad arguments");
  FPM_NEED_WS(ctx);
  const Workspace w = carve(ctx);
  const int rc = force_meshes(ctx, w, pos, n);
  if (rc != FPM_OK) return rc;
  ProfScope sc(&ctx->prof, K_READOUT);
  FPM_CUDA(ctx, readout3(w.F[0], w.F[1], w.F[2], pos, n, ctx->cfg.ng, force, order_of(ctx, n), ctx->stream));
  return FPM_OK;
}

const float* fpm_workspace_density(const fpm_ctx* ctx) {
  if (!ctx || !ctx->ws) return nullptr;
  return carve(ctx).rho;
}

int fpm_kick(fpm_ctx* ctx, float* mom, const float* force, int64_t n, double ai, double ac,
             double af) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_kick");
  FPM_REQUIRE(ctx, n >= 0 && ((mom && force) || n == 0), "fpm_kick: bad arguments");
  FPM_REQUIRE(ctx, ai > 0.0 && ac > 0.0 && af > 0.0, "fpm_kick: scale factors must be positive");
  const double k = kick_factor(ctx->cfg.omega_m, ai, ac, af, ctx->cfg.factor_mode);
  ProfScope sc(&ctx->prof, K_KICK);
  FPM_CUDA(ctx, kick(mom, force, 3 * n, (float)k, ctx->stream));
  return FPM_OK;
}

int fpm_drift(fpm_ctx* ctx, float* pos, const float* mom, int64_t n, double ai, double ac,
              double af) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_drift");
  FPM_REQUIRE(ctx, n >= 0 && ((pos && mom) || n == 0), "fpm_drift: bad arguments");
  FPM_REQUIRE(ctx, ai > 0.0 && ac > 0.0 && af > 0.0, "fpm_drift: scale factors must be positive");
  const double d = drift_factor(ctx->cfg.omega_m, ai, ac, af, ctx->cfg.factor_mode);
  ProfScope sc(&ctx->prof, K_DRIFT);
  FPM_CUDA(ctx, drift(pos, mom, 3 * n, (float)d, ctx->cfg.ng, ctx->stream));
  return FPM_OK;
}

}  // extern "C"

namespace {
int lpt_init_one(fpm_ctx* ctx, const float* delta_lin, double a0, int order, float* pos, float* mom);
}

extern "C" {

int fpm_lpt_init(fpm_ctx* ctx, const float* delta_lin, double a0, int order, float* pos,
                 float* mom) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, delta_lin && pos && mom, "fpm_lpt_init: null pointer");
  FPM_REQUIRE(ctx, order == 1 || order == 2, "fpm_lpt_init: order must be 1 or 2");
  FPM_REQUIRE(ctx, a0 > 0.0, "fpm_lpt_init: a0 must be positive");
  FPM_NEED_WS(ctx);
  // initial conditions are made once per run: the simulations of a batch take their turn (Alg. 4 each)
  const int64_t n3 = (int64_t)ctx->cfg.np * ctx->cfg.np * ctx->cfg.np;
  for (int b = 0; b < batch_of(ctx->cfg); ++b) {
    const int rc = lpt_init_one(ctx, delta_lin + b * n3, a0, order, pos + 3 * b * n3, mom + 3 * b * n3);
    if (rc != FPM_OK) return rc;
  }
  return FPM_OK;
}

}  // extern "C"

namespace {

int lpt_init_one(fpm_ctx* ctx, const float* delta_lin, double a0, int order, float* pos, float* mom) {
  const Workspace w = carve(ctx);
  cudaStream_t s = ctx->stream;
  const int np = ctx->cfg.np, ng = ctx->cfg.ng, bfac = ng / np;
  const int64_t n3 = (int64_t)np * np * np;
  const GrowthOut g = growth(ctx->cfg.omega_m, a0);
  const double pre = a0 * a0 * g.E;
  float2 *dk = w.dk, *tk = w.fk[0], *sk = w.fk[1];
  float *ra = w.F[0], *rb = w.F[1], *rc = w.F[2], *src = w.rho;

  FPM_CUDA(ctx, fft_r2c(ctx->fft_p, delta_lin, dk, s, &ctx->prof));
  // psi1_d = c2r(i k_d delta / k^2);  x = q + D1 psi1,  p = a^2 E f1 D1 psi1   (1LPT / Zel'dovich)
  for (int d = 0; d < 3; ++d) {
    ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, dk, tk, d, -1, -1.f, s));
    FPM_CUDA(ctx, fft_c2r(ctx->fft_p, tk, ra, s, &ctx->prof));
    ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_displace(ra, np, bfac, d, (float)g.D1, (float)(pre * g.f1 * g.D1), true,
                               pos + d * n3, mom + d * n3, s));
  }
  if (order == 2) {
    // S = sum_{i<j} (phi,ii phi,jj - phi,ij^2), phi,ij = c2r(k_i k_j delta / k^2)
    ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, dk, tk, 0, 0, 1.f, s));
    FPM_CUDA(ctx, fft_c2r(ctx->fft_p, tk, ra, s, &ctx->prof));
    ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, dk, tk, 1, 1, 1.f, s));
    FPM_CUDA(ctx, fft_c2r(ctx->fft_p, tk, rb, s, &ctx->prof));
    ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_source(src, ra, rb, nullptr, n3, 0, s));
    ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, dk, tk, 2, 2, 1.f, s));
    FPM_CUDA(ctx, fft_c2r(ctx->fft_p, tk, rc, s, &ctx->prof));
    ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_source(src, ra, rb, rc, n3, 1, s));
    const int pairs[3][2] = {{0, 1}, {0, 2}, {1, 2}};
    for (auto& pr : pairs) {
      ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, dk, tk, pr[0], pr[1], 1.f, s));
      FPM_CUDA(ctx, fft_c2r(ctx->fft_p, tk, ra, s, &ctx->prof));
      ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_source(src, ra, nullptr, nullptr, n3, 2, s));
    }
    FPM_CUDA(ctx, fft_r2c(ctx->fft_p, src, sk, s, &ctx->prof));
    // psi2_d = c2r(-i k_d S / k^2);  x += D2 psi2,  p += a^2 E f2 D2 psi2
    for (int d = 0; d < 3; ++d) {
      ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, sk, tk, d, -1, 1.f, s));
      FPM_CUDA(ctx, fft_c2r(ctx->fft_p, tk, ra, s, &ctx->prof));
      ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_displace(ra, np, bfac, d, (float)g.D2, (float)(pre * g.f2 * g.D2), false,
                                 pos + d * n3, mom + d * n3, s));
    }
  }
  ctx->prof.launches += 1; FPM_CUDA(ctx, lpt_wrap(pos, 3 * n3, ng, s));
  return FPM_OK;
}

// the n_steps + 1 PM steps of a run, enqueued kernel by kernel on ctx->stream
int run_steps(fpm_ctx* ctx, float* pos, float* mom, const std::vector<double>& kf, const std::vector<double>& dr,
              float* traj) {
  const Workspace w = carve(ctx);
  const int64_t n = (int64_t)ctx->cfg.np * ctx->cfg.np * ctx->cfg.np;
  const size_t state = sizeof(float) * 3 * (size_t)n * batch_of(ctx->cfg);
  for (size_t j = 0; j < kf.size(); ++j) {
    if (traj)
      FPM_CUDA(ctx, cudaMemcpyAsync(reinterpret_cast<char*>(traj) + j * state, pos, state, cudaMemcpyDeviceToDevice,
                                    ctx->stream));
    const int rc = pm_step(ctx, w, pos, mom, n, kf[j], dr[j]);
    if (rc != FPM_OK) return rc;
  }
  return FPM_OK;
}

// The same run as ONE CUDA graph launch (fpm.h FPM_GRAPH_*): a small configuration spends its step in launch
// latency (C1: 8 launches of 6-24 us for 0.1 ms of work), so the run is captured once -- on an internal stream:
// the caller's may be the legacy default stream, which cannot be captured -- and replayed on ctx->stream.
// Graphs are cached per (pos, mom, traj, factors).  Capture + instantiation cost more than the launches one
// replay saves, so under FPM_GRAPH_AUTO an argument set is captured only the second time in a row it is seen
// (`always` = FPM_GRAPH_ALWAYS captures at once).  Returns FPM_ENOTIMPL when no graph is used or capture is not
// possible (the caller then enqueues kernel by kernel); nothing has been enqueued in that case.
int run_graph(fpm_ctx* ctx, float* pos, float* mom, const std::vector<double>& kf, const std::vector<double>& dr,
              float* traj, bool always) {
  for (auto& g : ctx->graphs)
    if (g.pos == pos && g.mom == mom && g.traj == traj && g.kf == kf && g.dr == dr) {
      FPM_CUDA(ctx, cudaGraphLaunch(g.exec, ctx->stream));
      ctx->prof.launches += g.launches;
      return FPM_OK;
    }
  if (!always) {
    auto& sn = ctx->seen;
    const bool again = sn.valid && sn.pos == pos && sn.mom == mom && sn.traj == traj && sn.kf == kf && sn.dr == dr;
    if (!again) {
      sn.pos = pos; sn.mom = mom; sn.traj = traj; sn.kf = kf; sn.dr = dr; sn.valid = true;
      return FPM_ENOTIMPL;
    }
    sn.valid = false;
  }
  if (!ctx->capture_stream &&
      cudaStreamCreateWithFlags(&ctx->capture_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    return FPM_ENOTIMPL;
  }
  cudaStream_t user = ctx->stream;
  const long long before = ctx->prof.launches;
  if (cudaStreamBeginCapture(ctx->capture_stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
    cudaGetLastError();
    return FPM_ENOTIMPL;
  }
  ctx->stream = ctx->capture_stream;
  ctx->prof.stream = ctx->capture_stream;
  const int rc = run_steps(ctx, pos, mom, kf, dr, traj);
  ctx->stream = user;
  ctx->prof.stream = user;
  cudaGraph_t graph = nullptr;
  const cudaError_t e = cudaStreamEndCapture(ctx->capture_stream, &graph);
  const long long nodes = ctx->prof.launches - before;
  ctx->prof.launches = before;
  cudaGraphExec_t exec = nullptr;
  if (rc != FPM_OK || e != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    ctx->sticky = false;                 // a failed capture enqueued nothing; the eager path reports real errors
    return FPM_ENOTIMPL;
  }
  cudaGraphDestroy(graph);
  if (ctx->graphs.size() >= 8) {         // small cache: drop the oldest
    cudaGraphExecDestroy(ctx->graphs.front().exec);
    ctx->graphs.erase(ctx->graphs.begin());
  }
  ctx->graphs.push_back(fpm_ctx::RunGraph{pos, mom, traj, kf, dr, exec, nodes});
  FPM_CUDA(ctx, cudaGraphLaunch(exec, ctx->stream));
  ctx->prof.launches += nodes;
  return FPM_OK;
}

}  // namespace

extern "C" {

int fpm_nbody(fpm_ctx* ctx, float* pos, float* mom, const double* a_stages, int n_steps,
              float* traj) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, pos && mom && a_stages && n_steps >= 0, "fpm_nbody: bad arguments");
  for (int j = 0; j <= n_steps; ++j)
    FPM_REQUIRE(ctx, a_stages[j] > 0.0, "fpm_nbody: scale factors must be positive");
  FPM_NEED_WS(ctx);
  std::vector<double> kf(n_steps + 1), dr(n_steps + 1);
  step_factors(ctx, a_stages, n_steps, kf.data(), dr.data());
  const int64_t cells = (int64_t)batch_of(ctx->cfg) * ctx->cfg.ng * ctx->cfg.ng * ctx->cfg.ng;
  const bool want_graph = ctx->graph_mode == FPM_GRAPH_ALWAYS ||
                          (ctx->graph_mode == FPM_GRAPH_AUTO && cells <= (int64_t(1) << 24));
  // Inside the CALLER's own stream capture (e.g. torch.cuda.graph) the run must stay plain launches on
  // ctx->stream, which the caller's graph then records: creating a stream, capturing or instantiating here could
  // be refused or invalidate that capture.  (On the legacy default stream the query itself fails while another
  // stream captures in global mode -- without harming that capture; treated the same way.)
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(ctx->stream, &cap) != cudaSuccess) {
    cudaGetLastError();
    cap = cudaStreamCaptureStatusActive;
  }
  if (want_graph && !ctx->prof.enabled && cap == cudaStreamCaptureStatusNone) {   // (event timing needs kernel by kernel)
    const int rc = run_graph(ctx, pos, mom, kf, dr, traj, ctx->graph_mode == FPM_GRAPH_ALWAYS);
    if (rc != FPM_ENOTIMPL) return rc;
  }
  return run_steps(ctx, pos, mom, kf, dr, traj);
}

int fpm_nbody_host(fpm_ctx* ctx, float* h_pos, float* h_mom, float* d_pos, float* d_mom,
                   const double* a_stages, int n_steps) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_nbody_host");
  FPM_REQUIRE(ctx, h_pos && h_mom && d_pos && d_mom, "fpm_nbody_host: null pointer");
  const int64_t n = (int64_t)ctx->cfg.np * ctx->cfg.np * ctx->cfg.np;
  const size_t bytes = sizeof(float) * 3 * (size_t)n;
  cudaStream_t s = ctx->stream;
  FPM_CUDA(ctx, cudaMemcpyAsync(d_pos, h_pos, bytes, cudaMemcpyHostToDevice, s));
  FPM_CUDA(ctx, cudaMemcpyAsync(d_mom, h_mom, bytes, cudaMemcpyHostToDevice, s));
  const int rc = fpm_nbody(ctx, d_pos, d_mom, a_stages, n_steps, nullptr);
  if (rc != FPM_OK) return rc;
  FPM_CUDA(ctx, cudaMemcpyAsync(h_pos, d_pos, bytes, cudaMemcpyDeviceToHost, s));
  FPM_CUDA(ctx, cudaMemcpyAsync(h_mom, d_mom, bytes, cudaMemcpyDeviceToHost, s));
  FPM_CUDA(ctx, cudaStreamSynchronize(s));
  return FPM_OK;
}

int fpm_pm_step(fpm_ctx* ctx, float* pos, float* mom, int64_t n, double kick_fac, double drift_fac) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, n >= 0 && ((pos && mom) || n == 0), "fpm_pm_step: bad arguments");
  FPM_REQUIRE(ctx, std::isfinite(kick_fac) && std::isfinite(drift_fac), "fpm_pm_step: non-finite factor");
  FPM_NEED_WS(ctx);
  return pm_step(ctx, carve(ctx), pos, mom, n, kick_fac, drift_fac);
}

int fpm_pm_step_host(fpm_ctx* ctx, float* h_pos, float* h_mom, float* d_pos, float* d_mom, int64_t n,
                     double kick_fac, double drift_fac) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_pm_step_host");
  FPM_REQUIRE(ctx, n >= 0 && h_pos && h_mom && d_pos && d_mom, "fpm_pm_step_host: bad arguments");
  const size_t bytes = sizeof(float) * 3 * (size_t)n;
  cudaStream_t s = ctx->stream;
  FPM_CUDA(ctx, cudaMemcpyAsync(d_pos, h_pos, bytes, cudaMemcpyHostToDevice, s));
  FPM_CUDA(ctx, cudaMemcpyAsync(d_mom, h_mom, bytes, cudaMemcpyHostToDevice, s));
  const int rc = fpm_pm_step(ctx, d_pos, d_mom, n, kick_fac, drift_fac);
  if (rc != FPM_OK) return rc;
  FPM_CUDA(ctx, cudaMemcpyAsync(h_pos, d_pos, bytes, cudaMemcpyDeviceToHost, s));
  FPM_CUDA(ctx, cudaMemcpyAsync(h_mom, d_mom, bytes, cudaMemcpyDeviceToHost, s));
  FPM_CUDA(ctx, cudaStreamSynchronize(s));
  return FPM_OK;
}

int fpm_force_vjp(fpm_ctx* ctx, const float* pos, int64_t n, const float* v, double coef,
                  float* grad_pos) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_force_vjp");
  FPM_REQUIRE(ctx, n >= 0 && ((pos && v && grad_pos) || n == 0), "fpm_force_vjp: bad arguments");
  FPM_REQUIRE(ctx, std::isfinite(coef), "fpm_force_vjp: non-finite coefficient");
  FPM_NEED_WS(ctx);
  return force_vjp(ctx, carve(ctx), pos, n, v, coef, grad_pos);
}

int fpm_nbody_vjp(fpm_ctx* ctx, const float* traj, const double* a_stages, int n_steps,
                  float* grad_pos, float* grad_mom, int flags) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_nbody_vjp");
  FPM_REQUIRE(ctx, traj && a_stages && grad_pos && grad_mom && n_steps >= 0, "fpm_nbody_vjp: bad arguments");
  FPM_REQUIRE(ctx, (flags & ~FPM_VJP_GRAD_MOM_ZERO) == 0, "fpm_nbody_vjp: unknown flag");
  for (int j = 0; j <= n_steps; ++j)
    FPM_REQUIRE(ctx, a_stages[j] > 0.0, "fpm_nbody_vjp: scale factors must be positive");
  FPM_NEED_WS(ctx);
  const Workspace w = carve(ctx);
  const int np = ctx->cfg.np;
  const int64_t n = (int64_t)np * np * np;
  // the same merged factors as fpm_nbody: step j is  p += kf_j f(x_j);  x = wrap(x + dr_j p)
  std::vector<double> kf(n_steps + 1), dr(n_steps + 1);
  step_factors(ctx, a_stages, n_steps, kf.data(), dr.data());
  for (int j = n_steps; j >= 0; --j) {
    // x' = wrap(x + dr p'):  p'_bar += dr x'_bar   (wrap has unit derivative)
    if (dr[j] != 0.0) {
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, axpy(grad_mom, grad_pos, (float)dr[j], 3 * n, ctx->stream));
    }
    // p' = p + kf f(x_j):  x_bar += kf J_f(x_j)^T p'_bar
    // (with a loss on the final positions only, p'_bar of the last step is identically zero: nothing to add)
    if (j == n_steps && (flags & FPM_VJP_GRAD_MOM_ZERO)) continue;
    if (kf[j] != 0.0) {
      const int rc = force_vjp(ctx, w, traj + (int64_t)j * 3 * n, n, grad_mom, kf[j], grad_pos);
      if (rc != FPM_OK) return rc;
    }
  }
  return FPM_OK;
}

int fpm_lpt_init_vjp(fpm_ctx* ctx, const float* delta_lin, double a0, int order,
                     const float* grad_pos, const float* grad_mom, float* grad_delta) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_lpt_init_vjp");
  FPM_REQUIRE(ctx, delta_lin && grad_pos && grad_mom && grad_delta, "fpm_lpt_init_vjp: null pointer");
  FPM_REQUIRE(ctx, order == 1 || order == 2, "fpm_lpt_init_vjp: order must be 1 or 2");
  FPM_REQUIRE(ctx, a0 > 0.0, "fpm_lpt_init_vjp: a0 must be positive");
  FPM_NEED_WS(ctx);
  const Workspace w = carve(ctx);
  cudaStream_t s = ctx->stream;
  Profiler* pr = &ctx->prof;
  const int np = ctx->cfg.np, bfac = ctx->cfg.ng / np;
  const int64_t n3 = (int64_t)np * np * np;
  const GrowthOut g = growth(ctx->cfg.omega_m, a0);
  const double pre = a0 * a0 * g.E;
  float2 *dk = w.dk, *tk = w.fk[0], *acck = w.fk[1];
  float* bar = reinterpret_cast<float*>(w.fk[2]);
  float* sbar = w.rho;
  // x = q B + (D1 psi1 + D2 psi2) B,  p = a^2 E (f1 D1 psi1 + f2 D2 psi2) B
  // psi1_d = T[i k_d / k^2] delta  ->  delta_bar_k += (-i k_d / k^2) psi1bar_d,k
  for (int d = 0; d < 3; ++d) {
    ctx->prof.launches += 1;
    FPM_CUDA(ctx, lincomb2(bar, grad_pos + d * n3, (float)(bfac * g.D1), grad_mom + d * n3,
                           (float)(bfac * pre * g.f1 * g.D1), n3, s));
    FPM_CUDA(ctx, fft_r2c(ctx->fft_p, bar, tk, s, pr));
    ctx->prof.launches += 1;
    FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, tk, acck, d, -1, 1.f, s, d > 0));
  }
  if (order == 2) {
    // psi2_d = T[-i k_d / k^2] S  ->  S_bar_k = sum_d (+i k_d / k^2) psi2bar_d,k
    for (int d = 0; d < 3; ++d) {
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, lincomb2(bar, grad_pos + d * n3, (float)(bfac * g.D2), grad_mom + d * n3,
                             (float)(bfac * pre * g.f2 * g.D2), n3, s));
      FPM_CUDA(ctx, fft_r2c(ctx->fft_p, bar, tk, s, pr));
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, tk, dk, d, -1, -1.f, s, d > 0));
    }
    FPM_CUDA(ctx, fft_c2r(ctx->fft_p, dk, sbar, s, pr));
    // S = sum_{i<j} (phi,ii phi,jj - phi,ij^2), phi,ij = T[k_i k_j / k^2] delta (real, even: self-adjoint)
    FPM_CUDA(ctx, fft_r2c(ctx->fft_p, delta_lin, dk, s, pr));
    for (int c = 0; c < 3; ++c) {
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, dk, tk, c, c, 1.f, s));
      FPM_CUDA(ctx, fft_c2r(ctx->fft_p, tk, w.F[c], s, pr));
    }
    for (int c = 0; c < 3; ++c) {
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, lpt_phibar(bar, sbar, w.F[(c + 1) % 3], w.F[(c + 2) % 3], n3, s));
      FPM_CUDA(ctx, fft_r2c(ctx->fft_p, bar, tk, s, pr));
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, tk, acck, c, c, 1.f, s, true));
    }
    const int pairs[3][2] = {{0, 1}, {0, 2}, {1, 2}};
    for (auto& pq : pairs) {
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, dk, tk, pq[0], pq[1], 1.f, s));
      FPM_CUDA(ctx, fft_c2r(ctx->fft_p, tk, w.F[0], s, pr));
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, lpt_phibar(bar, sbar, w.F[0], nullptr, n3, s));
      FPM_CUDA(ctx, fft_r2c(ctx->fft_p, bar, tk, s, pr));
      ctx->prof.launches += 1;
      FPM_CUDA(ctx, lpt_spectral(ctx->kt_p, tk, acck, pq[0], pq[1], 1.f, s, true));
    }
  }
  FPM_CUDA(ctx, fft_c2r(ctx->fft_p, acck, grad_delta, s, pr));
  return FPM_OK;
}

size_t fpm_recon_scratch_bytes(const fpm_config* cfg, int n_steps) {
  if (!config_ok(cfg) || n_steps < 0) return 0;
  const size_t n = (size_t)cfg->np * cfg->np * cfg->np;
  return sizeof(float) * 3 * n * ((size_t)n_steps + 5);
}

int fpm_recon_loss_grad(fpm_ctx* ctx, const float* s_lin, const float* data, double sigma,
                        const float* inv_power, const double* a_stages, int n_steps, int lpt_order,
                        void* scratch, size_t scratch_bytes, float* grad, double* loss) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_recon_loss_grad");
  FPM_REQUIRE(ctx, s_lin && data && inv_power && a_stages && scratch && grad && loss && n_steps >= 0,
              "fpm_recon_loss_grad: bad arguments");
  FPM_REQUIRE(ctx, sigma > 0.0, "fpm_recon_loss_grad: sigma must be positive");
  FPM_REQUIRE(ctx, (reinterpret_cast<uintptr_t>(scratch) & 15) == 0, "fpm_recon_loss_grad: scratch must be 16-byte aligned");
  if (scratch_bytes < fpm_recon_scratch_bytes(&ctx->cfg, n_steps))
    return fail(ctx, FPM_ENOMEM, "fpm_recon_loss_grad: scratch too small (fpm_recon_scratch_bytes)");
  FPM_NEED_WS(ctx);
  const Workspace w = carve(ctx);
  cudaStream_t st = ctx->stream;
  Profiler* pr = &ctx->prof;
  const int np = ctx->cfg.np, ng = ctx->cfg.ng;
  const int64_t n = (int64_t)np * np * np, g3 = (int64_t)ng * ng * ng;
  float* pos = static_cast<float*>(scratch);
  float *mom = pos + 3 * n, *gx = mom + 3 * n, *gp = gx + 3 * n, *traj = gp + 3 * n;
  FPM_CUDA(ctx, cudaMemsetAsync(ctx->d_acc, 0, 2 * sizeof(double), st));
  // forward model F(s) (Listing 7.1 "model = FLOWPM(var, ...)")
  int rc = fpm_lpt_init(ctx, s_lin, a_stages[0], lpt_order, pos, mom);
  if (rc != FPM_OK) return rc;
  rc = fpm_nbody(ctx, pos, mom, a_stages, n_steps, traj);
  if (rc != FPM_OK) return rc;
  { ProfScope sc(pr, K_PAINT);
    FPM_CUDA(ctx, paint(pos, nullptr, particle_mass(ctx), n, ng, w.rho, true, order_of(ctx, n), st)); }
  // likelihood term and its cotangent on the mesh
  ctx->prof.launches += 1;
  FPM_CUDA(ctx, recon_residual(w.rho, data, (float)(1.0 / (sigma * sigma)), g3, w.F[0], ctx->d_acc, st));
  // reverse: paint -> run -> initial conditions
  { ProfScope sc(pr, K_READOUT_GRAD);
    FPM_CUDA(ctx, readout_grad(w.F[0], pos, nullptr, particle_mass(ctx), n, ng, gx, nullptr, st)); }
  FPM_CUDA(ctx, cudaMemsetAsync(gp, 0, sizeof(float) * 3 * n, st));
  rc = fpm_nbody_vjp(ctx, traj, a_stages, n_steps, gx, gp, FPM_VJP_GRAD_MOM_ZERO);
  if (rc != FPM_OK) return rc;
  rc = fpm_lpt_init_vjp(ctx, s_lin, a_stages[0], lpt_order, gx, gp, grad);
  if (rc != FPM_OK) return rc;
  // prior term (Listing 7.1 "prior = sum(r2c(var)^2 / power)") and its gradient n^3 c2r(inv_power s_k)
  FPM_CUDA(ctx, fft_r2c(ctx->fft_p, s_lin, w.dk, st, pr));
  ctx->prof.launches += 1;
  FPM_CUDA(ctx, recon_prior(w.dk, inv_power, np, w.fk[0], ctx->d_acc + 1, st));
  FPM_CUDA(ctx, fft_c2r(ctx->fft_p, w.fk[0], w.F[0], st, pr));
  ctx->prof.launches += 1;
  FPM_CUDA(ctx, axpy(grad, w.F[0], 1.f, n, st));
  double acc[2];
  FPM_CUDA(ctx, cudaMemcpyAsync(acc, ctx->d_acc, sizeof acc, cudaMemcpyDeviceToHost, st));
  FPM_CUDA(ctx, cudaStreamSynchronize(st));
  loss[0] = 0.5 * acc[0] / (sigma * sigma);
  loss[1] = 0.5 * acc[1];
  return FPM_OK;
}

int fpm_adam_step(fpm_ctx* ctx, float* x, const float* grad, float* m, float* v, int64_t n, double lr,
                  double beta1, double beta2, double eps, int t) {
  FPM_ENTER(ctx);
  FPM_REQUIRE(ctx, n >= 0 && ((x && grad && m && v) || n == 0), "fpm_adam_step: bad arguments");
  FPM_REQUIRE(ctx, t >= 1 && beta1 >= 0.0 && beta1 < 1.0 && beta2 >= 0.0 && beta2 < 1.0, "fpm_adam_step: bad hyper-parameters");
  if (n == 0) return FPM_OK;
  const double c1 = 1.0 - std::pow(beta1, t), c2 = 1.0 - std::pow(beta2, t);
  ctx->prof.launches += 1;
  FPM_CUDA(ctx, adam_update(x, grad, m, v, n, lr, beta1, beta2, eps, 1.0 / c1, 1.0 / c2, ctx->stream));
  return FPM_OK;
}

}  // extern "C"

namespace {

inline int64_t cube(int64_t n) { return n * n * n; }

// REDUCE in (n^3) by `levels` levels into out; scratch: n^3 floats (3/4 + 1/8 of each level's mesh)
int pyr_reduce(fpm_ctx* ctx, const float* in, int n, int levels, float* scratch, float* out) {
  if (levels == 0) {
    FPM_CUDA(ctx, cudaMemcpyAsync(out, in, sizeof(float) * cube(n), cudaMemcpyDeviceToDevice, ctx->stream));
    return FPM_OK;
  }
  const float* cur = in;
  for (int l = 0; l < levels; ++l) {
    float* tmp = scratch;
    float* dst = (l == levels - 1) ? out : scratch + 3 * cube(n) / 4;
    ctx->prof.launches += 3;
    FPM_CUDA(ctx, pyramid_reduce_level(cur, n, tmp, dst, ctx->stream));
    scratch += 3 * cube(n) / 4 + cube(n / 2);
    cur = dst;
    n /= 2;
  }
  return FPM_OK;
}

// EXPAND in (m^3) by `levels` levels into out ((m << levels)^3); scratch: (m << levels)^3 floats
int pyr_expand(fpm_ctx* ctx, const float* in, int m, int levels, float* scratch, float* out) {
  if (levels == 0) {
    FPM_CUDA(ctx, cudaMemcpyAsync(out, in, sizeof(float) * cube(m), cudaMemcpyDeviceToDevice, ctx->stream));
    return FPM_OK;
  }
  const float* cur = in;
  for (int l = 0; l < levels; ++l) {
    float* tmp = scratch;
    float* dst = (l == levels - 1) ? out : scratch + 6 * cube(m);
    ctx->prof.launches += 3;
    FPM_CUDA(ctx, pyramid_expand_level(cur, m, tmp, dst, ctx->stream));
    scratch += 6 * cube(m) + 8 * cube(m);
    cur = dst;
    m *= 2;
  }
  return FPM_OK;
}

bool pyramid_levels_ok(const fpm_ctx* ctx, int levels) {
  return levels >= 0 && levels < 8 && (ctx->cfg.ng >> levels) >= 8;
}

}  // namespace

extern "C" {

int fpm_reduce(fpm_ctx* ctx, const float* in, int levels, float* out) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_reduce");
  FPM_REQUIRE(ctx, in && out && in != out, "fpm_reduce: bad arguments");
  FPM_REQUIRE(ctx, pyramid_levels_ok(ctx, levels), "fpm_reduce: levels out of range (ng >> levels >= 8)");
  FPM_NEED_WS(ctx);
  return pyr_reduce(ctx, in, ctx->cfg.ng, levels, reinterpret_cast<float*>(carve(ctx).dk), out);
}

int fpm_expand(fpm_ctx* ctx, const float* in, int levels, float* out) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_expand");
  FPM_REQUIRE(ctx, in && out && in != out, "fpm_expand: bad arguments");
  FPM_REQUIRE(ctx, pyramid_levels_ok(ctx, levels), "fpm_expand: levels out of range (ng >> levels >= 8)");
  FPM_NEED_WS(ctx);
  return pyr_expand(ctx, in, ctx->cfg.ng >> levels, levels, reinterpret_cast<float*>(carve(ctx).dk), out);
}

int fpm_force_pyramid(fpm_ctx* ctx, const float* pos, int64_t n, int levels, float* force) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_force_pyramid");
  FPM_REQUIRE(ctx, n >= 0 && ((pos && force) || n == 0), "fpm_force_pyramid: bad arguments");
  FPM_REQUIRE(ctx, pyramid_levels_ok(ctx, levels), "fpm_force_pyramid: levels out of range (ng >> levels >= 8)");
  FPM_NEED_WS(ctx);
  const Workspace w = carve(ctx);
  cudaStream_t s = ctx->stream;
  Profiler* pr = &ctx->prof;
  const int ng = ctx->cfg.ng, nc = ng >> levels;
  const float scale = (float)(1.5 * ctx->cfg.omega_m);
  if (ctx->coarse_n != nc) {                      // plans of the coarse mesh, kept for the next call
    fft_tables_destroy(&ctx->fft_c);
    kernel_tables_destroy(&ctx->kt_c);
    ctx->coarse_n = 0;
    FPM_CUDA(ctx, fft_tables_create(nc, &ctx->fft_c));
    FPM_CUDA(ctx, kernel_tables_create(nc, ctx->cfg.kernel_mode, &ctx->kt_c));
    ctx->coarse_n = nc;
  }
  // F_S <= ForceGrids(H, local): the single-mesh force meshes, op by op (Alg. 3 ForceGrids)
  { ProfScope sc(pr, K_PAINT); FPM_CUDA(ctx, paint(pos, nullptr, particle_mass(ctx), n, ng, w.rho, true, order_of(ctx, n), s)); }
  FPM_CUDA(ctx, fft_r2c(ctx->fft_g, w.rho, w.dk, s, pr));
  { ProfScope sc(pr, K_GREEN); FPM_CUDA(ctx, apply_force_kernel(ctx->kt_g, w.dk, scale, w.fk[0], w.fk[1], w.fk[2], s)); }
  for (int d = 0; d < 3; ++d) FPM_CUDA(ctx, fft_c2r(ctx->fft_g, w.fk[d], w.F[d], s, pr));
  if (levels == 0) {     // no reduction: F_L = F_S and EXPAND = REDUCE = identity, so F = F_S exactly
    ProfScope sc(pr, K_READOUT);
    FPM_CUDA(ctx, readout3(w.F[0], w.F[1], w.F[2], pos, n, ng, force, order_of(ctx, n), s));
    return FPM_OK;
  }
  // the four half-complex regions are free now; each holds one real mesh (and a little more: padded pitch)
  const int64_t g3 = cube(ng), c3 = cube(nc);
  float* scratch = reinterpret_cast<float*>(w.dk);            // pyr_reduce / pyr_expand scratch (< g3 floats)
  float* up = w.rho;                                          // EXPAND(F_L): rho is dead once D is made
  float* lowup = reinterpret_cast<float*>(w.fk[0]);           // EXPAND(REDUCE(F_S))
  float* coarse = reinterpret_cast<float*>(w.fk[1]);          // D | F_L[3] | low   (5 c3 <= 5/8 g3 floats)
  float* D = coarse;
  float* FL[3] = {coarse + c3, coarse + 2 * c3, coarse + 3 * c3};
  float* low = coarse + 4 * c3;
  float2* ck = reinterpret_cast<float2*>(w.fk[2]);            // coarse spectra: dk | fk[3]  (~4 c3 floats)
  const int64_t ckn = (int64_t)nc * nc * (nc / 2 + 1);
  // D <= REDUCE(H);  F_L <= ForceGrids(D, distributed), in fine-cell units
  int rc = pyr_reduce(ctx, w.rho, ng, levels, scratch, D);
  if (rc != FPM_OK) return rc;
  FPM_CUDA(ctx, fft_r2c(ctx->fft_c, D, ck, s, pr));
  { ProfScope sc(pr, K_GREEN);
    FPM_CUDA(ctx, apply_force_kernel(ctx->kt_c, ck, scale * (float)(1 << levels), ck + ckn, ck + 2 * ckn, ck + 3 * ckn, s)); }
  for (int d = 0; d < 3; ++d) FPM_CUDA(ctx, fft_c2r(ctx->fft_c, ck + (d + 1) * ckn, FL[d], s, pr));
  for (int d = 0; d < 3; ++d) {
    rc = pyr_expand(ctx, FL[d], nc, levels, scratch, up);          // F_iL <= EXPAND(F_iL)
    if (rc != FPM_OK) return rc;
    rc = pyr_reduce(ctx, w.F[d], ng, levels, scratch, low);        // F_il <= REDUCE(F_iS)
    if (rc != FPM_OK) return rc;
    rc = pyr_expand(ctx, low, nc, levels, scratch, lowup);         // F_il <= EXPAND(F_il)
    if (rc != FPM_OK) return rc;
    ctx->prof.launches += 1;
    FPM_CUDA(ctx, pyramid_combine(w.F[d], up, lowup, g3, s));      // F_i <= F_iL + (F_iS - F_il)
  }
  ProfScope sc(pr, K_READOUT);
  FPM_CUDA(ctx, readout3(w.F[0], w.F[1], w.F[2], pos, n, ng, force, order_of(ctx, n), s));
  return FPM_OK;
}

int fpm_profile_enable(fpm_ctx* ctx, int on) {
  if (!ctx) return FPM_EINVAL;
  DeviceGuard device_guard__(ctx->device);
  ctx->prof.flush();
  ctx->prof.enabled = on != 0;
  return FPM_OK;
}

int fpm_profile_reset(fpm_ctx* ctx) {
  if (!ctx) return FPM_EINVAL;
  DeviceGuard device_guard__(ctx->device);
  ctx->prof.reset();
  return FPM_OK;
}

int fpm_profile_read(fpm_ctx* ctx, int kernel_id, const char** name, double* total_ms, int64_t* count) {
  if (!ctx || kernel_id < 0 || kernel_id >= K_COUNT) return FPM_EINVAL;
  DeviceGuard device_guard__(ctx->device);
  ctx->prof.flush();
  if (name) *name = kernel_name(kernel_id);
  if (total_ms) *total_ms = ctx->prof.ms[kernel_id];
  if (count) *count = ctx->prof.count[kernel_id];
  return FPM_OK;
}

int64_t fpm_launch_count(const fpm_ctx* ctx) { return ctx ? ctx->prof.launches : -1; }

int fpm_paint_adjoint(fpm_ctx* ctx, const float* pos, const float* mass, int64_t n,
                      const float* grad_mesh, float* grad_pos, float* grad_mass) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_paint_adjoint");
  FPM_REQUIRE(ctx, n >= 0 && grad_mesh && ((pos && grad_pos) || n == 0), "fpm_paint_adjoint: bad arguments");
  ProfScope sc(&ctx->prof, K_READOUT_GRAD);
  FPM_CUDA(ctx, readout_grad(grad_mesh, pos, mass, particle_mass(ctx), n, ctx->cfg.ng, grad_pos,
                             grad_mass, ctx->stream));
  return FPM_OK;
}

int fpm_readout_adjoint(fpm_ctx* ctx, const float* mesh, const float* pos, int64_t n,
                        const float* grad_out, float* grad_mesh, float* grad_pos) {
  FPM_ENTER(ctx);
  FPM_NO_BATCH(ctx, "fpm_readout_adjoint");
  FPM_REQUIRE(ctx, n >= 0 && grad_mesh && ((pos && grad_out) || n == 0), "fpm_readout_adjoint: bad arguments");
  FPM_REQUIRE(ctx, !grad_pos || mesh, "fpm_readout_adjoint: grad_pos needs the forward mesh");
  { ProfScope sc(&ctx->prof, K_PAINT); FPM_CUDA(ctx, paint(pos, grad_out, 0.f, n, ctx->cfg.ng, grad_mesh, false, order_of(ctx, n), ctx->stream)); }
  if (grad_pos) {
    ProfScope sc(&ctx->prof, K_READOUT_GRAD);
    FPM_CUDA(ctx, readout_grad(mesh, pos, grad_out, 0.f, n, ctx->cfg.ng, grad_pos, nullptr, ctx->stream));
  }
  return FPM_OK;
}

}  // extern "C"
