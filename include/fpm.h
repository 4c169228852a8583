/* fpm.h -- C-ABI boundary of the B200-native FastPM particle-mesh step.
 *
 * One GPU, one stream, no collectives.  Every entry point follows the paper's statement of the
 * problem (FlowPM, arxiv 2010.11847; citations are PAPER.md:LINE) and SURVEY.md section 8(b).
 *
 * Conventions common to all calls
 *   - Return value: FPM_OK (0) or a negative fpm_status.  Argument validation is synchronous and
 *     has no side effects.  CUDA errors are sticky per context: once FPM_ECUDA is returned every
 *     later call on that context returns FPM_ECUDA; fpm_last_error() gives the text.  No
 *     exception crosses this boundary and the library never calls exit().
 *   - Unless a parameter is marked HOST, every array argument is a DEVICE pointer owned by the
 *     caller (e.g. a torch tensor's data_ptr()); the library never allocates, frees or keeps it.
 *     Scratch memory is also caller-owned: query fpm_workspace_bytes(), allocate, hand it over
 *     with fpm_set_workspace().  Only small plan tables (twiddles, per-axis kernel tables) are
 *     owned by the context.
 *   - All work is enqueued on the context's CUDA stream and the call returns without
 *     synchronising (except the *_host calls, which synchronise before returning).
 *   - Layouts.  Particles are structure-of-arrays: pos/mom/force are 3 contiguous planes
 *     [3][n] of float32; positions are in MESH-CELL units, wrapped to [0, ng); momenta are
 *     p = a^2 dx/dt / H0 in mesh cells.  Real meshes are [ng][ng][ng] float32, z fastest.
 *     k-space meshes are [ng][ng][ng/2+1] interleaved complex64 (the cuFFT r2c layout), integer
 *     frequency n_d in (-ng/2, ng/2], omega_d = 2 pi n_d / ng.
 *   - Sizes: ng and np are powers of two, 8 <= np <= ng <= 1024, ng % np == 0.
 *   - Performance paths: when n == np^3 particles are passed in lattice (Lagrangian) order -- what
 *     fpm_lpt_init produces and every later call preserves -- with np a multiple of 32 and 16-byte aligned
 *     arrays, paint, readout and the fused step walk the particles brick by brick (shared-memory paint
 *     window, cp.async-pipelined gathers); any other particle set takes the generic one-thread-per-particle
 *     kernels.  Gathers give the same values either way; for paint see FPM_PAINT_* below (the brick window
 *     is fixed point, within the stated quantum of the direct fp32 reductions).
 *   - Device: a context belongs to the CUDA device that was current in fpm_create; every later call runs
 *     there whatever device is current in the calling thread (which is restored on return).
 */
#ifndef FPM_H
#define FPM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  FPM_OK = 0,
  FPM_EINVAL = -1,   /* bad argument (null pointer, size, alignment, mode) */
  FPM_ENOMEM = -2,   /* workspace missing or too small */
  FPM_ECUDA = -3,    /* a CUDA call or kernel launch failed (sticky) */
  FPM_ENOTIMPL = -4
} fpm_status;

/* Transfer function nabla nabla^-2 (Eq. 3-5). */
enum {
  FPM_KERNEL_PAPER = 0, /* Eq. 4 (3-point Laplacian symbol) + Eq. 5 (4-point gradient) [default] */
  FPM_KERNEL_NAIVE = 1, /* -1/k^2 and i k ("the simplest way") */
  FPM_KERNEL_MIXED = 2  /* -1/k^2 and Eq. 5 */
};

/* Kick/drift operators (Eq. 1-2). */
enum {
  FPM_FACTORS_FASTPM = 0, /* growth-factor form (exact for a Zel'dovich flow) [default] */
  FPM_FACTORS_QUINN = 1   /* plain integrals  int da/(a^3 E), int da/(a^2 E) */
};

/* How the three force components are produced inside fpm_force / fpm_nbody. */
enum {
  FPM_FORCE_UNFUSED = 0, /* r2c, apply_force_kernel, 3x c2r, 3x readout as separate kernels */
  FPM_FORCE_FUSED = 1    /* Green's function fused into the FFT passes, readout+kick+drift fused */
};

/* How fpm_paint scatters.  DIRECT and BRICK_FLOAT agree within fp32 summation order.  BRICK_FIXED rounds every
 * deposit m_p W to a multiple of a per-brick (4096 lattice neighbours, 512 when ng = 2 np) power-of-two
 * quantum q: q <= 2^-19 m for the density paint of a run (mass == NULL), and
 * q <= max(2^-18 mean|m|, 2^-21 max|m|) over the brick with per-particle masses; a cell is off by at most
 * q/2 per deposit it receives (measured 1.5e-6 relative L2 on the density).  A brick holding a non-finite
 * mass, or whose max|m| exceeds 64 mean|m|, is deposited with plain fp32 reductions instead (so NaN/Inf
 * propagate and an outlier does not coarsen its neighbours).  Particles a brick's window cannot hold always
 * take plain fp32 reductions: the result is defined for any input. */
enum {
  FPM_PAINT_AUTO = 0,        /* BRICK_FIXED when the particles are a full np^3 lattice set and ng == np or 2 np, else DIRECT */
  FPM_PAINT_DIRECT = 1,      /* one thread per particle, 8 global fp32 reductions */
  FPM_PAINT_BRICK_FLOAT = 2, /* shared-memory window per lattice brick, fp32 accumulation */
  FPM_PAINT_BRICK_FIXED = 3  /* shared-memory window per lattice brick, 32-bit fixed-point accumulation */
};

typedef struct {
  int32_t ng;          /* mesh cells per side */
  int32_t np;          /* particles per side (np^3 particles on a lattice of spacing ng/np) */
  double omega_m;      /* flat LCDM: E(a)^2 = omega_m a^-3 + 1 - omega_m */
  double box;          /* Mpc/h, bookkeeping only */
  int32_t kernel_mode; /* FPM_KERNEL_* */
  int32_t factor_mode; /* FPM_FACTORS_* */
  int32_t force_path;  /* FPM_FORCE_* */
  int32_t paint_mode;  /* FPM_PAINT_* */
  int32_t batch;       /* independent simulations advanced together (0 or 1: one); see "Batches" below */
} fpm_config;

/* Batches ("splitting along the batch dimension is almost always the most
 * efficient"): with batch = B > 1 a context advances B independent simulations of the same
 * (ng, np, cosmology) in the SAME kernel launches -- every kernel's grid is extended over the batch, so small
 * configurations stop being bound by launch latency.  Particle arrays are then [B][3][n], the linear field of
 * fpm_lpt_init [B][np^3], meshes [B][ng^3]; `n` stays the particle count of ONE simulation.  Simulation b's
 * results equal those of a batch-1 run of the same inputs.  Calls that take a batch: fpm_lpt_init, fpm_paint,
 * fpm_pm_step, fpm_nbody (traj: [n_steps+1][B][3][n]); the batch needs FPM_FORCE_FUSED and a full np^3
 * lattice particle set (np a multiple of 32); every other call returns FPM_ENOTIMPL on a context with
 * batch > 1. */

typedef struct fpm_ctx fpm_ctx;

/* ---- context ---------------------------------------------------------------------------- */
const char* fpm_version(void);

/* cfg: HOST.  cuda_stream: a cudaStream_t (NULL = legacy default stream).  *out receives the
 * context.  FPM_EINVAL on bad sizes/modes, FPM_ECUDA if the plan tables cannot be created. */
int fpm_create(const fpm_config* cfg, void* cuda_stream, fpm_ctx** out);
int fpm_destroy(fpm_ctx* ctx);
/* Text of the last error on this context (HOST string owned by the context; "" if none). */
const char* fpm_last_error(const fpm_ctx* ctx);

/* Bytes of scratch needed by fpm_force / fpm_nbody / fpm_lpt_init / the adjoint driver for this
 * configuration (0 on invalid cfg).  The single-operator calls (paint, readout, fft, kick, drift,
 * apply_force_kernel, *_adjoint) need no workspace. */
size_t fpm_workspace_bytes(const fpm_config* cfg);
/* ws: DEVICE, 256-byte aligned, stays owned by the caller and must outlive its use. */
int fpm_set_workspace(fpm_ctx* ctx, void* ws, size_t bytes);

/* Changes cfg.paint_mode after creation.  FPM_EINVAL on an unknown mode. */
int fpm_set_paint_mode(fpm_ctx* ctx, int paint_mode);

/* Which tile movers the fused FFT passes (FPM_FORCE_FUSED, fpm_force_vjp's potential solve) use.  The
 * library holds exactly two chains and nothing but this call selects between them (no environment variable):
 * FPM_MOVERS_AUTO [default] moves tiles with TMA tensor maps (cp.async.bulk.tensor) when the driver provides
 * cuTensorMapEncodeTiled, FPM_MOVERS_GLOBAL forces the ld.global / st.global chain that otherwise runs only
 * when it does not (same arithmetic, results equal to round-off).  fpm_tile_movers reports what the context
 * runs now: FPM_MOVERS_TENSOR_MAPS or FPM_MOVERS_GLOBAL (the latter also before a workspace is set). */
enum { FPM_MOVERS_AUTO = 0, FPM_MOVERS_GLOBAL = 1, FPM_MOVERS_TENSOR_MAPS = 2 };
int fpm_set_tile_movers(fpm_ctx* ctx, int tile_movers);
int fpm_tile_movers(const fpm_ctx* ctx);

/* How fpm_nbody enqueues its n_steps + 1 PM steps.  FPM_GRAPH_AUTO [default]: when one PM step is small enough
 * to be bound by launch latency (batch * ng^3 <= 2^24 cells), a run whose argument set (pos, mom, traj, schedule)
 * repeats the previous call's is captured into a CUDA graph (cached on the context, 8 entries) and replayed
 * with one launch from then on; a first or one-off argument set, and larger runs, enqueue kernel by kernel.
 * FPM_GRAPH_ALWAYS captures on the first call.  When the context's stream is itself being captured by the caller
 * (e.g. torch.cuda.graph), fpm_nbody never builds a graph of its own: it enqueues plain launches, which the
 * caller's capture records.  Results are identical either way. */
enum { FPM_GRAPH_OFF = 0, FPM_GRAPH_AUTO = 1, FPM_GRAPH_ALWAYS = 2 };
int fpm_set_graph_mode(fpm_ctx* ctx, int graph_mode);

/* ---- background cosmology (host, float64; paper defers to Feng et al. 2016) -- */
/* out: HOST double[7] = {D1, f1, D2, f2, E, Gf = a^3 E dD1/da, gf = dGf/da}, D1(1) = 1. */
int fpm_growth(const fpm_ctx* ctx, double a, double* out);
/* Drift factor multiplying p (epoch a_c) to move x from a_i to a_f; kick factor multiplying the
 * force (epoch a_c) to move p from a_i to a_f.  HOST doubles. */
int fpm_drift_factor(const fpm_ctx* ctx, double ai, double ac, double af, double* out);
int fpm_kick_factor(const fpm_ctx* ctx, double ai, double ac, double af, double* out);
/* The (kick_fac, drift_fac) pairs of the n_steps + 1 PM steps fpm_nbody performs for the schedule
 * a_stages[0 .. n_steps]: the half step sits at sqrt(a_j a_j+1), and the
 * two half kicks that use the same force evaluation are merged, so step j is
 *   mom += f(pos) * kick_fac[j];  pos = wrap(pos + mom * drift_fac[j]),   drift_fac[n_steps] = 0.
 * a_stages, kick_fac, drift_fac: HOST double arrays of n_steps + 1 entries.  fpm_nbody, fpm_nbody_vjp and
 * fpm_pm_step callers all use exactly these numbers. */
int fpm_step_factors(const fpm_ctx* ctx, const double* a_stages, int n_steps, double* kick_fac,
                     double* drift_fac);

/* ---- the operators of one PM step --------------------------------------------------------- */

/* Cloud-in-cell paint: mesh[c] = sum_p m_p prod_d max(0, 1 - |x_pd - c_d|),
 * periodic.  pos [3][n]; mass [n] or NULL (=> every particle has mass (ng/np)^3 so <mesh> = 1);
 * mesh [ng^3] is OVERWRITTEN.  n >= 0. */
int fpm_paint(fpm_ctx* ctx, const float* pos, const float* mass, int64_t n, float* mesh);

/* 3-D real-to-complex FFT: cplx(k) = sum_x real(x) exp(-2 pi i n.x/ng),
 * unnormalised.  real [ng^3] is read only; cplx [ng*ng*(ng/2+1)] complex64 (float2). */
int fpm_fft_r2c(fpm_ctx* ctx, const float* real, float* cplx);
/* Inverse: real(x) = ng^-3 sum_k cplx(k) exp(+2 pi i n.x/ng), with the
 * Hermitian half implied.  cplx is CLOBBERED (used as scratch for the in-place passes).
 * Input contract: cplx is the half-complex spectrum of a REAL field, i.e. on the planes kz = 0 and
 * kz = ng/2 it satisfies cplx(-kx, -ky, kz) = conj(cplx(kx, ky, kz)) (true of every spectrum this library
 * produces: fpm_fft_r2c output times a transfer function with the parity of Eq. 3-5).  On other inputs the
 * result is the real part of the inverse transform of the spectrum completed by
 * cplx(-kx, -ky, -kz) := conj(cplx(kx, ky, kz)) for 0 < kz < ng/2 and taken as stored on those two planes:
 * the component of the two planes that breaks the symmetry contributes its real part only. */
int fpm_fft_c2r(fpm_ctx* ctx, float* cplx, float* real);

/* Transfer function (Eq. 3-5): fk_d = scale * i g(omega_d) delta_k / K^2,
 * 1/K^2 := 0 at k = 0, g := 0 at the Nyquist index of axis d.  Outputs must not alias delta_k. */
int fpm_apply_force_kernel(fpm_ctx* ctx, const float* delta_k, float scale, float* fkx,
                           float* fky, float* fkz);

/* Cloud-in-cell readout, same window as paint: out[p] = sum_c mesh[c] W(x_p - c). */
int fpm_readout(fpm_ctx* ctx, const float* mesh, const float* pos, int64_t n, float* out);

/* One force evaluation at the particles (Alg. 3 ForceGrids local, between a
 * paint and three readouts): force [3][n] = -1.5 omega_m grad laplace^-1 delta at pos, i.e. already
 * multiplied by 1.5 omega_m.  Needs the workspace.  The painted density stays in the workspace
 * (fpm_workspace_density) until the next call. */
int fpm_force(fpm_ctx* ctx, const float* pos, int64_t n, float* force);
/* DEVICE pointer to the [ng^3] density painted by the last fpm_force / fpm_nbody force evaluation
 * (valid only with FPM_FORCE_UNFUSED or right after fpm_paint_density); NULL without workspace. */
const float* fpm_workspace_density(const fpm_ctx* ctx);

/* Kick (Eq. 2): mom += force * K(ai, ac, af); force [3][n] already holds 1.5 omega_m. */
int fpm_kick(fpm_ctx* ctx, float* mom, const float* force, int64_t n, double ai, double ac,
             double af);
/* Drift (Eq. 1): pos = wrap(pos + mom * D(ai, ac, af)) into [0, ng). */
int fpm_drift(fpm_ctx* ctx, float* pos, const float* mom, int64_t n, double ai, double ac,
              double af);

/* ---- initial conditions and the whole run -------------------------------------------------- */

/* LPT initial conditions (Alg. 4).  delta_lin [np^3]: real-space Gaussian
 * linear field at a = 1 on the particle lattice.  order 1 (Zel'dovich) or 2.  Outputs pos, mom
 * [3][np^3] in mesh cells at scale factor a0.  Needs the workspace. */
int fpm_lpt_init(fpm_ctx* ctx, const float* delta_lin, double a0, int order, float* pos,
                 float* mom);

/* Whole FastPM run (PAPER.md:37-45 leapfrog).  a_stages: HOST double
 * [n_steps+1] (a_0 .. a_n).  Force at a_0, then per step: half kick to sqrt(a_j a_j+1), drift to
 * a_j+1, force, half kick.  pos/mom [3][n] are updated in place, n = np^3.  traj: NULL, or DEVICE
 * [(n_steps+1)][3][n] receiving the positions at every force evaluation (for the backward pass).
 * Needs the workspace. */
int fpm_nbody(fpm_ctx* ctx, float* pos, float* mom, const double* a_stages, int n_steps,
              float* traj);

/* One PM step = one force evaluation + kick + drift (the loop body of
 * fpm_nbody): force at pos (paint, r2c, transfer function, 3 c2r, readout), mom += force *
 * kick_fac, pos = wrap(pos + mom * drift_fac).  kick_fac / drift_fac: HOST doubles from
 * fpm_kick_factor / fpm_drift_factor.  Needs the workspace. */
int fpm_pm_step(fpm_ctx* ctx, float* pos, float* mom, int64_t n, double kick_fac,
                double drift_fac);
/* The same step with HOST state: h_pos/h_mom [3][n] are copied to d_pos/d_mom (DEVICE,
 * caller-owned), stepped, copied back; synchronises before returning. */
int fpm_pm_step_host(fpm_ctx* ctx, float* h_pos, float* h_mom, float* d_pos, float* d_mom,
                     int64_t n, double kick_fac, double drift_fac);

/* The same run with HOST buffers: h_pos/h_mom [3][n] (pinned or pageable) are copied to the
 * device buffers d_pos/d_mom (DEVICE, caller-owned), evolved, copied back; synchronises. */
int fpm_nbody_host(fpm_ctx* ctx, float* h_pos, float* h_mom, float* d_pos, float* d_mom,
                   const double* a_stages, int n_steps);

/* ---- adjoints ("differentiable with respect to every component") ------ */

/* VJP of paint.  grad_mesh [ng^3] = dL/dmesh.  grad_pos [3][n] = m_p sum_c grad_mesh[c] dW/dx_d
 * (overwritten); grad_mass [n] = readout(grad_mesh) (overwritten) or NULL. */
int fpm_paint_adjoint(fpm_ctx* ctx, const float* pos, const float* mass, int64_t n,
                      const float* grad_mesh, float* grad_pos, float* grad_mass);
/* VJP of readout.  grad_out [n] = dL/dout.  grad_mesh [ng^3] is ACCUMULATED INTO (+= paint of
 * grad_out); grad_pos [3][n] = grad_out_p sum_c mesh[c] dW/dx_d (overwritten) or NULL. */
int fpm_readout_adjoint(fpm_ctx* ctx, const float* mesh, const float* pos, int64_t n,
                        const float* grad_out, float* grad_mesh, float* grad_pos);

/* ---- reverse mode through a force evaluation, a run and the initial conditions ---------------
 * (needed by BASELINE.json's C4 "backward pass: gradient of sum(final density x
 * weight field) with respect to the initial linear modes, via adjoint paint/readout/FFT").  All need
 * the workspace. */

/* grad_pos [3][n] += coef * J_f(pos)^T v, where f = fpm_force(pos) and v [3][n] is the cotangent of
 * the force: the direct dW/dx term of the three readouts plus the path through paint -> r2c ->
 * transfer function -> c2r (whose transpose is its negative: the kernel is odd and imaginary). */
int fpm_force_vjp(fpm_ctx* ctx, const float* pos, int64_t n, const float* v, double coef,
                  float* grad_pos);

/* Reverse of fpm_nbody.  traj: DEVICE [(n_steps+1)][3][n] as stored by fpm_nbody for the same HOST
 * a_stages.  grad_pos / grad_mom: DEVICE [3][n]; on entry dL/d(final pos, final mom), on return
 * dL/d(initial pos, initial mom) (updated in place).  The forward force meshes of every step are
 * recomputed from traj.  flags: 0, or FPM_VJP_GRAD_MOM_ZERO when the caller guarantees that grad_mom is all
 * zeros on entry (a loss on the final positions only): the force VJP of the last force evaluation, which
 * then adds exactly zero, is skipped (one of n_steps + 1 backward force evaluations). */
enum { FPM_VJP_GRAD_MOM_ZERO = 1 };
int fpm_nbody_vjp(fpm_ctx* ctx, const float* traj, const double* a_stages, int n_steps,
                  float* grad_pos, float* grad_mom, int flags);

/* Reverse of fpm_lpt_init.  grad_pos / grad_mom: DEVICE [3][np^3] (read only); grad_delta: DEVICE
 * [np^3] = dL/d(delta_lin) (overwritten).  delta_lin, a0, order as in the forward call. */
int fpm_lpt_init_vjp(fpm_ctx* ctx, const float* delta_lin, double a0, int order,
                     const float* grad_pos, const float* grad_mom, float* grad_delta);

/* ---- MAP reconstruction of the linear field (Eq. 12, Listing 7.1) -- */

/* Bytes of caller-owned DEVICE scratch fpm_recon_loss_grad needs for a forward model of n_steps steps:
 * pos, mom, their cotangents and the trajectory, (n_steps + 5) * 3 * np^3 floats (0 on invalid input). */
size_t fpm_recon_scratch_bytes(const fpm_config* cfg, int n_steps);

/* Negative log-posterior of the linear field s and its gradient (Eq. 12):
 *   loss = 1/2 sum_c ((rho_m[c] - data[c]) / sigma)^2 + 1/2 sum_k |s_k|^2 inv_power[k],
 *   rho_m = paint(nbody(lpt_init(s, a_stages[0], lpt_order), a_stages)), mean density 1,
 *   s_k the unnormalised DFT of s, the k sum over the full k-space.
 * s [np^3] DEVICE; data [ng^3] DEVICE (a mean-1 density); inv_power [np*np*(np/2+1)] DEVICE real table
 * 1/<|s_k|^2> (0 where a mode is unconstrained); a_stages HOST [n_steps+1]; scratch DEVICE, 16-byte
 * aligned; grad [np^3] DEVICE = d loss / d s (overwritten); loss HOST double[2] = {likelihood term,
 * prior term}.  Needs the workspace; synchronises the stream before returning (the loss is read back). */
int fpm_recon_loss_grad(fpm_ctx* ctx, const float* s, const float* data, double sigma,
                        const float* inv_power, const double* a_stages, int n_steps, int lpt_order,
                        void* scratch, size_t scratch_bytes, float* grad, double* loss);

/* One Adam update (Listing 7.1 "AdamOptimizer"), step t >= 1, all arrays DEVICE [n]:
 * m = b1 m + (1-b1) g; v = b2 v + (1-b2) g^2; x -= lr (m/(1-b1^t)) / (sqrt(v/(1-b2^t)) + eps). */
int fpm_adam_step(fpm_ctx* ctx, float* x, const float* grad, float* m, float* v, int64_t n, double lr,
                  double beta1, double beta2, double eps, int t);

/* ---- multi-grid pyramid (Eq. 6-9, Alg. 2-3) ------------
 * The paper's two-level force scheme, built for its distributed FFT; on one GPU it is strictly more work than
 * the single-mesh force, so it is offered for accuracy studies, not used by fpm_nbody.
 * BSpline(6) is read as the two-scale mask of the order-6 cardinal B-spline, [1, 6, 15, 20, 15, 6, 1]/64 per
 * axis (R14).  All three calls need the workspace; levels >= 0 with ng >> levels >= 8. */

/* Alg. 2 REDUCE: `levels` consecutive periodic stride-2 convolutions with the mask.  in [ng^3] -> out
 * [(ng >> levels)^3]; out must not alias in. */
int fpm_reduce(fpm_ctx* ctx, const float* in, int levels, float* out);
/* Alg. 2 EXPAND: `levels` consecutive transposed stride-2 convolutions with 8 x the mask.
 * in [(ng >> levels)^3] -> out [ng^3]. */
int fpm_expand(fpm_ctx* ctx, const float* in, int levels, float* out);
/* Alg. 3 Force: force [3][n] at pos from F = EXPAND(2^levels ForceGrids(REDUCE(rho))) + F_S - EXPAND(REDUCE(F_S)),
 * F_S = ForceGrids(rho) the single-mesh force meshes, rho = paint(pos); already x 1.5 omega_m like fpm_force.
 * (The factor 2^levels converts the coarse mesh's force per coarse cell spacing into fine-cell units.) */
int fpm_force_pyramid(fpm_ctx* ctx, const float* pos, int64_t n, int levels, float* force);

/* REDUCE for callers that cannot allocate device memory (no context, no workspace, no cudaMalloc anywhere on
 * its path).  Meant for code hosted where device memory already belongs to someone else -- a plug-in inside a
 * process whose framework pool or MIG/MPS budget holds all of it, so a fresh cudaMalloc fails or makes the pool
 * give memory back -- and for loops that cannot afford the device-wide synchronisation an allocation implies.
 * Same result as fpm_reduce: `levels` stride-2 convolutions, in [ng^3] -> out [(ng >> levels)^3], both DEVICE
 * arrays of the CURRENT device owned by the caller (in != out); cuda_stream: a cudaStream_t of that device
 * (NULL = legacy default stream); work is enqueued, not synchronised.
 *   - The intermediates of the axis passes live in an array built into the library image,
 *     FPM_REDUCE_STATIC_MAX_NG^3 floats = 8 MiB, which every GPU that loads libfpm's kernels holds until the
 *     process exits.  ng > FPM_REDUCE_STATIC_MAX_NG returns FPM_EINVAL (use fpm_reduce with a workspace).
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress); make that
 *     first call outside any stream capture.  Later calls only launch kernels.
 *   - All calls on a device share the one array.  It is never cleared and need not be (each pass writes what
 *     the next reads), but two calls whose kernels overlap on the GPU -- different streams, no dependency --
 *     race on it: keep calls on one stream or order them with events.
 * err: HOST buffer of err_len bytes receiving a message on failure ("" on success), or NULL.  Returns FPM_OK,
 * FPM_EINVAL (pointers, ng not a power of two in [8, FPM_REDUCE_STATIC_MAX_NG], levels with ng >> levels < 8)
 * or FPM_ECUDA. */
#define FPM_REDUCE_STATIC_MAX_NG 128
int fpm_reduce_static(const float* in, int ng, int levels, float* out, void* cuda_stream, char* err,
                      size_t err_len);

/* ---- measurement hooks -------------------------------------------------------------------- */
/* Per-kernel CUDA-event timing on the context's stream (off by default).  fpm_profile_read
 * synchronises the recorded events; kernel_id runs over 0 .. until FPM_EINVAL is returned.
 * name: HOST out (static string); total_ms / count: HOST out, accumulated since the last reset. */
int fpm_profile_enable(fpm_ctx* ctx, int on);
int fpm_profile_reset(fpm_ctx* ctx);
int fpm_profile_read(fpm_ctx* ctx, int kernel_id, const char** name, double* total_ms,
                     int64_t* count);
/* Kernels of this library launched on this context since the last fpm_profile_reset. */
int64_t fpm_launch_count(const fpm_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* FPM_H */
