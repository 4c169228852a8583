"""Thin Python binding of libfpm (include/fpm.h): argument marshalling only.

Every numerical step runs in the CUDA kernels of libfpm.so; PyTorch supplies device memory and
the stream.  There is no CPU fallback: importing this package without the built library, or
calling it with CPU tensors, raises.
"""
import ctypes
import os

import torch

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libfpm.so")

KERNEL_PAPER, KERNEL_NAIVE, KERNEL_MIXED = 0, 1, 2
FACTORS_FASTPM, FACTORS_QUINN = 0, 1
FORCE_UNFUSED, FORCE_FUSED = 0, 1
PAINT_AUTO, PAINT_DIRECT, PAINT_BRICK_FLOAT, PAINT_BRICK_FIXED = 0, 1, 2, 3
GRAPH_OFF, GRAPH_AUTO, GRAPH_ALWAYS = 0, 1, 2
MOVERS_AUTO, MOVERS_GLOBAL, MOVERS_TENSOR_MAPS = 0, 1, 2
VJP_GRAD_MOM_ZERO = 1
OK, EINVAL, ENOMEM, ECUDA, ENOTIMPL = 0, -1, -2, -3, -4


class FpmError(RuntimeError):
    pass


class _Config(ctypes.Structure):
    _fields_ = [("ng", ctypes.c_int32), ("np", ctypes.c_int32), ("omega_m", ctypes.c_double),
                ("box", ctypes.c_double), ("kernel_mode", ctypes.c_int32),
                ("factor_mode", ctypes.c_int32), ("force_path", ctypes.c_int32),
                ("paint_mode", ctypes.c_int32), ("batch", ctypes.c_int32)]


def _load():
    try:
        _build.build()            # no-op when libfpm.so matches the sources (content hash)
    except Exception as e:        # noqa: BLE001
        raise ImportError(f"cannot build {_LIB_PATH} with nvcc for sm_100a ({e}); "
                          "there is no CPU fallback") from e
    lib = ctypes.CDLL(_LIB_PATH)
    vp, i64, dbl, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
    sig = {
        "fpm_version": (ctypes.c_char_p, []),
        "fpm_create": (i32, [ctypes.POINTER(_Config), vp, ctypes.POINTER(vp)]),
        "fpm_destroy": (i32, [vp]),
        "fpm_last_error": (ctypes.c_char_p, [vp]),
        "fpm_workspace_bytes": (ctypes.c_size_t, [ctypes.POINTER(_Config)]),
        "fpm_set_workspace": (i32, [vp, vp, ctypes.c_size_t]),
        "fpm_set_paint_mode": (i32, [vp, i32]),
        "fpm_set_graph_mode": (i32, [vp, i32]),
        "fpm_set_tile_movers": (i32, [vp, i32]),
        "fpm_tile_movers": (i32, [vp]),
        "fpm_growth": (i32, [vp, dbl, ctypes.POINTER(dbl)]),
        "fpm_drift_factor": (i32, [vp, dbl, dbl, dbl, ctypes.POINTER(dbl)]),
        "fpm_kick_factor": (i32, [vp, dbl, dbl, dbl, ctypes.POINTER(dbl)]),
        "fpm_step_factors": (i32, [vp, ctypes.POINTER(dbl), i32, ctypes.POINTER(dbl), ctypes.POINTER(dbl)]),
        "fpm_paint": (i32, [vp, vp, vp, i64, vp]),
        "fpm_fft_r2c": (i32, [vp, vp, vp]),
        "fpm_fft_c2r": (i32, [vp, vp, vp]),
        "fpm_apply_force_kernel": (i32, [vp, vp, ctypes.c_float, vp, vp, vp]),
        "fpm_readout": (i32, [vp, vp, vp, i64, vp]),
        "fpm_force": (i32, [vp, vp, i64, vp]),
        "fpm_workspace_density": (vp, [vp]),
        "fpm_kick": (i32, [vp, vp, vp, i64, dbl, dbl, dbl]),
        "fpm_drift": (i32, [vp, vp, vp, i64, dbl, dbl, dbl]),
        "fpm_lpt_init": (i32, [vp, vp, dbl, i32, vp, vp]),
        "fpm_nbody": (i32, [vp, vp, vp, ctypes.POINTER(dbl), i32, vp]),
        "fpm_nbody_host": (i32, [vp, vp, vp, vp, vp, ctypes.POINTER(dbl), i32]),
        "fpm_pm_step": (i32, [vp, vp, vp, i64, dbl, dbl]),
        "fpm_pm_step_host": (i32, [vp, vp, vp, vp, vp, i64, dbl, dbl]),
        "fpm_profile_enable": (i32, [vp, i32]),
        "fpm_profile_reset": (i32, [vp]),
        "fpm_profile_read": (i32, [vp, i32, ctypes.POINTER(ctypes.c_char_p), ctypes.POINTER(dbl),
                                   ctypes.POINTER(i64)]),
        "fpm_launch_count": (i64, [vp]),
        "fpm_force_vjp": (i32, [vp, vp, i64, vp, dbl, vp]),
        "fpm_nbody_vjp": (i32, [vp, vp, ctypes.POINTER(dbl), i32, vp, vp, i32]),
        "fpm_lpt_init_vjp": (i32, [vp, vp, dbl, i32, vp, vp, vp]),
        "fpm_recon_scratch_bytes": (ctypes.c_size_t, [ctypes.POINTER(_Config), i32]),
        "fpm_recon_loss_grad": (i32, [vp, vp, vp, dbl, vp, ctypes.POINTER(dbl), i32, i32, vp, ctypes.c_size_t, vp,
                                      ctypes.POINTER(dbl)]),
        "fpm_adam_step": (i32, [vp, vp, vp, vp, vp, i64, dbl, dbl, dbl, dbl, i32]),
        "fpm_paint_adjoint": (i32, [vp, vp, vp, i64, vp, vp, vp]),
        "fpm_reduce": (i32, [vp, vp, i32, vp]),
        "fpm_expand": (i32, [vp, vp, i32, vp]),
        "fpm_reduce_static": (i32, [vp, i32, i32, vp, vp, ctypes.c_char_p, ctypes.c_size_t]),
        "fpm_force_pyramid": (i32, [vp, vp, i64, i32, vp]),
        "fpm_readout_adjoint": (i32, [vp, vp, vp, i64, vp, vp, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    return lib


_lib = _load()


def version():
    return _lib.fpm_version().decode()


def library_path():
    return _LIB_PATH


REDUCE_STATIC_MAX_NG = 128


def reduce_static(mesh, levels, out):
    """fpm_reduce_static: REDUCE `mesh` [ng^3] by `levels` levels into the caller's `out` [(ng >> levels)^3]
    without a context, a workspace or any device allocation -- for code that runs where device memory is
    already owned by something else (a framework pool, a fixed MIG/MPS budget) or that cannot take the
    device-wide synchronisation of cudaMalloc.  The intermediates use an 8 MiB array built into libfpm.so
    (meshes up to REDUCE_STATIC_MAX_NG^3; larger ones raise).  Enqueued on torch's current stream.  Calls share
    that array: do not let two of them overlap on the GPU.  The first call on a device does a one-time address
    lookup and should come before any stream capture.  Nothing is allocated here either: `out` is required."""
    shape = tuple(getattr(mesh, "shape", ()))
    if len(shape) != 3 or not (shape[0] == shape[1] == shape[2]):
        raise FpmError(f"mesh: expected an [ng][ng][ng] tensor, got shape {shape}")
    ng, levels = int(shape[0]), int(levels)
    nc = ng >> levels if 0 <= levels < 8 else 0
    err = ctypes.create_string_buffer(256)
    rc = _lib.fpm_reduce_static(_dev(mesh, what="mesh"), ng, levels,
                                _dev(out, numel=nc ** 3 if nc else None, what="out"),
                                ctypes.c_void_p(torch.cuda.current_stream(mesh.device).cuda_stream), err, len(err))
    if rc != OK:
        raise FpmError(f"fpm_reduce_static -> {rc}: {err.value.decode()}")
    return out


def _dev(t, dtype=torch.float32, numel=None, what="tensor"):
    """data_ptr of a contiguous CUDA tensor of the given dtype (and element count, when the C call assumes
    one): a wrong size would be an out-of-bounds device access behind the C-ABI, so it is refused here."""
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise FpmError(f"expected a contiguous CUDA {dtype} tensor (no CPU fallback), got "
                       f"{type(t).__name__} {getattr(t, 'dtype', None)} {getattr(t, 'device', None)}")
    if numel is not None and t.numel() != numel:
        raise FpmError(f"{what}: expected {numel} elements, got {t.numel()} (shape {tuple(t.shape)})")
    return ctypes.c_void_p(t.data_ptr())


def _particles(t, what="pos", batch=1):
    """[3][n] particle array ([batch][3][n] on a batched context) -> n, the particle count of one simulation."""
    shape = tuple(getattr(t, "shape", ()))
    if batch > 1:
        if not (isinstance(t, torch.Tensor) and len(shape) == 3 and shape[0] == batch and shape[1] == 3):
            raise FpmError(f"{what}: expected a [{batch}][3][n] tensor on a batched context, got shape {shape}")
        return int(shape[2])
    if not (isinstance(t, torch.Tensor) and len(shape) == 2 and shape[0] == 3):
        raise FpmError(f"{what}: expected a [3][n] tensor, got shape {shape}")
    return int(shape[1])


class FPM:
    """One context = one (ng, np, cosmology, kernel) configuration on one CUDA stream."""

    def __init__(self, ng, np_side=None, omega_m=0.3075, box=0.0, kernel_mode=KERNEL_PAPER,
                 factor_mode=FACTORS_FASTPM, force_path=FORCE_UNFUSED, device="cuda:0",
                 stream=None, workspace=True, paint_mode=PAINT_AUTO, batch=1):
        if not torch.cuda.is_available():
            raise FpmError("CUDA device required: libfpm has no CPU fallback")
        self.device = torch.device(device)
        self.ng, self.np_side = int(ng), int(np_side if np_side is not None else ng)
        self.n_particles = self.np_side ** 3
        self.nzh = self.ng // 2 + 1
        self.omega_m = float(omega_m)
        self.batch = int(batch)
        self._cfg = _Config(self.ng, self.np_side, self.omega_m, float(box), kernel_mode,
                            factor_mode, force_path, paint_mode, self.batch)
        with torch.cuda.device(self.device):
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = ctypes.c_void_p()
            rc = _lib.fpm_create(ctypes.byref(self._cfg), ctypes.c_void_p(self._stream.cuda_stream),
                                 ctypes.byref(h))
        if rc != OK:
            raise FpmError(f"fpm_create failed with status {rc}")
        self._h = h
        self._ws = None
        if workspace:
            nbytes = _lib.fpm_workspace_bytes(ctypes.byref(self._cfg))
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            off = (-self._ws.data_ptr()) % 256
            self._check(_lib.fpm_set_workspace(self._h, ctypes.c_void_p(self._ws.data_ptr() + off), nbytes))

    def close(self):
        if getattr(self, "_h", None):
            _lib.fpm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != OK:
            raise FpmError(f"libfpm status {rc}: {_lib.fpm_last_error(self._h).decode()}")

    def _empty(self, *shape, dtype=torch.float32):
        return torch.empty(*shape, dtype=dtype, device=self.device)

    def set_paint_mode(self, mode):
        self._check(_lib.fpm_set_paint_mode(self._h, int(mode)))

    def set_graph_mode(self, mode):
        self._check(_lib.fpm_set_graph_mode(self._h, int(mode)))

    def set_tile_movers(self, mode):
        self._check(_lib.fpm_set_tile_movers(self._h, int(mode)))

    def tile_movers(self):
        return int(_lib.fpm_tile_movers(self._h))

    # ---- cosmology ----------------------------------------------------------------------
    def growth(self, a):
        out = (ctypes.c_double * 7)()
        self._check(_lib.fpm_growth(self._h, a, out))
        return dict(zip(("D1", "f1", "D2", "f2", "E", "Gf", "gf"), list(out)))

    def drift_factor(self, ai, ac, af):
        out = ctypes.c_double()
        self._check(_lib.fpm_drift_factor(self._h, ai, ac, af, ctypes.byref(out)))
        return out.value

    def kick_factor(self, ai, ac, af):
        out = ctypes.c_double()
        self._check(_lib.fpm_kick_factor(self._h, ai, ac, af, ctypes.byref(out)))
        return out.value

    # ---- operators ------------------------------------------------------------------------
    # Every wrapper checks the element counts the C call assumes (a wrong shape would be a silent
    # out-of-bounds device access behind the C-ABI) and raises FpmError.
    @property
    def _n_g(self):
        return self.ng ** 3

    @property
    def _n_k(self):
        return self.ng * self.ng * self.nzh

    def paint(self, pos, mass=None, out=None):
        b = self.batch
        n = _particles(pos, batch=b)
        shape = (self.ng, self.ng, self.ng) if b <= 1 else (b, self.ng, self.ng, self.ng)
        mesh = out if out is not None else self._empty(*shape)
        self._check(_lib.fpm_paint(self._h, _dev(pos), _dev(mass, numel=n * max(b, 1), what="mass"), n,
                                   _dev(mesh, numel=self._n_g * max(b, 1), what="mesh")))
        return mesh

    def fft_r2c(self, real, out=None):
        cplx = out if out is not None else self._empty(self.ng, self.ng, self.nzh, dtype=torch.complex64)
        self._check(_lib.fpm_fft_r2c(self._h, _dev(real, numel=self._n_g, what="real mesh"),
                                     _dev(cplx, torch.complex64, self._n_k, "half-complex mesh")))
        return cplx

    def fft_c2r(self, cplx, out=None, clobber=False):
        work = cplx if clobber else cplx.clone()
        real = out if out is not None else self._empty(self.ng, self.ng, self.ng)
        self._check(_lib.fpm_fft_c2r(self._h, _dev(work, torch.complex64, self._n_k, "half-complex mesh"),
                                     _dev(real, numel=self._n_g, what="real mesh")))
        return real

    def apply_force_kernel(self, delta_k, scale=1.0):
        outs = [torch.empty_like(delta_k) for _ in range(3)]
        self._check(_lib.fpm_apply_force_kernel(self._h, _dev(delta_k, torch.complex64, self._n_k, "delta_k"),
                                                scale, *[_dev(o, torch.complex64) for o in outs]))
        return outs

    def readout(self, mesh, pos):
        n = _particles(pos)
        out = self._empty(n)
        self._check(_lib.fpm_readout(self._h, _dev(mesh, numel=self._n_g, what="mesh"), _dev(pos), n, _dev(out)))
        return out

    def force(self, pos):
        n = _particles(pos)
        f = self._empty(3, n)
        self._check(_lib.fpm_force(self._h, _dev(pos), n, _dev(f)))
        return f

    def workspace_density(self):
        """Copy of the density painted by the last force evaluation (unfused path)."""
        ptr = _lib.fpm_workspace_density(self._h)
        if not ptr:
            raise FpmError("no workspace")
        out = self._empty(self.ng, self.ng, self.ng)
        off = ptr - self._ws.data_ptr()
        out.view(-1).copy_(self._ws[off:off + out.numel() * 4].view(torch.float32))
        return out

    def kick(self, mom, force, ai, ac, af):
        n = _particles(mom, "mom")
        self._check(_lib.fpm_kick(self._h, _dev(mom), _dev(force, numel=3 * n, what="force"), n, ai, ac, af))
        return mom

    def drift(self, pos, mom, ai, ac, af):
        n = _particles(pos)
        self._check(_lib.fpm_drift(self._h, _dev(pos), _dev(mom, numel=3 * n, what="mom"), n, ai, ac, af))
        return pos

    def lpt_init(self, delta_lin, a0, order):
        b = max(self.batch, 1)
        shape = (3, self.n_particles) if b == 1 else (b, 3, self.n_particles)
        pos, mom = self._empty(*shape), self._empty(*shape)
        self._check(_lib.fpm_lpt_init(self._h, _dev(delta_lin, numel=b * self.n_particles, what="delta_lin"), a0,
                                      order, _dev(pos), _dev(mom)))
        return pos, mom

    def _stages(self, stages):
        if len(stages) < 1:
            raise FpmError("stages: need at least a_0")
        return (ctypes.c_double * len(stages))(*[float(a) for a in stages]), len(stages) - 1

    def nbody(self, pos, mom, stages, traj=None):
        st, n_steps = self._stages(stages)
        n3 = 3 * self.n_particles * max(self.batch, 1)
        self._check(_lib.fpm_nbody(self._h, _dev(pos, numel=n3, what="pos"), _dev(mom, numel=n3, what="mom"), st,
                                   n_steps, _dev(traj, numel=(n_steps + 1) * n3, what="traj")))
        return pos, mom

    def pm_step(self, pos, mom, kick_fac, drift_fac):
        """One PM step: force at pos, mom += f * kick_fac, pos = wrap(pos + mom * drift_fac)."""
        n = _particles(pos, batch=self.batch)
        self._check(_lib.fpm_pm_step(self._h, _dev(pos), _dev(mom, numel=pos.numel(), what="mom"), n, kick_fac,
                                     drift_fac))
        return pos, mom

    def pm_step_host(self, h_pos, h_mom, d_pos, d_mom, kick_fac, drift_fac):
        """The same step on HOST float32 tensors: H2D, step, D2H, synchronise."""
        n = _particles(h_pos, "h_pos")
        for t in (h_pos, h_mom):
            if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or t.numel() != 3 * n:
                raise FpmError("pm_step_host expects contiguous CPU float32 [3][n] tensors")
        self._check(_lib.fpm_pm_step_host(self._h, ctypes.c_void_p(h_pos.data_ptr()),
                                          ctypes.c_void_p(h_mom.data_ptr()), _dev(d_pos, numel=3 * n, what="d_pos"),
                                          _dev(d_mom, numel=3 * n, what="d_mom"), n, kick_fac, drift_fac))
        return h_pos, h_mom

    def step_factors(self, stages):
        """[(kick_fac, drift_fac)] of the n+1 PM steps fpm_nbody performs for stages a_0..a_n
        (fpm_step_factors: the schedule arithmetic lives behind the C-ABI, not here)."""
        st, n_steps = self._stages(stages)
        kf, dr = (ctypes.c_double * (n_steps + 1))(), (ctypes.c_double * (n_steps + 1))()
        self._check(_lib.fpm_step_factors(self._h, st, n_steps, kf, dr))
        return list(zip(list(kf), list(dr)))

    # ---- measurement hooks ----------------------------------------------------------------
    def profile_enable(self, on=True):
        self._check(_lib.fpm_profile_enable(self._h, int(bool(on))))

    def profile_reset(self):
        self._check(_lib.fpm_profile_reset(self._h))

    def profile_read(self):
        """{kernel name: (total ms, launches timed)} since the last reset (synchronises)."""
        out, kid = {}, 0
        while True:
            name, ms, cnt = ctypes.c_char_p(), ctypes.c_double(), ctypes.c_int64()
            rc = _lib.fpm_profile_read(self._h, kid, ctypes.byref(name), ctypes.byref(ms), ctypes.byref(cnt))
            if rc != OK:
                break
            out[name.value.decode()] = (ms.value, cnt.value)
            kid += 1
        return out

    def launch_count(self):
        return int(_lib.fpm_launch_count(self._h))

    def nbody_host(self, h_pos, h_mom, d_pos, d_mom, stages):
        """Whole run on HOST float32 tensors (pinned for full PCIe speed); synchronises."""
        n3 = 3 * self.n_particles
        for t in (h_pos, h_mom):
            if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or t.numel() != n3:
                raise FpmError("nbody_host expects contiguous CPU float32 [3][np^3] tensors")
        st, n_steps = self._stages(stages)
        self._check(_lib.fpm_nbody_host(self._h, ctypes.c_void_p(h_pos.data_ptr()),
                                        ctypes.c_void_p(h_mom.data_ptr()), _dev(d_pos, numel=n3, what="d_pos"),
                                        _dev(d_mom, numel=n3, what="d_mom"), st, n_steps))
        return h_pos, h_mom

    def paint_adjoint(self, pos, grad_mesh, mass=None, want_grad_mass=True):
        n = _particles(pos)
        gpos = self._empty(3, n)
        gmass = self._empty(n) if want_grad_mass else None
        self._check(_lib.fpm_paint_adjoint(self._h, _dev(pos), _dev(mass, numel=n, what="mass"), n,
                                           _dev(grad_mesh, numel=self._n_g, what="grad_mesh"), _dev(gpos),
                                           _dev(gmass)))
        return gpos, gmass

    def readout_adjoint(self, mesh, pos, grad_out, grad_mesh=None, want_grad_pos=True):
        n = _particles(pos)
        gm = grad_mesh if grad_mesh is not None else torch.zeros(self.ng, self.ng, self.ng,
                                                                  dtype=torch.float32, device=self.device)
        gpos = self._empty(3, n) if want_grad_pos else None
        self._check(_lib.fpm_readout_adjoint(self._h, _dev(mesh, numel=self._n_g, what="mesh"), _dev(pos), n,
                                             _dev(grad_out, numel=n, what="grad_out"),
                                             _dev(gm, numel=self._n_g, what="grad_mesh"), _dev(gpos)))
        return gm, gpos

    # ---- reverse mode --------------------------------------------------
    def force_vjp(self, pos, v, coef=1.0, grad_pos=None):
        """grad_pos += coef * J_f(pos)^T v for f = force(pos); returns grad_pos [3][n]."""
        n = _particles(pos)
        g = grad_pos if grad_pos is not None else torch.zeros(3, n, dtype=torch.float32, device=self.device)
        self._check(_lib.fpm_force_vjp(self._h, _dev(pos), n, _dev(v, numel=3 * n, what="v"), float(coef),
                                       _dev(g, numel=3 * n, what="grad_pos")))
        return g

    def nbody_vjp(self, traj, stages, grad_pos, grad_mom, grad_mom_is_zero=False):
        """Cotangents of the final (pos, mom) -> of the initial (pos, mom), in place.  grad_mom_is_zero: the
        caller guarantees grad_mom holds zeros (loss on the final positions only): FPM_VJP_GRAD_MOM_ZERO."""
        st, n_steps = self._stages(stages)
        n3 = 3 * self.n_particles
        self._check(_lib.fpm_nbody_vjp(self._h, _dev(traj, numel=(n_steps + 1) * n3, what="traj"), st, n_steps,
                                       _dev(grad_pos, numel=n3, what="grad_pos"),
                                       _dev(grad_mom, numel=n3, what="grad_mom"),
                                       VJP_GRAD_MOM_ZERO if grad_mom_is_zero else 0))
        return grad_pos, grad_mom

    def lpt_init_vjp(self, delta_lin, a0, order, grad_pos, grad_mom):
        out = self._empty(self.np_side, self.np_side, self.np_side)
        n3 = 3 * self.n_particles
        self._check(_lib.fpm_lpt_init_vjp(self._h, _dev(delta_lin, numel=self.n_particles, what="delta_lin"), a0,
                                          order, _dev(grad_pos, numel=n3, what="grad_pos"),
                                          _dev(grad_mom, numel=n3, what="grad_mom"), _dev(out)))
        return out

    # ---- multi-grid pyramid (Alg. 2-3) -----------------------------------
    def reduce(self, mesh, levels=2):
        nc = self.ng >> levels
        out = self._empty(nc, nc, nc)
        self._check(_lib.fpm_reduce(self._h, _dev(mesh, numel=self._n_g, what="mesh"), int(levels), _dev(out)))
        return out

    def expand(self, mesh, levels=2):
        nc = self.ng >> levels
        out = self._empty(self.ng, self.ng, self.ng)
        self._check(_lib.fpm_expand(self._h, _dev(mesh, numel=nc ** 3, what="coarse mesh"), int(levels), _dev(out)))
        return out

    def force_pyramid(self, pos, levels=2):
        n = _particles(pos)
        f = self._empty(3, n)
        self._check(_lib.fpm_force_pyramid(self._h, _dev(pos), n, int(levels), _dev(f)))
        return f

    # ---- MAP reconstruction (Eq. 12, Listing 7.1) -------------------
    def recon_loss_grad(self, s, data, sigma, inv_power, stages, lpt_order=2, scratch=None):
        """((likelihood term, prior term), gradient [np^3]) of the negative log-posterior of s."""
        st, n_steps = self._stages(stages)
        need = _lib.fpm_recon_scratch_bytes(ctypes.byref(self._cfg), n_steps)
        if scratch is None:
            scratch = getattr(self, "_recon_scratch", None)      # reuse the one a previous call allocated
        if scratch is None or scratch.numel() * scratch.element_size() < need:
            scratch = torch.empty(need // 4, dtype=torch.float32, device=self.device)
        self._recon_scratch = scratch
        grad = self._empty(self.np_side, self.np_side, self.np_side)
        loss = (ctypes.c_double * 2)()
        n_kp = self.np_side * self.np_side * (self.np_side // 2 + 1)
        self._check(_lib.fpm_recon_loss_grad(self._h, _dev(s, numel=self.n_particles, what="s"),
                                             _dev(data, numel=self._n_g, what="data"), float(sigma),
                                             _dev(inv_power, numel=n_kp, what="inv_power"), st,
                                             n_steps, int(lpt_order), ctypes.c_void_p(scratch.data_ptr()),
                                             scratch.numel() * scratch.element_size(), _dev(grad), loss))
        return (loss[0], loss[1]), grad

    def adam_step(self, x, grad, m, v, lr, t, beta1=0.9, beta2=0.999, eps=1e-8):
        n = x.numel()
        self._check(_lib.fpm_adam_step(self._h, _dev(x), _dev(grad, numel=n, what="grad"), _dev(m, numel=n, what="m"),
                                       _dev(v, numel=n, what="v"), n, lr, beta1, beta2, eps, int(t)))
        return x
