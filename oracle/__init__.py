"""ctypes front-end of the float64 CPU oracle (oracle/fpm_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The product package paper_2010_11847_b200 never does, and this package
never imports it.  All arrays are host numpy float64 in the layouts of include/fpm.h.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fpm_oracle.cpp")
_LIB = os.path.join(_HERE, "libfpm_oracle.so")

KERNEL_PAPER, KERNEL_NAIVE, KERNEL_MIXED = 0, 1, 2
FACTORS_FASTPM, FACTORS_QUINN = 0, 1


def build(force=False):
    """Compile the oracle with g++ (C++17, -O2, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_drift_factor.restype = ctypes.c_double
        _lib.orc_kick_factor.restype = ctypes.c_double
        _lib.orc_num_threads.restype = ctypes.c_int
        for name in ("orc_drift_factor", "orc_kick_factor"):
            getattr(_lib, name).argtypes = [ctypes.c_double] * 4 + [ctypes.c_int]
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def num_threads():
    return int(_load().orc_num_threads())


def growth(omega_m, a):
    """dict D1, f1, D2, f2, E, Gf, gf at scale factor a (R5)."""
    out = np.zeros(7)
    _load().orc_growth(ctypes.c_double(omega_m), ctypes.c_double(a), _p(out))
    return dict(zip(("D1", "f1", "D2", "f2", "E", "Gf", "gf"), out.tolist()))


def drift_factor(omega_m, ai, ac, af, factor_mode=FACTORS_FASTPM):
    return float(_load().orc_drift_factor(omega_m, ai, ac, af, factor_mode))


def kick_factor(omega_m, ai, ac, af, factor_mode=FACTORS_FASTPM):
    return float(_load().orc_kick_factor(omega_m, ai, ac, af, factor_mode))


def fft_r2c(real, force_naive=False):
    real = _f64(real)
    ng = real.shape[0]
    out = np.zeros((ng, ng, ng // 2 + 1, 2))
    _load().orc_fft_r2c(_p(real), ctypes.c_int(ng), _p(out), ctypes.c_int(int(force_naive)))
    return out[..., 0] + 1j * out[..., 1]


def _split(c):
    c = np.asarray(c, dtype=np.complex128)
    return np.ascontiguousarray(np.stack([c.real, c.imag], axis=-1))


def fft_c2r(cplx, force_naive=False):
    ng = cplx.shape[0]
    inp = _split(cplx)
    out = np.zeros((ng, ng, ng))
    _load().orc_fft_c2r(_p(inp), ctypes.c_int(ng), _p(out), ctypes.c_int(int(force_naive)))
    return out


def paint(pos, ng, mass=None, mass_const=1.0):
    pos = _f64(pos)
    n = pos.shape[1]
    m = None if mass is None else _f64(mass)
    mesh = np.zeros((ng, ng, ng))
    _load().orc_paint(_p(pos), _p(m), ctypes.c_double(mass_const), ctypes.c_int64(n),
                      ctypes.c_int(ng), _p(mesh))
    return mesh


def readout(mesh, pos):
    mesh, pos = _f64(mesh), _f64(pos)
    n = pos.shape[1]
    out = np.zeros(n)
    _load().orc_readout(_p(mesh), _p(pos), ctypes.c_int64(n), ctypes.c_int(mesh.shape[0]), _p(out))
    return out


def apply_force_kernel(delta_k, mode=KERNEL_PAPER, scale=1.0):
    ng = delta_k.shape[0]
    inp = _split(delta_k)
    outs = [np.zeros_like(inp) for _ in range(3)]
    _load().orc_apply_force_kernel(_p(inp), ctypes.c_int(ng), ctypes.c_int(mode),
                                   ctypes.c_double(scale), *[_p(o) for o in outs])
    return [o[..., 0] + 1j * o[..., 1] for o in outs]


def force_grids(rho, mode=KERNEL_PAPER, scale=1.0):
    """Alg. 3 ForceGrids(G, local): three force meshes from a density mesh."""
    rho = _f64(rho)
    ng = rho.shape[0]
    outs = [np.zeros((ng, ng, ng)) for _ in range(3)]
    _load().orc_force_grids(_p(rho), ctypes.c_int(ng), ctypes.c_int(mode), ctypes.c_double(scale),
                            *[_p(o) for o in outs])
    return outs


def force(pos, ng, mode=KERNEL_PAPER, scale=1.0, mass=1.0, return_rho=False):
    pos = _f64(pos)
    n = pos.shape[1]
    f = np.zeros((3, n))
    rho = np.zeros((ng, ng, ng)) if return_rho else None
    _load().orc_force(_p(pos), ctypes.c_int64(n), ctypes.c_int(ng), ctypes.c_int(mode),
                      ctypes.c_double(scale), ctypes.c_double(mass), _p(f), _p(rho))
    return (f, rho) if return_rho else f


def kick(mom, force_, factor):
    mom = _f64(mom).copy()
    force_ = _f64(force_)
    _load().orc_kick(_p(mom), _p(force_), ctypes.c_int64(mom.shape[1]), ctypes.c_double(factor))
    return mom


def drift(pos, mom, factor, ng):
    pos = _f64(pos).copy()
    mom = _f64(mom)
    _load().orc_drift(_p(pos), _p(mom), ctypes.c_int64(pos.shape[1]), ctypes.c_double(factor),
                      ctypes.c_int(ng))
    return pos


def lpt_displacements(delta_lin, order=2):
    d = _f64(delta_lin)
    np_side = d.shape[0]
    psi1 = np.zeros((3,) + d.shape)
    psi2 = np.zeros((3,) + d.shape)
    _load().orc_lpt_displacements(_p(d), ctypes.c_int(np_side), ctypes.c_int(order), _p(psi1), _p(psi2))
    return psi1, psi2


def lpt_init(delta_lin, ng, omega_m, a0, order):
    d = _f64(delta_lin)
    np_side = d.shape[0]
    n = np_side ** 3
    pos, mom = np.zeros((3, n)), np.zeros((3, n))
    _load().orc_lpt_init(_p(d), ctypes.c_int(np_side), ctypes.c_int(ng), ctypes.c_double(omega_m),
                         ctypes.c_double(a0), ctypes.c_int(order), _p(pos), _p(mom))
    return pos, mom


def nbody(pos, mom, ng, np_side, omega_m, stages, mode=KERNEL_PAPER, factor_mode=FACTORS_FASTPM,
          return_traj=False):
    pos, mom = _f64(pos).copy(), _f64(mom).copy()
    n = pos.shape[1]
    st = _f64(stages)
    n_steps = len(st) - 1
    traj = np.zeros((n_steps + 1, 3, n)) if return_traj else None
    _load().orc_nbody(_p(pos), _p(mom), ctypes.c_int64(n), ctypes.c_int(ng), ctypes.c_int(np_side),
                      ctypes.c_double(omega_m), ctypes.c_int(mode), ctypes.c_int(factor_mode),
                      _p(st), ctypes.c_int(n_steps), _p(traj))
    return (pos, mom, traj) if return_traj else (pos, mom)


def reduce(mesh, levels=2):
    """Alg. 2 REDUCE (reading R14): f stride-2 convolutions with the order-6 B-spline mask."""
    m = _f64(mesh)
    n = m.shape[0]
    out = np.zeros((n >> levels,) * 3)
    _load().orc_reduce(_p(m), ctypes.c_int(n), ctypes.c_int(levels), _p(out))
    return out


def expand(mesh, levels=2):
    """Alg. 2 EXPAND: f transposed stride-2 convolutions with 8 x the same mask."""
    m = _f64(mesh)
    n = m.shape[0]
    out = np.zeros((n << levels,) * 3)
    _load().orc_expand(_p(m), ctypes.c_int(n), ctypes.c_int(levels), _p(out))
    return out


def force_grids_pyramid(rho, levels=2, mode=KERNEL_PAPER, scale=1.0):
    """Alg. 3 Force(H, f): the three force meshes of the two-level pyramid scheme."""
    rho = _f64(rho)
    ng = rho.shape[0]
    outs = [np.zeros((ng, ng, ng)) for _ in range(3)]
    _load().orc_force_grids_pyramid(_p(rho), ctypes.c_int(ng), ctypes.c_int(mode), ctypes.c_double(scale),
                                    ctypes.c_int(levels), *[_p(o) for o in outs])
    return outs


def force_pyramid(pos, ng, levels=2, mode=KERNEL_PAPER, scale=1.0, mass=1.0):
    pos = _f64(pos)
    n = pos.shape[1]
    f = np.zeros((3, n))
    _load().orc_force_pyramid(_p(pos), ctypes.c_int64(n), ctypes.c_int(ng), ctypes.c_int(mode),
                              ctypes.c_double(scale), ctypes.c_double(mass), ctypes.c_int(levels), _p(f))
    return f


def nbody_batch(pos, mom, ng, np_side, omega_m, stages, mode=KERNEL_PAPER, factor_mode=FACTORS_FASTPM):
    """SURVEY.md 8(f) N2 (the batch dimension): a batch of B simulations IS B independent
    runs -- the definition written out as the loop it is.  pos, mom: [B][3][n]; returns the final [B][3][n]."""
    pos, mom = _f64(pos), _f64(mom)
    out_p, out_m = np.empty_like(pos), np.empty_like(mom)
    for b in range(pos.shape[0]):
        out_p[b], out_m[b] = nbody(pos[b], mom[b], ng, np_side, omega_m, stages, mode, factor_mode)
    return out_p, out_m


def power(mesh_a, box, mesh_b=None):
    """(k_mean, P(k), N_modes) in bins centred on integer multiples of k_f (R13)."""
    a = _f64(mesh_a)
    b = None if mesh_b is None else _f64(mesh_b)
    ng = a.shape[0]
    nb = ng // 2
    pk, km, nm = np.zeros(nb), np.zeros(nb), np.zeros(nb)
    _load().orc_power(_p(a), _p(b), ctypes.c_int(ng), ctypes.c_double(box), _p(pk), _p(km), _p(nm))
    return km, pk, nm


def paint_adjoint(pos, ng, grad_mesh, mass=None, mass_const=1.0):
    pos, g = _f64(pos), _f64(grad_mesh)
    n = pos.shape[1]
    m = None if mass is None else _f64(mass)
    gpos, gmass = np.zeros((3, n)), np.zeros(n)
    _load().orc_paint_adjoint(_p(pos), _p(m), ctypes.c_double(mass_const), ctypes.c_int64(n),
                              ctypes.c_int(ng), _p(g), _p(gpos), _p(gmass))
    return gpos, gmass


def readout_adjoint(mesh, pos, grad_out, grad_mesh=None):
    mesh, pos, go = _f64(mesh), _f64(pos), _f64(grad_out)
    n = pos.shape[1]
    gm = np.zeros_like(mesh) if grad_mesh is None else _f64(grad_mesh).copy()
    gpos = np.zeros((3, n))
    _load().orc_readout_adjoint(_p(mesh), _p(pos), ctypes.c_int64(n), ctypes.c_int(mesh.shape[0]),
                                _p(go), _p(gm), _p(gpos))
    return gm, gpos


def force_vjp(pos, ng, v, mode=KERNEL_PAPER, scale=1.0, mass=1.0):
    """J_f(pos)^T v for f = force(pos) (R12); v, result [3][n]."""
    pos, v = _f64(pos), _f64(v)
    n = pos.shape[1]
    gx = np.zeros((3, n))
    _load().orc_force_vjp(_p(pos), ctypes.c_int64(n), ctypes.c_int(ng), ctypes.c_int(mode),
                          ctypes.c_double(scale), ctypes.c_double(mass), _p(v), _p(gx))
    return gx


def nbody_vjp(traj, ng, np_side, omega_m, stages, gx, gp, mode=KERNEL_PAPER,
              factor_mode=FACTORS_FASTPM):
    """Reverse of nbody (R12): cotangents of the final (pos, mom) -> of the initial (pos, mom)."""
    traj = _f64(traj)
    gx, gp = _f64(gx).copy(), _f64(gp).copy()
    n = traj.shape[2]
    st = _f64(stages)
    _load().orc_nbody_vjp(_p(traj), ctypes.c_int64(n), ctypes.c_int(ng), ctypes.c_int(np_side),
                          ctypes.c_double(omega_m), ctypes.c_int(mode), ctypes.c_int(factor_mode),
                          _p(st), ctypes.c_int(len(st) - 1), _p(gx), _p(gp))
    return gx, gp


def lpt_init_vjp(delta_lin, ng, omega_m, a0, order, gx, gp):
    """Reverse of lpt_init (R12): cotangents of (pos, mom) -> of delta_lin [np^3]."""
    d, gx, gp = _f64(delta_lin), _f64(gx), _f64(gp)
    np_side = d.shape[0]
    out = np.zeros(d.shape)
    _load().orc_lpt_init_vjp(_p(d), ctypes.c_int(np_side), ctypes.c_int(ng), ctypes.c_double(omega_m),
                             ctypes.c_double(a0), ctypes.c_int(order), _p(gx), _p(gp), _p(out))
    return out


def recon_loss_grad(s, ng, omega_m, a0, order, stages, data, sigma, inv_power, mode=KERNEL_PAPER,
                    factor_mode=FACTORS_FASTPM):
    """N1 (Eq. 12): (chi2 term, prior term), gradient w.r.t. the real linear field s [np^3]."""
    s, data, ip = _f64(s), _f64(data), _f64(inv_power)
    np_side = s.shape[0]
    st = _f64(stages)
    grad, loss2 = np.zeros(s.shape), np.zeros(2)
    _load().orc_recon_loss_grad(_p(s), ctypes.c_int(np_side), ctypes.c_int(ng), ctypes.c_double(omega_m),
                                ctypes.c_int(mode), ctypes.c_int(factor_mode), ctypes.c_double(a0),
                                ctypes.c_int(order), _p(st), ctypes.c_int(len(st) - 1), _p(data),
                                ctypes.c_double(sigma), _p(ip), _p(grad), _p(loss2))
    return (float(loss2[0]), float(loss2[1])), grad


def adam_step(x, g, m, v, lr, t, b1=0.9, b2=0.999, eps=1e-8):
    """One Adam update (in float64); returns new (x, m, v)."""
    x, m, v, g = _f64(x).copy(), _f64(m).copy(), _f64(v).copy(), _f64(g)
    _load().orc_adam_step(_p(x), _p(g), _p(m), _p(v), ctypes.c_int64(x.size), ctypes.c_double(lr),
                          ctypes.c_double(b1), ctypes.c_double(b2), ctypes.c_double(eps), ctypes.c_int(t))
    return x, m, v
