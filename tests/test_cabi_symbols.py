"""The C-ABI library builds, loads without a GPU and exports every symbol include/fpm.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "fpm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fpm_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for required in ("fpm_lpt_init", "fpm_paint", "fpm_fft_r2c", "fpm_fft_c2r", "fpm_apply_force_kernel",
                     "fpm_readout", "fpm_kick", "fpm_drift", "fpm_nbody", "fpm_paint_adjoint",
                     "fpm_readout_adjoint"):
        assert required in names


def test_library_exports_every_declared_symbol():
    from paper_2010_11847_b200 import build as fpm_build
    lib = ctypes.CDLL(fpm_build.build())
    for name in declared_functions():
        assert hasattr(lib, name), f"libfpm.so does not export {name}"
    lib.fpm_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.fpm_version()


def test_argument_validation_needs_no_gpu():
    from paper_2010_11847_b200 import build as fpm_build
    lib = ctypes.CDLL(fpm_build.build())

    class Cfg(ctypes.Structure):
        _fields_ = [("ng", ctypes.c_int32), ("np", ctypes.c_int32), ("omega_m", ctypes.c_double),
                    ("box", ctypes.c_double), ("kernel_mode", ctypes.c_int32),
                    ("factor_mode", ctypes.c_int32), ("force_path", ctypes.c_int32),
                    ("paint_mode", ctypes.c_int32), ("batch", ctypes.c_int32)]

    lib.fpm_workspace_bytes.restype = ctypes.c_size_t
    good = Cfg(512, 512, 0.3075, 1000.0, 0, 0, 0, 0)
    nk = 512 * 512 * 272          # half-complex scratch rows are padded to 16 elements (128 bytes)
    assert lib.fpm_workspace_bytes(ctypes.byref(good)) == 4 * 512 ** 3 * 4 + 4 * nk * 8
    for bad in (Cfg(500, 500, 0.3, 0, 0, 0, 0, 0), Cfg(64, 128, 0.3, 0, 0, 0, 0, 0),
                Cfg(2048, 2048, 0.3, 0, 0, 0, 0, 0), Cfg(64, 64, -1.0, 0, 0, 0, 0, 0),
                Cfg(64, 64, 0.3, 0, 7, 0, 0, 0), Cfg(64, 64, 0.3, 0, 0, 0, 0, 9), Cfg(64, 64, 0.3, 0, 0, 0, 5, 0),
                Cfg(64, 64, 0.3, 0, 0, 0, 0, 0, -1), Cfg(64, 64, 0.3, 0, 0, 0, 0, 0, 4),      # a batch needs the fused path
                Cfg(64, 16, 0.3, 0, 0, 0, 1, 0, 4), Cfg(1024, 1024, 0.3, 0, 0, 0, 1, 0, 64)):
        assert lib.fpm_workspace_bytes(ctypes.byref(bad)) == 0
        h = ctypes.c_void_p()
        assert lib.fpm_create(ctypes.byref(bad), None, ctypes.byref(h)) == -1
    batched = Cfg(128, 128, 0.3075, 200.0, 0, 0, 1, 0, 16)
    assert lib.fpm_workspace_bytes(ctypes.byref(batched)) == 16 * (4 * 128 ** 3 * 4 + 4 * 128 * 128 * 80 * 8)
    assert lib.fpm_destroy(None) == -1
    assert lib.fpm_paint(None, None, None, ctypes.c_int64(0), None) == -1
    # calls added for the backward pass and N1 validate the same way
    lib.fpm_recon_scratch_bytes.restype = ctypes.c_size_t
    assert lib.fpm_recon_scratch_bytes(ctypes.byref(good), 5) == 4 * 3 * 512 ** 3 * (5 + 5)
    assert lib.fpm_recon_scratch_bytes(ctypes.byref(good), -1) == 0
    assert lib.fpm_recon_scratch_bytes(ctypes.byref(Cfg(500, 500, 0.3, 0, 0, 0, 0, 0)), 5) == 0
    assert lib.fpm_force_vjp(None, None, ctypes.c_int64(0), None, ctypes.c_double(1.0), None) == -1
    assert lib.fpm_nbody_vjp(None, None, None, 0, None, None, 0) == -1
    assert lib.fpm_step_factors(None, None, 0, None, None) == -1
    assert lib.fpm_lpt_init_vjp(None, None, ctypes.c_double(0.1), 2, None, None, None) == -1
    assert lib.fpm_adam_step(None, None, None, None, None, ctypes.c_int64(0), ctypes.c_double(0.1),
                             ctypes.c_double(0.9), ctypes.c_double(0.999), ctypes.c_double(1e-8), 1) == -1


def test_reduce_static_validates_without_a_gpu():
    """fpm_reduce_static checks its arguments before it touches CUDA, and says why it refuses."""
    from paper_2010_11847_b200 import build as fpm_build
    lib = ctypes.CDLL(fpm_build.build())
    vp = ctypes.c_void_p
    lib.fpm_reduce_static.argtypes = [vp, ctypes.c_int, ctypes.c_int, vp, vp, ctypes.c_char_p, ctypes.c_size_t]
    err = ctypes.create_string_buffer(200)
    a, b = vp(256), vp(512)                   # never dereferenced: every case below fails validation first
    assert lib.fpm_reduce_static(None, 64, 1, b, None, err, len(err)) == -1 and b"distinct" in err.value
    assert lib.fpm_reduce_static(a, 256, 1, b, None, err, len(err)) == -1
    assert b"exceeds the built-in scratch (meshes up to 128^3)" in err.value
    assert lib.fpm_reduce_static(a, 96, 1, b, None, err, len(err)) == -1 and b"power of two" in err.value
    assert lib.fpm_reduce_static(a, 32, 3, b, None, err, len(err)) == -1 and b"levels" in err.value
    assert lib.fpm_reduce_static(a, 32, 3, b, None, None, 0) == -1      # the message buffer is optional
