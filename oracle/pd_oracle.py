"""ctypes front end of the CPU oracle (oracle/pd_oracle.cpp).

TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  Argument marshalling only: every number is
computed by the C++ in pd_oracle.cpp.  Layout: arrays are [batch][ny][nx] (x fastest) or [ny][nx].
"""
import ctypes as C
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

B0_X, B0_Y, B0_ANGLE = 0, 1, 2
REG_TV, REG_L1 = 0, 1
TV_ISO, TV_ANISO = 0, 1
LAMBDA_REG, LAMBDA_DATA = 0, 1


class Params(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("batch", C.c_int), ("b0_dir", C.c_int),
        ("lambda_", C.c_double), ("sigma", C.c_double), ("tau", C.c_double), ("theta", C.c_double),
        ("max_iters", C.c_int), ("tol", C.c_double),
        ("tv_mode", C.c_int), ("lambda_conv", C.c_int), ("check_every", C.c_int),
        ("regulariser", C.c_int), ("b0_angle", C.c_double),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        spec = importlib.util.spec_from_file_location("_pd_oracle_build", os.path.join(_HERE, "build.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        _lib = C.CDLL(mod.build())
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_float))


def _i(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_int))


def _c64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _c32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError("oracle %s failed with code %d" % (what, rc))


def fft2(a, inverse=False, bruteforce=False):
    """2-D DFT of a complex [ny][nx] array (unnormalised forward, 1/(nx*ny) inverse)."""
    a = np.asarray(a)
    ny, nx = a.shape
    re, im = _c64(a.real), _c64(a.imag)
    ore, oim = np.empty_like(re), np.empty_like(re)
    fn = lib().pdo_dft2_bruteforce if bruteforce else lib().pdo_fft2
    _check(fn(nx, ny, _d(re), _d(im), _d(ore), _d(oim), int(inverse)), "fft2")
    return ore + 1j * oim


def dipole(nx, ny, b0_dir=B0_Y):
    D = np.empty((ny, nx), np.float64)
    _check(lib().pdo_dipole(nx, ny, b0_dir, _d(D)), "dipole")
    return D


def apply_K(a, b0_dir=B0_Y):
    a = _c64(a)
    ny, nx = a.shape
    out = np.empty_like(a)
    _check(lib().pdo_apply_K(nx, ny, b0_dir, _d(a), _d(out)), "apply_K")
    return out


def dipole_angle(nx, ny, angle):
    D = np.empty((ny, nx), np.float64)
    _check(lib().pdo_dipole_angle(nx, ny, C.c_double(angle), _d(D)), "dipole_angle")
    return D


def apply_K_angle(a, angle):
    a = _c64(a)
    ny, nx = a.shape
    out = np.empty_like(a)
    _check(lib().pdo_apply_K_angle(nx, ny, C.c_double(angle), _d(a), _d(out)), "apply_K_angle")
    return out


def shrink(v, t):
    v = _c64(v).copy()
    t = _c64(np.broadcast_to(t, v.shape))
    _check(lib().pdo_shrink(v.size, _d(v), _d(t)), "shrink")
    return v


def grad(a):
    a = _c64(a)
    ny, nx = a.shape
    gx, gy = np.empty_like(a), np.empty_like(a)
    _check(lib().pdo_grad(nx, ny, _d(a), _d(gx), _d(gy)), "grad")
    return gx, gy


def gradT(qx, qy):
    qx, qy = _c64(qx), _c64(qy)
    ny, nx = qx.shape
    out = np.empty_like(qx)
    _check(lib().pdo_gradT(nx, ny, _d(qx), _d(qy), _d(out)), "gradT")
    return out


def prox_p(p, r, sigma, lambda_=1.0, lambda_conv=LAMBDA_REG):
    p = _c64(p).copy()
    r = _c64(r)
    _check(lib().pdo_prox_p(p.size, _d(p), _d(r), C.c_double(sigma), C.c_double(lambda_), lambda_conv), "prox_p")
    return p


def prox_q(tx, ty, radius, tv_mode=TV_ISO):
    tx, ty = _c64(tx).copy(), _c64(ty).copy()
    _check(lib().pdo_prox_q(tx.size, _d(tx), _d(ty), C.c_double(radius), tv_mode), "prox_q")
    return tx, ty


def make_params(nx, ny, batch, lambda_, sigma, tau, theta=1.0, max_iters=100, tol=0.0, b0_dir=B0_Y,
                tv_mode=TV_ISO, lambda_conv=LAMBDA_REG, check_every=1, regulariser=REG_TV, b0_angle=None):
    if b0_angle is not None:
        b0_dir = B0_ANGLE
    return Params(nx, ny, batch, b0_dir, lambda_, sigma, tau, theta, max_iters, tol, tv_mode, lambda_conv,
                  check_every, regulariser, 0.0 if b0_angle is None else float(b0_angle))


def solve(field, mask=None, weight=None, *, lambda_, sigma, tau, theta=1.0, max_iters=100, tol=0.0,
          b0_dir=B0_Y, tv_mode=TV_ISO, lambda_conv=LAMBDA_REG, check_every=1, precision="f64",
          want_state=False, want_hist=True, regulariser=REG_TV, b0_angle=None):
    """Run the PD iteration slice after slice.  field/mask/weight: [batch][ny][nx] (or [ny][nx]).

    Returns a dict: chi (float64 [batch][ny][nx]), chi32, iters_done, relgap/relres ([batch][max_iters],
    entry n = value computed in 0-based iteration n, -1 where not run), and p, qx, qy, chibar if want_state.
    """
    field = _c32(field)
    if field.ndim == 2:
        field = field[None]
    batch, ny, nx = field.shape
    mask = _c32(mask)
    weight = _c32(weight)
    for name, arr in (("mask", mask), ("weight", weight)):
        if arr is not None and arr.size != field.size:
            raise ValueError("%s must have the shape of field" % name)
    prm = make_params(nx, ny, batch, lambda_, sigma, tau, theta, max_iters, tol, b0_dir, tv_mode, lambda_conv,
                      check_every, regulariser, b0_angle)
    chi64 = np.empty((batch, ny, nx), np.float64)
    chi32 = np.empty((batch, ny, nx), np.float32)
    iters = np.zeros(batch, np.int32)
    gap = np.empty((batch, max(max_iters, 1)), np.float64) if want_hist else None
    res = np.empty((batch, max(max_iters, 1)), np.float64) if want_hist else None
    st = [np.empty((batch, ny, nx), np.float64) if want_state else None for _ in range(4)]
    fn = {"f64": lib().pdo_solve_f64, "f32": lib().pdo_solve_f32}[precision]
    _check(fn(C.byref(prm), _f(field), _f(mask), _f(weight), _d(chi64), _f(chi32), _i(iters), _d(gap), _d(res),
              _d(st[0]), _d(st[1]), _d(st[2]), _d(st[3])), "solve")
    out = {"chi": chi64, "chi32": chi32, "iters_done": iters}
    if want_hist:
        out["relgap"] = gap[:, :max_iters]
        out["relres"] = res[:, :max_iters]
    if want_state:
        out.update(p=st[0], qx=st[1], qy=st[2], chibar=st[3])
    return out


def trace(field, mask=None, weight=None, *, lambda_, sigma, tau, theta=1.0, max_iters=10, b0_dir=B0_Y,
          tv_mode=TV_ISO, lambda_conv=LAMBDA_REG, regulariser=REG_TV, b0_angle=None):
    """Single slice; returns trace[n][c] for n=0..max_iters, c = (chi, p, qx, qy)."""
    field = _c32(field)
    ny, nx = field.shape
    prm = make_params(nx, ny, 1, lambda_, sigma, tau, theta, max_iters, 0.0, b0_dir, tv_mode, lambda_conv, 1,
                      regulariser, b0_angle)
    tr = np.empty((max_iters + 1, 4, ny, nx), np.float64)
    _check(lib().pdo_trace_f64(C.byref(prm), _f(field), _f(_c32(mask)), _f(_c32(weight)), _d(tr)), "trace")
    return tr


def forward3d(chi):
    chi = _c64(chi)
    n = chi.shape[0]
    assert chi.shape == (n, n, n)
    out = np.empty_like(chi)
    _check(lib().pdo_forward3d(n, _d(chi), _d(out)), "forward3d")
    return out
