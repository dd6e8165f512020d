"""Thin ctypes binding of the C ABI in include/pd.h (argument marshalling only).

PyTorch is used by callers for device memory and streams; this module only passes raw pointers.
There is no CPU fallback: if libpd_b200.so is missing or cannot be loaded, every entry point raises.
Names mirror the C ABI: pd_plan -> Plan(...), pd_solve -> Plan.solve, pd_solve_host -> Plan.solve_host,
pd_set_weight / pd_set_option / pd_set_steps / pd_get_stats(_host) / pd_destroy likewise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpd_b200.so")

B0_X, B0_Y = 0, 1
OK, EINVAL, ESIZE, ESTEP, ENOMEM, ECUDA, EVARIANT, ESTATIC = 0, -1, -2, -3, -4, -5, -6, -7
STATIC_MAX_N, STATIC_MAX_BATCH, STATIC_MAX_CELLS = 256, 32, 65536   # limits of pd_solve_static (include/pd.h)
OPT_TV_MODE, OPT_LAMBDA_CONV, OPT_VARIANT, OPT_CHECK_EVERY, OPT_MASK_SHARED, OPT_UNSAFE_STEPS, OPT_KERNEL_TIMING, OPT_FOURIER_DUAL, OPT_HYBRID_TAIL, OPT_GRAPH_LOOP, OPT_REGULARISER, OPT_HOST_CHUNKING = range(12)
REG_TV, REG_L1 = 0, 1
KERNEL_CLASSES = ["init", "dual_rows", "dipole_cols", "primal_rows", "finish", "resident", "fd_cols", "fd_rows"]
TV_ISO, TV_ANISO = 0, 1
LAMBDA_REG, LAMBDA_DATA = 0, 1
VARIANT_AUTO, VARIANT_STREAMING, VARIANT_RESIDENT = 0, 1, 2

# every symbol include/pd.h declares (tests/test_abi.py checks the header against this list and the built library)
SYMBOLS = ["pd_plan", "pd_solve", "pd_solve_host", "pd_set_weight", "pd_set_steps", "pd_set_option", "pd_get_stats",
           "pd_get_stats_host", "pd_get_kernel_times", "pd_last_launch_count", "pd_get_info", "pd_get_hybrid_tail", "pd_hybrid_tail_rule", "pd_line_factors", "pd_get_hybrid_rho", "pd_set_b0_angle", "pd_set_norm_bounds", "pd_destroy", "pd_strerror",
           "pd_solve_static", "pd_preprocess", "pd_combine_coils", "pd_plan3d", "pd_solve3d", "pd_set_weight3d", "pd_last_launch_count3d",
           "pd_destroy3d"]

_lib = None


class PdError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("pd error %d: %s" % (code, text))
        self.code = code


def lib():
    """Load libpd_b200.so (built in-tree by paper_2006_09808_b200/build.py).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("CUDA library %s is not built (run `python -m paper_2006_09808_b200.build`); "
                               "there is no CPU fallback" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, fp, ip = C.c_void_p, C.c_float, C.c_int
        L.pd_plan.argtypes = [C.POINTER(vp), ip, ip, ip, ip, fp, fp, fp, fp]
        L.pd_solve.argtypes = [vp, vp, vp, vp, ip, fp, vp]
        L.pd_solve_host.argtypes = [vp, vp, vp, vp, ip, fp, vp]
        L.pd_set_weight.argtypes = [vp, vp]
        L.pd_set_steps.argtypes = [vp, fp, fp, fp, fp]
        L.pd_set_option.argtypes = [vp, ip, ip]
        L.pd_set_b0_angle.argtypes = [vp, fp]
        L.pd_set_norm_bounds.argtypes = [vp, fp, fp]
        L.pd_get_stats.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.pd_get_stats_host.argtypes = [vp, vp, vp, vp, vp]
        L.pd_get_kernel_times.argtypes = [vp, vp, vp]
        L.pd_last_launch_count.argtypes = [vp]
        L.pd_get_info.argtypes = [vp, C.POINTER(ip), C.POINTER(ip), C.POINTER(ip)]
        L.pd_get_hybrid_tail.argtypes = [vp, C.POINTER(ip)]
        L.pd_hybrid_tail_rule.argtypes = [ip, ip, fp]
        L.pd_line_factors.argtypes = [ip, C.POINTER(ip), C.POINTER(ip)]
        L.pd_get_hybrid_rho.argtypes = [vp, C.POINTER(fp)]
        L.pd_destroy.argtypes = [vp]
        L.pd_preprocess.argtypes = [vp, vp, C.c_longlong, fp, fp, fp, vp, vp, vp, vp, vp]
        L.pd_combine_coils.argtypes = [vp, vp, ip, ip, ip, ip, vp, vp]
        L.pd_plan3d.argtypes = [C.POINTER(vp), ip, ip, ip, ip, ip, fp, fp, fp, fp]
        L.pd_solve3d.argtypes = [vp, vp, vp, vp, ip, vp]
        L.pd_set_weight3d.argtypes = [vp, vp]
        L.pd_last_launch_count3d.argtypes = [vp]
        L.pd_destroy3d.argtypes = [vp]
        L.pd_solve_static.argtypes = [ip, ip, ip, ip, fp, fp, fp, fp, vp, vp, vp, ip, fp, vp, vp, vp, vp]
        L.pd_strerror.argtypes = [ip]
        L.pd_strerror.restype = C.c_char_p
        for name in SYMBOLS:
            if name != "pd_strerror":
                getattr(L, name).restype = ip
        _lib = L
    return _lib


def strerror(code):
    return lib().pd_strerror(code).decode()


def _check(code):
    if code != OK:
        raise PdError(code, strerror(code))


def _ptr(t):
    """Raw device pointer of a torch tensor (or None)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous() or t.dtype.__str__() != "torch.float32":
        raise ValueError("expected a contiguous float32 CUDA tensor")
    if t.data_ptr() % 16:
        raise ValueError("tensor must be 16-byte aligned")
    return C.c_void_p(t.data_ptr())


def _stream_handle(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return C.c_void_p(stream)
    return C.c_void_p(stream.cuda_stream)


def hybrid_tail_rule(npairs, clusters, rho):
    """pd_hybrid_tail_rule: the automatic tail of the hybrid schedule for `npairs` slice pairs, `clusters` clusters and
    a streaming side that finishes rho * clusters pairs per resident wave."""
    return lib().pd_hybrid_tail_rule(int(npairs), int(clusters), float(rho))


def line_factors(n):
    """pd_line_factors: (tuned, n1, n2) -- how a line of length n is transformed (host arithmetic only)."""
    a, b = C.c_int(), C.c_int()
    rc = lib().pd_line_factors(int(n), C.byref(a), C.byref(b))
    if rc < 0:
        raise PdError(rc, strerror(rc))
    return bool(rc), a.value, b.value


class Plan3D:
    """pd_plan3d(nx, ny, nz, nvol, B0_axis, lambda, sigma, tau, theta): the true 3-D variant, one problem per volume."""

    def __init__(self, nx, ny, nz, nvol=1, b0_axis=2, lambda_=0.01, sigma=0.25, tau=0.25, theta=1.0):
        self._h = C.c_void_p()
        self.shape = (nvol, nz, ny, nx)
        _check(lib().pd_plan3d(C.byref(self._h), nx, ny, nz, nvol, b0_axis, lambda_, sigma, tau, theta))

    def solve(self, field, mask, chi_out, max_iters, stream=None):
        """field, mask (or None), chi_out: float32 CUDA tensors [nvol][nz][ny][nx]."""
        for t in (field, mask, chi_out):
            if t is not None and tuple(t.shape) != self.shape:
                raise ValueError("expected shape %r" % (self.shape,))
        _check(lib().pd_solve3d(self._h, _ptr(field), _ptr(mask), _ptr(chi_out), int(max_iters), _stream_handle(stream)))

    def set_weight(self, weight):
        """pd_set_weight3d: W [nvol][nz][ny][nx] (float32 CUDA tensor, kept alive here) or None."""
        if weight is not None and tuple(weight.shape) != self.shape:
            raise ValueError("expected shape %r" % (self.shape,))
        self._keep = weight
        _check(lib().pd_set_weight3d(self._h, _ptr(weight)))

    @property
    def last_launch_count(self):
        return lib().pd_last_launch_count3d(self._h)

    def destroy(self):
        if self._h:
            _check(lib().pd_destroy3d(self._h))
            self._h = C.c_void_p()


def preprocess(s0, s1, fscale, threshold, wscale=0.0, field=None, weight=None, mask=None, wmax=None, stream=None):
    """pd_preprocess: s0, s1 complex64 CUDA tensors [batch][ny][nx] (without / with the echo shift); field, weight, mask:
    float32 CUDA tensors of the same shape or None; wmax: float32 CUDA tensor of one element (needed when wscale <= 0)."""
    for t in (s0, s1):
        if not t.is_cuda or not t.is_contiguous() or str(t.dtype) != "torch.complex64" or t.data_ptr() % 16:
            raise ValueError("expected contiguous, 16-byte aligned complex64 CUDA tensors")
    if s0.shape != s1.shape or any(t is not None and t.shape != s0.shape for t in (field, weight, mask)):
        raise ValueError("s0, s1 and the outputs must have the same shape")
    _check(lib().pd_preprocess(C.c_void_p(s0.data_ptr()), C.c_void_p(s1.data_ptr()), s0.numel(), float(fscale), float(wscale),
                               float(threshold), _ptr(field), _ptr(weight), _ptr(mask), _ptr(wmax), _stream_handle(stream)))


def combine_coils(chi, weight, ncoils, chi_out, stream=None):
    """pd_combine_coils: chi, weight [nslices*ncoils][ny][nx] -> chi_out [nslices][ny][nx] (float32 CUDA tensors)."""
    batch, ny, nx = chi.shape
    if batch % ncoils or weight.shape != chi.shape or tuple(chi_out.shape) != (batch // ncoils, ny, nx):
        raise ValueError("chi, weight: [nslices*ncoils][ny][nx]; chi_out: [nslices][ny][nx]")
    _check(lib().pd_combine_coils(_ptr(chi), _ptr(weight), batch // ncoils, ncoils, ny, nx, _ptr(chi_out), _stream_handle(stream)))


def solve_static(field, mask, chi_out, max_iters, tol=0.0, b0_dir=B0_Y, lambda_=0.01, sigma=0.25, tau=0.25, theta=1.0,
                 iters_done=None, relgap=None, relres=None, stream=None):
    """pd_solve_static: the allocation-free entry point (workspace in a static device array inside the library; limits
    STATIC_MAX_*).  field, mask (or None), chi_out: float32 CUDA tensors [batch][ny][nx]; iters_done (int32), relgap,
    relres (float32): optional CUDA tensors [batch].  Enqueues on `stream` (default: torch's current stream)."""
    batch, ny, nx = field.shape
    if chi_out.shape != field.shape or (mask is not None and mask.shape != field.shape):
        raise ValueError("field, mask and chi_out must have the same [batch][ny][nx] shape")
    for t in (iters_done, relgap, relres):
        if t is not None and (not t.is_cuda or not t.is_contiguous() or t.numel() < batch or t.element_size() != 4):
            raise ValueError("statistics outputs must be contiguous 4-byte CUDA tensors of length batch")
    raw = lambda t: None if t is None else C.c_void_p(t.data_ptr())
    _check(lib().pd_solve_static(nx, ny, batch, b0_dir, lambda_, sigma, tau, theta, _ptr(field), _ptr(mask), _ptr(chi_out),
                                 int(max_iters), float(tol), raw(iters_done), raw(relgap), raw(relres),
                                 _stream_handle(stream)))


class Plan:
    """pd_plan(nx, ny, batch, B0_dir, lambda, sigma, tau, theta) -- owns the device workspace."""

    def __init__(self, nx, ny, batch, b0_dir=B0_Y, lambda_=0.01, sigma=0.25, tau=0.25, theta=1.0):
        self._h = C.c_void_p()
        self.nx, self.ny, self.batch = nx, ny, batch
        self._mask_shared = 0
        self._keep = None
        _check(lib().pd_plan(C.byref(self._h), nx, ny, batch, b0_dir, lambda_, sigma, tau, theta))

    def set_option(self, key, value):
        _check(lib().pd_set_option(self._h, key, value))
        if key == OPT_MASK_SHARED:
            self._mask_shared = value

    def set_steps(self, lambda_, sigma, tau, theta=1.0):
        _check(lib().pd_set_steps(self._h, lambda_, sigma, tau, theta))

    def set_norm_bounds(self, max_abs_w, max_abs_m):
        """pd_set_norm_bounds: bounds on |W| and |M| for the automatic steps and the PD_ESTEP check."""
        _check(lib().pd_set_norm_bounds(self._h, float(max_abs_w), float(max_abs_m)))

    def set_b0_angle(self, angle_rad):
        """pd_set_b0_angle: B0 along (cos a, sin a) in the slice plane."""
        _check(lib().pd_set_b0_angle(self._h, float(angle_rad)))

    def set_weight(self, weight):
        if weight is not None and weight.numel() != self.batch * self.ny * self.nx:
            raise ValueError("weight must be [batch][ny][nx]")
        self._keep = weight
        _check(lib().pd_set_weight(self._h, _ptr(weight)))

    def solve(self, field, mask, chi_out, max_iters, tol=0.0, stream=None):
        """pd_solve: device tensors [batch][ny][nx] float32; enqueues on `stream` (default: torch's current stream)."""
        n = self.batch * self.ny * self.nx
        if field.numel() != n or chi_out.numel() != n:
            raise ValueError("field and chi_out must be [batch][ny][nx]")
        if mask is not None and mask.numel() != (self.ny * self.nx if self._mask_shared else n):
            raise ValueError("mask has the wrong number of elements")
        _check(lib().pd_solve(self._h, _ptr(field), _ptr(mask), _ptr(chi_out), int(max_iters), float(tol),
                              _stream_handle(stream)))
        return chi_out

    def solve_host(self, field, mask, chi_out, max_iters, tol=0.0, stream=None):
        """pd_solve_host: numpy float32 arrays (or pinned torch CPU tensors); H2D + solve + D2H + stream sync."""
        def hp(a):
            if a is None:
                return None
            if isinstance(a, np.ndarray):
                assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"]
                return C.c_void_p(a.ctypes.data)
            assert a.dtype.__str__() == "torch.float32" and a.is_contiguous() and not a.is_cuda
            return C.c_void_p(a.data_ptr())
        _check(lib().pd_solve_host(self._h, hp(field), hp(mask), hp(chi_out), int(max_iters), float(tol),
                                   _stream_handle(stream)))
        return chi_out

    def stats(self, stream=None):
        """pd_get_stats_host: (iters_done int32[batch], relgap float32[batch], relres float32[batch]) on the host."""
        it = np.empty(self.batch, np.int32)
        gap = np.empty(self.batch, np.float32)
        res = np.empty(self.batch, np.float32)
        _check(lib().pd_get_stats_host(self._h, C.c_void_p(it.ctypes.data), C.c_void_p(gap.ctypes.data),
                                       C.c_void_p(res.ctypes.data), _stream_handle(stream)))
        return it, gap, res

    def stats_device_ptrs(self):
        """pd_get_stats: raw device pointers (iters_done, relgap, relres)."""
        a, b, c = C.c_void_p(), C.c_void_p(), C.c_void_p()
        _check(lib().pd_get_stats(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return a.value, b.value, c.value

    def kernel_times(self):
        """pd_get_kernel_times: {class name: (total ms, launches)} of the last solve (needs OPT_KERNEL_TIMING = 1)."""
        ms = np.zeros(len(KERNEL_CLASSES), np.float32)
        cnt = np.zeros(len(KERNEL_CLASSES), np.int32)
        _check(lib().pd_get_kernel_times(self._h, C.c_void_p(ms.ctypes.data), C.c_void_p(cnt.ctypes.data)))
        return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(KERNEL_CLASSES)}

    def info(self):
        """pd_get_info: {"variant": "streaming"|"resident", "clusters": n, "cluster_size": c} of the next solve."""
        v, n, c = C.c_int(), C.c_int(), C.c_int()
        _check(lib().pd_get_info(self._h, C.byref(v), C.byref(n), C.byref(c)))
        return {"variant": "resident" if v.value == VARIANT_RESIDENT else "streaming", "clusters": n.value,
                "cluster_size": c.value}

    def hybrid_tail(self):
        """pd_get_hybrid_tail: slice pairs the next solve runs through the streaming kernels beside the resident clusters."""
        n = C.c_int()
        _check(lib().pd_get_hybrid_tail(self._h, C.byref(n)))
        return n.value

    def hybrid_rho(self):
        """pd_get_hybrid_rho: the streaming-to-resident rate ratio pd_plan measured for the hybrid schedule."""
        r = C.c_float()
        _check(lib().pd_get_hybrid_rho(self._h, C.byref(r)))
        return r.value

    @property
    def last_launch_count(self):
        return lib().pd_last_launch_count(self._h)

    def destroy(self):
        if self._h:
            lib().pd_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
