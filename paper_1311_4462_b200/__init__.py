"""Thin Python binding of the C-ABI library declared in include/tm.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libtm_b200.so; PyTorch supplies device memory
(field storage is a torch.uint8 tensor the library borrows) and the stream.  There is no CPU fallback:
importing works without a GPU (so the symbol table can be checked), but any compute call needs one, and a
missing library is a hard error.

Functions carry the C names (tm_init, tm_field_alloc, tm_gauge_load, tm_dslash_apply, tm_mat_pc,
tm_reconstruct_odd, ...) and raise TmError on a non-zero status.  Host arrays are numpy complex128 in the
canonical order of include/tm.h:  spinor [nf, V or V/2, 4, 3],  gauge [4, V, 3, 3].
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtm_b200.so")

# enums of include/tm.h
TM_OK = 0
TM_ERR_ARG, TM_ERR_DIMS, TM_ERR_MISMATCH, TM_ERR_ALIAS = -1, -2, -3, -4
TM_ERR_PARAM, TM_ERR_NOMEM, TM_ERR_CUDA, TM_ERR_UNSUPPORTED = -5, -6, -7, -8
TM_DOUBLE, TM_SINGLE, TM_HALF = 8, 4, 2
TM_RECON_18, TM_RECON_12, TM_RECON_8 = 18, 12, 8
TM_EVEN, TM_ODD = 0, 1
TM_TWIST_INV_DSLASH, TM_TWIST_INV_DSLASH_XPAY, TM_DSLASH_TWIST_XPAY, TM_RECONSTRUCT = 0, 1, 2, 3
TM_DSLASH_XPAY, TM_DSLASH_AXPY = 4, 5
TM_TWIST_INV_DSLASH_TWIST_INV, TM_RECONSTRUCT_TWIST_INV, TM_DSLASH_TWIST_INV_AXPY = 6, 7, 8
TM_MATPC_ASYM, TM_MATPC_SYM = 0, 1
TM_BASIS_NONREL, TM_BASIS_CHIRAL, TM_BASIS_CUSTOM = 0, 1, 2

EXPORTS = [
    "tm_init", "tm_set_stream", "tm_sync", "tm_finalize", "tm_field_bytes", "tm_field_alloc", "tm_field_free",
    "tm_field_device_ptr", "tm_set_host_basis", "tm_field_upload", "tm_field_download", "tm_field_upload_cb", "tm_field_download_cb", "tm_field_upload_cb_async", "tm_field_download_cb_async", "tm_field_upload_cb_async_f32", "tm_field_download_cb_async_f32",
    "tm_gauge_load", "tm_gauge_free", "tm_dslash_apply", "tm_mat_pc", "tm_reconstruct_odd", "tm_twist_apply",
    "tm_prepare_rhs", "tm_set_open_time", "tm_set_open_dirs", "tm_halo_bytes", "tm_halo_pack", "tm_halo_apply", "tm_field_axpby", "tm_field_redot", "tm_field_redot_noalloc", "tm_invert_cg", "tm_cg_release", "tm_set_allreduce", "tm_last_error",
    "tm_launch_count", "tm_last_kernel_name", "tm_set_path", "tm_set_tuning", "tm_timing_enable", "tm_timing_read",
]


class TmError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("tm status %d: %s" % (status, message))
        self.status = status


class tm_params(ctypes.Structure):
    _fields_ = [("kappa", ctypes.c_double), ("mu", ctypes.c_double), ("epsilon", ctypes.c_double),
                ("twist_flavor", ctypes.c_int), ("t_boundary", ctypes.c_int)]


# int op(out_e, in_e, tmp_o, gauge, params, matpc type, dagger, user)  /  int allreduce(dev_sums, n, cuda_stream, user)
TM_CG_OP_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.POINTER(tm_params),
                               ctypes.c_int, ctypes.c_int, ctypes.c_void_p)
TM_ALLREDUCE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p)


class tm_cg_params(ctypes.Structure):
    _fields_ = [("tol", ctypes.c_double), ("max_iter", ctypes.c_int), ("sloppy_precision", ctypes.c_int),
                ("delta", ctypes.c_double), ("op", TM_CG_OP_FN), ("op_user", ctypes.c_void_p)]


class tm_cg_info(ctypes.Structure):
    _fields_ = [("iterations", ctypes.c_int), ("restarts", ctypes.c_int), ("residual", ctypes.c_double),
                ("converged", ctypes.c_int)]


def params(kappa, mu, epsilon=0.0, twist_flavor=1, t_boundary=-1):
    return tm_params(float(kappa), float(mu), float(epsilon), int(twist_flavor), int(t_boundary))


_lib = None


def lib():
    """Load libtm_b200.so (built in-tree by paper_1311_4462_b200.build); fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: run `python -m paper_1311_4462_b200.build` (there is no CPU fallback)"
                          % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, i, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    pp = ctypes.POINTER(tm_params)
    L.tm_init.argtypes = [ctypes.POINTER(i), i, ctypes.POINTER(vp)]
    L.tm_set_stream.argtypes = [vp, vp]
    L.tm_sync.argtypes = [vp]
    L.tm_finalize.argtypes = [vp]
    L.tm_finalize.restype = None
    L.tm_field_bytes.argtypes = [vp, i, i]
    L.tm_field_bytes.restype = ctypes.c_size_t
    L.tm_field_alloc.argtypes = [vp, i, i, vp, ctypes.c_size_t, ctypes.POINTER(vp)]
    L.tm_field_free.argtypes = [vp]
    L.tm_field_free.restype = None
    L.tm_field_device_ptr.argtypes = [vp]
    L.tm_field_device_ptr.restype = vp
    for name in ("tm_field_upload", "tm_field_download", "tm_field_upload_cb", "tm_field_download_cb",
                 "tm_field_upload_cb_async", "tm_field_download_cb_async", "tm_field_upload_cb_async_f32", "tm_field_download_cb_async_f32"):
        getattr(L, name).argtypes = [vp, i, vp]
    L.tm_gauge_load.argtypes = [vp, vp, i, i, ctypes.POINTER(vp)]
    L.tm_gauge_free.argtypes = [vp]
    L.tm_gauge_free.restype = None
    L.tm_dslash_apply.argtypes = [vp, vp, vp, vp, pp, i, i, i, i]
    L.tm_mat_pc.argtypes = [vp, vp, vp, vp, pp, i, i]
    L.tm_reconstruct_odd.argtypes = [vp, vp, vp, vp, pp]
    L.tm_twist_apply.argtypes = [vp, vp, pp, i, i]
    L.tm_prepare_rhs.argtypes = [vp, vp, vp, vp, vp, pp, i]
    L.tm_set_open_time.argtypes = [vp, i]
    L.tm_set_open_dirs.argtypes = [vp, i]
    L.tm_halo_bytes.argtypes = [vp, i, i, i]
    L.tm_halo_bytes.restype = ctypes.c_size_t
    L.tm_halo_pack.argtypes = [vp, vp, i, i, i, vp, vp, vp, vp, ctypes.c_uint]
    L.tm_halo_apply.argtypes = [vp, vp, vp, vp, pp, i, i, i, i, i, i, vp, vp, ctypes.c_uint]
    L.tm_field_axpby.argtypes = [vp, d, vp, d, vp]
    L.tm_field_redot.argtypes = [vp, vp, ctypes.POINTER(d)]
    L.tm_field_redot_noalloc.argtypes = [vp, vp, vp]
    L.tm_invert_cg.argtypes = [vp, vp, vp, vp, pp, i, ctypes.POINTER(tm_cg_params), ctypes.POINTER(tm_cg_info)]
    L.tm_cg_release.argtypes = [vp]
    L.tm_cg_release.restype = None
    L.tm_set_allreduce.argtypes = [vp, TM_ALLREDUCE_FN, vp]
    L.tm_last_error.restype = ctypes.c_char_p
    L.tm_launch_count.argtypes = [vp]
    L.tm_launch_count.restype = ctypes.c_long
    L.tm_last_kernel_name.argtypes = [vp]
    L.tm_last_kernel_name.restype = ctypes.c_char_p
    L.tm_set_path.argtypes = [vp, i]
    L.tm_set_host_basis.argtypes = [vp, i, vp]
    L.tm_set_tuning.argtypes = [vp, ctypes.c_char_p, i]
    L.tm_timing_enable.argtypes = [vp, i]
    L.tm_timing_read.argtypes = [vp, i, ctypes.POINTER(ctypes.c_char_p), ctypes.POINTER(ctypes.c_float),
                                 ctypes.POINTER(i)]
    _lib = L
    return L


def _check(rc):
    if rc != TM_OK:
        raise TmError(rc, lib().tm_last_error().decode())


def _host(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if shape is not None and tuple(a.shape) != tuple(shape):
        raise ValueError("host array has shape %s, expected %s" % (a.shape, tuple(shape)))
    return a


# ---- the C entry points, same names --------------------------------------------------------------------

def tm_init(dims, cuda_device=0):
    arr = (ctypes.c_int * 4)(*[int(x) for x in dims])
    h = ctypes.c_void_p()
    _check(lib().tm_init(arr, int(cuda_device), ctypes.byref(h)))
    return h


def tm_set_stream(ctx, cuda_stream):
    _check(lib().tm_set_stream(ctx, ctypes.c_void_p(int(cuda_stream))))


def tm_sync(ctx):
    _check(lib().tm_sync(ctx))


def tm_finalize(ctx):
    lib().tm_finalize(ctx)


def tm_field_bytes(ctx, prec, n_flavor):
    return int(lib().tm_field_bytes(ctx, int(prec), int(n_flavor)))


def tm_field_alloc(ctx, prec, n_flavor, ext_dev_ptr=None, ext_bytes=0):
    h = ctypes.c_void_p()
    _check(lib().tm_field_alloc(ctx, int(prec), int(n_flavor),
                                ctypes.c_void_p(ext_dev_ptr) if ext_dev_ptr else None, int(ext_bytes),
                                ctypes.byref(h)))
    return h


def tm_field_free(f):
    lib().tm_field_free(f)


def tm_field_upload(f, parity, host_full):
    _check(lib().tm_field_upload(f, int(parity), host_full.ctypes.data_as(ctypes.c_void_p)))


def tm_field_download(f, parity, host_full):
    _check(lib().tm_field_download(f, int(parity), host_full.ctypes.data_as(ctypes.c_void_p)))


def tm_field_upload_cb(f, parity, host_cb):
    ptr = host_cb if isinstance(host_cb, int) else host_cb.ctypes.data
    _check(lib().tm_field_upload_cb(f, int(parity), ctypes.c_void_p(ptr)))


def tm_field_download_cb(f, parity, host_cb):
    ptr = host_cb if isinstance(host_cb, int) else host_cb.ctypes.data
    _check(lib().tm_field_download_cb(f, int(parity), ctypes.c_void_p(ptr)))


def tm_field_upload_cb_async(f, parity, host_cb):
    """host_cb: address (int) of PINNED host memory, or a numpy array backed by it; valid until tm_sync."""
    ptr = host_cb if isinstance(host_cb, int) else host_cb.ctypes.data
    _check(lib().tm_field_upload_cb_async(f, int(parity), ctypes.c_void_p(ptr)))


def tm_field_download_cb_async(f, parity, host_cb):
    ptr = host_cb if isinstance(host_cb, int) else host_cb.ctypes.data
    _check(lib().tm_field_download_cb_async(f, int(parity), ctypes.c_void_p(ptr)))


def tm_field_upload_cb_async_f32(f, parity, host_cb):
    """The same from a float32 host array (address of PINNED memory or a numpy array backed by it)."""
    ptr = host_cb if isinstance(host_cb, int) else host_cb.ctypes.data
    _check(lib().tm_field_upload_cb_async_f32(f, int(parity), ctypes.c_void_p(ptr)))


def tm_field_download_cb_async_f32(f, parity, host_cb):
    ptr = host_cb if isinstance(host_cb, int) else host_cb.ctypes.data
    _check(lib().tm_field_download_cb_async_f32(f, int(parity), ctypes.c_void_p(ptr)))


def tm_gauge_load(ctx, host_links, prec, recon):
    h = ctypes.c_void_p()
    _check(lib().tm_gauge_load(ctx, host_links.ctypes.data_as(ctypes.c_void_p), int(prec), int(recon),
                               ctypes.byref(h)))
    return h


def tm_gauge_free(g):
    lib().tm_gauge_free(g)


def tm_dslash_apply(out, inp, x, gauge, p, parity, dagger, kernel_type, prec):
    _check(lib().tm_dslash_apply(out, inp, x, gauge, ctypes.byref(p), int(parity), int(dagger),
                                 int(kernel_type), int(prec)))


def tm_mat_pc(out_e, in_e, tmp_o, gauge, p, matpc_type, dagger=0):
    _check(lib().tm_mat_pc(out_e, in_e, tmp_o, gauge, ctypes.byref(p), int(matpc_type), int(dagger)))


def tm_reconstruct_odd(psi_o, psi_e, b_o, gauge, p):
    _check(lib().tm_reconstruct_odd(psi_o, psi_e, b_o, gauge, ctypes.byref(p)))


def tm_twist_apply(out, inp, p, inverse=0, dagger=0):
    _check(lib().tm_twist_apply(out, inp, ctypes.byref(p), int(inverse), int(dagger)))


def tm_prepare_rhs(rhs_e, b_e, b_o, tmp_o, gauge, p, matpc_type):
    _check(lib().tm_prepare_rhs(rhs_e, b_e, b_o, tmp_o, gauge, ctypes.byref(p), int(matpc_type)))


def tm_set_open_time(ctx, on):
    _check(lib().tm_set_open_time(ctx, int(on)))


def tm_set_open_dirs(ctx, mask):
    _check(lib().tm_set_open_dirs(ctx, int(mask)))


def tm_halo_bytes(ctx, prec, n_flavor, direction=3):
    return lib().tm_halo_bytes(ctx, int(prec), int(n_flavor), int(direction))


def tm_halo_pack(inp, gauge, out_parity, dagger, dev_to_prev, dev_to_next, direction=3, flag_prev=None, flag_next=None, epoch=0):
    _check(lib().tm_halo_pack(inp, gauge, int(out_parity), int(dagger), int(direction), ctypes.c_void_p(dev_to_prev),
                              ctypes.c_void_p(dev_to_next), ctypes.c_void_p(flag_prev), ctypes.c_void_p(flag_next), int(epoch)))


def tm_halo_apply(out, dev_from_prev, dev_from_next, gauge, p, out_parity, dagger, kernel_type, sign_prev, sign_next, direction=3,
                  wait_prev=None, wait_next=None, epoch=0):
    _check(lib().tm_halo_apply(out, ctypes.c_void_p(dev_from_prev), ctypes.c_void_p(dev_from_next), gauge, ctypes.byref(p),
                               int(out_parity), int(dagger), int(kernel_type), int(direction), int(sign_prev), int(sign_next),
                               ctypes.c_void_p(wait_prev), ctypes.c_void_p(wait_next), int(epoch)))


def tm_field_axpby(z, a, x, b, y):
    _check(lib().tm_field_axpby(z, float(a), x, float(b), y))


def tm_field_redot(x, y):
    r = ctypes.c_double(0.0)
    _check(lib().tm_field_redot(x, y, ctypes.byref(r)))
    return r.value


TM_NOALLOC_MAX_SITES = 8388608      # include/tm.h: sites per parity the fixed scratch array of tm_field_redot_noalloc covers


def tm_field_redot_noalloc(x, y, dev_result):
    """dev_result: DEVICE address of one double (e.g. torch tensor .data_ptr()); nothing is allocated or synchronised."""
    _check(lib().tm_field_redot_noalloc(x, y, ctypes.c_void_p(int(dev_result))))


def tm_invert_cg(x_e, b_e, g_precise, g_sloppy, p, matpc_type, tol, max_iter, sloppy_precision, delta, op=None):
    """-> dict(iterations, restarts, residual, converged).  op: a TM_CG_OP_FN (the caller's operator, e.g. a sharded one)."""
    cp = tm_cg_params(float(tol), int(max_iter), int(sloppy_precision), float(delta), op if op is not None else TM_CG_OP_FN(), None)
    info = tm_cg_info()
    _check(lib().tm_invert_cg(x_e, b_e, g_precise, g_sloppy, ctypes.byref(p), int(matpc_type), ctypes.byref(cp),
                              ctypes.byref(info)))
    return dict(iterations=info.iterations, restarts=info.restarts, residual=info.residual, converged=bool(info.converged))


def tm_cg_release(ctx):
    lib().tm_cg_release(ctx)


def tm_set_allreduce(ctx, fn):
    """fn: a TM_ALLREDUCE_FN instance (keep a reference to it while it is set) or None."""
    _check(lib().tm_set_allreduce(ctx, fn if fn is not None else TM_ALLREDUCE_FN(), None))


def tm_launch_count(ctx):
    return int(lib().tm_launch_count(ctx))


def tm_last_kernel_name(ctx):
    return lib().tm_last_kernel_name(ctx).decode()


def tm_set_host_basis(ctx, basis, custom=None):
    """custom: complex 4x4 (numpy) for TM_BASIS_CUSTOM."""
    ptr = None
    if custom is not None:
        custom = np.ascontiguousarray(custom, dtype=np.complex128).reshape(4, 4)
        ptr = custom.ctypes.data_as(ctypes.c_void_p)
    _check(lib().tm_set_host_basis(ctx, int(basis), ptr))


def tm_set_path(ctx, path):
    _check(lib().tm_set_path(ctx, int(path)))


def tm_set_tuning(ctx, key, value):
    _check(lib().tm_set_tuning(ctx, key.encode(), int(value)))


def tm_timing_enable(ctx, on):
    _check(lib().tm_timing_enable(ctx, int(on)))


def tm_timing_read(ctx, max_records=1 << 16):
    """-> list of (kernel name, milliseconds) per dslash launch since the last read, in launch order."""
    names = (ctypes.c_char_p * max_records)()
    ms = (ctypes.c_float * max_records)()
    n = ctypes.c_int(0)
    _check(lib().tm_timing_read(ctx, max_records, names, ms, ctypes.byref(n)))
    return [(names[k].decode(), float(ms[k])) for k in range(n.value)]


# ---- handle owners: torch supplies the memory and the stream -------------------------------------------

class Lattice:
    """A tm_ctx bound to torch's current stream on `device`."""

    def __init__(self, dims, device=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1311_4462_b200 needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.dims = tuple(int(d) for d in dims)
        self.V = int(np.prod(self.dims))
        self.Vh = self.V // 2
        self.device = int(device)
        torch.cuda.set_device(self.device)
        self.ctx = tm_init(self.dims, self.device)
        self.use_stream(torch.cuda.current_stream(self.device))

    def use_stream(self, stream):
        self.stream = stream
        tm_set_stream(self.ctx, stream.cuda_stream)

    def field(self, prec, n_flavor=1):
        return Field(self, prec, n_flavor)

    def gauge(self, host_links, prec, recon):
        return Gauge(self, host_links, prec, recon)

    def sync(self):
        tm_sync(self.ctx)

    def launches(self):
        return tm_launch_count(self.ctx)

    def close(self):
        if self.ctx is not None:
            tm_finalize(self.ctx)
            self.ctx = None


class Field:
    """One single-parity spinor field; storage is a torch.uint8 tensor borrowed by the library."""

    def __init__(self, lat, prec, n_flavor=1):
        torch = lat.torch
        self.lat, self.prec, self.nf = lat, int(prec), int(n_flavor)
        self.nbytes = tm_field_bytes(lat.ctx, prec, n_flavor)
        self.storage = torch.zeros(self.nbytes, dtype=torch.uint8, device="cuda:%d" % lat.device)
        self.h = tm_field_alloc(lat.ctx, prec, n_flavor, self.storage.data_ptr(), self.nbytes)

    def upload(self, parity, host_full):
        tm_field_upload(self.h, parity, _host(host_full, (self.nf, self.lat.V, 4, 3)))
        return self

    def download(self, parity, out=None):
        if out is None:
            out = np.zeros((self.nf, self.lat.V, 4, 3), dtype=np.complex128)
        tm_field_download(self.h, parity, out)
        return out

    def upload_cb(self, parity, host_cb):
        tm_field_upload_cb(self.h, parity, _host(host_cb, (self.nf, self.lat.Vh, 4, 3)))
        return self

    def download_cb(self, parity):
        out = np.zeros((self.nf, self.lat.Vh, 4, 3), dtype=np.complex128)
        tm_field_download_cb(self.h, parity, out)
        return out

    def __del__(self):
        try:
            if getattr(self, "h", None) is not None:
                tm_field_free(self.h)
                self.h = None
        except Exception:
            pass


class Gauge:
    def __init__(self, lat, host_links, prec, recon):
        self.lat, self.prec, self.recon = lat, int(prec), int(recon)
        self.h = tm_gauge_load(lat.ctx, _host(host_links, (4, lat.V, 3, 3)), prec, recon)

    def __del__(self):
        try:
            if getattr(self, "h", None) is not None:
                tm_gauge_free(self.h)
                self.h = None
        except Exception:
            pass


def dslash_apply(out, inp, x, gauge, p, parity, dagger, kernel_type):
    tm_dslash_apply(out.h, inp.h, None if x is None else x.h, gauge.h, p, parity, dagger, kernel_type, out.prec)


def mat_pc(out_e, in_e, tmp_o, gauge, p, matpc_type, dagger=0):
    tm_mat_pc(out_e.h, in_e.h, tmp_o.h, gauge.h, p, matpc_type, dagger)


def reconstruct_odd(psi_o, psi_e, b_o, gauge, p):
    tm_reconstruct_odd(psi_o.h, psi_e.h, b_o.h, gauge.h, p)


def twist_apply(out, inp, p, inverse=0, dagger=0):
    tm_twist_apply(out.h, inp.h, p, inverse, dagger)


def prepare_rhs(rhs_e, b_e, b_o, tmp_o, gauge, p, matpc_type):
    tm_prepare_rhs(rhs_e.h, b_e.h, b_o.h, tmp_o.h, gauge.h, p, matpc_type)


def field_axpby(z, a, x, b=0.0, y=None):
    tm_field_axpby(z.h, a, x.h, b, None if y is None else y.h)


def field_redot(x, y):
    return tm_field_redot(x.h, y.h)


def invert_cg(x_e, b_e, g_precise, g_sloppy, p, matpc_type, tol=1e-10, max_iter=10000, sloppy_precision=TM_SINGLE, delta=0.1, op=None):
    return tm_invert_cg(x_e.h, b_e.h, g_precise.h, None if g_sloppy is None else g_sloppy.h, p, matpc_type, tol, max_iter,
                        sloppy_precision, delta, op)
