"""ctypes binding of liblgf (include/lgf.h) -- argument marshalling only.

Every function has the name and the meaning of the C entry point it wraps; every step of the hot path
runs inside the CUDA kernels of liblgf.so.  PyTorch is used here only to own device memory and to
provide the stream.  There is no CPU fallback: if liblgf.so is missing the import of the library
fails with an instruction to build it, and without a CUDA device ``lgf_create`` raises ``LgfError``.

Tensors passed as ``links`` are in the canonical layout of include/lgf.h: shape
[Lt, Lz, Ly, Lx, 4, 3, 3, 2] real (or [Lt, Lz, Ly, Lx, 4, 3, 3] complex), dtype matching the
context's precision, contiguous; CUDA tensors go to the device entry points, CPU tensors / numpy
arrays to the ``*_host`` ones.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

LGF_FP32, LGF_FP64 = 4, 8
LGF_LINKS_18, LGF_LINKS_12 = 18, 12
LGF_OK, LGF_EINVAL, LGF_ENOMEM, LGF_ECUDA, LGF_ESTATE, LGF_ENAN = 0, -1, -2, -3, -4, -5
LGF_K_DELTA, LGF_K_FFT, LGF_K_UPDATE, LGF_K_GBUILD, LGF_K_CONVERT, LGF_K_PLAQ, LGF_K_HEATBATH, LGF_K_COUNT = 0, 1, 2, 3, 4, 5, 6, 7
LGF_K_ITERATION = 100
KERNEL_CLASSES = ("delta", "fft", "update", "gbuild", "convert", "plaquette", "heatbath")

_LIBPATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "liblgf.so")
_lib = None

# name -> (restype, argtypes); the list of symbols include/lgf.h declares
_vp, _i, _d, _ll = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_longlong
_dp, _llp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_longlong)
SIGNATURES = {
    "lgf_create": (_i, [ctypes.POINTER(ctypes.c_int), _i, _i, ctypes.POINTER(_vp)]),
    "lgf_destroy": (_i, [_vp]),
    "lgf_set_stream": (_i, [_vp, _vp]),
    "lgf_set_links": (_i, [_vp, _vp]),
    "lgf_get_links": (_i, [_vp, _vp]),
    "lgf_set_links_host": (_i, [_vp, _vp]),
    "lgf_get_links_host": (_i, [_vp, _vp]),
    "lgf_iterate": (_i, [_vp, _d, _i]),
    "lgf_measure": (_i, [_vp, _dp, _dp, _dp]),
    "lgf_fix": (_ll, [_vp, _vp, _d, _d, _ll]),
    "lgf_fix_host": (_ll, [_vp, _vp, _d, _d, _ll]),
    "lgf_history": (_i, [_vp, _ll, _ll, _dp, _dp]),
    "lgf_history_length": (_ll, [_vp]),
    "lgf_iterations": (_ll, [_vp]),
    "lgf_step_delta": (_i, [_vp, _dp, _dp]),
    "lgf_step_accelerate": (_i, [_vp]),
    "lgf_step_update": (_i, [_vp, _d]),
    "lgf_get_field": (_i, [_vp, _vp]),
    "lgf_set_field": (_i, [_vp, _vp]),
    "lgf_thermalize": (_i, [_vp, _d, _i, ctypes.c_ulonglong]),
    "lgf_overrelax": (_i, [_vp, _i]),
    "lgf_track_transform": (_i, [_vp, _i]),
    "lgf_get_transform": (_i, [_vp, _vp]),
    "lgf_gluon_field": (_i, [_vp, _i, _vp]),
    "lgf_apply_transform": (_i, [_vp, _vp]),
    "lgf_tune": (_i, [_vp, ctypes.c_char_p, _i]),
    "lgf_fft_passes": (_i, [_vp]),
    "lgf_set_profiling": (_i, [_vp, _i]),
    "lgf_kernel_times": (_i, [_vp, _dp, _llp]),
    "lgf_kernel_names": (_i, [_vp, ctypes.c_char_p, _i]),
    "lgf_launch_count": (_ll, [_vp]),
    "lgf_algorithmic_bytes": (_d, [_vp, _i]),
    "lgf_last_error": (ctypes.c_char_p, [_vp]),
    "lgf_version": (ctypes.c_char_p, []),
    "lgf_measure_static": (_i, [ctypes.POINTER(ctypes.c_int), _i, _vp, _vp, _vp]),
    "lgf_static_last_error": (ctypes.c_char_p, []),
    # one configuration sharded over several GPUs (per-rank entry points; exchanges in slab.py)
    "lgf_slab_create": (_i, [ctypes.POINTER(ctypes.c_int), _i, _i, _i, _i, ctypes.POINTER(_vp)]),
    "lgf_slab_destroy": (_i, [_vp]),
    "lgf_slab_set_stream": (_i, [_vp, _vp]),
    "lgf_slab_set_links": (_i, [_vp, _vp]),
    "lgf_slab_get_links": (_i, [_vp, _vp]),
    "lgf_slab_halo_elems": (_ll, [_vp, _i]),
    "lgf_slab_halo_pack": (_i, [_vp, _i, _vp]),
    "lgf_slab_halo_unpack": (_i, [_vp, _i, _vp]),
    "lgf_slab_delta": (_i, [_vp, _vp]),
    "lgf_slab_fft_forward": (_i, [_vp, _vp]),
    "lgf_slab_fft_t": (_i, [_vp, _vp, _vp]),
    "lgf_slab_fft_inverse": (_i, [_vp, _vp]),
    "lgf_slab_fft_inverse_g": (_i, [_vp, _vp, _d]),
    "lgf_slab_by_component": (_i, [_vp]),
    "lgf_slab_fft_forward_comp": (_i, [_vp, _vp, _i]),
    "lgf_slab_fft_t_comp": (_i, [_vp, _vp, _vp, _i]),
    "lgf_slab_fft_zinv_comp": (_i, [_vp, _vp, _i]),
    "lgf_slab_fft_xyinv": (_i, [_vp, _i, _d]),
    "lgf_slab_gbuild": (_i, [_vp, _d]),
    "lgf_slab_update": (_i, [_vp]),
    "lgf_slab_sweep": (_i, [_vp, _vp]),
    "lgf_slab_finalize": (_i, [_vp, _vp, _d, _i, _i]),
    "lgf_slab_clear_done": (_i, [_vp]),
    "lgf_slab_poll": (_i, [_vp]),
    "lgf_slab_poll_wait": (_i, [_vp, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int), _llp, _dp, _dp]),
    "lgf_slab_history_length": (_ll, [_vp]),
    "lgf_slab_history": (_i, [_vp, _ll, _ll, _dp, _dp]),
    "lgf_slab_get_field": (_i, [_vp, _vp]),
    "lgf_slab_launch_count": (_ll, [_vp]),
    "lgf_slab_last_error": (ctypes.c_char_p, [_vp]),
}
LGF_HALO_LINKS, LGF_HALO_G, LGF_HALO_G_UP = 0, 1, 2


class LgfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("liblgf error %d: %s" % (code, msg))
        self.code = code


def library_path() -> str:
    return _LIBPATH


def load():
    """Load liblgf.so (built by ``python -m paper_1206_0675_b200.build``).  Never falls back."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise ImportError("%s is missing: build the CUDA library with `python -m paper_1206_0675_b200.build` "
                              "(there is no CPU fallback)" % _LIBPATH)
        lib = ctypes.CDLL(_LIBPATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _check(ctx, rc):
    if rc < 0:
        msg = load().lgf_last_error(ctx)
        raise LgfError(int(rc), msg.decode() if msg else "")
    return rc


def _dev_ptr(t, ctx_prec, nreal):
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("expected a CUDA torch tensor")
    if t.is_complex():
        t = torch.view_as_real(t)
    want = torch.float64 if ctx_prec == LGF_FP64 else torch.float32
    if t.dtype != want or not t.is_contiguous() or t.numel() != nreal:
        raise ValueError("tensor must be contiguous %s with %d reals (got %s, %d)" % (want, nreal, t.dtype, t.numel()))
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(a, ctx_prec, nreal):
    import torch

    if isinstance(a, torch.Tensor):
        if a.is_cuda:
            raise TypeError("expected host memory")
        if a.is_complex():
            a = torch.view_as_real(a)
        want = torch.float64 if ctx_prec == LGF_FP64 else torch.float32
        if a.dtype != want or not a.is_contiguous() or a.numel() != nreal:
            raise ValueError("host tensor must be contiguous %s with %d reals" % (want, nreal))
        return ctypes.c_void_p(a.data_ptr())
    want = {LGF_FP64: (np.float64, np.complex128), LGF_FP32: (np.float32, np.complex64)}[ctx_prec]
    if not isinstance(a, np.ndarray) or a.dtype not in want or not a.flags.c_contiguous:
        raise ValueError("host array must be a C-contiguous numpy array of %s" % (want,))
    if a.size * (2 if np.iscomplexobj(a) else 1) != nreal:
        raise ValueError("host array has the wrong size")
    return ctypes.c_void_p(a.ctypes.data)


class Context:
    """Owns one lgf_ctx.  Methods are the C entry points minus the ``lgf_`` prefix and ``ctx`` argument."""

    def __init__(self, dims, precision=LGF_FP64, link_storage=LGF_LINKS_18, stream=None):
        self.dims = tuple(int(v) for v in dims)
        self.precision, self.link_storage = int(precision), int(link_storage)
        self.V = int(np.prod(self.dims))
        self._h = ctypes.c_void_p()
        lib = load()
        rc = lib.lgf_create((ctypes.c_int * 4)(*self.dims), self.precision, self.link_storage, ctypes.byref(self._h))
        if rc < 0:
            msg = lib.lgf_last_error(None)
            raise LgfError(rc, msg.decode() if msg else "")
        if stream is not None:
            self.set_stream(stream)

    # -- lifetime ---------------------------------------------------------------------------------
    def destroy(self):
        if self._h:
            load().lgf_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    # -- plumbing ---------------------------------------------------------------------------------
    def set_stream(self, stream):
        ptr = stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)
        _check(self._h, load().lgf_set_stream(self._h, ctypes.c_void_p(ptr)))

    def set_links(self, links):
        _check(self._h, load().lgf_set_links(self._h, _dev_ptr(links, self.precision, self.V * 72)))

    def get_links(self, out):
        _check(self._h, load().lgf_get_links(self._h, _dev_ptr(out, self.precision, self.V * 72)))
        return out

    def set_links_host(self, links):
        _check(self._h, load().lgf_set_links_host(self._h, _host_ptr(links, self.precision, self.V * 72)))

    def get_links_host(self, out):
        _check(self._h, load().lgf_get_links_host(self._h, _host_ptr(out, self.precision, self.V * 72)))
        return out

    # -- the path ---------------------------------------------------------------------------------
    def iterate(self, alpha, n):
        _check(self._h, load().lgf_iterate(self._h, float(alpha), int(n)))

    def measure(self, plaquette=True):
        F, th, P = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        _check(self._h, load().lgf_measure(self._h, ctypes.byref(F), ctypes.byref(th),
                                           ctypes.byref(P) if plaquette else None))
        return F.value, th.value, (P.value if plaquette else None)

    def fix(self, links, alpha, tol, max_iter):
        return int(_check(self._h, load().lgf_fix(self._h, _dev_ptr(links, self.precision, self.V * 72), float(alpha),
                                                  float(tol), int(max_iter))))

    def fix_host(self, links, alpha, tol, max_iter):
        return int(_check(self._h, load().lgf_fix_host(self._h, _host_ptr(links, self.precision, self.V * 72),
                                                       float(alpha), float(tol), int(max_iter))))

    def history_length(self):
        return int(_check(self._h, load().lgf_history_length(self._h)))

    def history(self, first=0, count=None):
        if count is None:
            count = self.history_length() - first
        F = np.zeros(count)
        th = np.zeros(count)
        _check(self._h, load().lgf_history(self._h, int(first), int(count), F.ctypes.data_as(_dp), th.ctypes.data_as(_dp)))
        return F, th

    def iterations(self):
        return int(_check(self._h, load().lgf_iterations(self._h)))

    # -- single steps -----------------------------------------------------------------------------
    def step_delta(self, want_values=True):
        if not want_values:
            _check(self._h, load().lgf_step_delta(self._h, None, None))
            return None
        F, th = ctypes.c_double(), ctypes.c_double()
        _check(self._h, load().lgf_step_delta(self._h, ctypes.byref(F), ctypes.byref(th)))
        return F.value, th.value

    def step_accelerate(self):
        _check(self._h, load().lgf_step_accelerate(self._h))

    def step_update(self, alpha):
        _check(self._h, load().lgf_step_update(self._h, float(alpha)))

    def get_field(self, out):
        _check(self._h, load().lgf_get_field(self._h, _dev_ptr(out, self.precision, self.V * 18)))
        return out

    def set_field(self, field):
        _check(self._h, load().lgf_set_field(self._h, _dev_ptr(field, self.precision, self.V * 18)))

    # -- thermalisation --------------------------------------------------------------------------
    def thermalize(self, beta, nsweeps, seed):
        _check(self._h, load().lgf_thermalize(self._h, float(beta), int(nsweeps), int(seed)))

    def overrelax(self, nsweeps):
        _check(self._h, load().lgf_overrelax(self._h, int(nsweeps)))

    # -- accumulated gauge transformation ----------------------------------------------------------
    def track_transform(self, on=True):
        _check(self._h, load().lgf_track_transform(self._h, int(bool(on))))

    def get_transform(self, out):
        _check(self._h, load().lgf_get_transform(self._h, _dev_ptr(out, self.precision, self.V * 18)))
        return out

    def gluon_field(self, mu, out):
        _check(self._h, load().lgf_gluon_field(self._h, int(mu), _dev_ptr(out, self.precision, self.V * 18)))
        return out

    def apply_transform(self, transform):
        _check(self._h, load().lgf_apply_transform(self._h, _dev_ptr(transform, self.precision, self.V * 18)))

    # -- tuning -----------------------------------------------------------------------------------
    def tune(self, key, value):
        _check(self._h, load().lgf_tune(self._h, key.encode(), int(value)))

    def fft_passes(self):
        return int(load().lgf_fft_passes(self._h))

    # -- instrumentation --------------------------------------------------------------------------
    def set_profiling(self, on):
        _check(self._h, load().lgf_set_profiling(self._h, int(bool(on))))

    def kernel_times(self):
        ms = (ctypes.c_double * LGF_K_COUNT)()
        n = (ctypes.c_longlong * LGF_K_COUNT)()
        _check(self._h, load().lgf_kernel_times(self._h, ms, n))
        return {k: (ms[i], int(n[i])) for i, k in enumerate(KERNEL_CLASSES)}

    def launch_count(self):
        return int(load().lgf_launch_count(self._h))

    def kernel_names(self):
        """{kernel class: [instantiation names]} of one iteration, as a profiler prints them"""
        buf = ctypes.create_string_buffer(1024)
        _check(self._h, load().lgf_kernel_names(self._h, buf, 1024))
        return {k: v.split("|") for k, v in (kv.split("=", 1) for kv in buf.value.decode().split(";"))}

    def algorithmic_bytes(self, kernel_class):
        return float(load().lgf_algorithmic_bytes(self._h, int(kernel_class)))


class SlabContext:
    """Owns one lgf_slab: rank `rank` of `nranks` of ONE configuration sharded over t (include/lgf.h, last section).
    Methods are the C entry points minus the ``lgf_slab_`` prefix; all local to this rank -- the exchanges
    between ranks are paper_1206_0675_b200.slab's."""

    def __init__(self, dims, precision, link_storage, rank, nranks, stream=None):
        self.dims = tuple(int(v) for v in dims)
        self.precision, self.link_storage = int(precision), int(link_storage)
        self.rank, self.nranks = int(rank), int(nranks)
        self._h = ctypes.c_void_p()
        lib = load()
        rc = lib.lgf_slab_create((ctypes.c_int * 4)(*self.dims), self.precision, self.link_storage, self.rank,
                                 self.nranks, ctypes.byref(self._h))
        if rc < 0:
            msg = lib.lgf_slab_last_error(None)
            raise LgfError(rc, msg.decode() if msg else "")
        self.T = self.dims[3] // self.nranks
        self.V = self.dims[0] * self.dims[1] * self.dims[2] * self.T       # local sites
        if stream is not None:
            self.set_stream(stream)

    def destroy(self):
        if self._h:
            load().lgf_slab_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _ck(self, rc):
        if rc < 0:
            msg = load().lgf_slab_last_error(self._h)
            raise LgfError(int(rc), msg.decode() if msg else "")
        return rc

    def set_stream(self, stream):
        ptr = stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)
        self._ck(load().lgf_slab_set_stream(self._h, ctypes.c_void_p(ptr)))

    def set_links(self, links):
        self._ck(load().lgf_slab_set_links(self._h, _dev_ptr(links, self.precision, self.V * 72)))

    def get_links(self, out):
        self._ck(load().lgf_slab_get_links(self._h, _dev_ptr(out, self.precision, self.V * 72)))
        return out

    def halo_elems(self, which):
        return int(self._ck(load().lgf_slab_halo_elems(self._h, int(which))))

    def halo_pack(self, which, send):
        self._ck(load().lgf_slab_halo_pack(self._h, int(which), _dev_ptr(send, self.precision, self.halo_elems(which))))

    def halo_unpack(self, which, recv):
        self._ck(load().lgf_slab_halo_unpack(self._h, int(which), _dev_ptr(recv, self.precision, self.halo_elems(which))))

    def delta(self, sums):
        self._ck(load().lgf_slab_delta(self._h, _dev_ptr(sums, LGF_FP64, 2)))

    def fft_forward(self, send):
        self._ck(load().lgf_slab_fft_forward(self._h, _dev_ptr(send, self.precision, self.V * 8)))

    def fft_t(self, recv, send):
        self._ck(load().lgf_slab_fft_t(self._h, _dev_ptr(recv, self.precision, self.V * 8),
                                       _dev_ptr(send, self.precision, self.V * 8)))

    def fft_inverse(self, recv):
        self._ck(load().lgf_slab_fft_inverse(self._h, _dev_ptr(recv, self.precision, self.V * 8)))

    def fft_inverse_g(self, recv, alpha):
        self._ck(load().lgf_slab_fft_inverse_g(self._h, _dev_ptr(recv, self.precision, self.V * 8), float(alpha)))

    def by_component(self):
        return bool(self._ck(load().lgf_slab_by_component(self._h)))

    def fft_forward_comp(self, send, comp):
        self._ck(load().lgf_slab_fft_forward_comp(self._h, _dev_ptr(send, self.precision, self.V * 8), int(comp)))

    def fft_t_comp(self, recv, send, comp):
        self._ck(load().lgf_slab_fft_t_comp(self._h, _dev_ptr(recv, self.precision, self.V * 8),
                                            _dev_ptr(send, self.precision, self.V * 8), int(comp)))

    def fft_zinv_comp(self, recv, comp):
        self._ck(load().lgf_slab_fft_zinv_comp(self._h, _dev_ptr(recv, self.precision, self.V * 8), int(comp)))

    def fft_xyinv(self, with_g, alpha=0.0):
        self._ck(load().lgf_slab_fft_xyinv(self._h, int(bool(with_g)), float(alpha)))

    def gbuild(self, alpha):
        self._ck(load().lgf_slab_gbuild(self._h, float(alpha)))

    def update(self):
        self._ck(load().lgf_slab_update(self._h))

    def sweep(self, sums):
        self._ck(load().lgf_slab_sweep(self._h, _dev_ptr(sums, LGF_FP64, 2)))

    def finalize(self, sums, tol, after_sweep, record):
        self._ck(load().lgf_slab_finalize(self._h, _dev_ptr(sums, LGF_FP64, 2), float(tol), int(after_sweep), int(record)))

    def clear_done(self):
        self._ck(load().lgf_slab_clear_done(self._h))

    def poll(self):
        self._ck(load().lgf_slab_poll(self._h))

    def poll_wait(self):
        """(done, nan_seen, n_updates, F, theta) of the oldest outstanding look"""
        done, nan, n = ctypes.c_int(), ctypes.c_int(), ctypes.c_longlong()
        F, th = ctypes.c_double(), ctypes.c_double()
        self._ck(load().lgf_slab_poll_wait(self._h, ctypes.byref(done), ctypes.byref(nan), ctypes.byref(n), ctypes.byref(F),
                                           ctypes.byref(th)))
        return bool(done.value), bool(nan.value), int(n.value), F.value, th.value

    def history_length(self):
        return int(self._ck(load().lgf_slab_history_length(self._h)))

    def history(self, first=0, count=None):
        if count is None:
            count = self.history_length() - first
        F, th = np.zeros(count), np.zeros(count)
        self._ck(load().lgf_slab_history(self._h, int(first), int(count), F.ctypes.data_as(_dp), th.ctypes.data_as(_dp)))
        return F, th

    def get_field(self, out):
        self._ck(load().lgf_slab_get_field(self._h, _dev_ptr(out, self.precision, self.V * 18)))
        return out

    def launch_count(self):
        return int(load().lgf_slab_launch_count(self._h))


LGF_STATIC_MAX_SITES = 2097152


def measure_static(dims, precision, links, out, stream=None):
    """lgf_measure_static: (F, theta) of a canonical-layout CUDA tensor into `out` (CUDA tensor of two float64),
    asynchronously; allocates nothing on the device.  Returns `out`."""
    dims = tuple(int(v) for v in dims)
    V = int(np.prod(dims))
    lib = load()
    sp = 0 if stream is None else (stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))
    rc = lib.lgf_measure_static((ctypes.c_int * 4)(*dims), int(precision), _dev_ptr(links, precision, V * 72),
                                _dev_ptr(out, LGF_FP64, 2), ctypes.c_void_p(sp))
    if rc < 0:
        msg = lib.lgf_static_last_error()
        raise LgfError(int(rc), msg.decode() if msg else "")
    return out


def lgf_version() -> str:
    return load().lgf_version().decode()


# C-style aliases with the header's names
def lgf_create(dims, precision, link_storage):
    return Context(dims, precision, link_storage)


def lgf_destroy(ctx):
    ctx.destroy()


def lgf_iterate(ctx, alpha, n):
    ctx.iterate(alpha, n)


def lgf_measure(ctx):
    return ctx.measure()


def lgf_fix(ctx, links, alpha, tol, max_iter):
    return ctx.fix(links, alpha, tol, max_iter)
