"""Thin Python binding of libmvd.so (include/mvd.h): argument marshalling only.

Every step of the deconvolution runs in the library's CUDA kernels; PyTorch is used here only to
own device memory (views, workspace, results) and to supply the stream.  There is no CPU path: if
libmvd.so is missing or no CUDA device is present, constructing a Deconvolver raises.
The function names mirror the C ABI (mvd_create / mvd_iterate / mvd_get_estimate ...).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmvd.so")

VARIANTS = {"independent": 0, "efficient": 1, "osem": 2}
N_KERNEL_CLASSES = 7      # MVD_K_COUNT
KERNEL_MODES = {"auto": 0, "plain": 1, "compound": 2, "opt1": 3, "opt2": 4}

# every symbol include/mvd.h declares (tests check that the library exports them all)
SYMBOLS = (
    "mvd_options_init", "mvd_workspace_size", "mvd_plan_dims", "mvd_create", "mvd_iterate",
    "mvd_get_estimate", "mvd_set_estimate", "mvd_restart", "mvd_get_stats", "mvd_get_back_projector", "mvd_convolve",
    "mvd_launch_count", "mvd_profile", "mvd_profile_read", "mvd_kernel_class_name", "mvd_blocked_workspace_size", "mvd_deconvolve_blocked", "mvd_destroy",
    "mvd_status_string", "mvd_last_error",
    "mvd_compare", "mvd_partial_product", "mvd_get_product", "mvd_apply_product", "mvd_reduce_scratch_bytes", "mvd_reduce_sum",
    "mvd_reduce_sum_static", "mvd_reduce_sum_static_max", "mvd_reduce_sum_static_error",
)


class MvdError(RuntimeError):
    pass


class mvd_options(C.Structure):
    _fields_ = [
        ("struct_size", C.c_size_t),
        ("kernel_mode", C.c_int),
        ("literal_product", C.c_int),
        ("eps", C.c_float),
        ("psi_floor", C.c_float),
        ("psi0", C.c_void_p),
        ("fft_dims", C.c_int * 3),
        ("workspace", C.c_void_p),
        ("workspace_bytes", C.c_size_t),
        ("stream", C.c_void_p),
        ("use_graph", C.c_int),
        ("weights", C.c_void_p),
        ("local_views", C.c_void_p),
        ("n_local", C.c_int),
        ("psi0_value", C.c_float),
        ("views_ready", C.c_void_p),
        ("tikhonov_lambda", C.c_float),
        ("block_rank", C.c_int),
        ("block_world", C.c_int),
    ]


_Int3 = C.c_int * 3
_lib = None


def load_library():
    """dlopen libmvd.so (built in-tree by ``python -m paper_1308_0730_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MvdError("%s not found: build it with `python -m paper_1308_0730_b200.build` "
                       "(there is no CPU fallback)" % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    vp, ip = C.c_void_p, C.POINTER(C.c_int)
    lib.mvd_options_init.argtypes = [C.POINTER(mvd_options)]
    lib.mvd_options_init.restype = None
    lib.mvd_workspace_size.argtypes = [C.c_int, _Int3, vp, C.c_int, C.POINTER(mvd_options)]
    lib.mvd_workspace_size.restype = C.c_size_t
    lib.mvd_plan_dims.argtypes = [C.c_int, _Int3, vp, C.POINTER(mvd_options), _Int3]
    lib.mvd_plan_dims.restype = C.c_int
    lib.mvd_create.argtypes = [C.POINTER(vp), C.c_int, C.POINTER(vp), _Int3, C.POINTER(vp), vp, C.c_int,
                               C.POINTER(mvd_options)]
    lib.mvd_create.restype = C.c_int
    lib.mvd_iterate.argtypes = [vp, C.c_int]
    lib.mvd_iterate.restype = C.c_int
    lib.mvd_get_estimate.argtypes = [vp, vp, C.c_int]
    lib.mvd_get_estimate.restype = C.c_int
    lib.mvd_set_estimate.argtypes = [vp, vp]
    lib.mvd_set_estimate.restype = C.c_int
    lib.mvd_restart.argtypes = [vp, vp]
    lib.mvd_restart.restype = C.c_int
    lib.mvd_get_stats.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), ip]
    lib.mvd_get_stats.restype = C.c_int
    lib.mvd_get_back_projector.argtypes = [vp, C.c_int, vp]
    lib.mvd_get_back_projector.restype = C.c_int
    lib.mvd_convolve.argtypes = [vp, C.c_int, C.c_int, vp, vp]
    lib.mvd_convolve.restype = C.c_int
    lib.mvd_launch_count.argtypes = [vp]
    lib.mvd_launch_count.restype = C.c_longlong
    lib.mvd_profile.argtypes = [vp, C.c_int]
    lib.mvd_profile.restype = C.c_int
    lib.mvd_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    lib.mvd_profile_read.restype = C.c_int
    lib.mvd_kernel_class_name.argtypes = [C.c_int]
    lib.mvd_kernel_class_name.restype = C.c_char_p
    lib.mvd_blocked_workspace_size.argtypes = [C.c_int, _Int3, vp, C.c_int, C.POINTER(mvd_options), _Int3, vp]
    lib.mvd_blocked_workspace_size.restype = C.c_size_t
    lib.mvd_deconvolve_blocked.argtypes = [C.c_int, C.POINTER(vp), _Int3, C.POINTER(vp), vp, C.c_int,
                                           C.POINTER(mvd_options), _Int3, vp, C.c_int, vp,
                                           C.POINTER(C.c_longlong)]
    lib.mvd_deconvolve_blocked.restype = C.c_int
    lib.mvd_destroy.argtypes = [vp]
    lib.mvd_destroy.restype = None
    lib.mvd_status_string.argtypes = [C.c_int]
    lib.mvd_status_string.restype = C.c_char_p
    lib.mvd_last_error.argtypes = [vp]
    lib.mvd_last_error.restype = C.c_char_p
    lib.mvd_compare.argtypes = [vp, vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.mvd_compare.restype = C.c_int
    lib.mvd_partial_product.argtypes = [vp]
    lib.mvd_partial_product.restype = C.c_int
    lib.mvd_get_product.argtypes = [vp, C.POINTER(vp)]
    lib.mvd_get_product.restype = C.c_int
    lib.mvd_apply_product.argtypes = [vp, C.c_int]
    lib.mvd_apply_product.restype = C.c_int
    lib.mvd_reduce_scratch_bytes.argtypes = []
    lib.mvd_reduce_scratch_bytes.restype = C.c_size_t
    lib.mvd_reduce_sum.argtypes = [vp, C.c_longlong, vp, vp, C.POINTER(C.c_double)]
    lib.mvd_reduce_sum.restype = C.c_int
    lib.mvd_reduce_sum_static.argtypes = [vp, C.c_longlong, vp, C.POINTER(C.c_double)]
    lib.mvd_reduce_sum_static.restype = C.c_int
    lib.mvd_reduce_sum_static_max.argtypes = []
    lib.mvd_reduce_sum_static_max.restype = C.c_longlong
    lib.mvd_reduce_sum_static_error.argtypes = []
    lib.mvd_reduce_sum_static_error.restype = C.c_char_p
    _lib = lib
    return lib


def _check(status, ctx=None, what=""):
    if status != 0:
        lib = load_library()
        msg = lib.mvd_status_string(status).decode()
        detail = lib.mvd_last_error(ctx).decode() if ctx else ""
        raise MvdError("%s: %s%s" % (what, msg, (" (" + detail + ")") if detail else ""))


def _psf_args(psfs):
    """Host PSF arrays (Kz,Ky,Kx) -> (keepalive arrays, void* array, int[V][3] of {Kx,Ky,Kz})."""
    arrs = [np.ascontiguousarray(p, dtype=np.float32) for p in psfs]
    for a in arrs:
        if a.ndim != 3:
            raise MvdError("a PSF must be a 3-D array (Kz, Ky, Kx)")
    ptrs = (C.c_void_p * len(arrs))(*[a.ctypes.data for a in arrs])
    dims = (C.c_int * (3 * len(arrs)))()
    for v, a in enumerate(arrs):
        dims[3 * v + 0], dims[3 * v + 1], dims[3 * v + 2] = a.shape[2], a.shape[1], a.shape[0]
    return arrs, ptrs, dims


def _make_options(kernel_mode, literal_product, eps, psi_floor, fft_dims, use_graph, tikhonov_lambda=None):
    lib = load_library()
    opt = mvd_options()
    lib.mvd_options_init(C.byref(opt))
    opt.kernel_mode = KERNEL_MODES[kernel_mode]
    opt.literal_product = int(bool(literal_product))
    if eps is not None:
        opt.eps = float(eps)
    if psi_floor is not None:
        opt.psi_floor = float(psi_floor)
    if fft_dims is not None:
        opt.fft_dims[:] = [int(x) for x in fft_dims]
    opt.use_graph = int(bool(use_graph))
    if tikhonov_lambda is not None:
        opt.tikhonov_lambda = float(tikhonov_lambda)
    return opt


def plan_dims(dims, psfs_or_dims, kernel_mode="auto", fft_dims=None):
    """FFT lengths (Mx2, My, Mz) the library uses for volume dims (Nx,Ny,Nz) and PSF boxes
    [(Kx,Ky,Kz), ...].  Pure host logic: works without a GPU."""
    lib = load_library()
    boxes = [tuple(int(x) for x in b) for b in psfs_or_dims]
    pd = (C.c_int * (3 * len(boxes)))(*[x for b in boxes for x in b])
    opt = _make_options(kernel_mode, False, None, None, fft_dims, False)
    out = _Int3()
    _check(lib.mvd_plan_dims(len(boxes), _Int3(*dims), C.cast(pd, C.c_void_p), C.byref(opt), out), None, "mvd_plan_dims")
    return tuple(out)


def workspace_size(dims, boxes, variant="osem", kernel_mode="auto", fft_dims=None):
    lib = load_library()
    pd = (C.c_int * (3 * len(boxes)))(*[int(x) for b in boxes for x in b])
    opt = _make_options(kernel_mode, False, None, None, fft_dims, False)
    return int(lib.mvd_workspace_size(len(boxes), _Int3(*dims), C.cast(pd, C.c_void_p), VARIANTS[variant], C.byref(opt)))


class Deconvolver:
    """One mvd_ctx.  ``views``: list of CUDA float32 torch tensors of shape (Nz,Ny,Nx) (borrowed, kept
    alive here); ``psfs``: list of host arrays (Kz,Ky,Kx)."""

    def __init__(self, views, psfs, variant="osem", kernel_mode="auto", literal_product=False,
                 eps=None, psi_floor=None, psi0=None, fft_dims=None, use_graph=False, stream=None,
                 weights=None, views_ready=None, local_views=None, psi0_value=None, tikhonov_lambda=None):
        import torch

        lib = load_library()
        if not torch.cuda.is_available():
            raise MvdError("no CUDA device: the multi-view deconvolution path has no CPU fallback")
        if local_views is not None:
            # view-parallel context: `views` holds this rank's views only, in the order of local_views
            local_views = [int(v) for v in local_views]
            if len(views) != len(local_views):
                raise MvdError("need one view per entry of local_views")
            full = [None] * len(psfs)
            for i, v in enumerate(local_views):
                full[v] = views[i]
            self._local = (C.c_int * len(local_views))(*local_views)
        else:
            full = list(views)
        if len(full) != len(psfs) or not views:
            raise MvdError("need one PSF per view")
        self._torch = torch
        self.views = [None if v is None else
                      (v if (v.is_cuda and v.dtype == torch.float32 and v.is_contiguous())
                       else v.to(device="cuda", dtype=torch.float32).contiguous()) for v in full]
        present = [v for v in self.views if v is not None]
        shape = tuple(present[0].shape)
        if len(shape) != 3 or any(tuple(v.shape) != shape for v in present):
            raise MvdError("views must be 3-D tensors of one shape (Nz, Ny, Nx)")
        self.shape = shape
        self.dims = (shape[2], shape[1], shape[0])
        self.device = present[0].device
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._psfs, psf_ptrs, psf_dims = _psf_args(psfs)
        self._psf_dims = psf_dims
        opt = _make_options(kernel_mode, literal_product, eps, psi_floor, fft_dims, use_graph, tikhonov_lambda)
        if local_views is not None:
            opt.local_views = C.cast(self._local, C.c_void_p)
            opt.n_local = len(local_views)
        if psi0_value is not None:
            opt.psi0_value = float(psi0_value)
        nbytes = lib.mvd_workspace_size(len(full), _Int3(*self.dims), C.cast(psf_dims, C.c_void_p),
                                        VARIANTS[variant], C.byref(opt))
        if nbytes == 0:
            raise MvdError("mvd_workspace_size: invalid or unsupported problem "
                           "(dims %s, PSF boxes %s)" % (self.dims, [tuple(p.shape[::-1]) for p in self._psfs]))
        with torch.cuda.stream(self.stream):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        opt.workspace = base
        opt.workspace_bytes = nbytes
        opt.stream = self.stream.cuda_stream
        self._psi0 = None
        if psi0 is not None:
            self._psi0 = psi0.to(device=self.device, dtype=torch.float32).contiguous()
            opt.psi0 = self._psi0.data_ptr()
        self._weights = None
        if weights is not None:
            if len(weights) != len(full):
                raise MvdError("need one weight image per view")
            self._weights = [w.to(device=self.device, dtype=torch.float32).contiguous() for w in weights]
            if any(tuple(w.shape) != shape for w in self._weights):
                raise MvdError("weight images must have the shape of the views")
            self._weight_ptrs = (C.c_void_p * len(full))(*[w.data_ptr() for w in self._weights])
            opt.weights = C.cast(self._weight_ptrs, C.c_void_p)
        if views_ready is not None:      # torch.cuda.Event recorded after the caller's copy of the views
            opt.views_ready = views_ready.cuda_event
        self.workspace_bytes = int(nbytes)
        view_ptrs = (C.c_void_p * len(full))(*[None if v is None else v.data_ptr() for v in self.views])
        ctx = C.c_void_p()
        # the conversions / copies above ran on torch's current stream: the library's stream waits for them
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        with torch.cuda.device(self.device):
            st = lib.mvd_create(C.byref(ctx), len(full), view_ptrs, _Int3(*self.dims), psf_ptrs,
                                C.cast(psf_dims, C.c_void_p), VARIANTS[variant], C.byref(opt))
        _check(st, None, "mvd_create")
        self._ctx = ctx
        self._lib = lib
        out = _Int3()
        lib.mvd_plan_dims(len(full), _Int3(*self.dims), C.cast(psf_dims, C.c_void_p), C.byref(opt), out)
        self.fft_dims = tuple(out)

    # -- C ABI mirrors --------------------------------------------------------------------------
    def iterate(self, n=1):
        with self._torch.cuda.device(self.device):
            _check(self._lib.mvd_iterate(self._ctx, int(n)), self._ctx, "mvd_iterate")

    def compare(self, ref):
        """mvd_compare: (average absolute difference, cross-correlation) of psi against a reference volume."""
        r = ref.to(device=self.device, dtype=self._torch.float32).contiguous()
        self.stream.wait_stream(self._torch.cuda.current_stream(self.device))
        a, x = C.c_double(), C.c_double()
        with self._torch.cuda.device(self.device):
            _check(self._lib.mvd_compare(self._ctx, r.data_ptr(), C.byref(a), C.byref(x)), self._ctx, "mvd_compare")
        return a.value, x.value

    def partial_product(self):
        """mvd_partial_product: acc <- product over this context's views of max(f_v, 0), psi unchanged."""
        with self._torch.cuda.device(self.device):
            _check(self._lib.mvd_partial_product(self._ctx), self._ctx, "mvd_partial_product")

    def product_tensor(self):
        """The product accumulator as a float32 tensor (Nz,Ny,Nx) aliasing the workspace (mvd_get_product)."""
        p = C.c_void_p()
        _check(self._lib.mvd_get_product(self._ctx, C.byref(p)), self._ctx, "mvd_get_product")
        off = p.value - self.workspace.data_ptr()
        n = self.shape[0] * self.shape[1] * self.shape[2]
        return self.workspace[off:off + 4 * n].view(self._torch.float32).view(self.shape)

    def apply_product(self, total_views):
        with self._torch.cuda.device(self.device):
            _check(self._lib.mvd_apply_product(self._ctx, int(total_views)), self._ctx, "mvd_apply_product")

    def get_estimate(self, out=None):
        """Device tensor (Nz,Ny,Nx) with a copy of psi (asynchronous on the stream)."""
        torch = self._torch
        if out is None:
            with torch.cuda.stream(self.stream):
                out = torch.empty(self.shape, dtype=torch.float32, device=self.device)
        _check(self._lib.mvd_get_estimate(self._ctx, out.data_ptr(), 1), self._ctx, "mvd_get_estimate")
        return out

    def get_estimate_host(self, out=None):
        """numpy array (Nz,Ny,Nx); synchronises.  ``out`` may be a (pinned) float32 array."""
        if out is None:
            out = np.empty(self.shape, dtype=np.float32)
        _check(self._lib.mvd_get_estimate(self._ctx, out.ctypes.data, 0), self._ctx, "mvd_get_estimate")
        return out

    def set_estimate(self, psi):
        t = psi.to(device=self.device, dtype=self._torch.float32).contiguous()
        if tuple(t.shape) != self.shape:
            raise MvdError("estimate has the wrong shape")
        self.stream.wait_stream(self._torch.cuda.current_stream(self.device))
        _check(self._lib.mvd_set_estimate(self._ctx, t.data_ptr()), self._ctx, "mvd_set_estimate")
        self.stream.synchronize()

    def restart(self, views_ready=None):
        """mvd_restart: the view buffers hold a new time-point (same PSFs); `views_ready` is a torch.cuda.Event
        recorded after the caller's copy into them."""
        ev = views_ready.cuda_event if views_ready is not None else None
        with self._torch.cuda.device(self.device):
            _check(self._lib.mvd_restart(self._ctx, ev), self._ctx, "mvd_restart")

    def get_stats(self):
        f, l, it = C.c_double(), C.c_double(), C.c_int()
        _check(self._lib.mvd_get_stats(self._ctx, C.byref(f), C.byref(l), C.byref(it)), self._ctx, "mvd_get_stats")
        return {"flux": f.value, "l1_change": l.value, "iterations_done": it.value}

    def get_back_projector(self, view):
        p = self._psfs[view]
        out = np.empty(p.shape, dtype=np.float64)
        _check(self._lib.mvd_get_back_projector(self._ctx, int(view), out.ctypes.data), self._ctx, "mvd_get_back_projector")
        return out

    def convolve(self, view, which, src):
        """crop(src (*) P_view) (which=0) or crop(src (*) K_view) (which=1) through the FFT path."""
        torch = self._torch
        s = src.to(device=self.device, dtype=torch.float32).contiguous()
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        with torch.cuda.stream(self.stream):
            dst = torch.empty(self.shape, dtype=torch.float32, device=self.device)
        _check(self._lib.mvd_convolve(self._ctx, int(view), int(which), s.data_ptr(), dst.data_ptr()), self._ctx, "mvd_convolve")
        self.stream.synchronize()
        return dst

    def profile(self, enable=True):
        _check(self._lib.mvd_profile(self._ctx, int(bool(enable))), self._ctx, "mvd_profile")

    def profile_read(self):
        """{kernel class: (total device ms, launches)} since the last read; synchronises."""
        ms = (C.c_double * N_KERNEL_CLASSES)()
        n = (C.c_longlong * N_KERNEL_CLASSES)()
        _check(self._lib.mvd_profile_read(self._ctx, ms, n), self._ctx, "mvd_profile_read")
        return {self._lib.mvd_kernel_class_name(k).decode(): (ms[k], int(n[k])) for k in range(N_KERNEL_CLASSES)}

    @property
    def launch_count(self):
        return int(self._lib.mvd_launch_count(self._ctx))

    def close(self):
        if getattr(self, "_ctx", None):
            self.stream.synchronize()
            self._lib.mvd_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def deconvolve_blocked(views, psfs, block_dims, iterations, variant="osem", kernel_mode="auto",
                       halo=None, eps=None, psi_floor=None, literal_product=False, stream=None,
                       block_rank=0, block_world=0, out=None, tikhonov_lambda=None):
    """mvd_deconvolve_blocked: block_dims / halo are (x,y,z).  Returns (device tensor, launches).
    block_world > 1: only the blocks with index % block_world == block_rank are processed (blocks dealt
    over GPUs); the other voxels of the result keep what `out` held (zeros if out is None)."""
    import torch

    lib = load_library()
    if not torch.cuda.is_available():
        raise MvdError("no CUDA device: the multi-view deconvolution path has no CPU fallback")
    views = [v.to(device="cuda", dtype=torch.float32).contiguous() for v in views]
    shape = tuple(views[0].shape)
    dims = (shape[2], shape[1], shape[0])
    device = views[0].device
    stream = stream if stream is not None else torch.cuda.current_stream(device)
    keep, psf_ptrs, psf_dims = _psf_args(psfs)
    opt = _make_options(kernel_mode, literal_product, eps, psi_floor, None, False, tikhonov_lambda)
    opt.block_rank, opt.block_world = int(block_rank), int(block_world)
    halo_arg = C.cast(_Int3(*halo), C.c_void_p) if halo is not None else None
    nbytes = lib.mvd_blocked_workspace_size(len(views), _Int3(*dims), C.cast(psf_dims, C.c_void_p),
                                            VARIANTS[variant], C.byref(opt), _Int3(*block_dims), halo_arg)
    if nbytes == 0:
        raise MvdError("mvd_blocked_workspace_size: invalid or unsupported problem")
    with torch.cuda.stream(stream):
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
        if out is not None:
            if tuple(out.shape) != shape or out.dtype != torch.float32 or not out.is_cuda or not out.is_contiguous():
                raise MvdError("out must be a contiguous CUDA float32 tensor of the views' shape")
            dst = out
        else:
            dst = (torch.zeros if block_world > 1 else torch.empty)(shape, dtype=torch.float32, device=device)
    opt.workspace = (ws.data_ptr() + 255) // 256 * 256
    opt.workspace_bytes = nbytes
    opt.stream = stream.cuda_stream
    view_ptrs = (C.c_void_p * len(views))(*[v.data_ptr() for v in views])
    launches = C.c_longlong(0)
    stream.wait_stream(torch.cuda.current_stream(device))
    with torch.cuda.device(device):
        st = lib.mvd_deconvolve_blocked(len(views), view_ptrs, _Int3(*dims), psf_ptrs,
                                        C.cast(psf_dims, C.c_void_p), VARIANTS[variant], C.byref(opt),
                                        _Int3(*block_dims), halo_arg, int(iterations), dst.data_ptr(),
                                        C.byref(launches))
    _check(st, None, "mvd_deconvolve_blocked")
    stream.synchronize()
    del keep
    return dst, int(launches.value)


def reduce_sum(t, stream=None):
    """mvd_reduce_sum: fp64 sum of a CUDA float32 tensor through the library's reduction kernels."""
    import torch
    lib = load_library()
    t = t.contiguous()
    stream = stream if stream is not None else torch.cuda.current_stream(t.device)
    with torch.cuda.device(t.device):
        nscratch = int(lib.mvd_reduce_scratch_bytes())
    with torch.cuda.stream(stream):
        scratch = torch.empty(nscratch, dtype=torch.uint8, device=t.device)
    stream.wait_stream(torch.cuda.current_stream(t.device))      # t may have been produced on the current stream
    out = C.c_double(0.0)
    with torch.cuda.device(t.device):
        _check(lib.mvd_reduce_sum(t.data_ptr(), t.numel(), scratch.data_ptr(), stream.cuda_stream, C.byref(out)),
               None, "mvd_reduce_sum")
    return float(out.value)


def reduce_sum_static(t, stream=None):
    """mvd_reduce_sum_static: the same fp64 sum as reduce_sum, for callers that must not allocate.

    reduce_sum asks torch for a scratch tensor on every call.  A job whose workspace already fills the GPU, a time-lapse
    loop that cannot afford the allocator's device-wide synchronisation between time-points, or an embedding
    application that forbids allocations on its device cannot do that; this call allocates nothing, neither here nor in
    the library: the partial sums go to a fixed ~128 KB array inside libmvd.so's device image (include/mvd.h has the
    details).  Hence the rules: `t` is used where it lies (a non-contiguous tensor is refused rather than copied), at most
    2^30 elements (MvdError beyond that), and two calls whose GPU work could overlap must not be issued concurrently.
    The first call on a device also looks up the array's address; make it before capturing any stream of that device.
    """
    import torch
    lib = load_library()
    if t.dtype != torch.float32 or not t.is_cuda or not t.is_contiguous():
        raise MvdError("reduce_sum_static: needs a contiguous float32 CUDA tensor (no copy is made: that would allocate)")
    stream = stream if stream is not None else torch.cuda.current_stream(t.device)
    stream.wait_stream(torch.cuda.current_stream(t.device))
    out = C.c_double(0.0)
    with torch.cuda.device(t.device):
        st = lib.mvd_reduce_sum_static(t.data_ptr(), t.numel(), stream.cuda_stream, C.byref(out))
    if st != 0:
        raise MvdError("mvd_reduce_sum_static: %s (%s)" % (lib.mvd_status_string(st).decode(),
                                                           lib.mvd_reduce_sum_static_error().decode()))
    return float(out.value)


def split_views(n_views, world, rank):
    """Views of `rank` when n_views are dealt round-robin over `world` ranks (ascending indices)."""
    return [v for v in range(n_views) if v % world == rank]


class ViewParallelDeconvolver:
    """Combined variants (independent / efficient) with the views split over the ranks of a
    torch.distributed process group (all view contributions can be computed at the
    same time).  Every rank keeps the whole estimate; one iteration = each rank's partial product
    of its views' factors, ONE all-reduce(PRODUCT) of N floats, the same root update on every rank.
    `local_views_data`: this rank's views (CUDA tensors) in the order of split_views(); `psfs`:
    ALL PSFs (the compound kernels need them).  group=None and world 1 runs without torch.distributed."""

    def __init__(self, local_views_data, psfs, variant="efficient", rank=0, world=1, group=None, **kw):
        import torch
        if variant not in ("independent", "efficient"):
            raise MvdError("sequential updates (osem) do not split over ranks")
        self.rank, self.world, self.group = int(rank), int(world), group
        self.n_views = len(psfs)
        self.local = split_views(self.n_views, self.world, self.rank)
        if not self.local or len(local_views_data) != len(self.local):
            raise MvdError("rank %d owns views %s" % (self.rank, self.local))
        self._torch = torch
        stream = kw.pop("stream", None) or torch.cuda.current_stream(local_views_data[0].device)
        # psi^0 = mean over ALL views (L304, L421): local sums by the library, one all-reduce(SUM)
        tot = torch.tensor([sum(reduce_sum(v, stream) for v in local_views_data),
                            float(sum(v.numel() for v in local_views_data))], dtype=torch.float64)
        tot = self._all_reduce(tot, "sum")
        self.d = Deconvolver(local_views_data, psfs, variant=variant, local_views=self.local,
                             psi0_value=float(tot[0] / tot[1]), stream=stream, **kw)

    def _all_reduce(self, t, op):
        if self.world == 1:
            return t
        import torch.distributed as dist
        if t.device.type == "cpu" and dist.get_backend(self.group) == "nccl":
            t = t.cuda()
        dist.all_reduce(t, op=dist.ReduceOp.SUM if op == "sum" else dist.ReduceOp.PRODUCT, group=self.group)
        return t.cpu() if op == "sum" else t

    def iterate(self, n=1):
        torch = self._torch
        for _ in range(int(n)):
            self.d.partial_product()
            if self.world > 1:
                with torch.cuda.stream(self.d.stream):      # the collective is ordered after the kernels
                    self._all_reduce(self.d.product_tensor(), "product")
            self.d.apply_product(self.n_views)

    def get_estimate_host(self, out=None):
        return self.d.get_estimate_host(out)

    def get_stats(self):
        return self.d.get_stats()

    def close(self):
        self.d.close()
