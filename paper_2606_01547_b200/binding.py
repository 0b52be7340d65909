"""ctypes binding of include/jt.h -- argument marshalling only; every step runs in libjt's kernels.

Tensors are torch CUDA tensors (float32 -> JT_F32, float64 -> JT_F64), contiguous; the current
torch stream is passed through.  Names and argument meaning follow include/jt.h one to one.
"""
import ctypes
import functools
import inspect
import os
from dataclasses import dataclass

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libjt.so")
_lib = None

JT_F32, JT_F64 = 0, 1
_METHODS = {"auto": 0, "direct": 1, "fft": 2}
_STATUS = {0: "JT_OK", 1: "JT_ERR_INVALID_VALUE", 2: "JT_ERR_UNSUPPORTED", 3: "JT_ERR_WORKSPACE", 4: "JT_ERR_CUDA"}


class JtError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        extra = ""
        if self.status == 4 and _lib is not None:
            extra = " (cudaError %d)" % _lib.jt_last_cuda_error()
        super().__init__("%s failed: %s%s" % (where, _STATUS.get(self.status, str(status)), extra))


class _Grid(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("pixel_scale", ctypes.c_double),
                ("cx", ctypes.c_double), ("cy", ctypes.c_double), ("supersample", ctypes.c_int32)]


class _Lens(ctypes.Structure):
    _fields_ = [("has_sie", ctypes.c_int32), ("sie_theta_E", ctypes.c_double), ("sie_e1", ctypes.c_double),
                ("sie_e2", ctypes.c_double), ("sie_cx", ctypes.c_double), ("sie_cy", ctypes.c_double),
                ("has_shear", ctypes.c_int32), ("shear_gamma1", ctypes.c_double), ("shear_gamma2", ctypes.c_double),
                ("n_tnfw", ctypes.c_int64), ("tnfw_cx", ctypes.c_void_p), ("tnfw_cy", ctypes.c_void_p),
                ("tnfw_Rs", ctypes.c_void_p), ("tnfw_alpha_Rs", ctypes.c_void_p), ("tnfw_r_trunc", ctypes.c_void_p)]


_dp = ctypes.POINTER(ctypes.c_double)


class _Sources(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int32), ("amp", _dp), ("R_sersic", _dp), ("n_sersic", _dp), ("e1", _dp),
                ("e2", _dp), ("cx", _dp), ("cy", _dp)]


class _ConvPlan(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("method", "path", "tma", "z_split", "row_bands", "oy", "warps", "pad_y", "pad_x",
                                               "reserved")] + [("est_us", ctypes.c_double)]


class _TracePlan(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("rays_per_thread", "threads", "wide", "n_chunks", "tile_recs", "reserved")] + \
               [("chunk_len", ctypes.c_int64), ("n_ctas", ctypes.c_int64)]


class _Batch(ctypes.Structure):
    _fields_ = [("sie", ctypes.c_void_p), ("shear", ctypes.c_void_p), ("n_tnfw", ctypes.c_int32),
                ("tnfw", ctypes.c_void_p), ("n_src", ctypes.c_int32), ("sersic", ctypes.c_void_p),
                ("ky", ctypes.c_int32), ("kx", ctypes.c_int32), ("psf", ctypes.c_void_p)]


@dataclass
class Grid:
    """Definition G (include/jt.h jt_grid)."""
    nx: int
    ny: int
    pixel_scale: float
    cx: float = 0.0
    cy: float = 0.0
    supersample: int = 1

    def _c(self):
        return _Grid(self.nx, self.ny, self.pixel_scale, self.cx, self.cy, self.supersample)


def lib_path():
    return _LIB_PATH


def lib():
    """Loads libjt.so; raises (never falls back) when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError("libjt.so is missing: build it with `python -m paper_2606_01547_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(_LIB_PATH)
        vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
        L.jt_status_string.restype = ctypes.c_char_p
        L.jt_status_string.argtypes = [ctypes.c_int]
        L.jt_last_cuda_error.restype = ctypes.c_int
        L.jt_version.restype = ctypes.c_int
        L.jt_ray_shoot_workspace_bytes.restype = sz
        L.jt_ray_shoot_workspace_bytes.argtypes = [ctypes.c_int, i64, i64]
        L.jt_ray_shoot.argtypes = [ctypes.c_int, i64, vp, vp, ctypes.POINTER(_Lens), vp, sz, vp, vp, vp]
        L.jt_ray_shoot_noalloc_capacity.restype = sz
        L.jt_ray_shoot_noalloc_capacity.argtypes = []
        L.jt_ray_shoot_noalloc.argtypes = [ctypes.c_int, i64, vp, vp, ctypes.POINTER(_Lens), vp, vp, vp]
        L.jt_psf_convolve_plan.argtypes = [ctypes.c_int, i64, i32, i32, i32, i32, ctypes.c_int, vp, ctypes.POINTER(_ConvPlan)]
        L.jt_trace_plan_query.argtypes = [ctypes.c_int, ctypes.POINTER(_Grid), i64, i64, ctypes.POINTER(_TracePlan)]
        L.jt_source_brightness.argtypes = [ctypes.c_int, i64, vp, vp, ctypes.POINTER(_Sources), vp, vp]
        L.jt_psf_convolve_workspace_bytes.restype = sz
        L.jt_psf_convolve_workspace_bytes.argtypes = [ctypes.c_int, i32, i32, i32, i32, ctypes.c_int]
        L.jt_psf_convolve.argtypes = [ctypes.c_int, i32, i32, vp, i32, i32, vp, ctypes.c_int, vp, sz, vp, vp]
        L.jt_psf_convolve_batch_workspace_bytes.restype = sz
        L.jt_psf_convolve_batch_workspace_bytes.argtypes = [ctypes.c_int, i64, i32, i32, i32, i32, ctypes.c_int]
        L.jt_psf_convolve_batch.argtypes = [ctypes.c_int, i64, i32, i32, vp, i32, i32, vp, ctypes.c_int, vp, sz, vp, vp]
        L.jt_simulate_image_workspace_bytes.restype = sz
        L.jt_simulate_image_workspace_bytes.argtypes = [ctypes.c_int, ctypes.POINTER(_Grid), i64, i32, i32, ctypes.c_int]
        L.jt_simulate_image.argtypes = [ctypes.c_int, ctypes.POINTER(_Grid), ctypes.POINTER(_Lens),
                                        ctypes.POINTER(_Sources), i32, i32, vp, ctypes.c_int, vp, sz, vp, vp]
        L.jt_simulate_batch.argtypes = [ctypes.c_int, i64, ctypes.POINTER(_Grid), ctypes.POINTER(_Batch), vp, vp]
        dbl = ctypes.POINTER(ctypes.c_double)
        L.jt_chi2_batch.argtypes = [ctypes.c_int, i64, i32, i32, vp, vp, vp, vp, vp]
        L.jt_simulate_batch_chi2.argtypes = [ctypes.c_int, i64, ctypes.POINTER(_Grid), ctypes.POINTER(_Batch), vp, vp, vp, vp, vp]
        L.jt_lensing_maps.argtypes = [ctypes.c_int, i64, vp, vp, ctypes.POINTER(_Lens), vp, vp, vp, vp, vp]
        L.jt_ray_shoot_profiles.argtypes = [ctypes.c_int, i64, vp, vp, i64, vp, vp, vp, vp]
        L.jt_light_profiles.argtypes = [ctypes.c_int, i64, vp, vp, i64, vp, vp, vp]
        L.jt_light_core_sersic.argtypes = [ctypes.c_int, i64, vp, vp, dbl, vp, vp]
        L.jt_light_shapelets.argtypes = [ctypes.c_int, i64, vp, vp, i32, ctypes.c_double, ctypes.c_double, ctypes.c_double, vp, vp, vp]
        L.jt_simulate_image_supersampled_psf_workspace_bytes.restype = sz
        L.jt_simulate_image_supersampled_psf_workspace_bytes.argtypes = [ctypes.c_int, ctypes.POINTER(_Grid), i64, i32, i32, ctypes.c_int]
        L.jt_simulate_image_supersampled_psf.argtypes = [ctypes.c_int, ctypes.POINTER(_Grid), ctypes.POINTER(_Lens),
                                                         ctypes.POINTER(_Sources), i32, i32, vp, ctypes.c_int, vp, sz, vp, vp]
        del dbl
        L.jt_kernel_launches.restype = ctypes.c_uint64
        L.jt_profile_enable.argtypes = [ctypes.c_int]
        L.jt_profile_read.argtypes = [ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_float)]
        L.jt_profile_tiers.argtypes = [ctypes.POINTER(ctypes.c_uint64)]
        _lib = L
    return _lib


def version():
    return lib().jt_version()


def kernel_launches():
    """jt_kernel_launches: kernels launched by libjt from this host thread so far."""
    return int(lib().jt_kernel_launches())


def profile_enable(on=True):
    """jt_profile_enable: record events around the ray-tracing and convolution phases of jt_simulate_image."""
    _check(lib().jt_profile_enable(1 if on else 0), "jt_profile_enable")


def profile_read():
    """jt_profile_read: (trace_ms, conv_ms) of the last profiled jt_simulate_image call."""
    a, b = ctypes.c_float(), ctypes.c_float()
    _check(lib().jt_profile_read(ctypes.byref(a), ctypes.byref(b)), "jt_profile_read")
    return a.value, b.value


def profile_tiers():
    """jt_profile_tiers: (far-far long / middle / short series, far, mid, cold) counts of (warp, subhalo record) pairs of
    the last profiled call (JT_N_TIERS = 6 values)."""
    c = (ctypes.c_uint64 * 6)()
    _check(lib().jt_profile_tiers(c), "jt_profile_tiers")
    return tuple(int(x) for x in c)


PROBE_KINDS = {"ffma": 0, "ffma2": 1, "dfma": 2, "mufu_rsq": 3}
_probe_lib = None


def probe_lib_path():
    return os.path.join(_HERE, "libjtprobe.so")


def _probe():
    """libjtprobe.so (include/jt_probe.h): measurement aid, separate from the product library."""
    global _probe_lib
    if _probe_lib is None:
        L = ctypes.CDLL(probe_lib_path())
        L.jt_probe_alu.argtypes = [ctypes.c_int32, ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p,
                                   ctypes.POINTER(ctypes.c_int64), ctypes.c_void_p]
        L.jt_probe_alu.restype = ctypes.c_int
        _probe_lib = L
    return _probe_lib


def probe_alu(kind, blocks=148 * 8, iters=4096, repeats=3):
    """jt_probe_alu timed with CUDA events: returns thread-level instructions of `kind` per second (best of repeats)."""
    sink = torch.zeros(4, dtype=torch.float32, device="cuda")
    n = ctypes.c_int64()
    st = torch.cuda.current_stream()
    best = 0.0
    for _ in range(repeats + 1):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(st)
        _check(_probe().jt_probe_alu(PROBE_KINDS[kind], blocks, iters, ctypes.c_void_p(sink.data_ptr()), ctypes.byref(n),
                                     ctypes.c_void_p(st.cuda_stream)), "jt_probe_alu")
        b.record(st)
        b.synchronize()
        best = max(best, n.value / (a.elapsed_time(b) * 1e-3))
    return best


# ------------------------------------------------------------------ marshalling helpers
def _dt(t):
    if t.dtype == torch.float32:
        return JT_F32
    if t.dtype == torch.float64:
        return JT_F64
    raise TypeError("jt tensors must be float32 or float64, got %s" % t.dtype)


def _torch_dtype(code):
    return torch.float32 if code == JT_F32 else torch.float64


def _code(dtype):
    if dtype in (torch.float32, "f32", JT_F32, np.float32):
        return JT_F32
    if dtype in (torch.float64, "f64", JT_F64, np.float64):
        return JT_F64
    raise TypeError("dtype must be f32 or f64")


def _dev(t, what):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA tensor" % what)
    return t


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _on_stream(fn):
    """Decorator of the wrappers that take `stream`: when a stream other than torch's current one is given, the wrapper
    body runs with that stream current, so every tensor it creates -- outputs, scratch workspace, uploaded profile
    records -- is allocated from, filled on and later recycled in order with the stream the kernels run on.  (Created on
    the current stream instead, an upload could still be in flight when the kernel starts, and the caching allocator
    could hand a temporary to someone else while the kernel still reads it.)  Inputs the caller made on another stream
    remain the caller's to order, as with any torch op on a side stream."""
    idx = list(inspect.signature(fn).parameters).index("stream")

    @functools.wraps(fn)
    def wrapper(*args, **kw):
        stream = kw["stream"] if "stream" in kw else (args[idx] if len(args) > idx else None)
        if stream is None or stream == torch.cuda.current_stream(stream.device):
            return fn(*args, **kw)
        with torch.cuda.stream(stream):
            return fn(*args, **kw)
    return wrapper


def _check(status, where):
    if status != 0:
        raise JtError(status, where)


def _lens(dtype_code, sie, shear, tnfw):
    L = _Lens()
    if sie is not None:
        L.has_sie = 1
        L.sie_theta_E, L.sie_e1, L.sie_e2, L.sie_cx, L.sie_cy = [float(v) for v in sie]
    if shear is not None:
        L.has_shear = 1
        L.shear_gamma1, L.shear_gamma2 = [float(v) for v in shear]
    if tnfw is not None and tnfw.numel() > 0:
        _dev(tnfw, "tnfw")
        if tnfw.dim() != 2 or tnfw.shape[0] != 5 or _dt(tnfw) != dtype_code:
            raise TypeError("tnfw must be a [5][M] tensor of the call's dtype")
        M = tnfw.shape[1]
        es = tnfw.element_size()
        base = tnfw.data_ptr()
        L.n_tnfw = M
        L.tnfw_cx, L.tnfw_cy, L.tnfw_Rs, L.tnfw_alpha_Rs, L.tnfw_r_trunc = [base + k * M * es for k in range(5)]
    return L


def _sources(sources):
    a = np.ascontiguousarray(np.asarray(sources, dtype=np.float64).reshape(-1, 7).T)   # [7][n]
    S = _Sources()
    S.n = a.shape[1]
    ptrs = [a[k].ctypes.data_as(_dp) for k in range(7)]
    S.amp, S.R_sersic, S.n_sersic, S.e1, S.e2, S.cx, S.cy = ptrs
    return S, a          # keep `a` alive during the call


def _workspace(nbytes, device, workspace, stream=None):
    """Caller's workspace, or a scratch tensor; a scratch tensor used on a non-current stream is tied to that stream
    (record_stream) so that the caching allocator cannot hand it out again while the kernels still run."""
    if nbytes == 0:
        return None, 0
    if workspace is None:
        workspace = torch.empty(nbytes, dtype=torch.uint8, device=device)
        if stream is not None:
            workspace.record_stream(stream)
    return workspace, workspace.numel() * workspace.element_size()


# ------------------------------------------------------------------ the five calls
def ray_shoot_workspace_bytes(dtype, n_rays, n_tnfw):
    return int(lib().jt_ray_shoot_workspace_bytes(_code(dtype), n_rays, n_tnfw))


@_on_stream
def ray_shoot(theta_x, theta_y, sie=None, shear=None, tnfw=None, workspace=None, stream=None):
    """jt_ray_shoot: beta = theta - alpha(theta).  Returns (beta_x, beta_y)."""
    _dev(theta_x, "theta_x"), _dev(theta_y, "theta_y")
    code = _dt(theta_x)
    n = theta_x.numel()
    L = _lens(code, sie, shear, tnfw)
    ws, wsb = _workspace(ray_shoot_workspace_bytes(code, n, L.n_tnfw), theta_x.device, workspace, stream)
    bx, by = torch.empty_like(theta_x), torch.empty_like(theta_y)
    _check(lib().jt_ray_shoot(code, n, _ptr(theta_x), _ptr(theta_y), ctypes.byref(L), _ptr(ws), wsb,
                              _ptr(bx), _ptr(by), _stream(stream)), "jt_ray_shoot")
    return bx, by


def ray_shoot_noalloc_capacity():
    """Bytes of the library's built-in scratch array (JT_NOALLOC_SCRATCH_BYTES, held on every GPU that uses libjt)."""
    return int(lib().jt_ray_shoot_noalloc_capacity())


@_on_stream
def ray_shoot_noalloc(theta_x, theta_y, beta_x, beta_y, sie=None, shear=None, tnfw=None, stream=None):
    """jt_ray_shoot_noalloc: jt_ray_shoot without a workspace, for code that may not allocate device memory where it calls
    us (a framework callback that only receives its input / output buffers, a process whose memory pool already owns the
    GPU).  Nothing is allocated here either: the caller passes the outputs beta_x, beta_y (same shape and dtype as theta),
    and the scratch is a fixed 32 MiB array inside libjt.  Problems whose ray_shoot_workspace_bytes exceeds
    ray_shoot_noalloc_capacity() are refused.  All calls on a GPU share that array: keep them on one stream (calls that
    overlap on the GPU corrupt each other), and make the first call on a device outside stream capture."""
    for t, name in ((theta_x, "theta_x"), (theta_y, "theta_y"), (beta_x, "beta_x"), (beta_y, "beta_y")):
        _dev(t, name)
    code = _dt(theta_x)
    n = theta_x.numel()
    if _dt(beta_x) != code or _dt(beta_y) != code or _dt(theta_y) != code or beta_x.numel() != n or beta_y.numel() != n:
        raise TypeError("beta_x, beta_y must match theta_x, theta_y in dtype and size")
    L = _lens(code, sie, shear, tnfw)
    need = ray_shoot_workspace_bytes(code, n, L.n_tnfw)
    if need > ray_shoot_noalloc_capacity():
        raise JtError(3, "jt_ray_shoot_noalloc (%d rays x %d subhalos need %d bytes of scratch, the built-in array holds %d)"
                      % (n, L.n_tnfw, need, ray_shoot_noalloc_capacity()))
    _check(lib().jt_ray_shoot_noalloc(code, n, _ptr(theta_x), _ptr(theta_y), ctypes.byref(L), _ptr(beta_x), _ptr(beta_y),
                                      _stream(stream)), "jt_ray_shoot_noalloc")
    return beta_x, beta_y


_CONV_PATHS = {0: "small", 1: "tile", 2: "fft"}


def psf_convolve_plan(dtype, ny, nx, ky, kx, method="auto", B=1, image=None):
    """jt_psf_convolve_plan: the launch path a convolution call with these arguments takes (host only).  Returns a dict:
    method ("direct"/"fft"), path ("small"/"tile"/"fft"), tma, z_split, row_bands, oy, warps, pad_y, pad_x, est_us."""
    p = _ConvPlan()
    _check(lib().jt_psf_convolve_plan(_code(dtype), B, ny, nx, ky, kx, _METHODS[method], _ptr(image), ctypes.byref(p)),
           "jt_psf_convolve_plan")
    d = {n: getattr(p, n) for n, _ in _ConvPlan._fields_ if n != "reserved"}
    d["method"] = "direct" if p.method == 1 else "fft"
    d["path"] = _CONV_PATHS[p.path]
    return d


def trace_plan(dtype, grid=None, n_rays=0, n_tnfw=0):
    """jt_trace_plan_query: launch shape of the ray-tracing kernel for jt_simulate_image (grid given) or jt_ray_shoot
    (n_rays given).  Returns a dict: rays_per_thread, threads, wide, n_chunks, tile_recs, chunk_len, n_ctas."""
    p = _TracePlan()
    g = grid._c() if grid is not None else None
    _check(lib().jt_trace_plan_query(_code(dtype), ctypes.byref(g) if g is not None else None, n_rays, n_tnfw, ctypes.byref(p)),
           "jt_trace_plan_query")
    return {n: getattr(p, n) for n, _ in _TracePlan._fields_ if n != "reserved"}


@_on_stream
def source_brightness(beta_x, beta_y, sources, stream=None):
    """jt_source_brightness: sum of elliptical Sersic components at (beta_x, beta_y)."""
    _dev(beta_x, "beta_x"), _dev(beta_y, "beta_y")
    code = _dt(beta_x)
    S, keep = _sources(sources)
    flux = torch.empty_like(beta_x)
    _check(lib().jt_source_brightness(code, beta_x.numel(), _ptr(beta_x), _ptr(beta_y), ctypes.byref(S),
                                      _ptr(flux), _stream(stream)), "jt_source_brightness")
    del keep
    return flux


def psf_convolve_workspace_bytes(dtype, ny, nx, ky, kx, method="auto"):
    return int(lib().jt_psf_convolve_workspace_bytes(_code(dtype), ny, nx, ky, kx, _METHODS[method]))


@_on_stream
def psf_convolve(image, kernel, method="auto", workspace=None, out=None, stream=None):
    """jt_psf_convolve: zero-padded 'same' true convolution of image [ny][nx] with kernel [ky][kx]."""
    _dev(image, "image"), _dev(kernel, "kernel")
    code = _dt(image)
    if _dt(kernel) != code:
        raise TypeError("image and kernel dtypes differ")
    ny, nx = image.shape
    ky, kx = kernel.shape
    ws, wsb = _workspace(psf_convolve_workspace_bytes(code, ny, nx, ky, kx, method), image.device, workspace, stream)
    if out is None:
        out = torch.empty_like(image)
    _check(lib().jt_psf_convolve(code, ny, nx, _ptr(image), ky, kx, _ptr(kernel), _METHODS[method], _ptr(ws), wsb,
                                 _ptr(out), _stream(stream)), "jt_psf_convolve")
    return out


def psf_convolve_batch_workspace_bytes(dtype, B, ny, nx, ky, kx, method="auto"):
    return int(lib().jt_psf_convolve_batch_workspace_bytes(_code(dtype), B, ny, nx, ky, kx, _METHODS[method]))


@_on_stream
def psf_convolve_batch(images, kernel, method="auto", workspace=None, out=None, stream=None):
    """jt_psf_convolve_batch: images [B][ny][nx], one kernel [ky][kx] for all of them."""
    _dev(images, "images"), _dev(kernel, "kernel")
    code = _dt(images)
    if _dt(kernel) != code:
        raise TypeError("images and kernel dtypes differ")
    B, ny, nx = images.shape
    ky, kx = kernel.shape
    ws, wsb = _workspace(psf_convolve_batch_workspace_bytes(code, B, ny, nx, ky, kx, method) if B > 0 else 0,
                         images.device, workspace, stream)
    if out is None:
        out = torch.empty_like(images)
    _check(lib().jt_psf_convolve_batch(code, B, ny, nx, _ptr(images), ky, kx, _ptr(kernel), _METHODS[method], _ptr(ws),
                                       wsb, _ptr(out), _stream(stream)), "jt_psf_convolve_batch")
    return out


def simulate_image_workspace_bytes(dtype, grid, n_tnfw, ky, kx, method="auto"):
    g = grid._c()
    return int(lib().jt_simulate_image_workspace_bytes(_code(dtype), ctypes.byref(g), n_tnfw, ky, kx, _METHODS[method]))


@_on_stream
def simulate_image(grid, sie, shear, tnfw, sources, psf, dtype=None, method="auto", workspace=None, out=None,
                   stream=None, device="cuda"):
    """jt_simulate_image: grid -> ray-shoot -> Sersic -> bin -> PSF convolution.  psf=None skips the convolution."""
    code = _code(dtype) if dtype is not None else (_dt(psf) if psf is not None else _dt(tnfw))
    g = grid._c()
    L = _lens(code, sie, shear, tnfw)
    S, keep = _sources(sources)
    ky, kx = (0, 0) if psf is None else psf.shape
    if psf is not None:
        _dev(psf, "psf")
        if _dt(psf) != code:
            raise TypeError("psf dtype differs from the call's dtype")
        device = psf.device
    elif tnfw is not None:
        device = tnfw.device
    ws, wsb = _workspace(simulate_image_workspace_bytes(code, grid, L.n_tnfw, ky, kx, method), device, workspace, stream)
    if out is None:
        out = torch.empty((grid.ny, grid.nx), dtype=_torch_dtype(code), device=device)
    _check(lib().jt_simulate_image(code, ctypes.byref(g), ctypes.byref(L), ctypes.byref(S), ky, kx, _ptr(psf),
                                   _METHODS[method], _ptr(ws), wsb, _ptr(out), _stream(stream)), "jt_simulate_image")
    del keep
    return out


class PreparedImage:
    """jt_simulate_image with the argument marshalling done ONCE: the C structs, the workspace, the output tensor and the
    stream handle are built at construction, and each call is a single ctypes call (PAPER.md:89 is about exactly this
    per-call overhead; C0 spends 10 us on the device and several times that in marshalling through simulate_image()).
    Marshalling only: every step still runs in libjt's kernels.  The tensors passed in (tnfw, psf) are referenced, not
    copied: updating them IN PLACE between calls is how a caller changes subhalos or PSF; SIE / shear / sources are
    frozen (build another PreparedImage to change them).  Calls go to the stream given here (default: the stream current
    at construction); the returned tensor is the same `out` every time."""

    def __init__(self, grid, sie, shear, tnfw, sources, psf, dtype=None, method="auto", workspace=None, out=None, stream=None,
                 device="cuda"):
        code = _code(dtype) if dtype is not None else (_dt(psf) if psf is not None else _dt(tnfw))
        self._g = grid._c()
        self._L = _lens(code, sie, shear, tnfw)
        self._S, self._keep = _sources(sources)
        ky, kx = (0, 0) if psf is None else psf.shape
        if psf is not None:
            _dev(psf, "psf")
            if _dt(psf) != code:
                raise TypeError("psf dtype differs from the call's dtype")
            device = psf.device
        elif tnfw is not None:
            device = tnfw.device
        self._stream = torch.cuda.current_stream(device) if stream is None else stream
        with torch.cuda.stream(self._stream):
            self._ws, wsb = _workspace(simulate_image_workspace_bytes(code, grid, self._L.n_tnfw, ky, kx, method), device, workspace)
            self.out = out if out is not None else torch.empty((grid.ny, grid.nx), dtype=_torch_dtype(code), device=device)
        self._tensors = (tnfw, psf)                                    # keep the referenced device memory alive
        fn = lib().jt_simulate_image
        args = (code, ctypes.byref(self._g), ctypes.byref(self._L), ctypes.byref(self._S), ky, kx, _ptr(psf), _METHODS[method],
                _ptr(self._ws), wsb, _ptr(self.out), ctypes.c_void_p(self._stream.cuda_stream))
        self._call = functools.partial(fn, *args)

    def __call__(self):
        status = self._call()
        if status != 0:
            raise JtError(status, "jt_simulate_image")
        return self.out


def _batch_struct(sie, shear, tnfw, sersic, psf):
    _dev(sie, "sie"), _dev(shear, "shear")
    code = _dt(sie)
    P = _Batch()
    P.sie, P.shear = sie.data_ptr(), shear.data_ptr()
    if tnfw is not None and tnfw.numel() > 0:
        _dev(tnfw, "tnfw")
        P.n_tnfw, P.tnfw = tnfw.shape[2], tnfw.data_ptr()
    if sersic is not None and sersic.numel() > 0:
        _dev(sersic, "sersic")
        P.n_src, P.sersic = sersic.shape[1], sersic.data_ptr()
    if psf is not None:
        _dev(psf, "psf")
        P.ky, P.kx, P.psf = psf.shape[1], psf.shape[2], psf.data_ptr()
    for t in (shear, tnfw, sersic, psf):
        if t is not None and t.numel() > 0 and _dt(t) != code:
            raise TypeError("all batch tensors must share one dtype")
    return code, P


@_on_stream
def simulate_batch(grid, sie, shear, tnfw, sersic, psf, out=None, stream=None):
    """jt_simulate_batch: B independent systems.  sie [B][5], shear [B][2], tnfw [B][5][M], sersic [B][n][7], psf [B][ky][kx]."""
    code, P = _batch_struct(sie, shear, tnfw, sersic, psf)
    B = sie.shape[0]
    g = grid._c()
    if out is None:
        out = torch.empty((B, grid.ny, grid.nx), dtype=_torch_dtype(code), device=sie.device)
    _check(lib().jt_simulate_batch(code, B, ctypes.byref(g), ctypes.byref(P), _ptr(out), _stream(stream)),
           "jt_simulate_batch")
    return out


# ------------------------------------------------------------------ SURVEY section 8(f) rows
@_on_stream
def chi2_batch(models, data, sigma, out=None, stream=None):
    """jt_chi2_batch: chi2[b] = sum ((models[b] - data) / sigma)^2 as a float64 tensor [B]."""
    _dev(models, "models"), _dev(data, "data"), _dev(sigma, "sigma")
    code = _dt(models)
    if _dt(data) != code or _dt(sigma) != code:
        raise TypeError("models, data and sigma must share one dtype")
    B, ny, nx = models.shape
    if out is None:
        out = torch.empty(B, dtype=torch.float64, device=models.device)
    _check(lib().jt_chi2_batch(code, B, ny, nx, _ptr(models), _ptr(data), _ptr(sigma), _ptr(out), _stream(stream)), "jt_chi2_batch")
    return out


@_on_stream
def simulate_batch_chi2(grid, sie, shear, tnfw, sersic, psf, data, sigma, images=False, chi2=None, stream=None):
    """jt_simulate_batch_chi2: the batch kernel with the chi^2 against (data, sigma) accumulated in the same thread block.
    Returns chi2 [B] (float64), or (chi2, images) with images=True / an images tensor."""
    code, P = _batch_struct(sie, shear, tnfw, sersic, psf)
    _dev(data, "data"), _dev(sigma, "sigma")
    if _dt(data) != code or _dt(sigma) != code:
        raise TypeError("data and sigma must have the batch's dtype")
    B = sie.shape[0]
    g = grid._c()
    img = None
    if images is True:
        img = torch.empty((B, grid.ny, grid.nx), dtype=_torch_dtype(code), device=sie.device)
    elif isinstance(images, torch.Tensor):
        img = images
    if chi2 is None:
        chi2 = torch.empty(B, dtype=torch.float64, device=sie.device)
    _check(lib().jt_simulate_batch_chi2(code, B, ctypes.byref(g), ctypes.byref(P), _ptr(data), _ptr(sigma), _ptr(img), _ptr(chi2),
                                        _stream(stream)), "jt_simulate_batch_chi2")
    return chi2 if img is None else (chi2, img)


@_on_stream
def lensing_maps(theta_x, theta_y, sie=None, shear=None, tnfw=None, stream=None):
    """jt_lensing_maps: (kappa, gamma1, gamma2, mu) of SIE + shear + TNFW at the given points."""
    _dev(theta_x, "theta_x"), _dev(theta_y, "theta_y")
    code = _dt(theta_x)
    L = _lens(code, sie, shear, tnfw)
    out = [torch.empty_like(theta_x) for _ in range(4)]
    _check(lib().jt_lensing_maps(code, theta_x.numel(), _ptr(theta_x), _ptr(theta_y), ctypes.byref(L), _ptr(out[0]), _ptr(out[1]),
                                 _ptr(out[2]), _ptr(out[3]), _stream(stream)), "jt_lensing_maps")
    return tuple(out)


DEFLECTOR_TYPES = {"CONVERGENCE": 0, "SIS": 1, "NFW": 2, "HERNQUIST": 3, "PJAFFE": 4, "SIE": 5, "SHEAR": 6, "TNFW": 7,
                   "NIE": 8, "EPL": 9, "MULTIPOLE": 10, "CSE": 11, "PJAFFE_ELLIPSE_POTENTIAL": 12}
LIGHT_TYPES = {"SERSIC_ELLIPSE": 0, "GAUSSIAN_ELLIPSE": 1}
_PROFILE_DT = np.dtype([("type", np.int32), ("reserved", np.int32), ("p", np.float64, 8)])     # jt_profile, 72 bytes


def profile_records(records, table, device="cuda"):
    """[(name, [params...]), ...] -> device array of jt_profile (a uint8 tensor of 72-byte records)."""
    a = np.zeros(len(records), dtype=_PROFILE_DT)
    for k, (name, p) in enumerate(records):
        a[k]["type"] = table[name]
        a[k]["p"][:len(p)] = p
    return torch.as_tensor(a.view(np.uint8).reshape(-1).copy(), device=device)


@_on_stream
def ray_shoot_profiles(theta_x, theta_y, deflectors, stream=None):
    """jt_ray_shoot_profiles: beta = theta - sum of typed deflectors [(name, params), ...] (or a profile_records tensor)."""
    _dev(theta_x, "theta_x"), _dev(theta_y, "theta_y")
    code = _dt(theta_x)
    recs = deflectors if isinstance(deflectors, torch.Tensor) else profile_records(deflectors, DEFLECTOR_TYPES, theta_x.device)
    bx, by = torch.empty_like(theta_x), torch.empty_like(theta_y)
    _check(lib().jt_ray_shoot_profiles(code, theta_x.numel(), _ptr(theta_x), _ptr(theta_y), recs.numel() // 72,
                                       _ptr(recs) if recs.numel() else None, _ptr(bx), _ptr(by), _stream(stream)),
           "jt_ray_shoot_profiles")
    return bx, by


@_on_stream
def light_profiles(beta_x, beta_y, components, stream=None):
    """jt_light_profiles: sum of typed light components [(name, params), ...] at (beta_x, beta_y)."""
    _dev(beta_x, "beta_x"), _dev(beta_y, "beta_y")
    code = _dt(beta_x)
    recs = components if isinstance(components, torch.Tensor) else profile_records(components, LIGHT_TYPES, beta_x.device)
    flux = torch.empty_like(beta_x)
    _check(lib().jt_light_profiles(code, beta_x.numel(), _ptr(beta_x), _ptr(beta_y), recs.numel() // 72,
                                   _ptr(recs) if recs.numel() else None, _ptr(flux), _stream(stream)), "jt_light_profiles")
    return flux


@_on_stream
def light_core_sersic(beta_x, beta_y, params, stream=None):
    """jt_light_core_sersic: params = (amp, R_sersic, n_sersic, Rb, gamma, alpha, e1, e2, cx, cy)."""
    _dev(beta_x, "beta_x"), _dev(beta_y, "beta_y")
    p = (ctypes.c_double * 10)(*[float(v) for v in params])
    flux = torch.empty_like(beta_x)
    _check(lib().jt_light_core_sersic(_dt(beta_x), beta_x.numel(), _ptr(beta_x), _ptr(beta_y), p, _ptr(flux), _stream(stream)),
           "jt_light_core_sersic")
    return flux


@_on_stream
def light_shapelets(beta_x, beta_y, n_max, beta, cx, cy, coef, stream=None):
    """jt_light_shapelets: coef is a device tensor [(n_max+1)(n_max+2)/2] of the call's dtype (N ascending, n2 = 0..N)."""
    _dev(beta_x, "beta_x"), _dev(beta_y, "beta_y"), _dev(coef, "coef")
    if _dt(coef) != _dt(beta_x) or coef.numel() != (n_max + 1) * (n_max + 2) // 2:
        raise TypeError("coef: wrong dtype or length")
    flux = torch.empty_like(beta_x)
    _check(lib().jt_light_shapelets(_dt(beta_x), beta_x.numel(), _ptr(beta_x), _ptr(beta_y), int(n_max), float(beta), float(cx),
                                    float(cy), _ptr(coef), _ptr(flux), _stream(stream)), "jt_light_shapelets")
    return flux


@_on_stream
def simulate_image_supersampled_psf(grid, sie, shear, tnfw, sources, psf_fine, dtype=None, method="auto", workspace=None, out=None,
                                    stream=None):
    """jt_simulate_image_supersampled_psf (NEXT-4): psf_fine is sampled on the RAY grid [ky][kx]."""
    _dev(psf_fine, "psf_fine")
    code = _code(dtype) if dtype is not None else _dt(psf_fine)
    g = grid._c()
    L = _lens(code, sie, shear, tnfw)
    S, keep = _sources(sources)
    ky, kx = psf_fine.shape
    nb = int(lib().jt_simulate_image_supersampled_psf_workspace_bytes(code, ctypes.byref(g), L.n_tnfw, ky, kx, _METHODS[method]))
    ws, wsb = _workspace(nb, psf_fine.device, workspace, stream)
    if out is None:
        out = torch.empty((grid.ny, grid.nx), dtype=_torch_dtype(code), device=psf_fine.device)
    _check(lib().jt_simulate_image_supersampled_psf(code, ctypes.byref(g), ctypes.byref(L), ctypes.byref(S), ky, kx, _ptr(psf_fine),
                                                    _METHODS[method], _ptr(ws), wsb, _ptr(out), _stream(stream)),
           "jt_simulate_image_supersampled_psf")
    del keep
    return out
