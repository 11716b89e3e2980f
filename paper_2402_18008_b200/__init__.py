"""paper_2402_18008_b200 -- thin Python binding of libhg (include/hg.h).

Batched minimal 4-point homography by the ACA and SKS decompositions of arXiv 2402.18008 on one
B200.  Every function below only marshals arguments (torch tensors -> device pointers, the
current CUDA stream -> ``cuda_stream``) and calls the C entry point of the same name; all
arithmetic runs in the hand-written sm_100a kernels of ``csrc/``.  There is no CPU or PyTorch
fallback: if ``libhg.so`` cannot be built/loaded, or a tensor is not where the entry point expects
it, the call raises.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import torch

from . import _build

__all__ = [
    "HgError", "lib", "lib_path", "SOA", "AOS", "NORM_NONE", "NORM_H33", "NORM_FROBENIUS",
    "PREC_F64", "PREC_F32", "hg_aca_batched", "hg_sks_batched", "hg_aca_batched_host",
    "hg_sks_batched_host", "hg_offsets_to_grid", "hg_offsets_to_warp", "hg_aca_rect_batched", "hg_aca_rect_backward", "hg_aca_rect_backward_soa",
    "hg_affine_batched", "hg_sk_batched", "hg_aca_batched_f64", "hg_sks_batched_f64",
    "hg_ransac_workspace_bytes", "hg_ransac_hypothesize_score", "hg_ransac_hypothesize_score_host", "hg_ransac_adaptive",
    "hg_ransac_hypothesize_score_ex", "hg_ransac_adaptive_ex", "RANSAC_REJECT_DEGENERATE", "RANSAC_DECIDE_ALL_F64",
    "hg_ransac_hypothesize_score_noalloc", "RANSAC_NOALLOC_MAX_PTS", "RANSAC_NOALLOC_MAX_HYP",
    "hg_status_string", "hg_version", "hg_built_for_sm", "EXPORTS",
]

# include/hg.h enums
HG_OK = 0
SOA, AOS = 0, 1
NORM_NONE, NORM_H33, NORM_FROBENIUS = 0, 1, 2
PREC_F64, PREC_F32 = 0, 1
RANSAC_STAT_WORDS = 6
RANSAC_REJECT_DEGENERATE, RANSAC_DECIDE_ALL_F64 = 1, 2
HG_ERR_TOO_LARGE = -5
RANSAC_NOALLOC_MAX_PTS, RANSAC_NOALLOC_MAX_HYP = 4096, 9472

# every symbol include/hg.h declares
EXPORTS = [
    "hg_aca_batched", "hg_sks_batched", "hg_aca_batched_host", "hg_sks_batched_host",
    "hg_offsets_to_grid", "hg_offsets_to_warp", "hg_aca_rect_batched", "hg_aca_rect_backward", "hg_aca_rect_backward_soa", "hg_offsets_to_grid_backward", "hg_affine_batched",
    "hg_sk_batched", "hg_aca_batched_f64", "hg_sks_batched_f64", "hg_ransac_workspace_bytes", "hg_ransac_hypothesize_score",
    "hg_ransac_hypothesize_score_host", "hg_ransac_adaptive", "hg_ransac_hypothesize_score_ex", "hg_ransac_adaptive_ex",
    "hg_ransac_hypothesize_score_noalloc", "hg_status_string", "hg_version", "hg_built_for_sm",
]


class _RansacOptions(ctypes.Structure):
    """hg_ransac_options_t"""
    _fields_ = [("flags", ctypes.c_uint32), ("min_area_px2", ctypes.c_float)]


class HgError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        super().__init__("%s failed: %s (%d)" % (where, hg_status_string(status), status))


_lib = None
_c_int, _c_i32, _c_i64, _c_f32 = ctypes.c_int, ctypes.c_int32, ctypes.c_int64, ctypes.c_float
_vp = ctypes.c_void_p


def lib_path() -> Path:
    return _build.LIB


def lib() -> ctypes.CDLL:
    """Load libhg.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(str(path))
        solve_args = [_vp, _vp, _vp, _c_i64, _c_int, _c_int, _c_int, _vp]
        L.hg_aca_batched.argtypes = solve_args
        L.hg_sks_batched.argtypes = solve_args
        host_args = [_vp, _vp, _vp, _c_i64, _c_int, _c_int, _c_int, _c_i64]
        L.hg_aca_batched_host.argtypes = host_args
        L.hg_sks_batched_host.argtypes = host_args
        L.hg_offsets_to_grid.argtypes = [_vp, _c_f32, _c_f32, _c_f32, _c_f32, _c_i32, _c_i32, _vp, _vp,
                                         _c_i64, _c_int, _vp]
        L.hg_aca_rect_batched.argtypes = [_vp, _c_f32, _c_f32, _c_f32, _c_f32, _vp, _c_i64, _c_int, _c_int, _c_int, _vp]
        L.hg_aca_rect_backward.argtypes = [_vp, _c_f32, _c_f32, _c_f32, _c_f32, _vp, _vp, _c_i64, _vp]
        L.hg_aca_rect_backward_soa.argtypes = [_vp, _c_f32, _c_f32, _c_f32, _c_f32, _vp, _vp, _c_i64, _vp]
        L.hg_offsets_to_grid_backward.argtypes = [_vp, _c_f32, _c_f32, _c_f32, _c_f32, _c_i32, _c_i32, _vp, _vp, _vp, _c_i64, _vp]
        L.hg_offsets_to_warp.argtypes = [_vp, _c_f32, _c_f32, _c_f32, _c_f32, _c_i32, _c_i32, _vp, _c_i32, _c_i32, _c_i32,
                                         _vp, _vp, _c_i64, _c_int, _vp]
        L.hg_affine_batched.argtypes = solve_args
        _c_f64 = ctypes.c_double
        L.hg_sk_batched.argtypes = [_c_f64, _c_f64, _c_f64, _c_f64, _vp, _vp, _c_i64, _c_int, _c_int, _c_int, _vp]
        L.hg_aca_batched_f64.argtypes = [_vp, _vp, _vp, _c_i64, _c_int, _c_int, _vp]
        L.hg_sks_batched_f64.argtypes = [_vp, _vp, _vp, _c_i64, _c_int, _c_int, _vp]
        L.hg_ransac_workspace_bytes.argtypes = [_c_i32, _c_i64]
        L.hg_ransac_workspace_bytes.restype = ctypes.c_size_t
        L.hg_ransac_hypothesize_score.argtypes = [_vp, _vp, _c_i32, _vp, _c_i64, _c_f32, _vp, _vp, _vp, _vp,
                                                  _vp, ctypes.c_size_t, _vp]
        L.hg_ransac_hypothesize_score_ex.argtypes = [_vp, _vp, _c_i32, _vp, _c_i64, _c_f32, _vp, _vp, _vp, _vp, _vp,
                                                     _vp, ctypes.c_size_t, _vp]
        L.hg_ransac_adaptive.argtypes = [_vp, _vp, _c_i32, ctypes.c_uint64, _c_i64, _c_i64, _c_f32, _c_f32, _vp, _vp, _vp, _vp, _vp,
                                         _vp, _vp, ctypes.c_size_t, _vp]
        L.hg_ransac_adaptive_ex.argtypes = [_vp, _vp, _c_i32, ctypes.c_uint64, _c_i64, _c_i64, _c_f32, _c_f32, _vp, _vp, _vp, _vp, _vp,
                                            _vp, _vp, _vp, ctypes.c_size_t, _vp]
        L.hg_ransac_hypothesize_score_host.argtypes = [_vp, _vp, _c_i32, _vp, _c_i64, _c_f32, _vp, _vp, _vp, _vp]
        L.hg_ransac_hypothesize_score_noalloc.argtypes = [_vp, _vp, _c_i32, _vp, _c_i64, _c_f32, _vp, _vp, _vp, _vp, _vp]
        L.hg_status_string.argtypes = [_c_int]
        L.hg_status_string.restype = ctypes.c_char_p
        for name in ("hg_aca_batched", "hg_sks_batched", "hg_aca_batched_host", "hg_sks_batched_host",
                     "hg_offsets_to_grid", "hg_offsets_to_warp", "hg_aca_rect_batched", "hg_aca_rect_backward",
                     "hg_aca_rect_backward_soa", "hg_offsets_to_grid_backward", "hg_affine_batched", "hg_sk_batched", "hg_aca_batched_f64", "hg_sks_batched_f64",
                     "hg_ransac_hypothesize_score", "hg_ransac_hypothesize_score_host", "hg_ransac_adaptive",
                     "hg_ransac_hypothesize_score_ex", "hg_ransac_adaptive_ex", "hg_ransac_hypothesize_score_noalloc",
                     "hg_version", "hg_built_for_sm"):
            getattr(L, name).restype = _c_int
        _lib = L
    return _lib


def hg_status_string(status: int) -> str:
    return lib().hg_status_string(int(status)).decode()


def hg_version() -> int:
    return int(lib().hg_version())


def hg_built_for_sm() -> int:
    return int(lib().hg_built_for_sm())


# ---- recorded calls: the latency path without the marshalling ---------------------------------------
_plan = None          # the CallPlan being recorded, if any


class CallPlan:
    """Records the C calls the binding makes inside `with hg.CallPlan() as plan:` -- function, pointers, sizes, stream, as
    marshalled and checked once -- and re-issues exactly those calls on `plan()`.  For loops that call the library on the
    same buffers every iteration (the paper's Table 6 / Table 7 regime): a 1 us kernel then costs a ctypes call, not the
    8 us of tensor checks and conversions.  The plan holds a reference to every tensor whose address it recorded (the caller's
    and the ones the wrappers allocated: outputs, workspaces), so dropping a returned dict cannot hand that memory to another
    tensor while the plan lives; each call is replayed with the device that was current when it was recorded, on the stream
    that was current then.  One plan is recorded at a time, by one thread.  (A CUDA graph of the same calls is cheaper still;
    this needs no capture.)"""

    def __init__(self):
        self._calls = []
        self._keep = []

    def __enter__(self):
        global _plan
        if _plan is not None:
            raise RuntimeError("a CallPlan is already being recorded")
        _plan = self
        return self

    def __exit__(self, *exc):
        global _plan
        _plan = None
        return False

    def __len__(self):
        return len(self._calls)

    def __call__(self):
        for f, args, name, dev in self._calls:
            if dev != torch.cuda.current_device():
                with torch.cuda.device(dev):
                    st = f(*args)
            else:
                st = f(*args)
            if st != HG_OK:
                raise HgError(st, name)


def _c(name: str):
    """The C entry point `name`; while a CallPlan is being recorded, a wrapper that also notes the call."""
    f = getattr(lib(), name)
    if _plan is None:
        return f
    plan = _plan

    def recorded(*args):
        plan._calls.append((f, args, name, torch.cuda.current_device()))     # (called inside `with _on(dev)`)
        return f(*args)
    return recorded


# ---- argument marshalling -----------------------------------------------------------------------
def _ptr(t, dtype, device_type: str, name: str):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor):
        raise TypeError("%s must be a torch.Tensor" % name)
    if t.dtype != dtype:
        raise TypeError("%s must be %s, got %s" % (name, dtype, t.dtype))
    if t.device.type != device_type:
        raise ValueError("%s must live on %s, got %s (no fallback path exists)" % (name, device_type, t.device))
    if not t.is_contiguous():
        raise ValueError("%s must be contiguous" % name)
    if _plan is not None:
        _plan._keep.append(t)             # a recorded call holds this address: the plan keeps the tensor alive
    return _vp(t.data_ptr())


_raw_stream = getattr(torch._C, "_cuda_getCurrentRawStream", None)


def _stream(stream=None):
    """cudaStream_t of `stream`, or of torch's current stream on the current device (the cheap raw query when torch has it)."""
    if stream is None:
        if _raw_stream is not None:
            return _vp(int(_raw_stream(torch.cuda.current_device())))
        stream = torch.cuda.current_stream()
    return _vp(int(stream.cuda_stream))


def _same_device(*tensors):
    """Every device tensor of one call must live on one GPU: the kernels dereference all of them on the first one's device."""
    dev = None
    for x in tensors:
        if x is None or not isinstance(x, torch.Tensor):
            continue
        if dev is None:
            dev = x.device
        elif x.device != dev:
            raise ValueError("all tensors of a call must be on one device, got %s and %s" % (dev, x.device))
    return dev


class _NoCtx:
    def __enter__(self):
        return None

    def __exit__(self, *a):
        return False


_NOCTX = _NoCtx()


def _on(device):
    """Context that makes `device` current; free when it already is (the common case on the latency-bound C1 path)."""
    idx = device.index
    if idx is None or idx == torch.cuda.current_device():
        return _NOCTX
    return torch.cuda.device(device)


def _check(status: int, where: str):
    if status != HG_OK:
        raise HgError(status, where)


def _n_sets(src: torch.Tensor, layout: int) -> int:
    if layout == SOA:
        if src.dim() != 2 or src.shape[0] != 8:
            raise ValueError("SoA point sets are float32 [8, n]")
        return int(src.shape[1])
    if src.dim() != 3 or tuple(src.shape[1:]) != (4, 2):
        raise ValueError("AoS point sets are float32 [n, 4, 2]")
    return int(src.shape[0])


def _h_shape(n: int, layout: int):
    return (9, n) if layout == SOA else (n, 3, 3)


def _solve(fn_name: str, src, dst, H, layout, norm, prec, stream):
    n = _n_sets(src, layout)
    if tuple(dst.shape) != tuple(src.shape):
        raise ValueError("src and dst shapes differ")
    if H is None:
        H = torch.empty(_h_shape(n, layout), dtype=torch.float32, device=src.device)
    elif tuple(H.shape) != _h_shape(n, layout):
        raise ValueError("H must have shape %s" % (_h_shape(n, layout),))
    fn = _c(fn_name)
    ps, pd, ph = (_ptr(src, torch.float32, "cuda", "src"), _ptr(dst, torch.float32, "cuda", "dst"),
                  _ptr(H, torch.float32, "cuda", "H"))
    _same_device(src, dst, H)
    with _on(src.device):
        st = fn(ps, pd, ph, n, int(layout), int(norm), int(prec), _stream(stream))
    _check(st, fn_name)
    return H


def hg_aca_batched(src, dst, H=None, layout: int = SOA, norm: int = NORM_NONE, prec: int = PREC_F64,
                   stream=None) -> torch.Tensor:
    """ACA solve of n sets on the current device/stream.  SoA: src, dst [8,n] -> H [9,n];
    AoS: [n,4,2] -> [n,3,3].  Returns H (allocated if not given).  Asynchronous."""
    return _solve("hg_aca_batched", src, dst, H, layout, norm, prec, stream)


def hg_sks_batched(src, dst, H=None, layout: int = SOA, norm: int = NORM_NONE, prec: int = PREC_F64,
                   stream=None) -> torch.Tensor:
    """SKS solve; same contract as hg_aca_batched."""
    return _solve("hg_sks_batched", src, dst, H, layout, norm, prec, stream)


def _solve_host(fn_name: str, src, dst, H, layout, norm, prec, chunk_sets):
    n = _n_sets(src, layout)
    if tuple(dst.shape) != tuple(src.shape):
        raise ValueError("src and dst shapes differ")
    if H is None:
        H = torch.empty(_h_shape(n, layout), dtype=torch.float32, pin_memory=True)
    elif tuple(H.shape) != _h_shape(n, layout):
        raise ValueError("H must have shape %s" % (_h_shape(n, layout),))
    st = _c(fn_name)(_ptr(src, torch.float32, "cpu", "src"), _ptr(dst, torch.float32, "cpu", "dst"),
                                 _ptr(H, torch.float32, "cpu", "H"), n, int(layout), int(norm), int(prec),
                                 int(chunk_sets))
    _check(st, fn_name)
    return H


def hg_aca_batched_host(src, dst, H=None, layout: int = SOA, norm: int = NORM_NONE, prec: int = PREC_F64,
                        chunk_sets: int = 0) -> torch.Tensor:
    """Host-buffer ACA solve (CPU tensors, ideally pinned): chunked H2D -> kernel -> D2H pipeline
    inside the library on the current CUDA device.  Synchronous."""
    return _solve_host("hg_aca_batched_host", src, dst, H, layout, norm, prec, chunk_sets)


def hg_sks_batched_host(src, dst, H=None, layout: int = SOA, norm: int = NORM_NONE, prec: int = PREC_F64,
                        chunk_sets: int = 0) -> torch.Tensor:
    return _solve_host("hg_sks_batched_host", src, dst, H, layout, norm, prec, chunk_sets)


def hg_offsets_to_grid(offsets, x0: float, y0: float, w: float, h: float, grid_w: int, grid_h: int,
                       want_H: bool = True, want_grid: bool = True, H=None, grid=None,
                       norm: int = NORM_H33, stream=None):
    """offsets float32 [n,4,2] (corners TL,TR,BR,BL) -> (H [n,3,3] or None, grid [n,grid_h,grid_w,2] or None)."""
    if offsets.dim() != 3 or tuple(offsets.shape[1:]) != (4, 2):
        raise ValueError("offsets are float32 [n, 4, 2]")
    n = int(offsets.shape[0])
    po = _ptr(offsets, torch.float32, "cuda", "offsets")
    if want_H and H is None:
        H = torch.empty((n, 3, 3), dtype=torch.float32, device=offsets.device)
    if want_grid and grid is None:
        grid = torch.empty((n, grid_h, grid_w, 2), dtype=torch.float32, device=offsets.device)
    if H is not None and tuple(H.shape) != (n, 3, 3):
        raise ValueError("H must be [n,3,3]")
    if grid is not None and tuple(grid.shape) != (n, grid_h, grid_w, 2):
        raise ValueError("grid must be [n,grid_h,grid_w,2]")
    _same_device(offsets, H, grid)
    with _on(offsets.device):
        st = _c("hg_offsets_to_grid")(po, x0, y0, w, h,
                                      int(grid_w), int(grid_h), _ptr(H, torch.float32, "cuda", "H"),
                                      _ptr(grid, torch.float32, "cuda", "grid"), n, int(norm), _stream(stream))
    _check(st, "hg_offsets_to_grid")
    return H, grid


def hg_offsets_to_warp(offsets, x0: float, y0: float, w: float, h: float, out_w: int, out_h: int, image,
                       warped=None, want_H: bool = False, norm: int = NORM_H33, stream=None):
    """offsets [n,4,2] + image [n,C,img_h,img_w] -> (warped [n,C,out_h,out_w], H [n,3,3] or None)."""
    if offsets.dim() != 3 or tuple(offsets.shape[1:]) != (4, 2):
        raise ValueError("offsets are float32 [n, 4, 2]")
    n = int(offsets.shape[0])
    if image.dim() != 4 or image.shape[0] != n:
        raise ValueError("image is float32 [n, C, img_h, img_w]")
    C, ih, iw = int(image.shape[1]), int(image.shape[2]), int(image.shape[3])
    if warped is None:
        warped = torch.empty((n, C, out_h, out_w), dtype=torch.float32, device=offsets.device)
    elif tuple(warped.shape) != (n, C, out_h, out_w):
        raise ValueError("warped must be [n,C,out_h,out_w]")
    H = torch.empty((n, 3, 3), dtype=torch.float32, device=offsets.device) if want_H else None
    _same_device(offsets, image, warped, H)
    with _on(offsets.device):
        st = _c("hg_offsets_to_warp")(_ptr(offsets, torch.float32, "cuda", "offsets"), x0, y0, w, h, int(out_w), int(out_h),
                                      _ptr(image, torch.float32, "cuda", "image"), C, iw, ih,
                                      _ptr(warped, torch.float32, "cuda", "warped"), _ptr(H, torch.float32, "cuda", "H"),
                                      n, int(norm), _stream(stream))
    _check(st, "hg_offsets_to_warp")
    return warped, H


def hg_aca_rect_batched(offsets, x0: float, y0: float, w: float, h: float, H=None, layout: int = AOS,
                        norm: int = NORM_NONE, prec: int = PREC_F64, stream=None) -> torch.Tensor:
    """Algorithm 1 (rectangular source).  AoS: offsets [n,4,2] -> H [n,3,3]; SoA: [8,n] -> [9,n]."""
    n = _n_sets(offsets, layout)
    if H is None:
        H = torch.empty(_h_shape(n, layout), dtype=torch.float32, device=offsets.device)
    elif tuple(H.shape) != _h_shape(n, layout):
        raise ValueError("H must have shape %s" % (_h_shape(n, layout),))
    po, ph = _ptr(offsets, torch.float32, "cuda", "offsets"), _ptr(H, torch.float32, "cuda", "H")
    _same_device(offsets, H)
    with _on(offsets.device):
        st = _c("hg_aca_rect_batched")(po, x0, y0, w, h, ph, n, int(layout), int(norm), int(prec), _stream(stream))
    _check(st, "hg_aca_rect_batched")
    return H


def hg_aca_rect_backward(offsets, x0: float, y0: float, w: float, h: float, grad_H, grad_offsets=None,
                         stream=None) -> torch.Tensor:
    """dL/d offsets [n,4,2] of G = H/h33 (Algorithm 1) given dL/dG [n,3,3]."""
    n = _n_sets(offsets, AOS)
    if tuple(grad_H.shape) != (n, 3, 3):
        raise ValueError("grad_H must be [n,3,3]")
    if grad_offsets is None:
        grad_offsets = torch.empty((n, 4, 2), dtype=torch.float32, device=offsets.device)
    elif tuple(grad_offsets.shape) != (n, 4, 2):
        raise ValueError("grad_offsets must be [n,4,2]")
    po, pg, pr = (_ptr(offsets, torch.float32, "cuda", "offsets"), _ptr(grad_H, torch.float32, "cuda", "grad_H"),
                  _ptr(grad_offsets, torch.float32, "cuda", "grad_offsets"))
    _same_device(offsets, grad_H, grad_offsets)
    with _on(offsets.device):
        st = _c("hg_aca_rect_backward")(po, x0, y0, w, h, pg, pr, n, _stream(stream))
    _check(st, "hg_aca_rect_backward")
    return grad_offsets


def hg_aca_rect_backward_soa(offsets, x0: float, y0: float, w: float, h: float, grad_H, grad_offsets=None,
                             stream=None) -> torch.Tensor:
    """The backward pass on planes: offsets [8,n], grad_H [9,n] -> grad_offsets [8,n]."""
    n = _n_sets(offsets, SOA)
    if tuple(grad_H.shape) != (9, n):
        raise ValueError("grad_H must be [9,n]")
    if grad_offsets is None:
        grad_offsets = torch.empty((8, n), dtype=torch.float32, device=offsets.device)
    elif tuple(grad_offsets.shape) != (8, n):
        raise ValueError("grad_offsets must be [8,n]")
    po, pg, pr = (_ptr(offsets, torch.float32, "cuda", "offsets"), _ptr(grad_H, torch.float32, "cuda", "grad_H"),
                  _ptr(grad_offsets, torch.float32, "cuda", "grad_offsets"))
    _same_device(offsets, grad_H, grad_offsets)
    with _on(offsets.device):
        st = _c("hg_aca_rect_backward_soa")(po, x0, y0, w, h, pg, pr, n, _stream(stream))
    _check(st, "hg_aca_rect_backward_soa")
    return grad_offsets


def _n_generic(t: torch.Tensor, layout: int, scalars: int, what: str) -> int:
    if layout == SOA:
        if t.dim() != 2 or t.shape[0] != scalars:
            raise ValueError("SoA %s are [%d, n]" % (what, scalars))
        return int(t.shape[1])
    if t.dim() != 3 or tuple(t.shape[1:]) != (scalars // 2, 2):
        raise ValueError("AoS %s are [n, %d, 2]" % (what, scalars // 2))
    return int(t.shape[0])


def hg_offsets_to_grid_backward(offsets, x0: float, y0: float, w: float, h: float, grad_grid, grad_offsets=None,
                                want_grad_G: bool = False, stream=None):
    """Backward of hg_offsets_to_grid: offsets float32 [n,4,2], grad_grid float32 [n,grid_h,grid_w,2] (GPU) ->
    grad_offsets float32 [n,4,2] (and, if want_grad_G, dL/dG [n,3,3] for G = H/h33 as a second return value)."""
    n = int(offsets.shape[0])
    if tuple(offsets.shape) != (n, 4, 2):
        raise ValueError("offsets are float32 [n, 4, 2]")
    if grad_grid.dim() != 4 or int(grad_grid.shape[0]) != n or int(grad_grid.shape[3]) != 2:
        raise ValueError("grad_grid is float32 [n, grid_h, grid_w, 2]")
    gh, gw = int(grad_grid.shape[1]), int(grad_grid.shape[2])
    if grad_offsets is None:
        grad_offsets = torch.empty((n, 4, 2), dtype=torch.float32, device=offsets.device)
    elif tuple(grad_offsets.shape) != (n, 4, 2):
        raise ValueError("grad_offsets must have shape [n, 4, 2]")
    gG = torch.empty((n, 3, 3), dtype=torch.float32, device=offsets.device) if want_grad_G else None
    po, pg, pr, pG = (_ptr(offsets, torch.float32, "cuda", "offsets"), _ptr(grad_grid, torch.float32, "cuda", "grad_grid"),
                      _ptr(grad_offsets, torch.float32, "cuda", "grad_offsets"), _ptr(gG, torch.float32, "cuda", "grad_G"))
    _same_device(offsets, grad_grid, grad_offsets, gG)
    with _on(offsets.device):
        st = _c("hg_offsets_to_grid_backward")(po, x0, y0, w, h, gw, gh, pg, pr, pG, n, _stream(stream))
    _check(st, "hg_offsets_to_grid_backward")
    return (grad_offsets, gG) if want_grad_G else grad_offsets


def hg_affine_batched(src3, dst3, H=None, layout: int = SOA, norm: int = NORM_NONE, prec: int = PREC_F64,
                      stream=None) -> torch.Tensor:
    """Affine H_A from three correspondences (Eq. 41).  SoA: [6,n] x2 -> [9,n]; AoS: [n,3,2] x2 -> [n,3,3]."""
    n = _n_generic(src3, layout, 6, "3-point sets")
    if tuple(dst3.shape) != tuple(src3.shape):
        raise ValueError("src3 and dst3 shapes differ")
    if H is None:
        H = torch.empty(_h_shape(n, layout), dtype=torch.float32, device=src3.device)
    elif tuple(H.shape) != _h_shape(n, layout):
        raise ValueError("H must have shape %s" % (_h_shape(n, layout),))
    ps, pd, ph = (_ptr(src3, torch.float32, "cuda", "src3"), _ptr(dst3, torch.float32, "cuda", "dst3"),
                  _ptr(H, torch.float32, "cuda", "H"))
    _same_device(src3, dst3, H)
    with _on(src3.device):
        st = _c("hg_affine_batched")(ps, pd, ph, n, int(layout), int(norm), int(prec), _stream(stream))
    _check(st, "hg_affine_batched")
    return H


def hg_sk_batched(P3, Q3, dst, H=None, layout: int = SOA, norm: int = NORM_NONE, prec: int = PREC_F64,
                  stream=None) -> torch.Tensor:
    """Simplified SK (Eq. 17): pattern points P3, Q3 = (x, y) in the anchor frame; dst as hg_aca_batched's dst."""
    n = _n_sets(dst, layout)
    if H is None:
        H = torch.empty(_h_shape(n, layout), dtype=torch.float32, device=dst.device)
    elif tuple(H.shape) != _h_shape(n, layout):
        raise ValueError("H must have shape %s" % (_h_shape(n, layout),))
    pd, ph = _ptr(dst, torch.float32, "cuda", "dst"), _ptr(H, torch.float32, "cuda", "H")
    _same_device(dst, H)
    with _on(dst.device):
        st = _c("hg_sk_batched")(float(P3[0]), float(P3[1]), float(Q3[0]), float(Q3[1]), pd, ph, n, int(layout),
                                 int(norm), int(prec), _stream(stream))
    _check(st, "hg_sk_batched")
    return H


def _solve_f64(fn_name: str, src, dst, H, layout, norm, stream):
    n = _n_sets(src, layout)
    if tuple(dst.shape) != tuple(src.shape):
        raise ValueError("src and dst shapes differ")
    if H is None:
        H = torch.empty(_h_shape(n, layout), dtype=torch.float64, device=src.device)
    elif tuple(H.shape) != _h_shape(n, layout):
        raise ValueError("H must have shape %s" % (_h_shape(n, layout),))
    ps, pd, ph = (_ptr(src, torch.float64, "cuda", "src"), _ptr(dst, torch.float64, "cuda", "dst"),
                  _ptr(H, torch.float64, "cuda", "H"))
    _same_device(src, dst, H)
    with _on(src.device):
        st = _c(fn_name)(ps, pd, ph, n, int(layout), int(norm), _stream(stream))
    _check(st, fn_name)
    return H


def hg_aca_batched_f64(src, dst, H=None, layout: int = SOA, norm: int = NORM_NONE, stream=None) -> torch.Tensor:
    """ACA with float64 storage (the paper's GPU precision)."""
    return _solve_f64("hg_aca_batched_f64", src, dst, H, layout, norm, stream)


def hg_sks_batched_f64(src, dst, H=None, layout: int = SOA, norm: int = NORM_NONE, stream=None) -> torch.Tensor:
    return _solve_f64("hg_sks_batched_f64", src, dst, H, layout, norm, stream)


def hg_ransac_workspace_bytes(n_pts: int, n_hyp: int) -> int:
    return int(lib().hg_ransac_workspace_bytes(int(n_pts), int(n_hyp)))


def _ransac_options(reject_degenerate, min_area_px2, decide_all_f64):
    """(hg_ransac_options_t or None): None when every option is at its default, so the plain entry point is called."""
    flags = (RANSAC_REJECT_DEGENERATE if reject_degenerate else 0) | (RANSAC_DECIDE_ALL_F64 if decide_all_f64 else 0)
    if not flags:
        return None
    return _RansacOptions(flags, float(min_area_px2))


def hg_ransac_hypothesize_score(src_xy, dst_xy, hyp_idx, threshold_px: float, counts=None, workspace=None,
                                want_counts: bool = True, stream=None, reject_degenerate: bool = False,
                                min_area_px2: float = 0.0, decide_all_f64: bool = False, best=None):
    """src_xy, dst_xy float32 [n_pts,2]; hyp_idx int32 [n_hyp,4] (all on the GPU).
    Returns dict(counts int32 [n_hyp] or None, best_H float32 [3,3], best_index int64 [1],
    best_count int32 [1], workspace uint8) -- device tensors, produced asynchronously.
    best: optional (best_H [3,3] f32, best_index [1] i64, best_count [1] i32) tensors to write into.
    reject_degenerate / min_area_px2 / decide_all_f64: hg_ransac_options_t (the call goes through
    hg_ransac_hypothesize_score_ex when any is set)."""
    n_pts, n_hyp = int(src_xy.shape[0]), int(hyp_idx.shape[0])
    if tuple(src_xy.shape) != (n_pts, 2) or tuple(dst_xy.shape) != (n_pts, 2):
        raise ValueError("src_xy, dst_xy are float32 [n_pts, 2]")
    if tuple(hyp_idx.shape) != (n_hyp, 4):
        raise ValueError("hyp_idx is int32 [n_hyp, 4]")
    dev = src_xy.device
    _ptr(src_xy, torch.float32, "cuda", "src_xy")
    if want_counts and counts is None:
        counts = torch.empty((n_hyp,), dtype=torch.int32, device=dev)
    need = hg_ransac_workspace_bytes(n_pts, n_hyp)
    if workspace is None:
        workspace = torch.empty((max(need, 16),), dtype=torch.uint8, device=dev)
    if best is not None:          # (best_H, best_index, best_count) of an earlier call, reused: no allocation on the latency path
        best_H, best_index, best_count = best
    else:
        best_H = torch.empty((3, 3), dtype=torch.float32, device=dev)
        best_index = torch.empty((1,), dtype=torch.int64, device=dev)
        best_count = torch.empty((1,), dtype=torch.int32, device=dev)
    _same_device(src_xy, dst_xy, hyp_idx, counts, workspace, best_H, best_index, best_count)
    opt = _ransac_options(reject_degenerate, min_area_px2, decide_all_f64)
    if _plan is not None and opt is not None:
        _plan._keep.append(opt)                  # the recorded call holds a pointer into it
    head = (_ptr(src_xy, torch.float32, "cuda", "src_xy"), _ptr(dst_xy, torch.float32, "cuda", "dst_xy"), n_pts,
            _ptr(hyp_idx, torch.int32, "cuda", "hyp_idx"), n_hyp, float(threshold_px))
    tail = (_ptr(counts, torch.int32, "cuda", "counts"), _ptr(best_H, torch.float32, "cuda", "best_H"),
            _ptr(best_index, torch.int64, "cuda", "best_index"), _ptr(best_count, torch.int32, "cuda", "best_count"),
            _ptr(workspace, torch.uint8, "cuda", "workspace"), int(workspace.numel()))
    with _on(dev):
        tail = tail + (_stream(stream),)          # the current stream OF THE TENSORS' DEVICE
        if opt is None:
            st = _c("hg_ransac_hypothesize_score")(*head, *tail)
        else:
            st = _c("hg_ransac_hypothesize_score_ex")(*head, ctypes.cast(ctypes.pointer(opt), _vp), *tail)
    _check(st, "hg_ransac_hypothesize_score")
    return {"counts": counts, "best_H": best_H, "best_index": best_index, "best_count": best_count,
            "workspace": workspace}


hg_ransac_hypothesize_score_ex = hg_ransac_hypothesize_score      # one Python function serves both C entry points


def hg_ransac_hypothesize_score_noalloc(src_xy, dst_xy, hyp_idx, threshold_px: float, counts=None, best=None, stream=None):
    """hg_ransac_hypothesize_score without a workspace, for code that must not allocate device memory while it runs
    (called from inside another application's frame loop or memory pool, under a latency budget, or beside threads
    that are capturing streams): the scratch is a fixed 28 KB array inside libhg, so the limits are
    n_pts <= RANSAC_NOALLOC_MAX_PTS (4096) and n_hyp <= RANSAC_NOALLOC_MAX_HYP (9472); larger calls raise HgError
    with status HG_ERR_TOO_LARGE (-5).  In keeping with that, this wrapper creates no tensor either: every output is
    the caller's -- counts int32 [n_hyp] or None, best = (best_H [3,3] f32, best_index [1] i64, best_count [1] i32) or
    None -- and the return value is None.  Results equal those of hg_ransac_hypothesize_score.  All calls of one
    device share the one array: keep them on one stream (or ordered by events); calls that overlap on the GPU race.
    The first call on a device looks up the array's address; make it at start-up, outside any stream capture."""
    n_pts, n_hyp = int(src_xy.shape[0]), int(hyp_idx.shape[0])
    if tuple(src_xy.shape) != (n_pts, 2) or tuple(dst_xy.shape) != (n_pts, 2):
        raise ValueError("src_xy, dst_xy are float32 [n_pts, 2]")
    if tuple(hyp_idx.shape) != (n_hyp, 4):
        raise ValueError("hyp_idx is int32 [n_hyp, 4]")
    if counts is not None and counts.numel() < n_hyp:
        raise ValueError("counts is int32 [n_hyp]")
    best_H, best_index, best_count = best if best is not None else (None, None, None)
    dev = _same_device(src_xy, dst_xy, hyp_idx, counts, best_H, best_index, best_count)
    args = (_ptr(src_xy, torch.float32, "cuda", "src_xy"), _ptr(dst_xy, torch.float32, "cuda", "dst_xy"), n_pts,
            _ptr(hyp_idx, torch.int32, "cuda", "hyp_idx"), n_hyp, float(threshold_px),
            _ptr(counts, torch.int32, "cuda", "counts"), _ptr(best_H, torch.float32, "cuda", "best_H"),
            _ptr(best_index, torch.int64, "cuda", "best_index"), _ptr(best_count, torch.int32, "cuda", "best_count"))
    with _on(dev):
        st = _c("hg_ransac_hypothesize_score_noalloc")(*args, _stream(stream))
    _check(st, "hg_ransac_hypothesize_score_noalloc")


def hg_ransac_adaptive(src_xy, dst_xy, seed: int, max_hyp: int, round_hyp: int, threshold_px: float, confidence: float,
                       want_counts: bool = True, want_idx: bool = False, workspace=None, stream=None,
                       reject_degenerate: bool = False, min_area_px2: float = 0.0, decide_all_f64: bool = False):
    """On-device sampling (Philox4x32-10) + rounds + adaptive termination.  Returns dict(counts [max_hyp] or None,
    hyp_idx [max_hyp,4] or None, best_H [3,3], best_index [1], best_count [1], n_evaluated [1], workspace) -- device tensors."""
    n_pts = int(src_xy.shape[0])
    if tuple(src_xy.shape) != (n_pts, 2) or tuple(dst_xy.shape) != (n_pts, 2):
        raise ValueError("src_xy, dst_xy are float32 [n_pts, 2]")
    dev = src_xy.device
    need = hg_ransac_workspace_bytes(n_pts, max_hyp)
    if workspace is None:
        workspace = torch.empty((max(need, 16),), dtype=torch.uint8, device=dev)
    counts = torch.zeros((max_hyp,), dtype=torch.int32, device=dev) if want_counts else None
    idx = torch.zeros((max_hyp, 4), dtype=torch.int32, device=dev) if want_idx else None
    best_H = torch.empty((3, 3), dtype=torch.float32, device=dev)
    best_index = torch.empty((1,), dtype=torch.int64, device=dev)
    best_count = torch.empty((1,), dtype=torch.int32, device=dev)
    n_eval = torch.empty((1,), dtype=torch.int64, device=dev)
    _same_device(src_xy, dst_xy, workspace)
    opt = _ransac_options(reject_degenerate, min_area_px2, decide_all_f64)
    if _plan is not None:
        _plan._keep.extend([opt, counts, idx, best_H, best_index, best_count, n_eval, workspace])
    head = (_ptr(src_xy, torch.float32, "cuda", "src_xy"), _ptr(dst_xy, torch.float32, "cuda", "dst_xy"), n_pts,
            int(seed) & 0xFFFFFFFFFFFFFFFF, int(max_hyp), int(round_hyp), float(threshold_px), float(confidence))
    tail = (_ptr(counts, torch.int32, "cuda", "counts"), _ptr(idx, torch.int32, "cuda", "hyp_idx_out"),
            _ptr(best_H, torch.float32, "cuda", "best_H"), _ptr(best_index, torch.int64, "cuda", "best_index"),
            _ptr(best_count, torch.int32, "cuda", "best_count"), _ptr(n_eval, torch.int64, "cuda", "n_evaluated"),
            _ptr(workspace, torch.uint8, "cuda", "workspace"), int(workspace.numel()))
    with _on(dev):
        tail = tail + (_stream(stream),)          # the current stream OF THE TENSORS' DEVICE
        if opt is None:
            st = _c("hg_ransac_adaptive")(*head, *tail)
        else:
            st = _c("hg_ransac_adaptive_ex")(*head, ctypes.cast(ctypes.pointer(opt), _vp), *tail)
    _check(st, "hg_ransac_adaptive")
    return {"counts": counts, "hyp_idx": idx, "best_H": best_H, "best_index": best_index, "best_count": best_count,
            "n_evaluated": n_eval, "workspace": workspace}


hg_ransac_adaptive_ex = hg_ransac_adaptive


def ransac_stats(workspace: torch.Tensor) -> dict:
    """Decode the statistics words a finished hg_ransac_hypothesize_score call left in its workspace."""
    w = workspace[: 8 * RANSAC_STAT_WORDS].cpu().view(torch.int64)
    return {"best_key": int(w[0]), "n_fixup": int(w[1]), "n_pairs_f64": int(w[2]), "n_evaluated": int(w[3]),
            "n_rejected": int(w[4]), "n_band": int(w[5])}


def hg_ransac_hypothesize_score_host(src_xy, dst_xy, hyp_idx, threshold_px: float, want_counts: bool = True):
    """Host-buffer form (CPU tensors in, CPU tensors out); synchronous."""
    n_pts, n_hyp = int(src_xy.shape[0]), int(hyp_idx.shape[0])
    counts = torch.empty((n_hyp,), dtype=torch.int32) if want_counts else None
    best_H = torch.empty((3, 3), dtype=torch.float32)
    best_index = torch.empty((1,), dtype=torch.int64)
    best_count = torch.empty((1,), dtype=torch.int32)
    st = _c("hg_ransac_hypothesize_score_host")(
        _ptr(src_xy, torch.float32, "cpu", "src_xy"), _ptr(dst_xy, torch.float32, "cpu", "dst_xy"), n_pts,
        _ptr(hyp_idx, torch.int32, "cpu", "hyp_idx"), n_hyp, float(threshold_px),
        _ptr(counts, torch.int32, "cpu", "counts"), _ptr(best_H, torch.float32, "cpu", "best_H"),
        _ptr(best_index, torch.int64, "cpu", "best_index"), _ptr(best_count, torch.int32, "cpu", "best_count"))
    _check(st, "hg_ransac_hypothesize_score_host")
    return {"counts": counts, "best_H": best_H, "best_index": best_index, "best_count": best_count}
