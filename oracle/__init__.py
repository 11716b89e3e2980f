"""ORACLE -- TEST INFRASTRUCTURE ONLY.

Thin ctypes/numpy access to the plain fp64 CPU oracle in ``hg_oracle.cpp`` /
``hg_oracle_core.hpp`` (written from /root/reference/PAPER.md, "P:<line>").

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with, and never
imports, the CUDA path ``paper_2402_18008_b200``.  Parity pins: tests/test_oracle_*.py;
nothing is "parity unpinned".

Layouts (AoS): src, dst float32 [n,4,2]; H float64 [n,3,3].
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_LIB_PATH = _HERE / "libhg_oracle.so"
_SOURCES = [_HERE / "hg_oracle.cpp", _HERE / "hg_oracle_core.hpp"]

METHOD_DLT, METHOD_ACA, METHOD_SKS, METHOD_CLOSED = 0, 1, 2, 3


def build(force: bool = False) -> Path:
    """Compile the oracle with g++ (-O2, no fast-math, no FMA contraction)."""
    stale = (not _LIB_PATH.exists()) or any(
        s.stat().st_mtime > _LIB_PATH.stat().st_mtime for s in _SOURCES)
    if force or stale:
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-shared", "-fPIC", "-o", str(_LIB_PATH), str(_SOURCES[0])]
        subprocess.run(cmd, check=True, cwd=str(_HERE))
    return _LIB_PATH


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(str(_LIB_PATH))
        _lib.hgo_num_threads.restype = ctypes.c_int
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _f32(a, shape_tail) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(a), dtype=np.float32)
    return a.reshape((-1,) + shape_tail)


def num_threads() -> int:
    return int(lib().hgo_num_threads())


def set_num_threads(n: int) -> None:
    lib().hgo_set_num_threads(ctypes.c_int(int(n)))


def solve(method: int, src, dst, return_ok: bool = False):
    """H (float64 [n,3,3]) of each 4-point set.  DLT returns h33 = 1; ACA/SKS/closed form raw scale."""
    s = _f32(src, (4, 2))
    d = _f32(dst, (4, 2))
    n = s.shape[0]
    assert d.shape[0] == n
    H = np.empty((n, 3, 3), dtype=np.float64)
    ok = np.empty((n,), dtype=np.uint8)
    lib().hgo_solve(ctypes.c_int(method), _p(s), _p(d), _p(H), ctypes.c_int64(n), _p(ok))
    return (H, ok.astype(bool)) if return_ok else H


def dlt(src, dst):
    return solve(METHOD_DLT, src, dst)


def aca(src, dst):
    return solve(METHOD_ACA, src, dst)


def sks(src, dst):
    return solve(METHOD_SKS, src, dst)


def closed_form(src, dst):
    return solve(METHOD_CLOSED, src, dst)


def solve_f64(method: int, src, dst) -> np.ndarray:
    s = np.ascontiguousarray(np.asarray(src, dtype=np.float64)).reshape(-1, 4, 2)
    d = np.ascontiguousarray(np.asarray(dst, dtype=np.float64)).reshape(-1, 4, 2)
    n = s.shape[0]
    H = np.empty((n, 3, 3), dtype=np.float64)
    lib().hgo_solve_f64(ctypes.c_int(method), _p(s), _p(d), _p(H), ctypes.c_int64(n))
    return H


def aca_core(src, dst) -> np.ndarray:
    """c11, c22, c33 of Eq. 32 (float64 [n,3])."""
    s = _f32(src, (4, 2)); d = _f32(dst, (4, 2))
    out = np.empty((s.shape[0], 3), dtype=np.float64)
    lib().hgo_aca_core(_p(s), _p(d), _p(out), ctypes.c_int64(s.shape[0]))
    return out


def sks_kernel(src, dst) -> np.ndarray:
    """a_K, b_K, u_K, v_K of Eq. 15 (float64 [n,4])."""
    s = _f32(src, (4, 2)); d = _f32(dst, (4, 2))
    out = np.empty((s.shape[0], 4), dtype=np.float64)
    lib().hgo_sks_kernel(_p(s), _p(d), _p(out), ctypes.c_int64(s.shape[0]))
    return out


def normal_form(H) -> np.ndarray:
    """Unit-Frobenius, sign-fixed copy of H (largest-|.| element positive)."""
    Hn = np.array(H, dtype=np.float64, order="C", copy=True).reshape(-1, 3, 3)
    lib().hgo_normal_form(_p(Hn), ctypes.c_int64(Hn.shape[0]))
    return Hn


def op_counts(method: int) -> dict:
    out = np.zeros(4, dtype=np.int64)
    lib().hgo_op_counts(ctypes.c_int(method), _p(out))
    return {"add": int(out[0]), "mul": int(out[1]), "div": int(out[2]), "flops": int(out[3])}


def aca_rect(offsets, x0: float, y0: float, w: float, h: float) -> np.ndarray:
    o = _f32(offsets, (4, 2))
    H = np.empty((o.shape[0], 3, 3), dtype=np.float64)
    lib().hgo_aca_rect(_p(o), ctypes.c_float(x0), ctypes.c_float(y0), ctypes.c_float(w),
                       ctypes.c_float(h), _p(H), ctypes.c_int64(o.shape[0]))
    return H


def aca_rect_backward(offsets, x0: float, y0: float, w: float, h: float, grad_G, want_jac: bool = False):
    """dL/d offsets [n,4,2] (float64) of G = H/h33 (Algorithm 1) given dL/dG [n,3,3]; optionally the
    Jacobian dG/d offsets [n,9,8]."""
    o = _f32(offsets, (4, 2))
    n = o.shape[0]
    g = np.ascontiguousarray(np.asarray(grad_G, dtype=np.float64)).reshape(n, 9)
    go = np.empty((n, 4, 2), dtype=np.float64)
    jac = np.empty((n, 9, 8), dtype=np.float64) if want_jac else None
    lib().hgo_aca_rect_backward(_p(o), ctypes.c_float(x0), ctypes.c_float(y0), ctypes.c_float(w),
                                ctypes.c_float(h), _p(g), _p(go), _p(jac) if want_jac else None,
                                ctypes.c_int64(n))
    return (go, jac) if want_jac else go


def affine(src3, dst3) -> np.ndarray:
    """H_A = H_A2^-1 H_A1 (Eq. 41) from three correspondences: float32 [n,3,2] x2 -> float64 [n,3,3]."""
    s, d = _f32(src3, (3, 2)), _f32(dst3, (3, 2))
    H = np.empty((s.shape[0], 3, 3), dtype=np.float64)
    lib().hgo_affine(_p(s), _p(d), _p(H), ctypes.c_int64(s.shape[0]))
    return H


def sk(P3, Q3, dst) -> np.ndarray:
    """Simplified SK (Eq. 17): pattern points P3, Q3 (x,y) in the anchor frame, dst float32 [n,4,2] -> Hbar [n,3,3]."""
    d = _f32(dst, (4, 2))
    H = np.empty((d.shape[0], 3, 3), dtype=np.float64)
    lib().hgo_sk(ctypes.c_double(P3[0]), ctypes.c_double(P3[1]), ctypes.c_double(Q3[0]), ctypes.c_double(Q3[1]),
                 _p(d), _p(H), ctypes.c_int64(d.shape[0]))
    return H


def offsets_to_grid(offsets, x0: float, y0: float, w: float, h: float, grid_w: int, grid_h: int,
                    want_grid: bool = True):
    """(H float64 [n,3,3] raw scale, grid float64 [n,grid_h,grid_w,2] or None)."""
    o = _f32(offsets, (4, 2))
    n = o.shape[0]
    H = np.empty((n, 3, 3), dtype=np.float64)
    grid = np.empty((n, grid_h, grid_w, 2), dtype=np.float64) if want_grid else None
    lib().hgo_offsets_to_grid(_p(o), ctypes.c_float(x0), ctypes.c_float(y0), ctypes.c_float(w),
                              ctypes.c_float(h), ctypes.c_int32(grid_w), ctypes.c_int32(grid_h),
                              _p(H), _p(grid) if want_grid else None, ctypes.c_int64(n))
    return H, grid


def offsets_to_grid_backward(offsets, x0: float, y0: float, w: float, h: float, grad_grid) -> np.ndarray:
    """dL/d offsets float64 [n,4,2] of the grid of offsets_to_grid given dL/d grid [n,grid_h,grid_w,2] (forward-mode dual
    numbers through the general ACA solve and the projection of every lattice point)."""
    o = _f32(offsets, (4, 2))
    n = o.shape[0]
    g = np.ascontiguousarray(np.asarray(grad_grid, dtype=np.float64))
    assert g.ndim == 4 and g.shape[0] == n and g.shape[3] == 2
    go = np.empty((n, 4, 2), dtype=np.float64)
    lib().hgo_offsets_to_grid_backward(_p(o), ctypes.c_float(x0), ctypes.c_float(y0), ctypes.c_float(w), ctypes.c_float(h),
                                       ctypes.c_int32(g.shape[2]), ctypes.c_int32(g.shape[1]), _p(g), _p(go), ctypes.c_int64(n))
    return go


def offsets_to_warp(offsets, x0: float, y0: float, w: float, h: float, out_w: int, out_h: int, image) -> np.ndarray:
    """image float32 [n,C,img_h,img_w] sampled bilinearly (zero padding, pixel units) at the grid of H: float64 [n,C,out_h,out_w]."""
    o = _f32(offsets, (4, 2))
    img = np.ascontiguousarray(np.asarray(image), dtype=np.float32)
    n, C, ih, iw = img.shape
    assert n == o.shape[0]
    out = np.empty((n, C, out_h, out_w), dtype=np.float64)
    lib().hgo_offsets_to_warp(_p(o), ctypes.c_float(x0), ctypes.c_float(y0), ctypes.c_float(w), ctypes.c_float(h),
                              ctypes.c_int32(out_w), ctypes.c_int32(out_h), _p(img), ctypes.c_int32(C),
                              ctypes.c_int32(iw), ctypes.c_int32(ih), _p(out), ctypes.c_int64(n))
    return out


def sample_check(src_xy, dst_xy, hyp_idx, min_area: float = 0.0) -> np.ndarray:
    """Reading R20: bool [n_hyp], True where the 4-point sample is rejected (degenerate on either plane within
    min_area px^2, or a triangle's orientation not preserved)."""
    s = _f32(src_xy, (2,)); d = _f32(dst_xy, (2,))
    idx = np.ascontiguousarray(np.asarray(hyp_idx), dtype=np.int32).reshape(-1, 4)
    out = np.zeros(idx.shape[0], dtype=np.uint8)
    lib().hgo_sample_check(_p(s), _p(d), _p(idx), ctypes.c_int64(idx.shape[0]), ctypes.c_double(float(np.float32(min_area))), _p(out))
    return out.astype(bool)


def ransac(src_xy, dst_xy, hyp_idx, threshold: float, band_rel: float = 1e-4, solver: int = METHOD_ACA,
           reject_degenerate: bool = False, min_area: float = 0.0):
    """Returns dict(counts int32 [n_hyp], band_counts, best_H [3,3] normal form, best_index, best_count).
    reject_degenerate: samples rejected by reading R20 (min_area in px^2) score 0."""
    s = _f32(src_xy, (2,)); d = _f32(dst_xy, (2,))
    idx = np.ascontiguousarray(np.asarray(hyp_idx), dtype=np.int32).reshape(-1, 4)
    n_pts, n_hyp = s.shape[0], idx.shape[0]
    assert d.shape[0] == n_pts
    if n_hyp:
        assert idx.min() >= 0 and idx.max() < n_pts
    counts = np.zeros(n_hyp, dtype=np.int32)
    band = np.zeros(n_hyp, dtype=np.int32)
    best_H = np.full((3, 3), np.nan, dtype=np.float64)
    best_index = ctypes.c_int64(-1)
    best_count = ctypes.c_int32(-1)
    lib().hgo_ransac_opt(_p(s), _p(d), ctypes.c_int32(n_pts), _p(idx), ctypes.c_int64(n_hyp),
                         ctypes.c_double(float(np.float32(threshold))), ctypes.c_double(band_rel),
                         ctypes.c_int(1 if solver == METHOD_ACA else 0),
                         ctypes.c_double(float(np.float32(min_area)) if reject_degenerate else -1.0),
                         _p(counts), _p(band), _p(best_H), ctypes.byref(best_index), ctypes.byref(best_count))
    return {"counts": counts, "band_counts": band, "best_H": best_H,
            "best_index": int(best_index.value), "best_count": int(best_count.value)}


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.ascontiguousarray(ctr, dtype=np.uint32); k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().hgo_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def ransac_sample(seed: int, h0: int, n: int, n_pts: int) -> np.ndarray:
    idx = np.zeros((n, 4), dtype=np.int32)
    lib().hgo_ransac_sample(ctypes.c_uint64(seed), ctypes.c_int64(h0), ctypes.c_int64(n), ctypes.c_int32(n_pts), _p(idx))
    return idx


def ransac_adaptive(src_xy, dst_xy, seed: int, max_hyp: int, round_hyp: int, threshold: float, confidence: float,
                    band_rel: float = 1e-4, reject_degenerate: bool = False, min_area: float = 0.0):
    """Sampling + rounds + adaptive termination (reading R19).  Returns dict(n_evaluated, hyp_idx [n_evaluated,4],
    counts, band_counts, best_H, best_index, best_count, margins [rounds])."""
    s = _f32(src_xy, (2,)); d = _f32(dst_xy, (2,))
    n_pts = s.shape[0]
    idx = np.zeros((max_hyp, 4), dtype=np.int32)
    counts = np.zeros(max_hyp, dtype=np.int32); band = np.zeros(max_hyp, dtype=np.int32)
    n_rounds = (max_hyp + round_hyp - 1) // round_hyp
    margins = np.full(n_rounds, np.nan)
    best_H = np.full((3, 3), np.nan)
    bi, bc, ne = ctypes.c_int64(-1), ctypes.c_int32(-1), ctypes.c_int64(0)
    lib().hgo_ransac_adaptive(_p(s), _p(d), ctypes.c_int32(n_pts), ctypes.c_uint64(seed), ctypes.c_int64(max_hyp),
                              ctypes.c_int64(round_hyp), ctypes.c_double(float(np.float32(threshold))),
                              ctypes.c_double(float(np.float32(confidence))), ctypes.c_double(band_rel),
                              ctypes.c_double(float(np.float32(min_area)) if reject_degenerate else -1.0), _p(idx), _p(counts),
                              _p(band), _p(best_H), ctypes.byref(bi), ctypes.byref(bc), ctypes.byref(ne), _p(margins))
    n = int(ne.value)
    return {"n_evaluated": n, "hyp_idx": idx[:n], "counts": counts[:n], "band_counts": band[:n], "best_H": best_H,
            "best_index": int(bi.value), "best_count": int(bc.value), "margins": margins}


def residuals(H, src_xy, dst_xy) -> np.ndarray:
    Hc = np.ascontiguousarray(np.asarray(H, dtype=np.float64)).reshape(3, 3)
    s = _f32(src_xy, (2,)); d = _f32(dst_xy, (2,))
    r = np.empty(s.shape[0], dtype=np.float64)
    lib().hgo_residuals(_p(Hc), _p(s), _p(d), ctypes.c_int32(s.shape[0]), _p(r))
    return r
