"""Pins of the oracle functions behind the SURVEY.md 8(f) rows (CPU only).

Backward of offsets -> G = H/h33 (Algorithm 1; "naturally differential") is pinned by
  (a) the implicit-function theorem on the DLT system A h = b (Eq. 2-3): dh/d(u_k, v_k) = w_k A^-1 e,
      with numpy's inverse -- shares nothing with the dual-number evaluation;
  (b) central finite differences of the forward oracle on offsets that are exact in fp32;
  (c) the translation invariant: shifting all four targets by delta maps G to T(delta) G.
"""
import numpy as np
import pytest

import hg_workloads as W
import oracle

RECTS = [(0.0, 0.0, 127.0, 127.0), (16.0, 40.0, 300.0, 120.0)]


def _quantised_offsets(n, seed, max_off):
    off = W.offsets_workload(n, seed=seed, max_offset=max_off).numpy()
    return (np.round(off * 16.0) / 16.0).astype(np.float32)           # multiples of 1/16: +-2^-6 steps stay exact


def _G(off, rect):
    H = oracle.aca_rect(off, *rect)
    return H / H[:, 2:3, 2:3]


@pytest.mark.parametrize("rect", RECTS)
def test_backward_jacobian_equals_implicit_function_theorem(rect):
    x0, y0, w, h = rect
    n = 200
    off = _quantised_offsets(n, 11, 0.2 * min(w, h))
    _, J = oracle.aca_rect_backward(off, x0, y0, w, h, np.zeros((n, 3, 3)), want_jac=True)
    src = W.patch_corners(x0, y0, w, h).numpy().astype(np.float64)
    G = _G(off, rect)
    for i in range(n):
        dst = src + off[i].astype(np.float64)
        A = np.zeros((8, 8))
        for k in range(4):
            x, y = src[k]; u, v = dst[k]
            A[2 * k] = [x, y, 1, 0, 0, 0, -u * x, -u * y]
            A[2 * k + 1] = [0, 0, 0, x, y, 1, -v * x, -v * y]
        wk = G[i, 2, 0] * src[:, 0] + G[i, 2, 1] * src[:, 1] + 1.0
        J_ift = np.linalg.inv(A) * np.repeat(wk, 2)[None, :]           # dh_r / d(dst coordinate c) = (A^-1)_rc * w_k(c)
        assert np.abs(J[i, :8] - J_ift).max() <= 1e-9 * max(1.0, np.abs(J_ift).max())
        assert np.all(J[i, 8] == 0.0)                                 # G33 == 1


@pytest.mark.parametrize("rect", RECTS)
def test_backward_matches_central_differences(rect):
    x0, y0, w, h = rect
    n = 64
    off = _quantised_offsets(n, 12, 0.2 * min(w, h))
    _, J = oracle.aca_rect_backward(off, x0, y0, w, h, np.zeros((n, 3, 3)), want_jac=True)
    step = 2.0 ** -6
    for k in range(8):
        d = np.zeros((4, 2), dtype=np.float32); d.reshape(8)[k] = step
        fd = (_G(off + d, rect) - _G(off - d, rect)).reshape(n, 9) / (2 * step)
        assert np.abs(J[:, :, k] - fd).max() <= 2e-6 * max(1.0, np.abs(J[:, :, k]).max())


def test_backward_translation_invariant_and_vjp():
    rect = RECTS[1]
    n = 128
    off = W.offsets_workload(n, seed=13, max_offset=20.0).numpy()
    rng = np.random.default_rng(5)
    g = rng.standard_normal((n, 3, 3))
    go, J = oracle.aca_rect_backward(off, *rect, g, want_jac=True)
    G = _G(off, rect)
    ones_x = np.array([1, 0, 1, 0, 1, 0, 1, 0.0]); ones_y = np.array([0, 1, 0, 1, 0, 1, 0, 1.0])
    ex = np.zeros((n, 9)); ex[:, 0] = G[:, 2, 0]; ex[:, 1] = G[:, 2, 1]; ex[:, 2] = 1.0      # T(dx) G: row 1 += dx * row 3
    ey = np.zeros((n, 9)); ey[:, 3] = G[:, 2, 0]; ey[:, 4] = G[:, 2, 1]; ey[:, 5] = 1.0
    assert np.abs(J @ ones_x - ex).max() <= 1e-10
    assert np.abs(J @ ones_y - ey).max() <= 1e-10
    # the vector-Jacobian product is J^T g with the (3,3) entry ignored
    gg = g.reshape(n, 9).copy(); gg[:, 8] = 0.0
    assert np.abs(go.reshape(n, 8) - np.einsum("nek,ne->nk", J, gg)).max() <= 1e-12 * np.abs(go).max()
