"""Test-side comparison helpers (numpy fp64; no oracle, no CUDA code)."""
import numpy as np


def unit_frobenius(H):
    """H / ||H||_F after a max-abs pre-scale (raw ACA scale ~1e23 squares beyond fp32/fp64 comfort)."""
    H = np.asarray(H, dtype=np.float64).reshape(-1, 3, 3)
    H = H / np.abs(H).max(axis=(1, 2), keepdims=True)
    return H / np.sqrt((H ** 2).sum(axis=(1, 2), keepdims=True))


def align_to(H, H_ref):
    """Comparison form of DESIGN.md: both unit-Frobenius; the sign of H is chosen so that the element
    where |H_ref| is largest has the sign it has in H_ref."""
    H = unit_frobenius(H)
    H_ref = unit_frobenius(H_ref)
    n = H.shape[0]
    idx = np.abs(H_ref).reshape(n, 9).argmax(axis=1)
    s_ref = np.sign(H_ref.reshape(n, 9)[np.arange(n), idx])
    s = np.sign(H.reshape(n, 9)[np.arange(n), idx])
    s[s == 0] = 1
    return H * (s * s_ref)[:, None, None], H_ref


def project(H, pts):
    """pi(H [x;y;1]) in fp64; H [n,3,3], pts [n,k,2]."""
    pts = np.asarray(pts, dtype=np.float64)
    p = np.concatenate([pts, np.ones(pts.shape[:-1] + (1,))], axis=-1)
    q = np.einsum("nij,nkj->nki", np.asarray(H, dtype=np.float64), p)
    return q[..., :2] / q[..., 2:3]


def rounding_sensitivity(H_ref, src):
    """Reading R12: first-order change (px) of the 4-point reprojection caused by rounding H to fp32,
    S = 2^-24 * max_k sum_{r in 1,2} ( sum_j |h_rj x_kj| + |pi_r(x_k)| sum_j |h_3j x_kj| ) / |w_k|."""
    H = np.asarray(H_ref, dtype=np.float64).reshape(-1, 3, 3)
    src = np.asarray(src, dtype=np.float64)
    x = np.concatenate([src, np.ones(src.shape[:-1] + (1,))], axis=-1)          # [n,4,3]
    terms = np.abs(H[:, None, :, :] * x[:, :, None, :])                          # [n,k,r,j]
    row = terms.sum(axis=-1)                                                     # [n,k,3]
    hx = np.einsum("nij,nkj->nki", H, x)
    w = hx[..., 2]
    pi = hx[..., :2] / w[..., None]
    S = ((row[..., 0] + np.abs(pi[..., 0]) * row[..., 2]) + (row[..., 1] + np.abs(pi[..., 1]) * row[..., 2])) / np.abs(w)
    return 2.0 ** -24 * S.max(axis=1)
