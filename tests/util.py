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


def reprojection_px(H, src, dst):
    """4-point reprojection error of each set: max over the four points of the EUCLIDEAN distance ||pi(H s_k) - d_k||_2, px."""
    e = project(np.asarray(H, dtype=np.float64), src) - np.asarray(dst, dtype=np.float64)
    return np.hypot(e[..., 0], e[..., 1]).max(axis=1)


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


# ---- the H parity rule of BASELINE.json north_star + DESIGN.md reading R12, used by every GPU solver test ----
REL_TOL, ABS_FLOOR, REPROJ_TOL, S_MAX = 1e-4, 1e-7, 1e-3, 1e-3
# On the sets R12 excludes from the 1e-3 px reprojection bound (own fp32-rounding sensitivity S > 1e-3 px) the
# reprojection error must still be explained by the one rounding of H to fp32: reproj <= EXCL_C * S + EXCL_ABS
# (S is the first-order bound of exactly that rounding; DESIGN.md section 8 states the constant and what was measured).
EXCL_C, EXCL_ABS = 1.0, 1e-6


def check_h_parity(H_gpu, src, dst, H_ref, H_dlt, require_frac=0.98, label=""):
    """H_gpu [n,3,3] (fp32 result, any scale) against the oracle's H_ref for fp32 sets src, dst [n,4,2] that passed the
    generator's area filter.  Asserted on EVERY set: finite, |dH_ij| <= 1e-4 |H_ij| + 1e-7 (unit Frobenius, sign
    aligned).  Reprojection (Euclidean distance, max over the four points): <= 1e-3 px on the well-conditioned sets (S <= 1e-3 px, R12), <= EXCL_C * S + EXCL_ABS on
    the others.  Returns the literal statistics over all sets."""
    H_gpu = np.asarray(H_gpu)
    n = H_gpu.shape[0]
    assert np.isfinite(H_gpu).all(), (label, "non-finite H", int((~np.isfinite(H_gpu)).any(axis=(1, 2)).sum()))
    Hg, Hr = align_to(H_gpu.astype(np.float64), H_ref)
    dH = np.abs(Hg - Hr)
    tol = REL_TOL * np.abs(Hr) + ABS_FLOOR
    ratio = (dH / tol).max(axis=(1, 2))
    assert (ratio <= 1.0).all(), (label, "elementwise", int((ratio > 1.0).sum()), float(ratio.max()))
    S = rounding_sensitivity(H_dlt, src)
    well = S <= S_MAX
    assert well.mean() >= require_frac, (label, "well-conditioned fraction", float(well.mean()))
    reproj = reprojection_px(H_gpu, src, dst)
    assert (reproj[well] <= REPROJ_TOL).all(), (label, "reproj", float(reproj[well].max()))
    excl = ~well
    if excl.any():
        bound = EXCL_C * S[excl] + EXCL_ABS
        assert (reproj[excl] <= bound).all(), (label, "reproj on R12-excluded sets", float((reproj[excl] / bound).max()))
    q = lambda a, p: float(np.quantile(a, p)) if a.size else 0.0
    return {"n": int(n), "well_frac": float(well.mean()), "excluded": int(excl.sum()),
            "max_elem_ratio_all": float(ratio.max()),
            "max_reproj_well": float(reproj[well].max()) if well.any() else 0.0,
            "max_reproj_all": float(reproj.max()), "reproj_p50_all": q(reproj, 0.5), "reproj_p999_all": q(reproj, 0.999),
            "frac_reproj_le_1e-3_all": float((reproj <= REPROJ_TOL).mean()),
            "max_reproj_over_S_excluded": float((reproj[excl] / S[excl]).max()) if excl.any() else 0.0,
            "max_S": float(S.max())}


def check_h_parity_lazy(H_gpu, src, dst, H_ref, dlt_fn, label=""):
    """The same rule as check_h_parity, evaluated so that a 2^22-set slab costs a second: the DLT solve and the sensitivity S
    (R12) are computed only for the sets whose reprojection error exceeds 1e-3 px -- those must have S > 1e-3 px (i.e. be
    R12-excluded) and satisfy reproj <= EXCL_C * S + EXCL_ABS; every other set satisfies the 1e-3 px bound whatever its S.
    The "well-conditioned fraction >= 0.98" of check_h_parity is implied by the stronger requirement asserted here: at
    least 98 % of ALL sets reproject within 1e-3 px.  dlt_fn(src_subset, dst_subset) -> H_dlt.  Returns literal statistics."""
    H_gpu = np.asarray(H_gpu)
    n = H_gpu.shape[0]
    assert np.isfinite(H_gpu).all(), (label, "non-finite H", int((~np.isfinite(H_gpu)).any(axis=(1, 2)).sum()))
    Hg, Hr = align_to(H_gpu.astype(np.float64), H_ref)
    ratio = (np.abs(Hg - Hr) / (REL_TOL * np.abs(Hr) + ABS_FLOOR)).max(axis=(1, 2))
    assert (ratio <= 1.0).all(), (label, "elementwise", int((ratio > 1.0).sum()), float(ratio.max()), int(ratio.argmax()))
    reproj = reprojection_px(H_gpu, src, dst)
    over = np.nonzero(reproj > REPROJ_TOL)[0]
    assert over.size <= 0.02 * n, (label, "fraction within 1e-3 px", 1.0 - over.size / n)
    worst = 0.0
    if over.size:
        S = rounding_sensitivity(dlt_fn(src[over], dst[over]), src[over])
        assert (S > S_MAX).all(), (label, "reproj > 1e-3 px on a well-conditioned set", float(reproj[over][S <= S_MAX].max()))
        bound = EXCL_C * S + EXCL_ABS
        assert (reproj[over] <= bound).all(), (label, "reproj on R12-excluded sets", float((reproj[over] / bound).max()))
        worst = float((reproj[over] / S).max())
    return {"n": int(n), "over_1e-3px": int(over.size), "max_elem_ratio": float(ratio.max()), "max_reproj": float(reproj.max()),
            "max_reproj_over_S_on_those": worst}
