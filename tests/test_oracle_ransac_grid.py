"""Pins of the oracle's RANSAC scorer and offsets->grid evaluation (readings R9, R10 of DESIGN.md)
against the definition in exact arithmetic, planted models and closed-form special cases."""
import itertools
import random
from fractions import Fraction

import numpy as np
import pytest
import torch

import hg_workloads as W
import oracle
from exact_ref import all_quads, apply_exact, exact_h_by_definition, exact_inlier_count
from util import project


# ---- brute force by the definition: N = 8 integer points, all C(8,4) = 70 hypotheses ------------
def _collinear(a, b, c):
    return (b[0] - a[0]) * (c[1] - a[1]) - (b[1] - a[1]) * (c[0] - a[0]) == 0


def test_ransac_brute_force_exact_rational():
    rng = random.Random(656)
    t = 2.5
    for trial in range(3):
        while True:
            src = [(rng.randint(0, 40), rng.randint(0, 30)) for _ in range(8)]
            dst = [(x + rng.randint(-3, 3) + (y // 7), y + rng.randint(-3, 3) - (x // 9)) for x, y in src]
            if not any(_collinear(*tr) for tr in itertools.combinations(src, 3)) and \
               not any(_collinear(*tr) for tr in itertools.combinations(dst, 3)):
                break
        hyps = all_quads(8)
        assert len(hyps) == 70
        exact_counts, usable = [], []
        for h in hyps:
            try:
                Hx = exact_h_by_definition([src[i] for i in h], [dst[i] for i in h])
            except ZeroDivisionError:           # true h33 == 0: not representable with h33 = 1
                exact_counts.append(-1); usable.append(False); continue
            exact_counts.append(exact_inlier_count(Hx, src, dst, Fraction(t)))
            # decisions that fp64 rounding could flip: exact |r^2 - t^2| tiny
            margin = min(abs(((X / Wd - u) ** 2 + (Y / Wd - v) ** 2) - Fraction(t) ** 2)
                         for (x, y), (u, v) in zip(src, dst)
                         for X, Y, Wd in [apply_exact(Hx, Fraction(x), Fraction(y))] if Wd != 0)
            usable.append(margin > Fraction(1, 10 ** 9))
        out = oracle.ransac(np.array(src, np.float32), np.array(dst, np.float32),
                            np.array(hyps, np.int32), t)
        exact_counts = np.array(exact_counts)
        usable = np.array(usable)
        assert usable.sum() >= 60
        assert np.array_equal(out["counts"][usable], exact_counts[usable])
        assert (out["counts"][usable] >= 4).all()          # the 4 sampled points are always inliers
        if usable.all():
            best = int(exact_counts.max())
            assert out["best_count"] == best
            assert out["best_index"] == int(np.argmax(exact_counts))      # ties -> lowest index (R9)


# ---- planted model, zero noise: an all-inlier hypothesis counts the points consistent with H_gt -
def test_ransac_planted_model():
    wl = W.ransac_workload(n_pts=400, n_hyp=4, seed=11, inlier_frac=0.6, noise_var=0.0)
    src, dst = wl["src_xy"].numpy(), wl["dst_xy"].numpy()
    mask = wl["inlier_mask"].numpy()
    Hgt = wl["H_gt"].numpy()
    t = 3.0
    r_gt = np.linalg.norm(project(Hgt[None], src[None].astype(np.float64))[0] - dst, axis=1)
    sure_in = r_gt <= t - 1e-2
    maybe = np.abs(r_gt - t) < 1e-2
    assert (r_gt[mask] < 1e-3).all()
    inl = np.flatnonzero(mask)
    rng = np.random.default_rng(5)
    hyps = []
    while len(hyps) < 300:
        h = rng.choice(inl, 4, replace=False)
        if float(W.min_triangle_area(torch.from_numpy(src[h][None]))) >= 5000.0:
            hyps.append(h)
    out = oracle.ransac(src, dst, np.array(hyps, np.int32), t)
    lo, hi = int(sure_in.sum()), int(sure_in.sum() + maybe.sum())
    assert lo >= mask.sum()
    assert ((out["counts"] >= lo) & (out["counts"] <= hi)).all()


# ---- ACA-H and DLT-H score identically outside the allowance band; band semantics ----------------
def test_ransac_aca_vs_dlt_and_band():
    wl = W.ransac_workload(n_pts=512, n_hyp=3000, seed=W.SEED_BASE + 4)
    src, dst, idx = wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy()
    a = oracle.ransac(src, dst, idx, 3.0, band_rel=1e-7, solver=oracle.METHOD_ACA)
    b = oracle.ransac(src, dst, idx, 3.0, band_rel=1e-7, solver=oracle.METHOD_DLT)
    assert (np.abs(a["counts"] - b["counts"]) <= a["band_counts"] + b["band_counts"]).all()
    assert (a["counts"] != b["counts"]).mean() < 0.01
    assert a["best_count"] == b["best_count"] and a["best_index"] == b["best_index"]
    assert (a["counts"] >= 4).all() and (a["counts"] <= 512).all()
    # the best hypothesis explains roughly the planted inlier fraction
    assert a["best_count"] >= 0.6 * wl["inlier_mask"].sum().item()
    # band_counts by the definition, from per-pair residuals of one hypothesis
    h = int(a["best_index"])
    H = oracle.aca(src[idx[h]][None], dst[idx[h]][None])[0]
    r = oracle.residuals(H, src, dst)
    r_np = np.linalg.norm(project(H[None], src[None])[0] - dst.astype(np.float64), axis=1)
    assert np.abs(r - r_np).max() <= 1e-9
    assert a["counts"][h] == int((r <= 3.0).sum())
    wide = oracle.ransac(src, dst, idx[h:h + 1], 3.0, band_rel=0.05)
    assert wide["band_counts"][0] == int((np.abs(r - 3.0) <= 0.15).sum())
    assert np.abs(oracle.normal_form(H[None])[0] - a["best_H"]).max() <= 1e-15


def test_ransac_ties_and_empty():
    wl = W.ransac_workload(n_pts=64, n_hyp=50, seed=3)
    src, dst, idx = wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy()
    one = oracle.ransac(src, dst, idx, 3.0)
    b = one["best_index"]
    dup = np.concatenate([idx[b:b + 1], idx, idx[b:b + 1]], axis=0)       # best now also at 0 and at the end
    two = oracle.ransac(src, dst, dup, 3.0)
    assert two["best_count"] == one["best_count"] and two["best_index"] == 0
    none = oracle.ransac(src, dst, np.zeros((0, 4), np.int32), 3.0)
    assert none["best_index"] == -1 and none["counts"].shape == (0,)


# ---- grid (reading R10) ---------------------------------------------------------------------------
def test_grid_zero_offsets_is_pixel_coordinates():
    off = np.zeros((3, 4, 2), np.float32)
    H, g = oracle.offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128)
    xs, ys = np.meshgrid(np.arange(128.0), np.arange(128.0))
    assert np.abs(g[..., 0] - xs).max() <= 1e-10 and np.abs(g[..., 1] - ys).max() <= 1e-10
    assert np.abs(oracle.normal_form(H) - np.eye(3) / np.sqrt(3)).max() <= 1e-12


@pytest.mark.parametrize("rect,gw,gh", [((0.0, 0.0, 127.0, 127.0), 128, 128),
                                        ((10.0, -4.0, 300.0, 90.0), 37, 11)])
def test_grid_corners_and_dlt(rect, gw, gh):
    x0, y0, w, h = rect
    off = W.offsets_workload(64, seed=W.SEED_BASE + 5).numpy()
    H, g = oracle.offsets_to_grid(off, x0, y0, w, h, gw, gh)
    corners = W.patch_corners(x0, y0, w, h).numpy().astype(np.float64)
    target = corners[None] + off.astype(np.float64)
    got = np.stack([g[:, 0, 0], g[:, 0, gw - 1], g[:, gh - 1, gw - 1], g[:, gh - 1, 0]], axis=1)
    assert np.abs(got - target).max() <= 1e-9             # corner pixels land on corner + offset
    # every pixel: same as projecting with the by-definition (DLT) homography
    src = np.broadcast_to(corners, (64, 4, 2)).copy()
    Hd = oracle.solve_f64(oracle.METHOD_DLT, src, target)
    xs = x0 + np.arange(gw) * w / (gw - 1)
    ys = y0 + np.arange(gh) * h / (gh - 1)
    X, Y = np.meshgrid(xs, ys)
    pts = np.stack([X.ravel(), Y.ravel()], axis=-1)
    ref = project(Hd, np.broadcast_to(pts, (64,) + pts.shape)).reshape(64, gh, gw, 2)
    assert np.abs(g - ref).max() <= 1e-8


def test_grid_affine_offsets_have_zero_second_differences():
    # offsets that make the target quad a parallelogram => H affine => the grid is an affine lattice
    rng = np.random.default_rng(10)
    a = rng.uniform(-20, 20, size=(16, 2)).astype(np.float32)
    b = rng.uniform(-20, 20, size=(16, 2)).astype(np.float32)
    c = rng.uniform(-20, 20, size=(16, 2)).astype(np.float32)
    off = np.stack([a, a + b, a + b + c, a + c], axis=1).astype(np.float32)
    # fp32 sums above are rounded: rebuild exact parallelograms from representable pieces
    off = np.round(off * 64) / 64
    off[:, 2] = off[:, 1] + off[:, 3] - off[:, 0]
    H, g = oracle.offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128)
    d2x = g[:, :, 2:] - 2 * g[:, :, 1:-1] + g[:, :, :-2]
    d2y = g[:, 2:] - 2 * g[:, 1:-1] + g[:, :-2]
    assert np.abs(d2x).max() <= 1e-9 and np.abs(d2y).max() <= 1e-9
    Hn = oracle.normal_form(H)
    assert np.abs(Hn[:, 2, :2]).max() <= 1e-13


def test_grid_degenerate_sizes():
    off = W.offsets_workload(2, seed=1).numpy()
    H, g = oracle.offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 1, 1)
    assert g.shape == (2, 1, 1, 2)
    assert np.abs(g[:, 0, 0] - off[:, 0].astype(np.float64)).max() <= 1e-9   # pixel (x0,y0) -> TL + offset
    H2, none = oracle.offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128, want_grid=False)
    assert none is None and np.array_equal(H, H2)


# ---- reading R20: the sample check (degenerate configurations of P:786 + orientation) -----------------------------
def _area2_int(p, i, j, k):
    return (p[j][0] - p[i][0]) * (p[k][1] - p[i][1]) - (p[j][1] - p[i][1]) * (p[k][0] - p[i][0])


def _rejected_by_definition(src, dst, lim2):
    """R20 written out on exact integers: lim2 = 2 * min_area."""
    for tri in ((0, 1, 2), (0, 1, 3), (0, 2, 3), (1, 2, 3)):
        a1, a2 = _area2_int(src, *tri), _area2_int(dst, *tri)
        if abs(a1) <= lim2 or abs(a2) <= lim2:
            return True
        if (a1 > 0) != (a2 > 0):
            return True
    return False


def test_sample_check_brute_force_on_integer_points():
    """Every 4-subset (in 3 different orders each) of a small seeded integer table, against the definition evaluated with
    Python integers (exact): same flags, same number of rejections."""
    import itertools, random
    rng = random.Random(20)
    n = 14
    src = [(rng.randint(-9, 9), rng.randint(-9, 9)) for _ in range(n)]
    dst = [(rng.randint(-9, 9), rng.randint(-9, 9)) for _ in range(n)]
    dst[:7] = [(2 * x - y + 3, x + 3 * y - 1) for x, y in src[:7]]          # an orientation-preserving affine map on half the table
    quads = []
    for q in itertools.combinations(range(n), 4):
        quads += [q, (q[2], q[0], q[3], q[1]), (q[3], q[2], q[1], q[0])]
    idx = np.array(quads, dtype=np.int32)
    for min_area in (0.0, 1.0, 7.5):
        want = np.array([_rejected_by_definition([src[i] for i in q], [dst[i] for i in q], 2 * min_area) for q in quads])
        got = oracle.sample_check(np.array(src, np.float32), np.array(dst, np.float32), idx, min_area)
        assert np.array_equal(got, want), (min_area, int((got != want).sum()))
        assert 0 < want.sum() < len(quads)
    # the planted affine half: accepted whenever the source quadruple itself is non-degenerate
    acc = [q for q in quads if max(q) < 7 and not _rejected_by_definition([src[i] for i in q], [dst[i] for i in q], 0)]
    assert len(acc) > 20


def test_sample_check_planted_cases_and_invariances():
    rect = np.array([[0, 0], [40, 0], [40, 30], [0, 30]], dtype=np.float32)
    import itertools
    perms = np.array(list(itertools.permutations(range(4))), dtype=np.int32)
    # all 24 orders of a rectangle mapped onto a translated, scaled copy of itself (same order): accepted
    assert not oracle.sample_check(rect, rect * 1.5 + 7.0, perms).any()
    assert oracle.sample_check(rect, rect * 1.5 + 7.0, perms, min_area=601.0).all()           # every triangle has area 600
    assert not oracle.sample_check(rect, rect * 1.5 + 7.0, perms, min_area=599.0).any()
    # mirrored target: all four orientations flip -> rejected; two target points swapped: mixed -> rejected
    mirror = rect * np.array([-1.0, 1.0], dtype=np.float32)
    assert oracle.sample_check(rect, mirror, perms).all()
    twisted = rect[[0, 2, 1, 3]]
    assert oracle.sample_check(rect, twisted, perms).all()
    # three collinear points / two coincident points on either plane
    col = np.array([[0, 0], [10, 10], [20, 20], [5, 30]], dtype=np.float32)
    dup = np.array([[0, 0], [40, 0], [40, 0], [0, 30]], dtype=np.float32)
    base = np.arange(4, dtype=np.int32)[None]
    assert oracle.sample_check(col, rect, base)[0] and oracle.sample_check(rect, col, base)[0]
    assert oracle.sample_check(dup, rect, base)[0] and oracle.sample_check(rect, dup, base)[0]
    nan = rect.copy(); nan[2, 0] = np.nan
    assert oracle.sample_check(nan, rect, base)[0]
    # invariances: the same permutation on both planes, exchanging the planes, a common translation
    s, d = W.general_sets(4096, seed=31)
    s, d = s.numpy().reshape(-1, 2), d.numpy().reshape(-1, 2)
    d[::3] = d[::3][:, ::-1]                                                  # make a third of the sets inconsistent
    idx = np.arange(4 * 4096, dtype=np.int32).reshape(-1, 4)
    f0 = oracle.sample_check(s, d, idx, 50.0)
    assert 0.2 < f0.mean() < 0.9
    assert np.array_equal(f0, oracle.sample_check(s, d, idx[:, [2, 0, 3, 1]], 50.0))
    assert np.array_equal(f0, oracle.sample_check(d, s, idx, 50.0))


def test_sample_check_means_w_keeps_one_sign():
    """What the orientation rule says about H (pins it against the homography itself, computed by the DLT oracle):
    sign(A_dst) = sign(det H) * sign(W_i W_j W_k) * sign(A_src) for every triangle, so all four orientations are
    preserved iff W has one sign on the four source points and det(H) * W^3 > 0."""
    s, d = W.general_sets(1 << 13, seed=41)
    s, d = s.numpy().copy(), d.numpy().copy()
    rng = np.random.default_rng(3)
    k = rng.integers(0, 4, size=s.shape[0])
    bad = rng.random(s.shape[0]) < 0.5
    d[bad, k[bad]] = rng.random((int(bad.sum()), 2)).astype(np.float32) * np.array([640.0, 480.0], dtype=np.float32)   # an outlier
    idx = np.arange(4 * s.shape[0], dtype=np.int32).reshape(-1, 4)
    rej = oracle.sample_check(s.reshape(-1, 2), d.reshape(-1, 2), idx, 0.0)
    H, ok = oracle.solve(oracle.METHOD_DLT, s, d, return_ok=True)
    x = np.concatenate([s.astype(np.float64), np.ones(s.shape[:2] + (1,))], axis=-1)
    Wk = np.einsum("nj,nkj->nk", H[:, 2, :], x)
    same = (np.sign(Wk) == np.sign(Wk[:, :1])).all(axis=1)
    keeps = same & (np.linalg.det(H) * Wk[:, 0] > 0)
    # compare away from the decision boundary (|W| tiny or a nearly collinear triple): there the two must agree exactly
    clear = ok & (np.abs(Wk).min(axis=1) > 1e-6 * np.abs(Wk).max(axis=1))
    assert clear.mean() > 0.95
    assert np.array_equal(~rej[clear], keeps[clear])
    assert 0.2 < rej.mean() < 0.8


def test_ransac_with_sample_check_scores_rejected_hypotheses_zero():
    wl = W.ransac_workload(n_pts=300, n_hyp=2000, seed=9)
    s, d, idx = wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy()
    plain = oracle.ransac(s, d, idx, 3.0)
    chk = oracle.ransac(s, d, idx, 3.0, reject_degenerate=True, min_area=25.0)
    rej = oracle.sample_check(s, d, idx, 25.0)
    assert 0.1 < rej.mean() < 0.9
    assert (chk["counts"][rej] == 0).all() and (chk["band_counts"][rej] == 0).all()
    assert np.array_equal(chk["counts"][~rej], plain["counts"][~rej])
    assert chk["best_count"] == chk["counts"].max() and not rej[chk["best_index"]]
    # all-inlier samples are never rejected for a small epsilon: the best model survives
    assert chk["best_count"] >= 0.9 * plain["best_count"]
