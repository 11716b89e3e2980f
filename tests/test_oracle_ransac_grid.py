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
