"""GPU parity of hg_offsets_to_grid and hg_ransac_hypothesize_score against the fp64 oracle.

Grid tolerance: 1e-3 px absolute, the reprojection tolerance of
north_star applied to every pixel.  RANSAC (north_star): counts exact except for correspondences
whose fp64 residual lies within 1e-4 relative of the threshold, i.e.
|count_gpu - count_oracle| <= band_count(hypothesis); best index equal unless the top counts tie
within their bands.
"""
import numpy as np
import pytest
import torch

import hg_workloads as W
import oracle
import paper_2402_18008_b200 as hg
from util import align_to

pytestmark = pytest.mark.gpu
DEV = "cuda"
GRID_TOL = 1e-3


# ---- offsets -> H -> grid --------------------------------------------------------------------
@pytest.mark.parametrize("rect,gw,gh,n", [((0.0, 0.0, 127.0, 127.0), 128, 128, 300),      # C5 shape
                                          ((10.0, -4.0, 300.0, 90.0), 37, 11, 65),          # odd width: 64-bit stores
                                          ((0.0, 0.0, 63.0, 31.0), 64, 32, 17),
                                          ((5.0, 5.0, 20.0, 20.0), 1, 1, 4),
                                          ((0.0, 0.0, 511.0, 3.0), 512, 4, 9),              # row wider than a block
                                          ((0.0, 0.0, 1.0, 1.0), 2, 2, 1000)])
def test_grid_matches_oracle(rect, gw, gh, n):
    x0, y0, w, h = rect
    scale = min(32.0, 0.2 * min(w, h))
    off = W.offsets_workload(n, seed=W.SEED_BASE + 5, max_offset=scale)
    H, g = hg.hg_offsets_to_grid(off.to(DEV), x0, y0, w, h, gw, gh, norm=hg.NORM_H33)
    H_ref, g_ref = oracle.offsets_to_grid(off.numpy(), x0, y0, w, h, gw, gh)
    g = g.cpu().numpy().astype(np.float64)
    assert g.shape == g_ref.shape
    assert np.abs(g - g_ref).max() <= GRID_TOL, np.abs(g - g_ref).max()
    Hg, Hr = align_to(H.cpu().numpy().astype(np.float64), H_ref)
    assert (np.abs(Hg - Hr) <= 1e-4 * np.abs(Hr) + 1e-7).all()
    assert np.all(H.cpu().numpy()[:, 2, 2] == 1.0)


def test_grid_config5_corners_and_h_only_and_grid_only():
    n = 2048
    off = W.offsets_workload(n, seed=W.SEED_BASE + 5).to(DEV)
    H, g = hg.hg_offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128)
    corners = W.patch_corners().to(DEV)
    got = torch.stack([g[:, 0, 0], g[:, 0, 127], g[:, 127, 127], g[:, 127, 0]], dim=1)
    assert (got - (corners[None] + off)).abs().max().item() <= GRID_TOL
    H_only, none = hg.hg_offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128, want_grid=False)
    assert none is None and torch.equal(H_only, H)
    none, g_only = hg.hg_offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128, want_H=False)
    assert none is None and torch.equal(g_only, g)
    # zero offsets: the grid is the pixel lattice itself
    _, g0 = hg.hg_offsets_to_grid(torch.zeros((3, 4, 2), device=DEV), 0.0, 0.0, 127.0, 127.0, 128, 128)
    xs = torch.arange(128.0, device=DEV)
    assert (g0[..., 0] - xs[None, None, :]).abs().max().item() <= 1e-4
    assert (g0[..., 1] - xs[None, :, None]).abs().max().item() <= 1e-4


def test_grid_config1_h_only_matches_oracle_and_general_solver():
    """C1 through the offsets entry point (H only, thread per item): equals the oracle's offsets->H,
    and the general ACA solver on the fp32-rounded corners up to that rounding."""
    off = W.offsets_workload(1024, seed=W.SEED_BASE + 1)
    H, _ = hg.hg_offsets_to_grid(off.to(DEV), 0.0, 0.0, 127.0, 127.0, 128, 128, want_grid=False, norm=hg.NORM_FROBENIUS)
    Hr, _ = oracle.offsets_to_grid(off.numpy(), 0.0, 0.0, 127.0, 127.0, 128, 128, want_grid=False)
    a, b = align_to(H.cpu().numpy().astype(np.float64), Hr)
    assert (np.abs(a - b) <= 1e-4 * np.abs(b) + 1e-7).all()
    assert np.abs(a - b).max() <= 2e-7
    s, d = W.offsets_to_sets(off)                       # corner + offset rounded to fp32
    Hg = hg.hg_aca_batched(s.to(DEV), d.to(DEV), layout=hg.AOS, norm=hg.NORM_FROBENIUS)
    assert (H - Hg).abs().max().item() <= 1e-5
    # Algorithm 1 (TensorACA-rect) evaluated by the oracle gives the same H
    Ha = oracle.aca_rect(off.numpy(), 0.0, 0.0, 127.0, 127.0)
    a2, b2 = align_to(H.cpu().numpy().astype(np.float64), Ha)
    assert np.abs(a2 - b2).max() <= 2e-7


def test_grid_full_config5_every_item():
    """C5 at BASELINE size: 8192 x 128 x 128 x 2 in the launch configuration bench.py times; EVERY pixel of EVERY item
    compared with the oracle (in slabs of 512 items), plus the corner property and every H."""
    n = 8192
    off = W.offsets_workload(n, seed=W.SEED_BASE + 5)
    H, g = hg.hg_offsets_to_grid(off.to(DEV), 0.0, 0.0, 127.0, 127.0, 128, 128)
    worst = 0.0
    for b0 in range(0, n, 512):
        H_ref, g_ref = oracle.offsets_to_grid(off.numpy()[b0:b0 + 512], 0.0, 0.0, 127.0, 127.0, 128, 128)
        worst = max(worst, float(np.abs(g[b0:b0 + 512].cpu().numpy() - g_ref).max()))
        Hg, Hr = align_to(H[b0:b0 + 512].cpu().numpy().astype(np.float64), H_ref)
        assert (np.abs(Hg - Hr) <= 1e-4 * np.abs(Hr) + 1e-7).all()
    assert worst <= GRID_TOL, worst
    corners = W.patch_corners().to(DEV)
    got = torch.stack([g[:, 0, 0], g[:, 0, 127], g[:, 127, 127], g[:, 127, 0]], dim=1)
    assert (got - (corners[None] + off.to(DEV))).abs().max().item() <= GRID_TOL
    assert torch.isfinite(g).all()
    print("C5 every item: max |grid - oracle| =", worst, "px")


# ---- RANSAC ------------------------------------------------------------------------------------
def check_ransac(wl, t, out, ref):
    counts = out["counts"].cpu().numpy()
    diff = np.abs(counts.astype(np.int64) - ref["counts"].astype(np.int64))
    assert (diff <= ref["band_counts"]).all(), (int((diff > ref["band_counts"]).sum()), int(diff.max()))
    bi, bc = int(out["best_index"].item()), int(out["best_count"].item())
    assert bc == counts.max() and bi == int(np.argmax(counts))            # argmax, ties -> lowest index
    if ref["band_counts"][[bi, ref["best_index"]]].sum() == 0 and (diff == 0).all():
        assert bi == ref["best_index"] and bc == ref["best_count"]
    else:
        assert abs(bc - ref["best_count"]) <= ref["band_counts"].max()
    idx = wl["hyp_idx"].numpy()[bi]
    H_ref = oracle.normal_form(oracle.aca(wl["src_xy"].numpy()[idx][None], wl["dst_xy"].numpy()[idx][None]))[0]
    Hb = out["best_H"].cpu().numpy().astype(np.float64)
    a, b = align_to(Hb[None], H_ref[None])
    assert np.abs(a - b).max() <= 2e-7
    assert abs(np.sqrt((Hb ** 2).sum()) - 1.0) <= 3e-7
    return diff


# operand paths of the score kernel: tables of <= 4096 points -> constant bank / uniform datapath (launches of fewer than
# 148 x 512 hypotheses also split the table over blockIdx.y); more points -> shared-memory stages (split likewise); small
# calls on small tables -> the one-kernel path
@pytest.mark.parametrize("n_pts,n_hyp,t", [(4096, 6000, 3.0), (1001, 5000, 3.0), (100, 777, 1.5),
                                           (4, 1, 3.0), (2500, 3000, 0.75), (9000, 1500, 3.0),
                                           (1001, 80000, 3.0), (4095, 76000, 1.0), (17, 75776, 3.0), (9001, 76000, 3.0),
                                           (4095, 30000, 3.0), (1001, 30001, 2.0), (8191, 20000, 3.0)])   # split: constant bank / staged
def test_ransac_counts_match_oracle(n_pts, n_hyp, t):
    wl = W.ransac_workload(n_pts=n_pts, n_hyp=n_hyp, seed=W.SEED_BASE + 4 + n_pts)
    out = hg.hg_ransac_hypothesize_score(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"].to(DEV), t)
    ref = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), t, band_rel=1e-4)
    diff = check_ransac(wl, t, out, ref)
    stats = hg.ransac_stats(out["workspace"])
    print(n_pts, n_hyp, "mismatching (all inside the band):", int((diff > 0).sum()), stats)


def test_ransac_duplicate_best_and_degenerate_hypotheses():
    wl = W.ransac_workload(n_pts=512, n_hyp=400, seed=11)
    src, dst, idx = wl["src_xy"].clone(), wl["dst_xy"].clone(), wl["hyp_idx"].clone()
    # degenerate data: correspondences 0..3 coincide pairwise -> a hypothesis on them gives H = 0 -> count 0
    src[1] = src[0]; dst[1] = dst[0]; src[3] = src[2]; dst[3] = dst[2]
    idx[7] = torch.tensor([0, 1, 2, 3], dtype=torch.int32)
    ref = oracle.ransac(src.numpy(), dst.numpy(), idx.numpy(), 3.0, band_rel=1e-4)
    b = ref["best_index"]
    idx2 = torch.cat([idx, idx[b:b + 1]], dim=0)                # a tie: the lower index must win
    out = hg.hg_ransac_hypothesize_score(src.to(DEV), dst.to(DEV), idx2.to(DEV), 3.0)
    ref2 = oracle.ransac(src.numpy(), dst.numpy(), idx2.numpy(), 3.0, band_rel=1e-4)
    check_ransac({"src_xy": src, "dst_xy": dst, "hyp_idx": idx2}, 3.0, out, ref2)
    assert out["counts"][7].item() == 0 == ref2["counts"][7]
    assert int(out["best_index"].item()) == b


def test_ransac_host_entry_point_and_no_counts():
    wl = W.ransac_workload(n_pts=777, n_hyp=2000, seed=5)
    dev = hg.hg_ransac_hypothesize_score(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"].to(DEV), 3.0)
    host = hg.hg_ransac_hypothesize_score_host(wl["src_xy"], wl["dst_xy"], wl["hyp_idx"], 3.0)
    assert torch.equal(host["counts"], dev["counts"].cpu())
    assert torch.equal(host["best_H"], dev["best_H"].cpu())
    assert host["best_index"].item() == dev["best_index"].item()
    nc = hg.hg_ransac_hypothesize_score(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"].to(DEV), 3.0,
                                        want_counts=False)
    assert nc["counts"] is None and nc["best_index"].item() == dev["best_index"].item()


def test_ransac_full_config4_every_hypothesis():
    """C4 at BASELINE size (4096 correspondences, 2^20 hypotheses, t = 3 px), in the launch configuration bench.py
    times; the oracle scores ALL 2^20 hypotheses (4.29e9 pairs, OpenMP) and every count, the best index, the best count
    and the best H are compared."""
    wl = W.ransac_workload(n_pts=4096, n_hyp=1 << 20, seed=W.SEED_BASE + 4)
    out = hg.hg_ransac_hypothesize_score(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"].to(DEV), 3.0)
    ref = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), 3.0, band_rel=1e-4)
    diff = check_ransac(wl, 3.0, out, ref)
    assert int(out["best_count"].item()) >= 0.6 * 0.7 * 4096
    print("C4 every hypothesis: counts differing (all inside the band)", int((diff > 0).sum()), "of", 1 << 20,
          "hypotheses with in-band pairs", int((ref["band_counts"] > 0).sum()), hg.ransac_stats(out["workspace"]))


@pytest.mark.parametrize("n_pts,n_hyp,t,scale", [(4096, 1 << 20, 3.0, 1.0),        # C4 in full, constant-bank path
                                                 (2001, 100000, 0.5, 1.0),          # odd table, tight threshold
                                                 (1000, 4096, 3.0, 1.0),            # one-kernel path
                                                 (3001, 30000, 3.0, 1.0),           # constant bank, split over the table
                                                 (6001, 9000, 3.0, 1.0),            # shared-memory stages, split over the table
                                                 (6001, 80000, 3.0, 1.0),           # staged shared-memory path
                                                 (1500, 90000, 3e6, 1e6)])          # coordinates x 1e6: the band scales
def test_ransac_fp32_sweep_equals_fp64_decisions(n_pts, n_hyp, t, scale):
    """The claim of DESIGN.md section 7, pinned directly: the fp32 sweep with its error band gives the SAME counts as
    deciding every pair by the definition in fp64 from the kernel's own fp64 H (HG_RANSAC_DECIDE_ALL_F64).  Bit-exact:
    no oracle, no H rounding between the two sides -- only the band is under test."""
    wl = W.ransac_workload(n_pts=n_pts, n_hyp=n_hyp, seed=W.SEED_BASE + 90 + n_pts)
    s, d, idx = (wl["src_xy"] * scale).to(DEV), (wl["dst_xy"] * scale).to(DEV), wl["hyp_idx"].to(DEV)
    fast = hg.hg_ransac_hypothesize_score(s, d, idx, t)
    slow = hg.hg_ransac_hypothesize_score(s, d, idx, t, decide_all_f64=True)
    assert torch.equal(fast["counts"], slow["counts"])
    assert fast["best_index"].item() == slow["best_index"].item() and fast["best_count"].item() == slow["best_count"].item()
    assert torch.equal(fast["best_H"], slow["best_H"])
    st = hg.ransac_stats(slow["workspace"])
    assert st["n_pairs_f64"] == n_pts * n_hyp                                  # the slow side really decided every pair in fp64
    print(n_pts, n_hyp, "fast path fp64 decisions:", hg.ransac_stats(fast["workspace"])["n_pairs_f64"], "of", n_pts * n_hyp)


def test_ransac_pairs_exactly_at_the_threshold():
    """Adversarial for the band: dst = src for half the points (so hypotheses drawn from them give H = identity up to fp64
    rounding) and dst = src + (t, 0) for the other half -- residual t (1 +- 1e-16), every such pair lies inside any band.
    The sweep must hand all of them to the fp64 decision and agree with the all-fp64 mode bit for bit."""
    n_pts, n_hyp, t = 1200, 80000, 2.0
    g = torch.Generator().manual_seed(7)
    s = torch.rand((n_pts, 2), generator=g) * 600.0
    d = s.clone()
    d[n_pts // 2:, 0] += t
    idx = torch.stack([torch.randperm(n_pts // 2, generator=g)[:4] for _ in range(n_hyp // 100)]).repeat(100, 1).to(torch.int32)
    fast = hg.hg_ransac_hypothesize_score(s.to(DEV), d.to(DEV), idx.to(DEV), t)
    slow = hg.hg_ransac_hypothesize_score(s.to(DEV), d.to(DEV), idx.to(DEV), t, decide_all_f64=True)
    assert torch.equal(fast["counts"], slow["counts"])
    assert (fast["counts"] >= n_pts // 2).all()
    st = hg.ransac_stats(fast["workspace"])
    assert st["n_pairs_f64"] >= 0.4 * n_pts * n_hyp                          # the at-threshold half went to the cold path
    ref = oracle.ransac(s.numpy(), d.numpy(), idx.numpy()[:2000], t, band_rel=1e-4)
    diff = np.abs(fast["counts"].cpu().numpy()[:2000].astype(np.int64) - ref["counts"])
    assert (diff <= ref["band_counts"]).all()


def test_ransac_degenerate_and_non_finite_inputs():
    """Edge cases of the scorer: a NaN correspondence (outlier for everyone, zero count for hypotheses built on it),
    coincident points (H = 0 everywhere), dst = src (everything an inlier), very small / very large thresholds, and
    coordinates scaled by 1e6 (the error band scales with them).  Each against the oracle, and none may hang."""
    wl = W.ransac_workload(n_pts=1000, n_hyp=4096, seed=1)
    idx = wl["hyp_idx"]

    def both(src, dst, t):
        out = hg.hg_ransac_hypothesize_score(src.to(DEV), dst.to(DEV), idx.to(DEV), t)
        ref = oracle.ransac(src.numpy(), dst.numpy(), idx.numpy(), t, band_rel=1e-4)
        counts = out["counts"].cpu().numpy()
        diff = np.abs(counts.astype(np.int64) - ref["counts"])
        assert (diff <= ref["band_counts"]).all(), int(diff.max())
        assert int(out["best_count"].item()) == counts.max() and int(out["best_index"].item()) == int(np.argmax(counts))
        return counts

    s, d = wl["src_xy"].clone(), wl["dst_xy"].clone()
    s_nan = s.clone(); s_nan[5] = float("nan")
    c = both(s_nan, d, 3.0)
    uses5 = (idx == 5).any(dim=1).numpy()
    assert uses5.any() and (c[uses5] == 0).all()
    assert (both(torch.zeros_like(s), torch.zeros_like(d), 3.0) == 0).all()
    assert (both(s, s.clone(), 3.0) == 1000).all()
    assert (both(s, d, 1e-6) >= 4).all()                         # the four sampled correspondences always fit exactly
    assert (both(s, d, 1e9) >= 999).all()
    both(s * 1e6, d * 1e6, 3e6)


# ---- reading R20: sample check (HG_RANSAC_REJECT_DEGENERATE) -----------------------------------------------------------
@pytest.mark.parametrize("n_pts,n_hyp,min_area", [(4096, 100000, 0.0),      # constant-bank path
                                                  (4096, 100000, 400.0),
                                                  (1000, 3000, 25.0),        # split shared-memory path
                                                  (6001, 80000, 100.0),      # staged shared-memory path
                                                  (4, 24, 0.0), (37, 513, 1e4)])
def test_ransac_sample_check_matches_oracle(n_pts, n_hyp, min_area):
    """Reject flags are integer/sign decisions on fp64 values both sides compute with the same IEEE operations: bit-exact.
    A rejected hypothesis scores 0; every other count equals the plain call's."""
    wl = W.ransac_workload(n_pts=n_pts, n_hyp=n_hyp, seed=W.SEED_BASE + 120 + n_pts)
    s, d, idx = wl["src_xy"], wl["dst_xy"], wl["hyp_idx"]
    if n_pts == 4:                                            # all 24 orders of the only sample
        import itertools
        idx = torch.tensor(list(itertools.permutations(range(4))), dtype=torch.int32)
    rej = oracle.sample_check(s.numpy(), d.numpy(), idx.numpy(), min_area)
    out = hg.hg_ransac_hypothesize_score(s.to(DEV), d.to(DEV), idx.to(DEV), 3.0, reject_degenerate=True, min_area_px2=min_area)
    plain = hg.hg_ransac_hypothesize_score(s.to(DEV), d.to(DEV), idx.to(DEV), 3.0)
    counts, pc = out["counts"].cpu().numpy(), plain["counts"].cpu().numpy()
    st = hg.ransac_stats(out["workspace"])
    assert st["n_rejected"] == int(rej.sum())
    assert (counts[rej] == 0).all()
    assert np.array_equal(counts[~rej], pc[~rej])            # same kernel arithmetic for the accepted ones: identical
    assert (counts[~rej] >= 4).all() or n_pts == 4           # an accepted sample fits its own four points
    ref = oracle.ransac(s.numpy(), d.numpy(), idx.numpy(), 3.0, band_rel=1e-4, reject_degenerate=True, min_area=min_area)
    diff = np.abs(counts.astype(np.int64) - ref["counts"])
    assert (diff <= ref["band_counts"]).all()
    bi, bc = int(out["best_index"].item()), int(out["best_count"].item())
    assert bc == counts.max() and bi == int(np.argmax(counts))
    print(n_pts, n_hyp, min_area, "rejected", int(rej.sum()), "of", len(rej))


def test_ransac_sample_check_all_rejected_and_adaptive():
    wl = W.ransac_workload(n_pts=800, n_hyp=5000, seed=77, inlier_frac=1.0, noise_var=1e-6)
    s, d, idx = wl["src_xy"], wl["dst_xy"].clone(), wl["hyp_idx"]
    d[:, 0] = 640.0 - d[:, 0]                                                   # mirrored target plane: every sample flips
    assert oracle.sample_check(s.numpy(), d.numpy(), idx.numpy(), 0.0).all()
    out = hg.hg_ransac_hypothesize_score(s.to(DEV), d.to(DEV), idx.to(DEV), 3.0, reject_degenerate=True)
    assert (out["counts"] == 0).all() and out["best_count"].item() == 0 and out["best_index"].item() == 0
    assert hg.ransac_stats(out["workspace"])["n_rejected"] == 5000
    # adaptive entry point with the check, against the oracle's loop with the same rule
    wl = W.ransac_workload(n_pts=3000, n_hyp=4, seed=78, inlier_frac=0.4)
    a = hg.hg_ransac_adaptive(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), 1234, 1 << 17, 1 << 16, 3.0, 0.0, want_idx=True,
                              reject_degenerate=True, min_area_px2=50.0)
    ref = oracle.ransac_adaptive(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), 1234, 1 << 17, 1 << 16, 3.0, 0.0,
                                 reject_degenerate=True, min_area=50.0)
    assert int(a["n_evaluated"].item()) == ref["n_evaluated"] == 1 << 17
    assert np.array_equal(a["hyp_idx"].cpu().numpy(), ref["hyp_idx"])
    rej = oracle.sample_check(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), ref["hyp_idx"], 50.0)
    counts = a["counts"].cpu().numpy()
    assert (counts[rej] == 0).all() and hg.ransac_stats(a["workspace"])["n_rejected"] == int(rej.sum())
    assert (np.abs(counts.astype(np.int64) - ref["counts"]) <= ref["band_counts"]).all()
    assert 0.3 < rej.mean() < 0.99


# ---- tiny calls (the scale of the paper's Table 6): zero kernel + clustered one-kernel path ---------------------
# (n_pts, n_hyp) chosen so that every cluster size of the tiny path is taken: 1 (many groups / tiny tables), 2, 4, 8
@pytest.mark.parametrize("n_pts,n_hyp", [(1000, 1024), (500, 256), (4096, 9472), (4096, 40), (999, 33), (4095, 2100),
                                         (64, 5000), (37, 31), (131, 200), (263, 96), (5, 7),
                                         (2000, 16384), (2047, 20480)])               # the wide range of the one-kernel path
def test_ransac_tiny_calls_every_cluster_size(n_pts, n_hyp):
    wl = W.ransac_workload(n_pts=n_pts, n_hyp=n_hyp, seed=W.SEED_BASE + 300 + n_pts + n_hyp)
    s, d, idx = wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"].to(DEV)
    out = hg.hg_ransac_hypothesize_score(s, d, idx, 3.0)
    ref = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), 3.0, band_rel=1e-4)
    check_ransac(wl, 3.0, out, ref)
    slow = hg.hg_ransac_hypothesize_score(s, d, idx, 3.0, decide_all_f64=True)            # the band, bit for bit
    assert torch.equal(out["counts"], slow["counts"]) and torch.equal(out["best_H"], slow["best_H"])
    assert out["best_index"].item() == slow["best_index"].item()
    assert hg.ransac_stats(slow["workspace"])["n_pairs_f64"] == n_pts * n_hyp
    rej = oracle.sample_check(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), 50.0)
    chk = hg.hg_ransac_hypothesize_score(s, d, idx, 3.0, reject_degenerate=True, min_area_px2=50.0)
    cc = chk["counts"].cpu().numpy()
    assert hg.ransac_stats(chk["workspace"])["n_rejected"] == int(rej.sum())
    assert (cc[rej] == 0).all() and np.array_equal(cc[~rej], out["counts"].cpu().numpy()[~rej])
    assert chk["best_count"].item() == cc.max() and chk["best_index"].item() == int(np.argmax(cc))


def test_ransac_generic_calls_in_a_graph_replayed_beside_an_eager_call():
    """A captured mid-size call must not touch the constant bank (hg.h: a call on a capturing stream stages its table in
    shared memory): a graph holding a 4096 x 100 000 and a 6001 x 9000 call is replayed three times on a side stream while
    eager 4096 x 2^18 calls (constant-bank path) run on another stream.  Every result equals the same call issued alone,
    and the captured calls match the oracle."""
    t = 3.0
    shapes = [(4096, 100000), (6001, 9000)]
    wls = [W.ransac_workload(n_pts=p, n_hyp=h, seed=W.SEED_BASE + 5000 + p) for p, h in shapes]
    big = W.ransac_workload(n_pts=4096, n_hyp=1 << 18, seed=W.SEED_BASE + 5999)
    dev_in = [tuple(wl[k].to(DEV) for k in ("src_xy", "dst_xy", "hyp_idx")) for wl in wls]
    bs, bd, bidx = (big[k].to(DEV) for k in ("src_xy", "dst_xy", "hyp_idx"))
    alone = [hg.hg_ransac_hypothesize_score(s, d, i, t) for s, d, i in dev_in]                      # eager, nothing else running
    big_alone = hg.hg_ransac_hypothesize_score(bs, bd, bidx, t)
    torch.cuda.synchronize()
    outs = []
    for (p, h), (s, d, i) in zip(shapes, dev_in):                                                   # outputs the graph writes into
        outs.append({"counts": torch.zeros(h, dtype=torch.int32, device=DEV), "best_H": torch.zeros(3, 3, device=DEV),
                     "best_index": torch.zeros(1, dtype=torch.int64, device=DEV), "best_count": torch.zeros(1, dtype=torch.int32, device=DEV),
                     "workspace": torch.empty(hg.hg_ransac_workspace_bytes(p, h), dtype=torch.uint8, device=DEV)})
    side, other = torch.cuda.Stream(), torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            for (s, d, i), o in zip(dev_in, outs):
                hg.hg_ransac_hypothesize_score(s, d, i, t, counts=o["counts"], workspace=o["workspace"],
                                               best=(o["best_H"], o["best_index"], o["best_count"]))
    torch.cuda.synchronize()
    for rep in range(3):
        for o in outs:
            o["counts"].fill_(-1)
        torch.cuda.synchronize()
        with torch.cuda.stream(other):
            eager = [hg.hg_ransac_hypothesize_score(bs, bd, bidx, t) for _ in range(3)]               # ~0.5 ms each, constant bank
        with torch.cuda.stream(side):
            g.replay()
        torch.cuda.synchronize()
        for o, a in zip(outs, alone):
            assert torch.equal(o["counts"], a["counts"]), rep
            assert o["best_index"].item() == a["best_index"].item() and o["best_count"].item() == a["best_count"].item()
            assert torch.equal(o["best_H"], a["best_H"])
        for e in eager:
            assert torch.equal(e["counts"], big_alone["counts"]), rep
            assert e["best_index"].item() == big_alone["best_index"].item() and torch.equal(e["best_H"], big_alone["best_H"])
    for wl, o in zip(wls, outs):
        ref = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), t, band_rel=1e-4)
        check_ransac(wl, t, o, ref)


def test_ransac_tiny_call_replayed_in_a_cuda_graph():
    """The zero kernel and its programmatic dependent are captured as two graph nodes; every replay must start from a
    clean header (ticket, packed maximum) and see the inputs of that replay."""
    n_pts, n_hyp = 1000, 1024
    wls = [W.ransac_workload(n_pts=n_pts, n_hyp=n_hyp, seed=900 + k) for k in range(3)]
    s, d, idx = (wls[0][k].to(DEV).clone() for k in ("src_xy", "dst_xy", "hyp_idx"))
    ws = torch.empty(hg.hg_ransac_workspace_bytes(n_pts, n_hyp), dtype=torch.uint8, device=DEV)
    first = hg.hg_ransac_hypothesize_score(s, d, idx, 3.0, workspace=ws)
    keep = (first["best_H"], first["best_index"], first["best_count"])
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            for _ in range(3):                                  # back-to-back calls on one workspace inside the graph
                hg.hg_ransac_hypothesize_score(s, d, idx, 3.0, counts=first["counts"], workspace=ws, best=keep)
    for wl in wls[::-1]:
        s.copy_(wl["src_xy"]); d.copy_(wl["dst_xy"]); idx.copy_(wl["hyp_idx"])
        g.replay()
        torch.cuda.synchronize()
        ref = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), 3.0, band_rel=1e-4)
        check_ransac(wl, 3.0, first, ref)


@pytest.mark.parametrize("n_pts,n_hyp", [(1200, 2048), (601, 320), (4096, 64)])
def test_ransac_tiny_call_pairs_exactly_at_the_threshold(n_pts, n_hyp):
    """The at-threshold adversary on the tiny path: half the points have residual t (1 +- 1e-16) under every hypothesis, so
    every thread's queue of noted pairs overflows and it recounts its slice in fp64; counts must equal the all-fp64 mode."""
    t = 2.0
    g = torch.Generator().manual_seed(11 + n_pts)
    s = torch.rand((n_pts, 2), generator=g) * 600.0
    d = s.clone()
    d[n_pts // 2:, 0] += t
    idx = torch.stack([torch.randperm(n_pts // 2, generator=g)[:4] for _ in range(n_hyp)]).to(torch.int32)
    fast = hg.hg_ransac_hypothesize_score(s.to(DEV), d.to(DEV), idx.to(DEV), t)
    slow = hg.hg_ransac_hypothesize_score(s.to(DEV), d.to(DEV), idx.to(DEV), t, decide_all_f64=True)
    assert torch.equal(fast["counts"], slow["counts"]) and torch.equal(fast["best_H"], slow["best_H"])
    assert fast["best_index"].item() == slow["best_index"].item() and (fast["counts"] >= n_pts // 2).all()
    assert hg.ransac_stats(fast["workspace"])["n_pairs_f64"] >= 0.4 * n_pts * n_hyp
    ref = oracle.ransac(s.numpy(), d.numpy(), idx.numpy(), t, band_rel=1e-4)
    assert (np.abs(fast["counts"].cpu().numpy().astype(np.int64) - ref["counts"]) <= ref["band_counts"]).all()


def test_ransac_calls_on_two_streams_share_the_constant_bank_safely():
    """The packed table of a call lives in the one 64 KB constant bank of the device; calls on different streams are
    ordered against each other by the library (ConstTableGuard).  Two streams issue interleaved calls on different data;
    every result must equal the one of the same call issued alone."""
    wls = [W.ransac_workload(n_pts=4096 - 7 * k, n_hyp=90000 + 1000 * k, seed=W.SEED_BASE + 700 + k) for k in range(4)]
    dev_wl = [{k: v.to(DEV) for k, v in wl.items() if isinstance(v, torch.Tensor)} for wl in wls]
    alone = [hg.hg_ransac_hypothesize_score(w["src_xy"], w["dst_xy"], w["hyp_idx"], 3.0) for w in dev_wl]
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [None] * 4
    for rep in range(3):
        for k in range(4):
            with torch.cuda.stream(streams[k % 2]):
                outs[k] = hg.hg_ransac_hypothesize_score(dev_wl[k]["src_xy"], dev_wl[k]["dst_xy"], dev_wl[k]["hyp_idx"], 3.0)
    torch.cuda.synchronize()
    for k in range(4):
        assert torch.equal(outs[k]["counts"], alone[k]["counts"]), k
        assert outs[k]["best_index"].item() == alone[k]["best_index"].item() and torch.equal(outs[k]["best_H"], alone[k]["best_H"])


def test_ransac_tiny_call_protocol_stress():
    """The one-kernel path synchronises through stamped slots and a ticket, with no fence between them: 3000 calls on one
    workspace, alternating between three inputs of different shapes (so every call sees the leftovers of a different
    one), each result checked against the one computed alone."""
    shapes = [(1000, 1024), (500, 256), (333, 4000)]
    wls = [W.ransac_workload(n_pts=a, n_hyp=b, seed=40 + a) for a, b in shapes]
    dev_wl = [{k: v.to(DEV) for k, v in wl.items() if isinstance(v, torch.Tensor)} for wl in wls]
    alone = [hg.hg_ransac_hypothesize_score(w["src_xy"], w["dst_xy"], w["hyp_idx"], 3.0) for w in dev_wl]
    want = [(int(o["best_index"].item()), int(o["best_count"].item()), o["best_H"].clone(), int(o["counts"].sum().item())) for o in alone]
    ws = torch.empty(max(hg.hg_ransac_workspace_bytes(a, b) for a, b in shapes), dtype=torch.uint8, device=DEV)
    ws.fill_(0xAB)                                                    # garbage in, as the contract allows
    outs = [dict(o) for o in alone]
    bad = 0
    for it in range(3000):
        k = (it * 7 + it // 5) % 3
        o = hg.hg_ransac_hypothesize_score(dev_wl[k]["src_xy"], dev_wl[k]["dst_xy"], dev_wl[k]["hyp_idx"], 3.0,
                                           counts=outs[k]["counts"], workspace=ws,
                                           best=(outs[k]["best_H"], outs[k]["best_index"], outs[k]["best_count"]))
        if it % 10 == 9 or it > 2950:                                 # most calls run back to back without a host sync
            bi, bc = int(o["best_index"].item()), int(o["best_count"].item())
            ok = (bi, bc) == want[k][:2] and torch.equal(o["best_H"], want[k][2]) and int(o["counts"].sum().item()) == want[k][3]
            bad += 0 if ok else 1
    assert bad == 0
