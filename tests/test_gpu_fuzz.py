"""Randomised parity sweep: random (ragged) sizes, layouts, normalisations and shapes through every entry point, each
case compared with the oracle at the tolerances of the dedicated tests.  Seeded: the same cases every run."""
import numpy as np
import pytest
import torch

import hg_workloads as W
import oracle
import paper_2402_18008_b200 as hg
from util import align_to, check_h_parity

pytestmark = pytest.mark.gpu
DEV = "cuda"
SIZES = [1, 2, 3, 4, 5, 7, 31, 32, 33, 255, 256, 257, 1023, 1025]


def test_random_sizes_solvers_rect_backward():
    rng = np.random.default_rng(123)
    for it in range(60):
        n = int(rng.choice(SIZES + [int(rng.integers(1, 9000))]))
        s, d = W.general_sets(n, seed=1000 + it)
        layout, norm, meth = int(rng.integers(0, 2)), int(rng.integers(0, 3)), int(rng.integers(0, 2))
        fn = hg.hg_aca_batched if meth == 0 else hg.hg_sks_batched
        if layout == hg.SOA:
            H = fn(W.to_soa(s).to(DEV), W.to_soa(d).to(DEV), layout=hg.SOA, norm=norm).t().reshape(n, 3, 3)
        else:
            H = fn(s.to(DEV), d.to(DEV), layout=hg.AOS, norm=norm)
        ref = oracle.solve(oracle.METHOD_ACA if meth == 0 else oracle.METHOD_SKS, s.numpy(), d.numpy())
        # every set: finite, element-wise bound, reprojection bound (1e-3 px, or S on the R12-excluded sets)
        check_h_parity(H.cpu().numpy(), s.numpy(), d.numpy(), ref, oracle.dlt(s.numpy(), d.numpy()), require_frac=0.0,
                       label=(n, layout, norm, meth))
        off = W.offsets_workload(n, seed=2000 + it)
        Hr = hg.hg_aca_rect_batched(off.to(DEV), 3.0, -2.0, 100.0, 60.0, norm=hg.NORM_FROBENIUS).cpu().numpy().astype(np.float64)
        a, b = align_to(Hr, oracle.aca_rect(off.numpy(), 3.0, -2.0, 100.0, 60.0))
        assert np.abs(a - b).max() <= 3e-7, (n, np.abs(a - b).max())
        g = torch.randn((n, 3, 3), generator=torch.Generator().manual_seed(it))
        go = hg.hg_aca_rect_backward(off.to(DEV), 3.0, -2.0, 100.0, 60.0, g.to(DEV)).cpu().numpy().astype(np.float64)
        gr = oracle.aca_rect_backward(off.numpy(), 3.0, -2.0, 100.0, 60.0, g.numpy().astype(np.float64))
        sc = np.abs(gr).reshape(n, 8).max(axis=1)[:, None, None]
        assert (np.abs(go - gr) <= 4e-7 * sc + 1e-30).all(), n


def test_random_shapes_ransac_and_warp():
    rng = np.random.default_rng(321)
    for it in range(16):
        npts, nh = int(rng.integers(4, 3000)), int(rng.integers(1, 3000))
        t = float(rng.choice([0.5, 1.0, 3.0, 7.5]))
        wl = W.ransac_workload(n_pts=npts, n_hyp=nh, seed=3000 + it)
        out = hg.hg_ransac_hypothesize_score(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"].to(DEV), t)
        rf = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), t, band_rel=1e-4)
        df = np.abs(out["counts"].cpu().numpy().astype(np.int64) - rf["counts"])
        assert (df <= rf["band_counts"]).all(), (npts, nh, t, int(df.max()))
        ow, oh = int(rng.integers(1, 70)), int(rng.integers(1, 50))
        iw, ih, C, m = int(rng.integers(2, 90)), int(rng.integers(2, 70)), int(rng.integers(1, 5)), int(rng.integers(1, 9))
        o2 = W.offsets_workload(m, seed=it, max_offset=5.0)
        img = torch.rand((m, C, ih, iw), generator=torch.Generator().manual_seed(it))
        wp, _ = hg.hg_offsets_to_warp(o2.to(DEV), 1.0, 1.0, 40.0, 30.0, ow, oh, img.to(DEV))
        wr = oracle.offsets_to_warp(o2.numpy(), 1.0, 1.0, 40.0, 30.0, ow, oh, img.numpy())
        assert np.abs(wp.cpu().numpy() - wr).max() <= 2e-3, (ow, oh, iw, ih, C, m)


def test_random_shapes_grid_backward_and_small_ransac_modes():
    """Random grid shapes through hg_offsets_to_grid_backward (even and odd widths, single rows and columns, grids smaller
    than one batch of the copy pipeline) and random small RANSAC calls through the one-kernel path in all three modes."""
    rng = np.random.default_rng(777)
    for it in range(24):
        gw, gh, m = int(rng.integers(1, 200)), int(rng.integers(1, 90)), int(rng.integers(1, 12))
        rect = (float(rng.uniform(-5, 5)), float(rng.uniform(-5, 5)), float(rng.uniform(20, 130)), float(rng.uniform(20, 130)))
        off = W.offsets_workload(m, seed=500 + it, max_offset=0.2 * min(rect[2], rect[3]))
        g = torch.randn((m, gh, gw, 2), generator=torch.Generator().manual_seed(it))
        go = hg.hg_offsets_to_grid_backward(off.to(DEV), *rect, g.to(DEV)).cpu().numpy().astype(np.float64)
        ref = oracle.offsets_to_grid_backward(off.numpy(), *rect, g.numpy().astype(np.float64))
        sc = g.abs().sum(dim=(1, 2, 3)).numpy().astype(np.float64)[:, None, None]
        assert (np.abs(go - ref) <= 2e-6 * sc).all(), (gw, gh, m, float((np.abs(go - ref) / sc).max()))
    for it in range(12):
        npts, nh = int(rng.integers(4, 4097)), int(rng.integers(1, 9000))
        wl = W.ransac_workload(n_pts=npts, n_hyp=nh, seed=7000 + it)
        s, d, idx = wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"].to(DEV)
        fast = hg.hg_ransac_hypothesize_score(s, d, idx, 2.0)
        slow = hg.hg_ransac_hypothesize_score(s, d, idx, 2.0, decide_all_f64=True)
        assert torch.equal(fast["counts"], slow["counts"]) and torch.equal(fast["best_H"], slow["best_H"]), (npts, nh)
        rej = oracle.sample_check(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), 10.0)
        chk = hg.hg_ransac_hypothesize_score(s, d, idx, 2.0, reject_degenerate=True, min_area_px2=10.0)
        cc = chk["counts"].cpu().numpy()
        assert (cc[rej] == 0).all() and np.array_equal(cc[~rej], fast["counts"].cpu().numpy()[~rej]), (npts, nh)
        assert hg.ransac_stats(chk["workspace"])["n_rejected"] == int(rej.sum())
