"""GPU test of hg_ransac_hypothesize_score_noalloc, the one entry point of libhg that needs no workspace.

Why it exists: some users of this library run where device memory cannot be allocated -- a filter inside another
program's frame loop whose memory pool is not theirs, a loop with a latency budget (cudaMalloc may wait for the whole
device), a process in which another thread is capturing streams.  They can pass the tensors they already own (inputs,
counts, best_*), but not a fresh workspace.  The entry point therefore keeps its scratch in a fixed 28 KB array inside
the library, which limits it to 4096 correspondences and 9472 hypotheses, and every call on a device shares that array.

What is checked: on calls made back to back (so each one starts from the scratch the previous one left behind: a
larger call first, then smaller ones whose slots are a subset), the outputs equal those of the ordinary entry point with
a caller-owned workspace -- counts, best index and best count exactly, best_H to the same 2e-7 the other RANSAC tests
allow (both run the same kernel) -- and match the oracle under the rule of the other RANSAC tests; sizes beyond the
limits are refused with HG_ERR_TOO_LARGE and leave the outputs untouched; the device's free memory does not move across
a call.  The file is named so that pytest collects it last, and it depends on nothing the other tests leave behind: it
passes alone in a fresh process and at the end of the whole run.
"""
import numpy as np
import pytest
import torch

import hg_workloads as W
import oracle
import paper_2402_18008_b200 as hg
from test_gpu_grid_ransac import check_ransac

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _outputs(n_hyp):
    counts = torch.full((n_hyp,), -7, dtype=torch.int32, device=DEV)
    best = (torch.full((3, 3), float("nan"), dtype=torch.float32, device=DEV),
            torch.full((1,), -7, dtype=torch.int64, device=DEV), torch.full((1,), -7, dtype=torch.int32, device=DEV))
    return counts, best


def test_noalloc_entry_point_matches_the_workspace_path_on_consecutive_calls():
    # sizes in the order they are issued: the full capacity first, then calls that reuse a part of its slots, an odd
    # table, a single cluster-split group, and the same size twice in a row
    shapes = [(4096, 9472), (1000, 1024), (999, 33), (500, 256), (500, 256), (2047, 9000), (5, 7)]
    t = 3.0
    for call, (n_pts, n_hyp) in enumerate(shapes):
        wl = W.ransac_workload(n_pts=n_pts, n_hyp=n_hyp, seed=W.SEED_BASE + 7000 + call)
        s, d, idx = wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"].to(DEV)
        counts, best = _outputs(n_hyp)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        assert hg.hg_ransac_hypothesize_score_noalloc(s, d, idx, t, counts=counts, best=best) is None
        torch.cuda.synchronize()
        if call > 0:                                   # (the very first use of a kernel may load its code)
            assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory"
        got = {"counts": counts, "best_H": best[0], "best_index": best[1], "best_count": best[2]}
        want = hg.hg_ransac_hypothesize_score(s, d, idx, t)             # the existing path, its own workspace
        torch.cuda.synchronize()
        assert torch.equal(got["counts"], want["counts"]), (n_pts, n_hyp)
        assert got["best_index"].item() == want["best_index"].item(), (n_pts, n_hyp)
        assert got["best_count"].item() == want["best_count"].item(), (n_pts, n_hyp)
        assert (got["best_H"] - want["best_H"]).abs().max().item() <= 2e-7, (n_pts, n_hyp)
        ref = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), wl["hyp_idx"].numpy(), t, band_rel=1e-4)
        check_ransac(wl, t, got, ref)


def test_noalloc_entry_point_optional_outputs_and_same_stream_ordering():
    """counts only / best only, and three calls enqueued on one side stream without a synchronisation in between: stream
    order is all the shared array needs."""
    wls = [W.ransac_workload(n_pts=777, n_hyp=n_hyp, seed=W.SEED_BASE + 7100 + n_hyp) for n_hyp in (640, 96, 2000)]
    side = torch.cuda.Stream()
    outs = []
    dev_in = [tuple(wl[k].to(DEV) for k in ("src_xy", "dst_xy", "hyp_idx")) for wl in wls]
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        for (s, d, idx), wl in zip(dev_in, wls):
            counts, best = _outputs(idx.shape[0])
            hg.hg_ransac_hypothesize_score_noalloc(s, d, idx, 2.0, counts=counts, best=best)
            outs.append((counts, best))
    side.synchronize()
    for (s, d, idx), (counts, best) in zip(dev_in, outs):
        want = hg.hg_ransac_hypothesize_score(s, d, idx, 2.0)
        assert torch.equal(counts, want["counts"])
        assert best[1].item() == want["best_index"].item() and best[2].item() == want["best_count"].item()
        assert (best[0] - want["best_H"]).abs().max().item() <= 2e-7
    s, d, idx = dev_in[0]
    counts, best = _outputs(idx.shape[0])
    hg.hg_ransac_hypothesize_score_noalloc(s, d, idx, 2.0, counts=counts)                  # no best_*
    hg.hg_ransac_hypothesize_score_noalloc(s, d, idx, 2.0, best=best)                      # no counts
    torch.cuda.synchronize()
    assert best[2].item() == counts.max().item() and best[1].item() == int(counts.argmax().item())


def test_noalloc_entry_point_refuses_what_the_fixed_array_cannot_hold():
    for n_pts, n_hyp in [(hg.RANSAC_NOALLOC_MAX_PTS + 1, 64), (64, hg.RANSAC_NOALLOC_MAX_HYP + 1), (8192, 1 << 20)]:
        s = torch.zeros((n_pts, 2), dtype=torch.float32, device=DEV)
        idx = torch.zeros((n_hyp, 4), dtype=torch.int32, device=DEV)
        counts, best = _outputs(n_hyp)
        with pytest.raises(hg.HgError) as e:
            hg.hg_ransac_hypothesize_score_noalloc(s, s, idx, 3.0, counts=counts, best=best)
        assert e.value.status == hg.HG_ERR_TOO_LARGE and "TOO_LARGE" in str(e.value)
        torch.cuda.synchronize()
        assert (counts == -7).all() and best[1].item() == -7 and best[2].item() == -7      # nothing was enqueued
    # the limits themselves are accepted (checked above at 4096 x 9472); an empty call is a no-op
    s = torch.zeros((16, 2), dtype=torch.float32, device=DEV)
    hg.hg_ransac_hypothesize_score_noalloc(s, s, torch.zeros((0, 4), dtype=torch.int32, device=DEV), 3.0)
