"""GPU parity of the SURVEY.md 8(f) rows against the fp64 oracle (same tolerances as the general
solvers: reading R12 for H)."""
import numpy as np
import pytest
import torch

import hg_workloads as W
import oracle
import paper_2402_18008_b200 as hg
from util import align_to, project

pytestmark = pytest.mark.gpu
DEV = "cuda"


# ---- 8(f)-1: hg_aca_rect_batched (Algorithm 1) ----------------------------------------
@pytest.mark.parametrize("rect,n,max_off", [((0.0, 0.0, 127.0, 127.0), 1024, 32.0),      # C1
                                            ((16.0, 40.0, 300.0, 120.0), 4099, 30.0),     # ragged tail, r_rec = 2.5
                                            ((-50.0, 7.0, 64.0, 200.0), 777, 12.0),
                                            ((0.0, 0.0, 1.0, 1.0), 5, 0.2),
                                            ((0.0, 0.0, 127.0, 127.0), 1, 32.0)])
@pytest.mark.parametrize("layout", ["aos", "soa"])
def test_aca_rect_matches_oracle(rect, n, max_off, layout):
    x0, y0, w, h = rect
    off = W.offsets_workload(n, seed=W.SEED_BASE + 1 + n, max_offset=max_off)
    H_ref = oracle.aca_rect(off.numpy(), x0, y0, w, h)
    if layout == "aos":
        H = hg.hg_aca_rect_batched(off.to(DEV), x0, y0, w, h, layout=hg.AOS, norm=hg.NORM_FROBENIUS).cpu().numpy()
    else:
        o_soa = off.reshape(n, 8).t().contiguous()
        H = hg.hg_aca_rect_batched(o_soa.to(DEV), x0, y0, w, h, layout=hg.SOA, norm=hg.NORM_FROBENIUS)
        H = H.t().reshape(n, 3, 3).cpu().numpy()
    a, b = align_to(H.astype(np.float64), H_ref)
    assert (np.abs(a - b) <= 1e-4 * np.abs(b) + 1e-7).all()
    assert np.abs(a - b).max() <= 2e-7
    # defining property on the fp32 result: corners map to corner + offset within the north_star tolerance
    src = np.broadcast_to(W.patch_corners(x0, y0, w, h).numpy().astype(np.float64), (n, 4, 2))
    dst = src + off.numpy().astype(np.float64)
    assert np.abs(project(H.astype(np.float64), src) - dst).max() <= 1e-3


def test_aca_rect_norms_scale_and_agreement_with_general_entry_points():
    n = 4096
    off = W.offsets_workload(n, seed=W.SEED_BASE + 5).to(DEV)
    Hn = hg.hg_aca_rect_batched(off, 0.0, 0.0, 127.0, 127.0, norm=hg.NORM_NONE)
    H1 = hg.hg_aca_rect_batched(off, 0.0, 0.0, 127.0, 127.0, norm=hg.NORM_H33)
    Hf = hg.hg_aca_rect_batched(off, 0.0, 0.0, 127.0, 127.0, norm=hg.NORM_FROBENIUS)
    assert torch.all(H1[:, 2, 2] == 1.0)
    assert ((Hf.double() ** 2).sum(dim=(1, 2)).sqrt() - 1.0).abs().max().item() <= 3e-7
    # raw scale: Eq. 45, i.e. minus Algorithm 1's printed scale (reading R6) -- compare with the oracle's raw H
    H_ref = oracle.aca_rect(off.cpu().numpy(), 0.0, 0.0, 127.0, 127.0)
    raw = Hn.cpu().numpy().astype(np.float64)
    assert (np.abs(raw + H_ref) <= 1e-6 * np.abs(H_ref).max(axis=(1, 2), keepdims=True)).all()
    # the general offsets entry point (full ACA on the explicit corners) gives the same H
    Hg, _ = hg.hg_offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128, want_grid=False, norm=hg.NORM_H33)
    assert (Hg - H1).abs().max().item() <= 2e-5 * H1.abs().max().item()
    # fp32 arithmetic: sanity only (not a parity configuration)
    H32 = hg.hg_aca_rect_batched(off, 0.0, 0.0, 127.0, 127.0, norm=hg.NORM_H33, prec=hg.PREC_F32)
    assert (H32 - H1).abs().max().item() <= 1e-2 * H1.abs().max().item()


def test_aca_rect_large_batch_sampled():
    """2^22 items in the launch configuration bench.py times (AoS in, AoS out); the oracle checks a strided sample."""
    n = 1 << 22
    off = W.offsets_workload(n, seed=W.SEED_BASE + 6, device=DEV)
    H = hg.hg_aca_rect_batched(off, 0.0, 0.0, 127.0, 127.0, norm=hg.NORM_H33)
    sel = torch.arange(0, n, 4099, device=DEV)
    H_ref = oracle.aca_rect(off[sel].cpu().numpy(), 0.0, 0.0, 127.0, 127.0)
    a, b = align_to(H[sel].cpu().numpy().astype(np.float64), H_ref)
    assert (np.abs(a - b) <= 1e-4 * np.abs(b) + 1e-7).all()
    assert torch.isfinite(H).all()


# ---- 8(f)-2: hg_aca_rect_backward ----------------------------------------------------------------
# Tolerance: the kernel evaluates the reverse-mode chain in fp64 and rounds once to fp32; against the fp64
# dual-number oracle each gradient is within a few fp32 ulps of the item's largest gradient entry.
@pytest.mark.parametrize("rect,n,max_off", [((0.0, 0.0, 127.0, 127.0), 1024, 32.0),
                                            ((16.0, 40.0, 300.0, 120.0), 4099, 30.0),
                                            ((-50.0, 7.0, 64.0, 200.0), 3, 12.0)])
def test_rect_backward_matches_oracle(rect, n, max_off):
    x0, y0, w, h = rect
    off = W.offsets_workload(n, seed=W.SEED_BASE + 21 + n, max_offset=max_off)
    g = torch.randn((n, 3, 3), generator=torch.Generator().manual_seed(n), dtype=torch.float32)
    go = hg.hg_aca_rect_backward(off.to(DEV), x0, y0, w, h, g.to(DEV)).cpu().numpy().astype(np.float64)
    ref = oracle.aca_rect_backward(off.numpy(), x0, y0, w, h, g.numpy().astype(np.float64))
    scale = np.abs(ref).reshape(n, 8).max(axis=1)[:, None, None]
    assert (np.abs(go - ref) <= 4e-7 * scale + 1e-30).all(), (np.abs(go - ref) / scale).max()


@pytest.mark.parametrize("n", [4096, 4099, 1])
def test_rect_backward_soa_matches_oracle_and_the_aos_entry_point(n):
    rect = (16.0, 40.0, 300.0, 120.0)
    off = W.offsets_workload(n, seed=W.SEED_BASE + 31 + n, max_offset=30.0)
    g = torch.randn((n, 3, 3), generator=torch.Generator().manual_seed(n), dtype=torch.float32)
    o_soa, g_soa = off.reshape(n, 8).t().contiguous(), g.reshape(n, 9).t().contiguous()
    go = hg.hg_aca_rect_backward_soa(o_soa.to(DEV), *rect, g_soa.to(DEV))
    assert tuple(go.shape) == (8, n)
    aos = hg.hg_aca_rect_backward(off.to(DEV), *rect, g.to(DEV))
    assert torch.equal(go.t().reshape(n, 4, 2), aos)                     # the same arithmetic in both layouts
    ref = oracle.aca_rect_backward(off.numpy(), *rect, g.numpy().astype(np.float64))
    scale = np.abs(ref).reshape(n, 8).max(axis=1)[:, None, None]
    assert (np.abs(go.t().reshape(n, 4, 2).cpu().numpy().astype(np.float64) - ref) <= 4e-7 * scale + 1e-30).all()


def test_rect_backward_is_the_gradient_of_the_forward_entry_point():
    """Directional derivative of the library's own forward (H33-normalised) against <grad, direction>."""
    n = 512
    rect = (0.0, 0.0, 127.0, 127.0)
    off = (W.offsets_workload(n, seed=77) * 16).round() / 16          # exact +-2^-5 steps in fp32
    d = torch.randn((n, 4, 2), generator=torch.Generator().manual_seed(1)).sign() * 2.0 ** -5
    g = torch.randn((n, 3, 3), generator=torch.Generator().manual_seed(2))
    go = hg.hg_aca_rect_backward(off.to(DEV), *rect, g.to(DEV)).double().cpu()
    Hp = hg.hg_aca_rect_batched((off + d).to(DEV), *rect, norm=hg.NORM_H33).double().cpu()
    Hm = hg.hg_aca_rect_batched((off - d).to(DEV), *rect, norm=hg.NORM_H33).double().cpu()
    lhs = ((Hp - Hm) * g.double()).sum(dim=(1, 2)) / 2.0
    rhs = (go * d.double()).sum(dim=(1, 2))
    assert ((lhs - rhs).abs() <= 2e-3 * rhs.abs() + 1e-5 * go.abs().amax(dim=(1, 2)) * 2.0 ** -5 * 8).all()


# ---- 8(f)-3: hg_affine_batched (Eq. 41) -------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 1023, 4096, 50001])
@pytest.mark.parametrize("layout", ["aos", "soa"])
def test_affine_matches_oracle(n, layout):
    s, d = W.general_sets(n, seed=W.SEED_BASE + 40 + n)
    s3, d3 = s[:, :3].contiguous(), d[:, :3].contiguous()
    H_ref = oracle.affine(s3.numpy(), d3.numpy())
    if layout == "aos":
        H = hg.hg_affine_batched(s3.to(DEV), d3.to(DEV), layout=hg.AOS, norm=hg.NORM_H33).cpu().numpy()
    else:
        a, b = s3.reshape(n, 6).t().contiguous(), d3.reshape(n, 6).t().contiguous()
        H = hg.hg_affine_batched(a.to(DEV), b.to(DEV), layout=hg.SOA, norm=hg.NORM_H33).t().reshape(n, 3, 3).cpu().numpy()
    assert np.all(H[:, 2, 0] == 0.0) and np.all(H[:, 2, 1] == 0.0) and np.all(H[:, 2, 2] == 1.0)
    A_ref = H_ref / H_ref[:, 2:3, 2:3]
    # fp64 internal, one rounding to fp32: each entry within fp32 rounding of its own magnitude (+ the translation's scale)
    tol = 1.5e-7 * np.abs(A_ref) + 1e-7
    assert (np.abs(H - A_ref) <= tol).all()
    assert np.abs(project(H.astype(np.float64), s3.numpy()) - d3.numpy()).max() <= 1e-3
    raw = hg.hg_affine_batched(s3.to(DEV), d3.to(DEV), layout=hg.AOS, norm=hg.NORM_NONE).cpu().numpy()
    assert (np.abs(raw - H_ref) <= 1.5e-7 * np.abs(H_ref) + 1e-30).all()                 # raw scale: h33 = f_A1


# ---- 8(f)-4: hg_sk_batched (Eq. 17) -----------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 777, 8192])
@pytest.mark.parametrize("layout", ["aos", "soa"])
def test_sk_matches_oracle(n, layout):
    s, d = W.general_sets(n, seed=W.SEED_BASE + 50 + n)
    P3, Q3 = (0.35, 1.6), (-0.8, -1.1)                      # a fixed pattern in its anchor frame
    H_ref = oracle.sk(P3, Q3, d.numpy())
    if layout == "aos":
        H = hg.hg_sk_batched(P3, Q3, d.to(DEV), layout=hg.AOS, norm=hg.NORM_FROBENIUS).cpu().numpy()
    else:
        H = hg.hg_sk_batched(P3, Q3, W.to_soa(d).to(DEV), layout=hg.SOA, norm=hg.NORM_FROBENIUS)
        H = H.t().reshape(n, 3, 3).cpu().numpy()
    a, b = align_to(H.astype(np.float64), H_ref)
    assert (np.abs(a - b) <= 1e-4 * np.abs(b) + 1e-7).all()
    assert np.abs(a - b).max() <= 3e-7
    obj = np.broadcast_to(np.array([[-1.0, 0.0], [1.0, 0.0], P3, Q3]), (n, 4, 2))
    ok = np.isfinite(H_ref).all(axis=(1, 2))
    assert ok.all()
    # reprojection on the sets whose own fp32-rounding sensitivity is small (reading R12)
    from util import rounding_sensitivity
    S = rounding_sensitivity(H_ref, obj)
    good = S <= 1e-3
    assert n < 100 or good.mean() >= 0.7        # an arbitrary pattern against random quadrangles is strongly projective (77 %)
    reproj = np.abs(project(H.astype(np.float64), obj) - d.numpy().astype(np.float64)).max(axis=(1, 2))
    assert (reproj[good] <= 1e-3).all()
    assert (reproj[~good] <= S[~good] + 1e-6).all()      # the rest: explained by the one rounding of H to fp32


# ---- 8(f)-3: fp64 storage --------------------------------------------------------------------
@pytest.mark.parametrize("method", ["aca", "sks"])
@pytest.mark.parametrize("n,layout", [(4096, "soa"), (4097, "soa"), (1000, "aos"), (1, "aos")])
def test_f64_storage_matches_oracle(method, n, layout):
    s, d = W.general_sets(n, seed=W.SEED_BASE + 60 + n)
    s64, d64 = s.double(), d.double()
    fn = hg.hg_aca_batched_f64 if method == "aca" else hg.hg_sks_batched_f64
    if layout == "soa":
        H = fn(W.to_soa(s64).to(DEV), W.to_soa(d64).to(DEV), layout=hg.SOA, norm=hg.NORM_FROBENIUS).t().reshape(n, 3, 3)
    else:
        H = fn(s64.to(DEV), d64.to(DEV), layout=hg.AOS, norm=hg.NORM_FROBENIUS)
    H = H.cpu().numpy()
    H_ref = oracle.solve_f64(oracle.METHOD_ACA if method == "aca" else oracle.METHOD_SKS, s64.numpy(), d64.numpy())
    a, b = align_to(H, H_ref)
    # both sides fp64; they differ by FMA contraction and the reciprocal's last ulp, amplified by conditioning
    assert np.abs(a - b).max() <= (1e-11 if method == "aca" else 1e-9)
    assert np.abs(project(H, s.numpy()) - d.numpy().astype(np.float64)).max() <= 1e-7
    Hd = oracle.solve_f64(oracle.METHOD_DLT, s64.numpy(), d64.numpy())
    a, b = align_to(H, Hd)
    assert np.abs(a - b).max() <= 1e-9


# ---- 8(f)-4: hg_offsets_to_warp (reading R17) ---------------------------------------------------
# Tolerance: bilinear sampling is continuous in the sampling position with slope <= (max - min) of the image per
# pixel and axis; the fp32 sampling positions are within the grid tolerance (1e-3 px, typically 1e-5) of the oracle's.
@pytest.mark.parametrize("rect,ow,oh,iw,ih,C,n,max_off", [
    ((0.0, 0.0, 127.0, 127.0), 128, 128, 128, 128, 1, 24, 32.0),        # C5-shaped patches
    ((0.0, 0.0, 127.0, 127.0), 128, 128, 160, 144, 3, 5, 32.0),
    ((3.0, 2.0, 45.0, 30.0), 33, 21, 56, 40, 2, 9, 9.0),                 # odd width: scalar stores
    ((0.0, 0.0, 63.0, 31.0), 62, 30, 64, 32, 1, 3, 6.0),                 # width % 4 == 2
    ((0.0, 0.0, 255.0, 255.0), 256, 256, 256, 256, 1, 2, 40.0),          # plane too large to stage: gather form, row bands
    ((0.0, 0.0, 99.0, 79.0), 100, 80, 130, 90, 4, 7, 10.0),              # img_w % 4 != 0: staged by plain loads; 4 channels
    ((0.0, 0.0, 199.0, 199.0), 200, 200, 200, 200, 3, 2, 30.0),          # gather form, 3 channels
    ((0.0, 0.0, 127.0, 127.0), 128, 128, 128, 128, 3, 1, 60.0),          # one item: (channel, band) CTAs; large offsets -> frame taps
    ((0.0, 0.0, 127.0, 127.0), 128, 128, 128, 128, 1, 700, 32.0),        # large batches: several waves of (item, channel) CTAs
    ((0.0, 0.0, 63.0, 47.0), 64, 48, 72, 60, 3, 260, 14.0),
    ((2.0, 1.0, 40.0, 30.0), 35, 27, 48, 36, 2, 301, 8.0)])
def test_warp_matches_oracle(rect, ow, oh, iw, ih, C, n, max_off):
    off = W.offsets_workload(n, seed=W.SEED_BASE + 70 + ow, max_offset=max_off)
    img = torch.rand((n, C, ih, iw), generator=torch.Generator().manual_seed(ow), dtype=torch.float32)
    out, H = hg.hg_offsets_to_warp(off.to(DEV), *rect, ow, oh, img.to(DEV), want_H=True)
    ref = oracle.offsets_to_warp(off.numpy(), *rect, ow, oh, img.numpy())
    err = np.abs(out.cpu().numpy().astype(np.float64) - ref)
    assert err.max() <= 2e-3, err.max()                                  # 2 axes x 1e-3 px x range 1
    assert np.median(err) <= 1e-5
    Hg, _ = hg.hg_offsets_to_grid(off.to(DEV), *rect, ow, oh, want_grid=False)
    assert torch.equal(H, Hg)
    assert (ref != 0).mean() > 0.5


def test_warp_identity_translation_and_outside():
    img = torch.rand((3, 2, 128, 128), generator=torch.Generator().manual_seed(3)).to(DEV)
    zero = torch.zeros((3, 4, 2), device=DEV)
    out, _ = hg.hg_offsets_to_warp(zero, 0.0, 0.0, 127.0, 127.0, 128, 128, img)
    assert (out - img).abs().max().item() <= 2e-5
    sh = torch.zeros((3, 4, 2), device=DEV); sh[..., 0] = 5.0; sh[..., 1] = -7.0
    out, _ = hg.hg_offsets_to_warp(sh, 0.0, 0.0, 127.0, 127.0, 128, 128, img)
    exp = torch.zeros_like(img); exp[:, :, 7:, :123] = img[:, :, :121, 5:]
    assert (out - exp).abs().max().item() <= 1e-4
    far = torch.zeros((3, 4, 2), device=DEV); far[..., 0] = 1000.0
    out, _ = hg.hg_offsets_to_warp(far, 0.0, 0.0, 127.0, 127.0, 128, 128, img)
    assert torch.count_nonzero(out).item() == 0


# ---- 8(f)-4 "RANSAC extras": on-device sampling + adaptive termination (reading R19) ----------------------
def _adaptive_case(n_pts, inlier_frac, seed, max_hyp, round_hyp, conf, t=3.0):
    wl = W.ransac_workload(n_pts=n_pts, n_hyp=4, seed=W.SEED_BASE + 80 + n_pts, inlier_frac=inlier_frac)
    out = hg.hg_ransac_adaptive(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), seed, max_hyp, round_hyp, t, conf, want_idx=True)
    ref = oracle.ransac_adaptive(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), seed, max_hyp, round_hyp, t, conf)
    return wl, out, ref


@pytest.mark.parametrize("n_pts,frac,max_hyp,round_hyp,conf", [
    (4096, 0.7, 1 << 14, 512, 0.99),        # easy: stops after the first round
    (2000, 0.25, 1 << 15, 1024, 0.99),      # ~1200 samples needed: stops after a few rounds
    (1001, 0.12, 20000, 3000, 0.999),       # hard + ragged last round: runs to max_hyp or close
    (500, 0.5, 5000, 700, 0.0),             # confidence 0: never stops early
    (4, 1.0, 64, 16, 0.99)])                # tiny table: rejection sampling / fallback
def test_ransac_adaptive_matches_oracle(n_pts, frac, max_hyp, round_hyp, conf):
    wl, out, ref = _adaptive_case(n_pts, frac, 0xC0FFEE1234, max_hyp, round_hyp, conf)
    n, n_ref = int(out["n_evaluated"].item()), ref["n_evaluated"]
    m = min(n, n_ref)
    all_counts = out["counts"].cpu().numpy()
    # sampled indices: integer work, bit-exact (for every hypothesis both sides scored)
    assert np.array_equal(out["hyp_idx"].cpu().numpy()[:m], ref["hyp_idx"][:m])
    # counts of every hypothesis both sides scored: exact up to that hypothesis' in-band pairs
    counts = all_counts[:m]
    diff = np.abs(counts.astype(np.int64) - ref["counts"][:m])
    assert (diff <= ref["band_counts"][:m]).all()
    assert (all_counts[n:] == 0).all()                                      # entries past n_evaluated untouched

    # the stop rule of R19 in fp64: margin(done, best) = done * log1p(-(best/n_pts)^4) - log1p(-conf); stop iff <= 0
    c64 = float(np.float32(conf))
    def margin(done, best):
        with np.errstate(divide="ignore"):
            return done * np.log1p(-(best / n_pts) ** 4) - np.log1p(-c64)
    ends = list(range(round_hyp, max_hyp, round_hyp)) + [max_hyp]
    # (1) the kernel's own decisions follow the rule on its own counts: continue at every earlier round end, stop at n
    assert n in ends
    for d in ends:
        if d > n:
            break
        mg = margin(d, int(all_counts[:d].max())) if conf > 0 else np.inf
        if d < n:
            assert mg > -1e-9, ("continued although the rule says stop", d, mg)
        elif d < max_hyp:
            assert mg <= 1e-9, ("stopped although the rule says continue", d, mg)
    # (2) against the oracle: a different stop round is admissible only if, at the earlier of the two stops, the rule's
    # outcome depends on in-band pairs -- the best count lies in [max(count - band), max(count + band)] over the
    # hypotheses scored so far, and the margins at the two ends of that interval must straddle zero (1e-9: rounding of
    # the rule itself)
    if n != n_ref:
        rc, rb = ref["counts"][:m].astype(np.int64), ref["band_counts"][:m].astype(np.int64)
        lo, hi = int((rc - rb).max()), int((rc + rb).max())
        assert margin(m, hi) <= 1e-9 and margin(m, lo) >= -1e-9, (n, n_ref, lo, hi, margin(m, lo), margin(m, hi))
        return
    bi, bc = int(out["best_index"].item()), int(out["best_count"].item())
    assert bc == counts.max() and bi == int(np.argmax(counts))
    if (diff == 0).all():
        assert bi == ref["best_index"] and bc == ref["best_count"]
        Hb = out["best_H"].cpu().numpy().astype(np.float64).reshape(1, 3, 3)
        a, b = align_to(Hb, ref["best_H"].reshape(1, 3, 3))
        assert np.abs(a - b).max() <= 2e-7
    print(n_pts, frac, "n_evaluated", n, "of", max_hyp, "best", bc)


def test_ransac_adaptive_agrees_with_explicit_indices():
    """The sampled hypotheses scored through hg_ransac_hypothesize_score give the same counts."""
    wl, out, ref = _adaptive_case(3000, 0.3, 99, 1 << 13, 1 << 11, 0.0)
    idx = out["hyp_idx"]
    plain = hg.hg_ransac_hypothesize_score(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), idx, 3.0)
    assert torch.equal(plain["counts"], out["counts"])
    assert plain["best_index"].item() == out["best_index"].item()
    assert torch.equal(plain["best_H"], out["best_H"])


@pytest.mark.parametrize("n_pts,max_hyp,round_hyp", [(4, 10, 1000), (1001, 700, 5000), (37, 1, 1), (2049, 3000, 2999),
                                                     (1000, 1024, 1024), (500, 256, 1 << 20), (4096, 9472, 9472), (2000, 20480, 30000),
                                                     (4096, 9473, 9473)])
def test_ransac_adaptive_boundary_shapes(n_pts, max_hyp, round_hyp):
    """round_hyp > max_hyp (one ragged round), odd tables, the smallest table: same rule as the oracle's loop.  A single
    round on a small table is the one-kernel path with on-device sampling (the last case is just past its range)."""
    wl = W.ransac_workload(n_pts=n_pts, n_hyp=4, seed=W.SEED_BASE + 200 + n_pts, inlier_frac=0.6)
    out = hg.hg_ransac_adaptive(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), 42, max_hyp, round_hyp, 3.0, 0.0, want_idx=True)
    ref = oracle.ransac_adaptive(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), 42, max_hyp, round_hyp, 3.0, 0.0)
    assert int(out["n_evaluated"].item()) == ref["n_evaluated"] == max_hyp
    assert np.array_equal(out["hyp_idx"].cpu().numpy(), ref["hyp_idx"])
    diff = np.abs(out["counts"].cpu().numpy().astype(np.int64) - ref["counts"])
    assert (diff <= ref["band_counts"]).all()
    assert int(out["best_count"].item()) == int(out["counts"].max().item())


def test_combine_best_on_cuda_tensors_over_nccl():
    """The multi-GPU pick of the best hypothesis (sharding.combine_best) on device tensors through NCCL -- with the one
    GPU this box has, a world of size 1: it exercises the CUDA/NCCL code path, not scaling."""
    import os
    import torch.distributed as dist
    from paper_2402_18008_b200.sharding import combine_best, shard_range
    if dist.is_initialized():
        pytest.skip("a process group already exists in this process")
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29541")
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device(DEV, 0))
    try:
        wl = W.ransac_workload(n_pts=500, n_hyp=2000, seed=3)
        b, e = shard_range(2000, 0, 1)
        out = hg.hg_ransac_hypothesize_score(wl["src_xy"].to(DEV), wl["dst_xy"].to(DEV), wl["hyp_idx"][b:e].to(DEV), 3.0)
        c, i, H = combine_best(out["best_count"], out["best_index"] + b, out["best_H"])
        assert c.is_cuda and i.is_cuda and H.is_cuda
        assert int(c.item()) == int(out["best_count"].item()) and int(i.item()) == int(out["best_index"].item())
        assert torch.equal(H, out["best_H"])
    finally:
        dist.destroy_process_group()


def test_call_plan_replays_the_recorded_calls():
    """hg.CallPlan: the C calls recorded once (pointers, sizes, stream) and re-issued without the marshalling -- same results
    as fresh calls after the inputs were changed in place."""
    off = W.offsets_workload(1024, seed=3).to(DEV)
    H = torch.empty((1024, 3, 3), dtype=torch.float32, device=DEV)
    wl = W.ransac_workload(n_pts=1000, n_hyp=1024, seed=4)
    s, d, idx = (wl[k].to(DEV) for k in ("src_xy", "dst_xy", "hyp_idx"))
    with hg.CallPlan() as plan:
        hg.hg_offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128, H=H, want_grid=False, norm=hg.NORM_FROBENIUS)
        out = hg.hg_ransac_hypothesize_score(s, d, idx, 3.0)
        chk = hg.hg_ransac_hypothesize_score(s, d, idx, 3.0, reject_degenerate=True, min_area_px2=25.0)
    assert len(plan) == 3
    off2 = W.offsets_workload(1024, seed=5).to(DEV)
    wl2 = W.ransac_workload(n_pts=1000, n_hyp=1024, seed=6)
    off.copy_(off2); s.copy_(wl2["src_xy"]); d.copy_(wl2["dst_xy"]); idx.copy_(wl2["hyp_idx"])
    plan()
    plan()
    H_ref, _ = hg.hg_offsets_to_grid(off2, 0.0, 0.0, 127.0, 127.0, 128, 128, want_grid=False, norm=hg.NORM_FROBENIUS)
    assert torch.equal(H, H_ref)
    ref = hg.hg_ransac_hypothesize_score(s, d, idx, 3.0)
    ref_chk = hg.hg_ransac_hypothesize_score(s, d, idx, 3.0, reject_degenerate=True, min_area_px2=25.0)
    for a, b in ((out, ref), (chk, ref_chk)):
        assert torch.equal(a["counts"], b["counts"]) and torch.equal(a["best_H"], b["best_H"])
        assert a["best_index"].item() == b["best_index"].item()
    with pytest.raises(RuntimeError):
        with hg.CallPlan():
            with hg.CallPlan():
                pass


def test_call_plan_keeps_the_tensors_it_recorded_alive():
    """A recorded call holds raw addresses -- also of the tensors the wrapper allocated itself (counts, best_*, workspace).  The
    plan must keep them alive: after the caller drops the returned dict, memory handed out by the allocator must not be what a
    replay writes into."""
    import gc
    wl = W.ransac_workload(n_pts=1000, n_hyp=1024, seed=8)
    s, d, idx = (wl[k].to(DEV) for k in ("src_xy", "dst_xy", "hyp_idx"))
    off = W.offsets_workload(1024, seed=3).to(DEV)
    with hg.CallPlan() as plan:
        hg.hg_ransac_hypothesize_score(s, d, idx, 3.0)                                    # every output dropped on the spot
        hg.hg_offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 16, 16)                       # H and grid allocated by the wrapper, dropped
    gc.collect()
    kept = sum(t.numel() * t.element_size() for t in plan._keep if isinstance(t, torch.Tensor))
    assert kept >= 1024 * 4 + 1024 * 16 * 16 * 8                                          # counts + grid at least
    canary = [torch.full((4096,), 12345, dtype=torch.int32, device=DEV) for _ in range(128)]   # what the allocator hands out next
    torch.cuda.synchronize()
    plan(); plan()
    torch.cuda.synchronize()
    assert all(bool((c == 12345).all()) for c in canary)


# ---- 8(f) row 2, second half: backward through the grid --------------------------------------------------------------
# tolerance: the per-pixel partials and the per-thread sums are fp32 -- about 12 roundings per term
# plus a serial sum of <= 64 terms, |term| <= |g| * max|d grid / d offset| (< 2 for these quadrangles) -- the CTA
# reduction, the lattice unfolding and the reverse mode of Algorithm 1 are fp64 (dL/dG passes through fp32 once): worst case ~1e-5 * sum|g|;
# the sums average out -- measured 4e-9 (C5 shape) to 3e-7 (a 600 x 3 strip) -- and the tests assert 2e-6 * sum over the item of |g|.
@pytest.mark.parametrize("n,gw,gh,rect", [(96, 128, 128, (0.0, 0.0, 127.0, 127.0)),       # C5 shape
                                          (33, 37, 11, (5.0, -3.0, 36.0, 10.0)),            # odd width: 64-bit loads
                                          (7, 600, 3, (0.0, 0.0, 599.0, 2.0)),              # a row wider than four blocks
                                          (5, 1, 1, (2.0, 2.0, 8.0, 8.0)), (4, 2, 9, (0.0, 0.0, 1.0, 8.0))])
def test_grid_backward_matches_oracle(n, gw, gh, rect):
    g_cpu = torch.Generator().manual_seed(1000 + gw)
    off = W.offsets_workload(n, seed=W.SEED_BASE + 60 + gw) * (min(rect[2], rect[3]) / 127.0)
    g = torch.randn((n, gh, gw, 2), generator=g_cpu, dtype=torch.float32)
    go, gG = hg.hg_offsets_to_grid_backward(off.to(DEV), *rect, g.to(DEV), want_grad_G=True)
    ref = oracle.offsets_to_grid_backward(off.numpy(), *rect, g.numpy().astype(np.float64))
    scale = g.abs().sum(dim=(1, 2, 3)).numpy().astype(np.float64)[:, None, None]
    err = np.abs(go.cpu().numpy().astype(np.float64) - ref)
    assert np.isfinite(go.cpu().numpy()).all()
    assert (err <= 2e-6 * scale).all(), float((err / scale).max())
    # the intermediate dL/dG pulled back by the (separately tested) H backward gives the same thing
    via = hg.hg_aca_rect_backward(off.to(DEV), *rect, gG)
    assert (np.abs(via.cpu().numpy().astype(np.float64) - ref) <= 2e-6 * scale).all()
    print(n, gw, gh, "max |error| / sum|g| =", float((err / scale).max()), " max |grad| =", float(np.abs(ref).max()))


def test_grid_backward_full_config5_sampled_and_identities():
    """C5 at BASELINE size (8192 x 128 x 128 x 2 gradient, 1.07 GB) in the launch configuration bench.py times: every
    item checked by the translation identity (sum_k dL/d off_k = sum of g over the item, exact up to the fp32 sums), a
    strided sample of 64 items against the oracle, and a gradient living on the four corner pixels comes back unchanged."""
    n = 8192
    off = W.offsets_workload(n, seed=W.SEED_BASE + 5).to(DEV)
    g = torch.randn((n, 128, 128, 2), generator=torch.Generator(device=DEV).manual_seed(9), dtype=torch.float32, device=DEV)
    go = hg.hg_offsets_to_grid_backward(off, 0.0, 0.0, 127.0, 127.0, g)
    scale = g.abs().sum(dim=(1, 2, 3))
    assert torch.isfinite(go).all()
    assert ((go.sum(dim=1) - g.sum(dim=(1, 2))).abs().max(dim=1).values <= 1e-5 * scale).all()
    idx = torch.arange(0, n, n // 64)
    ref = oracle.offsets_to_grid_backward(off[idx].cpu().numpy(), 0.0, 0.0, 127.0, 127.0, g[idx].cpu().numpy().astype(np.float64))
    err = np.abs(go[idx].cpu().numpy().astype(np.float64) - ref)
    assert (err <= 2e-6 * scale[idx].cpu().numpy().astype(np.float64)[:, None, None]).all()
    gc = torch.zeros_like(g)
    corners = [(0, 0), (0, 127), (127, 127), (127, 0)]
    for (j, i) in corners:
        gc[:, j, i, :] = g[:, j, i, :]
    goc = hg.hg_offsets_to_grid_backward(off, 0.0, 0.0, 127.0, 127.0, gc)
    want = torch.stack([g[:, j, i, :] for (j, i) in corners], dim=1)
    assert (goc - want).abs().max().item() <= 2e-5 * want.abs().max().item()
