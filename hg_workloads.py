"""Seeded synthetic workloads (BASELINE.json configs C1..C5; recipe in DESIGN.md "Inputs").

This module serves both the oracle and the CUDA path and holds NONE of the method's
arithmetic: it only draws points, applies a ground-truth projective map to synthesise
targets, adds noise and filters degenerate quads.  fp32 arrays are the canonical problem
instance; whichever side did not generate them receives a copy.

All generators are torch-based and run on the device they are given (CPU for the oracle
tests, CUDA for the 2^26 bench).  The CPU and CUDA generators are different random streams:
a workload is defined by (function, arguments, seed, device type).

AoS layouts: src, dst float32 [n,4,2]; SoA: float32 [8,n] planes x0,y0,x1,y1,x2,y2,x3,y3.
"""
from __future__ import annotations

import math

import torch

SEED_BASE = 240218008          # + config number
IMG_W, IMG_H = 640.0, 480.0    # image size of the paper's RANSAC experiment
PATCH = 127.0                  # 128x128 patch: corners (0,0),(127,0),(127,127),(0,127)
MIN_AREA = 100.0               # px^2, every triangle of both quads (reading R13)


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def patch_corners(x0: float = 0.0, y0: float = 0.0, w: float = PATCH, h: float = PATCH,
                  device="cpu") -> torch.Tensor:
    """Corners TL, TR, BR, BL of the source rectangle, float32 [4,2]."""
    return torch.tensor([[x0, y0], [x0 + w, y0], [x0 + w, y0 + h], [x0, y0 + h]],
                        dtype=torch.float32, device=device)


def offsets_workload(n: int, seed: int = SEED_BASE + 1, max_offset: float = 32.0,
                     device="cpu") -> torch.Tensor:
    """C1 / C5: i.i.d. uniform corner offsets in [-max_offset, max_offset] px, float32 [n,4,2]."""
    g = _gen(seed, device)
    u = torch.rand((n, 4, 2), generator=g, device=device, dtype=torch.float32)
    return (u * 2.0 - 1.0) * max_offset


def offsets_to_sets(offsets: torch.Tensor, x0=0.0, y0=0.0, w=PATCH, h=PATCH):
    """(src, dst) float32 [n,4,2] of an offsets workload: src = rectangle corners, dst = src + offsets."""
    c = patch_corners(x0, y0, w, h, device=offsets.device)
    src = c.unsqueeze(0).expand(offsets.shape[0], 4, 2).contiguous()
    return src, (src + offsets).contiguous()


def random_h_gt(n: int, g: torch.Generator, device, persp_sigma: float = 1e-4) -> torch.Tensor:
    """Ground-truth homographies float64 [n,3,3] (reading R13):
    H_gt = C * [[s R(theta) [[1,k],[0,1]], t], [v^T, 1]] * C^-1, C = translate(320,240);
    theta in +-30 deg, s in [0.8,1.2], shear k in +-0.1, t in +-50 px, v ~ N(0, persp_sigma^2)."""
    r = torch.rand((n, 5), generator=g, device=device, dtype=torch.float64)
    theta = (r[:, 0] * 2 - 1) * math.radians(30.0)
    s = 0.8 + 0.4 * r[:, 1]
    k = (r[:, 2] * 2 - 1) * 0.1
    tx = (r[:, 3] * 2 - 1) * 50.0
    ty = (r[:, 4] * 2 - 1) * 50.0
    v = torch.randn((n, 2), generator=g, device=device, dtype=torch.float64) * persp_sigma
    c, sn = torch.cos(theta), torch.sin(theta)
    A = torch.zeros((n, 3, 3), dtype=torch.float64, device=device)
    A[:, 0, 0] = s * c
    A[:, 0, 1] = s * (c * k - sn)
    A[:, 1, 0] = s * sn
    A[:, 1, 1] = s * (sn * k + c)
    A[:, 0, 2] = tx
    A[:, 1, 2] = ty
    A[:, 2, 0] = v[:, 0]
    A[:, 2, 1] = v[:, 1]
    A[:, 2, 2] = 1.0
    C = torch.eye(3, dtype=torch.float64, device=device)
    C[0, 2], C[1, 2] = IMG_W / 2, IMG_H / 2
    Ci = torch.eye(3, dtype=torch.float64, device=device)
    Ci[0, 2], Ci[1, 2] = -IMG_W / 2, -IMG_H / 2
    return C @ A @ Ci


def apply_h(H: torch.Tensor, pts: torch.Tensor) -> torch.Tensor:
    """pi(H * [x;y;1]) for pts [...,k,2] with H [...,3,3] (float64)."""
    x, y = pts[..., 0], pts[..., 1]
    X = H[..., 0, 0, None] * x + H[..., 0, 1, None] * y + H[..., 0, 2, None]
    Y = H[..., 1, 0, None] * x + H[..., 1, 1, None] * y + H[..., 1, 2, None]
    W = H[..., 2, 0, None] * x + H[..., 2, 1, None] * y + H[..., 2, 2, None]
    return torch.stack((X / W, Y / W), dim=-1)


def min_triangle_area(q: torch.Tensor) -> torch.Tensor:
    """Smallest area of the 4 triangles of each quad q [n,4,2] (any dtype), float64 [n]."""
    q = q.to(torch.float64)
    best = None
    for (a, b, c) in ((0, 1, 2), (0, 1, 3), (0, 2, 3), (1, 2, 3)):
        ab = q[:, b] - q[:, a]
        ac = q[:, c] - q[:, a]
        area = 0.5 * (ab[:, 0] * ac[:, 1] - ab[:, 1] * ac[:, 0]).abs()
        best = area if best is None else torch.minimum(best, area)
    return best


def _draw_general(n: int, g: torch.Generator, device, noise_sigma: float, persp_sigma: float):
    src = torch.rand((n, 4, 2), generator=g, device=device, dtype=torch.float64)
    src[..., 0] *= IMG_W
    src[..., 1] *= IMG_H
    src = src.to(torch.float32)                     # the fp32 array is the instance
    H = random_h_gt(n, g, device, persp_sigma)
    dst = apply_h(H, src.to(torch.float64))
    dst = dst + torch.randn((n, 4, 2), generator=g, device=device, dtype=torch.float64) * noise_sigma
    return src, dst.to(torch.float32)


def general_sets(n: int, seed: int = SEED_BASE + 2, device="cpu", noise_sigma: float = 1.0,
                 persp_sigma: float = 1e-4, chunk: int = 1 << 22, soa: bool = False):
    """C2 / C3: random general-position correspondences (recipe R13).  Sets whose source or
    (noisy) target quad has a triangle of area < MIN_AREA are redrawn.
    Returns (src, dst) float32 [n,4,2], or [8,n] planes each when soa=True."""
    g = _gen(seed, device)
    if soa:
        src_out = torch.empty((8, n), dtype=torch.float32, device=device)
        dst_out = torch.empty((8, n), dtype=torch.float32, device=device)
    else:
        src_out = torch.empty((n, 4, 2), dtype=torch.float32, device=device)
        dst_out = torch.empty((n, 4, 2), dtype=torch.float32, device=device)
    for a in range(0, n, chunk):
        m = min(chunk, n - a)
        src, dst = _draw_general(m, g, device, noise_sigma, persp_sigma)
        for _ in range(64):
            bad = (torch.minimum(min_triangle_area(src), min_triangle_area(dst)) < MIN_AREA)
            nb = int(bad.sum())
            if nb == 0:
                break
            s2, d2 = _draw_general(nb, g, device, noise_sigma, persp_sigma)
            src[bad] = s2
            dst[bad] = d2
        else:
            raise RuntimeError("area filter did not converge")
        if soa:
            src_out[:, a:a + m] = src.reshape(m, 8).t()
            dst_out[:, a:a + m] = dst.reshape(m, 8).t()
        else:
            src_out[a:a + m] = src
            dst_out[a:a + m] = dst
    return src_out, dst_out


def to_soa(a: torch.Tensor) -> torch.Tensor:
    """[n,4,2] -> [8,n] planes (x0,y0,...,x3,y3)."""
    return a.reshape(a.shape[0], 8).t().contiguous()


def to_aos(a: torch.Tensor) -> torch.Tensor:
    """[8,n] planes -> [n,4,2]."""
    return a.t().contiguous().reshape(a.shape[1], 4, 2)


def h_soa_to_aos(H: torch.Tensor) -> torch.Tensor:
    """[9,n] planes h11..h33 -> [n,3,3]."""
    return H.t().contiguous().reshape(H.shape[1], 3, 3)


def ransac_workload(n_pts: int = 4096, n_hyp: int = 1 << 20, seed: int = SEED_BASE + 4,
                    inlier_frac: float = 0.7, noise_var: float = 0.5, device="cpu"):
    """C4: n_pts correspondences in a 640x480 image, inlier_frac of them
    dst = H_gt(src) + N(0, noise_var px^2), the rest src, dst independent uniform;
    n_hyp hypotheses of 4 distinct int32 indices.
    Returns dict(src_xy [n_pts,2] f32, dst_xy [n_pts,2] f32, hyp_idx [n_hyp,4] i32,
                 inlier_mask [n_pts] bool, H_gt [3,3] f64)."""
    g = _gen(seed, device)
    H = random_h_gt(1, g, device)[0]
    src = torch.rand((n_pts, 2), generator=g, device=device, dtype=torch.float64)
    src[:, 0] *= IMG_W
    src[:, 1] *= IMG_H
    src = src.to(torch.float32)
    dst_in = apply_h(H, src.to(torch.float64).unsqueeze(0))[0]
    dst_in = dst_in + torch.randn((n_pts, 2), generator=g, device=device,
                                  dtype=torch.float64) * math.sqrt(noise_var)
    dst_out = torch.rand((n_pts, 2), generator=g, device=device, dtype=torch.float64)
    dst_out[:, 0] *= IMG_W
    dst_out[:, 1] *= IMG_H
    perm = torch.randperm(n_pts, generator=g, device=device)
    mask = torch.zeros(n_pts, dtype=torch.bool, device=device)
    mask[perm[: int(round(inlier_frac * n_pts))]] = True
    dst = torch.where(mask[:, None], dst_in, dst_out).to(torch.float32)
    idx = distinct_indices(n_hyp, n_pts, g, device)
    return {"src_xy": src.contiguous(), "dst_xy": dst.contiguous(), "hyp_idx": idx,
            "inlier_mask": mask, "H_gt": H}


def distinct_indices(n_hyp: int, n_pts: int, g: torch.Generator, device) -> torch.Tensor:
    """int32 [n_hyp,4], the 4 indices of a row pairwise distinct, uniform in [0,n_pts)."""
    assert n_pts >= 4
    idx = torch.randint(0, n_pts, (n_hyp, 4), generator=g, device=device, dtype=torch.int64)
    for _ in range(256):
        srt, _ = idx.sort(dim=1)
        bad = (srt[:, 1:] == srt[:, :-1]).any(dim=1)
        nb = int(bad.sum())
        if nb == 0:
            break
        idx[bad] = torch.randint(0, n_pts, (nb, 4), generator=g, device=device, dtype=torch.int64)
    else:
        raise RuntimeError("distinct index draw did not converge")
    return idx.to(torch.int32).contiguous()
