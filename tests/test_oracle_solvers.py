"""Pins of the fp64 oracle solvers (DLT-GE, ACA, SKS, closed form, Algorithm 1) against what the
paper and the mathematics fix -- never against the oracle itself and never against the CUDA path.
Every pin names the passage of /root/reference/PAPER.md ("P:<line>") or the DESIGN.md reading.
"""
import itertools
import random
from fractions import Fraction

import numpy as np
import pytest
import torch

import hg_workloads as W
import oracle
from exact_ref import defining_property_holds, exact_h_by_definition
from util import align_to

METHODS = {"dlt": oracle.METHOD_DLT, "aca": oracle.METHOD_ACA, "sks": oracle.METHOD_SKS,
           "closed": oracle.METHOD_CLOSED}


def project(H, pts):
    """pi(H [x;y;1]) in fp64; H [n,3,3], pts [n,4,2]."""
    p = np.concatenate([pts.astype(np.float64), np.ones(pts.shape[:-1] + (1,))], axis=-1)
    q = np.einsum("nij,nkj->nki", H, p)
    return q[..., :2] / q[..., 2:3]


@pytest.fixture(scope="module")
def general():
    s, d = W.general_sets(1 << 15, seed=W.SEED_BASE + 2)
    return s.numpy(), d.numpy()


# ---- (i) defining property, Eq. 1: H maps each source point onto its target ----------
@pytest.mark.parametrize("name", list(METHODS))
def test_defining_property(general, name):
    s, d = general
    H = oracle.solve(METHODS[name], s, d)
    err = np.abs(project(H, s) - d.astype(np.float64)).max()
    assert err <= 1e-9, (name, err)


# ---- (ii) all exact solvers of the minimal problem give the same H up to scale -----
def test_cross_method_equality(general):
    s, d = general
    Hs = {k: oracle.normal_form(oracle.solve(m, s, d)) for k, m in METHODS.items()}
    for a, b in itertools.combinations(Hs, 2):
        assert np.abs(Hs[a] - Hs[b]).max() <= 1e-9, (a, b)


# ---- brute force by the definition in exact rational arithmetic on tiny integer quads ----------
def _random_int_quads(rng, lim, count):
    out = []
    while len(out) < count:
        q = [(rng.randint(-lim, lim), rng.randint(-lim, lim)) for _ in range(8)]
        src, dst = q[:4], q[4:]
        ok = True
        for quad in (src, dst):
            for a, b, c in itertools.combinations(quad, 3):
                if (b[0] - a[0]) * (c[1] - a[1]) - (b[1] - a[1]) * (c[0] - a[0]) == 0:
                    ok = False
        if ok:
            out.append((src, dst))
    return out


def test_against_exact_rational_solution():
    rng = random.Random(2402)
    quads = _random_int_quads(rng, 16, 200)
    src = np.array([q[0] for q in quads], dtype=np.float32)
    dst = np.array([q[1] for q in quads], dtype=np.float32)
    exact = []
    keep = []
    for i, (s, d) in enumerate(quads):
        try:
            Hx = exact_h_by_definition(s, d)          # needs true h33 != 0
        except ZeroDivisionError:
            continue
        assert defining_property_holds(Hx, s, d)
        exact.append([[float(v) for v in row] for row in Hx])
        keep.append(i)
    assert len(keep) > 150
    exact = oracle.normal_form(np.array(exact))
    for name, m in METHODS.items():
        # (SKS included: no three points are collinear, so its five denominators are non-zero; its reciprocals round,
        # ACA / closed form are exact on these integers)
        H = oracle.normal_form(oracle.solve(m, src[keep], dst[keep]))
        assert np.abs(H - exact).max() <= 1e-11, name


def test_aca_is_exact_integer_polynomial():
    """(x) + Sec. 4.5: on small integers every intermediate of the 85-FLOP sequence is an
    exact integer < 2^53, so raw ACA equals the polynomial H exactly; that integer H satisfies the
    defining property exactly, and its ratio to the by-definition rational H is one common factor."""
    rng = random.Random(18008)
    quads = _random_int_quads(rng, 16, 200)
    src = np.array([q[0] for q in quads], dtype=np.float64)
    dst = np.array([q[1] for q in quads], dtype=np.float64)
    Ha = oracle.solve_f64(oracle.METHOD_ACA, src, dst)
    Hc = oracle.solve_f64(oracle.METHOD_CLOSED, src, dst)
    assert np.array_equal(Ha, np.round(Ha))
    assert np.array_equal(Ha, Hc)                         # two different evaluation orders, bit-equal
    for i, (s, d) in enumerate(quads):
        Hi = [[int(v) for v in row] for row in Ha[i]]
        assert defining_property_holds(Hi, s, d), i      # exact, in Python big ints


# ---- scale convention of the raw ACA output (Eq. 24, 28, 30-32; geometric meaning: doubled areas) -
def test_aca_raw_scale_and_core_structure(general):
    s, d = general
    s, d = s[:512], d[:512]
    H = oracle.aca(s, d)
    core = oracle.aca_core(s, d)
    hom = lambda p: np.concatenate([p.astype(np.float64), np.ones(p.shape[:-1] + (1,))], axis=-1)
    S, D = hom(s), hom(d)
    det = lambda a, b, c: np.linalg.det(np.stack([a, b, c], axis=-1))
    m1, n1, p1, q1 = (S[:, k] for k in range(4))
    m2, n2, p2, q2 = (D[:, k] for k in range(4))
    c33 = det(n2, p2, q2) * det(m1, q1, p1) * det(m1, n1, q1)      # reading R5
    c11 = det(n1, p1, q1) * det(m1, n1, q1) * det(m2, q2, p2)
    c22 = det(n1, p1, q1) * det(m1, q1, p1) * det(m2, n2, q2)
    ref = np.stack([c11, c22, c33], axis=1)
    assert np.abs(core / ref - 1).max() <= 1e-9
    # Proposition 4 / Eq. 26, 31: A2 * H * A1^-1 is the core transformation,
    # A_i = the affine map sending M_i,N_i,P_i to (0,0),(1,0),(0,1) (solved by the definition).
    canon = np.array([[0, 0, 1], [1, 0, 1], [0, 1, 1]], dtype=np.float64).T
    for i in range(64):
        A1 = canon @ np.linalg.inv(S[i, :3].T)
        A2 = canon @ np.linalg.inv(D[i, :3].T)
        C = A2 @ H[i] @ np.linalg.inv(A1)
        C = C / np.abs(C).max()
        assert abs(C[0, 1]) + abs(C[0, 2]) + abs(C[1, 0]) + abs(C[1, 2]) <= 1e-9
        assert abs(C[2, 0] - (C[0, 0] - C[2, 2])) <= 1e-9
        assert abs(C[2, 1] - (C[1, 1] - C[2, 2])) <= 1e-9
        k = core[i] / np.abs(core[i]).max()
        Cd = np.array([C[0, 0], C[1, 1], C[2, 2]])
        Cd = Cd / np.abs(Cd).max() * np.sign(Cd[np.abs(Cd).argmax()]) * np.sign(k[np.abs(k).argmax()])
        assert np.abs(Cd - k).max() <= 1e-9


# ---- (iii) identity ------------------------------------------------------------------------------
@pytest.mark.parametrize("name", list(METHODS))
def test_identity(general, name):
    s, _ = general
    H = oracle.normal_form(oracle.solve(METHODS[name], s[:2048], s[:2048]))
    I = np.eye(3) / np.sqrt(3.0)
    assert np.abs(H - I).max() <= 1e-9      # a dropped / mis-signed term would show at O(1)


# ---- (iv) affine configurations: Eq. 41, b_K = v_K = 0 ----------------------
def test_affine_configuration():
    g = torch.Generator().manual_seed(41)
    n = 2000
    src = (torch.randint(0, 640, (n, 4, 2), generator=g)).to(torch.float64)
    keep = W.min_triangle_area(src) >= W.MIN_AREA
    src = src[keep]
    n = src.shape[0]
    # integer affine maps keep the targets exactly representable in fp32
    A = torch.randint(-3, 4, (n, 2, 2), generator=g).to(torch.float64)
    A[:, 0, 0] += 5; A[:, 1, 1] += 5
    t = torch.randint(-50, 51, (n, 1, 2), generator=g).to(torch.float64)
    dst = src @ A.transpose(1, 2) + t
    keep = W.min_triangle_area(dst) >= W.MIN_AREA        # drops singular A
    src, dst, A, t = src[keep], dst[keep], A[keep], t[keep]
    n = src.shape[0]
    assert n > 1000
    s32, d32 = src.to(torch.float32).numpy(), dst.to(torch.float32).numpy()
    assert np.array_equal(d32.astype(np.float64), dst.numpy())
    expected = np.zeros((n, 3, 3))
    expected[:, :2, :2] = A.numpy()
    expected[:, :2, 2] = t.numpy()[:, 0]
    expected[:, 2, 2] = 1
    expected = oracle.normal_form(expected)
    for name, m in METHODS.items():
        H = oracle.solve(m, s32, d32)
        Hn = oracle.normal_form(H)
        assert np.abs(Hn[:, 2, :2]).max() <= 1e-12, name
        Ha, Er = align_to(H, expected)      # integer data: |t.x| == |t.y| ties make the sign rule ambiguous
        assert np.abs(Ha - Er).max() <= 1e-9, name
    core = oracle.aca_core(s32, d32)
    assert np.array_equal(core[:, 0], core[:, 2]) and np.array_equal(core[:, 1], core[:, 2])
    kern = oracle.sks_kernel(s32, d32)
    scale = np.abs(kern[:, [0, 2]]).max(axis=1)
    assert (np.abs(kern[:, 1]) <= 1e-11 * scale).all()
    assert (np.abs(kern[:, 3]) <= 1e-11 * scale).all()


# ---- (v) canonical anchors: H = H_C of Eq. 26 with a_C, b_C of Eq. 29 ---------------
def test_canonical_anchors():
    rng = np.random.default_rng(29)
    n = 500
    q1 = rng.uniform(0.2, 3.0, size=(n, 2)).astype(np.float32)
    q2 = rng.uniform(0.2, 3.0, size=(n, 2)).astype(np.float32)
    ok = (np.abs(1 - q1.sum(1)) > 0.1) & (np.abs(1 - q2.sum(1)) > 0.1)
    q1, q2 = q1[ok], q2[ok]
    n = q1.shape[0]
    anchors = np.array([[0, 0], [1, 0], [0, 1]], dtype=np.float32)
    s = np.concatenate([np.broadcast_to(anchors, (n, 3, 2)), q1[:, None]], axis=1)
    d = np.concatenate([np.broadcast_to(anchors, (n, 3, 2)), q2[:, None]], axis=1)
    Q3, Q4 = q1.astype(np.float64), q2.astype(np.float64)
    t1, t2 = 1 - Q3.sum(1), 1 - Q4.sum(1)
    aC = t1 * Q4[:, 0] / (t2 * Q3[:, 0])
    bC = t1 * Q4[:, 1] / (t2 * Q3[:, 1])
    HC = np.zeros((n, 3, 3))
    HC[:, 0, 0], HC[:, 1, 1] = aC, bC
    HC[:, 2, 0], HC[:, 2, 1], HC[:, 2, 2] = aC - 1, bC - 1, 1
    HC = oracle.normal_form(HC)
    for name in ("aca", "closed", "dlt"):
        H = oracle.normal_form(oracle.solve(METHODS[name], s, d))
        assert np.abs(H - HC).max() <= 1e-10, name


# ---- (vi) operation counts, Tables 3 and 4, counting rule P:193 ----------
def test_operation_counts():
    import json
    from pathlib import Path
    paper = json.loads((Path(__file__).parent / "golden" / "paper_constants.json").read_text())
    assert sum(paper["aca_table4"]["steps"].values()) == paper["aca_table4"]["sum"] == 85
    assert sum(paper["sks_table3"]["steps"].values()) == paper["sks_table3"]["sum"] == 157
    aca = oracle.op_counts(oracle.METHOD_ACA)
    assert aca["flops"] == paper["aca_table4"]["sum"] and aca["div"] == paper["aca_table4"]["divisions"]
    assert aca == {"add": 40, "mul": 45, "div": 0, "flops": 85}          # Table 4: 85, no division
    sks = oracle.op_counts(oracle.METHOD_SKS)
    # Table 3 prints 157; the formulas as printed (Eq. 6-16) evaluate in 160 with 5 reciprocals --
    # DESIGN.md reading R15.  11 of the 14 step counts of Table 3 are matched exactly.
    assert sks["div"] == 5 and sks["flops"] == 160
    # Algorithm 1 for a rectangle: 47 FLOPs; the 3 multiplications by r_rec vanish for a square (44)
    rect = oracle.op_counts(3)
    assert rect["flops"] == paper["aca_rect_flops"]["rectangle"] == 47 and rect["div"] == 0
    assert rect["flops"] - 3 == paper["aca_rect_flops"]["square"]


# ---- (vii) homogeneity degrees of the raw ACA output, Eq. 35 ------------------------
def test_homogeneity_degrees_bit_exact(general):
    s, d = general
    s, d = s[:4096].astype(np.float64), d[:4096].astype(np.float64)
    deg_src = np.array([[5, 5, 6]] * 3)
    deg_dst = np.array([[3, 3, 3], [3, 3, 3], [2, 2, 2]])
    import json
    from pathlib import Path
    paper = json.loads((Path(__file__).parent / "golden" / "paper_constants.json").read_text())
    assert np.array_equal(deg_src + deg_dst, np.array(paper["polynomial_degrees_eq35"]["total"]))  # Eq. 35
    for m in (oracle.METHOD_ACA, oracle.METHOD_CLOSED):
        H = oracle.solve_f64(m, s, d)
        for a, b in ((3, 0), (0, -2), (-4, 5)):
            H2 = oracle.solve_f64(m, s * 2.0 ** a, d * 2.0 ** b)
            assert np.array_equal(H2, H * 2.0 ** (a * deg_src + b * deg_dst)), (m, a, b)
    # every method: power-of-two scaling acts on H as diag(2^b,2^b,1) H diag(2^-a,2^-a,1)
    for m in METHODS.values():
        H = oracle.solve_f64(m, s, d)
        a, b = 3, -2
        H2 = oracle.normal_form(oracle.solve_f64(m, s * 2.0 ** a, d * 2.0 ** b))
        T = np.diag([2.0 ** b, 2.0 ** b, 1.0]) @ H @ np.diag([2.0 ** -a, 2.0 ** -a, 1.0])
        assert np.abs(H2 - oracle.normal_form(T)).max() <= 1e-13, m


# ---- (viii) the 24 relabelings of the correspondences give the same H (App. B) ----------
def test_relabeling_invariance(general):
    s, d = general
    s, d = s[:1024], d[:1024]
    ref = oracle.normal_form(oracle.dlt(s, d))
    for perm in itertools.permutations(range(4)):
        p = list(perm)
        for name in ("aca", "sks", "closed"):
            H = oracle.normal_form(oracle.solve(METHODS[name], s[:, p], d[:, p]))
            assert np.abs(H - ref).max() <= 1e-9, (name, perm)


def test_rectangle_all_vertex_orders():
    """App. B: RHO-GE divides by zero on 8 of the 24 orders of a rectangle; ACA/SKS/DLT must not.
    (SKS is singular only when P or Q lies on the anchor line MN, which no vertex order of a rectangle
    produces.)"""
    src = np.array([[0, 0], [127, 0], [127, 127], [0, 127]], dtype=np.float32)
    off = W.offsets_workload(64, seed=7).numpy()
    for perm in itertools.permutations(range(4)):
        p = list(perm)
        s = np.broadcast_to(src[p], (64, 4, 2)).copy()
        d = s + off[:, p]
        ref = oracle.normal_form(oracle.dlt(s, d))
        for name in ("aca", "sks", "closed"):
            H = oracle.solve(METHODS[name], s, d)
            assert np.isfinite(H).all(), (name, perm)
            assert np.abs(oracle.normal_form(H) - ref).max() <= 1e-10, (name, perm)


# ---- (ix) swapping source and target gives the inverse homography -------------------------------
@pytest.mark.parametrize("name", list(METHODS))
def test_swap_gives_inverse(general, name):
    s, d = general
    s, d = s[:2048], d[:2048]
    H = oracle.solve(METHODS[name], s, d)
    Hi = oracle.solve(METHODS[name], d, s)
    P = np.einsum("nij,njk->nik", oracle.normal_form(Hi), oracle.normal_form(H))
    P = oracle.normal_form(P)
    assert np.abs(P - np.eye(3) / np.sqrt(3)).max() <= 1e-8


# ---- degenerate input (reading R8): ACA stays finite, DLT reports the zero pivot ---------------
def test_degenerate_collinear():
    s = np.array([[[0, 0], [10, 0], [20, 0], [5, 7]]], dtype=np.float32)   # M, N, P collinear
    d = np.array([[[1, 1], [11, 2], [3, 9], [8, 8]]], dtype=np.float32)
    H = oracle.aca(s, d)
    assert np.isfinite(H).all()
    assert abs(np.linalg.det(H[0] / np.abs(H[0]).max())) <= 1e-12           # singular H
    _, ok = oracle.solve(oracle.METHOD_DLT, s, d, return_ok=True)
    assert not ok[0]
    s2 = np.array([[[0, 0], [10, 0], [5, 0], [5, 7]]], dtype=np.float32)    # P on the anchor line MN
    assert not np.isfinite(oracle.sks(s2, d)).all()                        # SKS divides by P3.y = 0


# ---- Algorithm 1 / Eq. 42-45: rectangle fast path equals general ACA ----------------
@pytest.mark.parametrize("rect", [(0.0, 0.0, 127.0, 127.0), (16.0, 40.0, 300.0, 120.0)])
def test_algorithm1_equals_general_aca(rect):
    x0, y0, w, h = rect
    off = W.offsets_workload(1024, seed=W.SEED_BASE + 1).numpy()
    # the instance is (rectangle, offsets): targets are corner + offset in exact (fp64) arithmetic
    src = np.broadcast_to(W.patch_corners(x0, y0, w, h).numpy().astype(np.float64), (1024, 4, 2)).copy()
    dst = src + off.astype(np.float64)
    H1 = oracle.aca_rect(off, x0, y0, w, h)
    assert np.abs(project(H1, src) - dst).max() <= 1e-9                       # defining property
    Hd = oracle.normal_form(oracle.solve_f64(oracle.METHOD_DLT, src, dst))
    assert np.abs(oracle.normal_form(H1) - Hd).max() <= 1e-11
    Ha = oracle.normal_form(oracle.solve_f64(oracle.METHOD_ACA, src, dst))
    assert np.abs(oracle.normal_form(H1) - Ha).max() <= 1e-12


# ---- normal form (comparison form of DESIGN.md) --------------------------------------------------
def test_normal_form_properties(general):
    s, d = general
    H = oracle.aca(s[:1000], d[:1000])
    Hn = oracle.normal_form(H)
    assert np.abs(np.sqrt((Hn ** 2).sum(axis=(1, 2))) - 1).max() <= 1e-14
    flat = Hn.reshape(-1, 9)
    assert (flat[np.arange(len(flat)), np.abs(flat).argmax(1)] > 0).all()
    assert np.abs(oracle.normal_form(-3.5e20 * H) - Hn).max() <= 1e-15        # scale and sign free
