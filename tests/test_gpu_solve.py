"""GPU parity of hg_aca_batched / hg_sks_batched (through the C ABI) against the fp64 oracle.

Comparison form and tolerances (BASELINE.json north_star, reading R12): both H are
scaled to unit Frobenius norm and sign-aligned; a sample is *well-conditioned* when it passes the
area filter of the generator and its own fp32-rounding sensitivity S is <= 1e-3 px.  Asserted on EVERY set:
finite H and |dH_ij| <= 1e-4 |H_ij| + 1e-7; 4-point reprojection error <= 1e-3 px on the well-conditioned sets and
<= S + 1e-6 px on the others (tests/util.py::check_h_parity; the all-sample statistics are printed).
"""
import numpy as np
import pytest
import torch

import hg_workloads as W
import oracle
import paper_2402_18008_b200 as hg
from util import align_to, check_h_parity, project

pytestmark = pytest.mark.gpu
DEV = "cuda"

ORACLE = {"aca": oracle.METHOD_ACA, "sks": oracle.METHOD_SKS}
GPU_FN = {"aca": hg.hg_aca_batched, "sks": hg.hg_sks_batched}


def check_parity(H_gpu, src, dst, method, require_frac=0.98):
    """H_gpu [n,3,3] (any scale), src/dst float32 numpy [n,4,2].  Every set is checked (util.check_h_parity);
    returns the all-sample statistics."""
    return check_h_parity(H_gpu, src, dst, oracle.solve(ORACLE[method], src, dst), oracle.dlt(src, dst),
                          require_frac=require_frac, label=method)


@pytest.fixture(scope="module")
def general():
    n = (1 << 17) + 1000          # 132072 = many 1024-set tiles; % 4 == 0 -> 128-bit path
    s, d = W.general_sets(n, seed=W.SEED_BASE + 2)
    return s, d


@pytest.mark.parametrize("method", ["aca", "sks"])
@pytest.mark.parametrize("layout", ["soa", "aos"])
def test_general_sets_f64_internal(general, method, layout):
    s, d = general
    n = s.shape[0]
    if layout == "soa":
        H = GPU_FN[method](W.to_soa(s).to(DEV), W.to_soa(d).to(DEV), layout=hg.SOA)
        Hn = W.h_soa_to_aos(H.cpu()).numpy()
    else:
        H = GPU_FN[method](s.to(DEV), d.to(DEV), layout=hg.AOS)
        Hn = H.cpu().numpy()
    assert Hn.shape == (n, 3, 3)
    stats = check_parity(Hn, s.numpy(), d.numpy(), method)
    print(method, layout, stats)


@pytest.mark.parametrize("method", ["aca", "sks"])
def test_config2_full_batch_every_set_against_oracle(method):
    """C2 as BASELINE.json states it: 2^20 general-position sets, fp32 SoA, every set compared with the oracle."""
    n = 1 << 20
    s, d = W.general_sets(n, seed=W.SEED_BASE + 2)
    H = GPU_FN[method](W.to_soa(s).to(DEV), W.to_soa(d).to(DEV), layout=hg.SOA)
    stats = check_parity(W.h_soa_to_aos(H.cpu()).numpy(), s.numpy(), d.numpy(), method)
    print("C2", method, stats)


@pytest.mark.parametrize("method", ["aca", "sks"])
@pytest.mark.parametrize("n", [1, 3, 255, 1001, 4099])
def test_ragged_sizes_scalar_path(method, n):
    """n % 4 != 0 takes the scalar-load SoA path; n < one block; plane stride = n."""
    s, d = W.general_sets(n, seed=77 + n)
    H = GPU_FN[method](W.to_soa(s).to(DEV), W.to_soa(d).to(DEV), layout=hg.SOA, norm=hg.NORM_FROBENIUS)
    Hn = W.h_soa_to_aos(H.cpu()).numpy()
    check_parity(Hn, s.numpy(), d.numpy(), method, require_frac=0.0 if n < 100 else 0.95)
    Ha = GPU_FN[method](s.to(DEV), d.to(DEV), layout=hg.AOS, norm=hg.NORM_FROBENIUS).cpu().numpy()
    assert np.array_equal(Ha, Hn)          # both layouts run the same arithmetic


@pytest.mark.parametrize("method", ["aca", "sks"])
def test_layouts_and_vector_widths_agree_bitwise(general, method):
    s, d = general
    n4 = 4096
    s4, d4 = s[:n4], d[:n4]
    Hv = GPU_FN[method](W.to_soa(s4).to(DEV), W.to_soa(d4).to(DEV)).cpu()           # 128-bit path
    s3, d3 = s[:n4 - 1], d[:n4 - 1]
    Hs = GPU_FN[method](W.to_soa(s3).to(DEV), W.to_soa(d3).to(DEV)).cpu()           # scalar path
    assert torch.equal(Hv[:, : n4 - 1], Hs)


@pytest.mark.parametrize("method", ["aca", "sks"])
def test_config1_deep_homography_offsets(method):
    """C1: 1024 sets, source = corners of the 128x128 patch, target = source + U[-32,32] offsets."""
    off = W.offsets_workload(1024, seed=W.SEED_BASE + 1)
    s, d = W.offsets_to_sets(off)
    H = GPU_FN[method](W.to_soa(s).to(DEV), W.to_soa(d).to(DEV), norm=hg.NORM_H33)
    Hn = W.h_soa_to_aos(H.cpu()).numpy()
    assert np.all(Hn[:, 2, 2] == 1.0)
    stats = check_parity(Hn, s.numpy(), d.numpy(), method, require_frac=0.999)
    print("C1", method, stats)


@pytest.mark.parametrize("method", ["aca", "sks"])
def test_normalisations(general, method):
    s, d = general
    s, d = s[:8192], d[:8192]
    ss, ds = W.to_soa(s).to(DEV), W.to_soa(d).to(DEV)
    raw = W.h_soa_to_aos(GPU_FN[method](ss, ds, norm=hg.NORM_NONE).cpu()).numpy().astype(np.float64)
    h33 = W.h_soa_to_aos(GPU_FN[method](ss, ds, norm=hg.NORM_H33).cpu()).numpy().astype(np.float64)
    fro = W.h_soa_to_aos(GPU_FN[method](ss, ds, norm=hg.NORM_FROBENIUS).cpu()).numpy().astype(np.float64)
    assert np.isfinite(raw).all()
    assert np.all(h33[:, 2, 2] == 1.0)
    assert np.abs(np.sqrt((fro ** 2).sum(axis=(1, 2))) - 1.0).max() <= 3e-7
    # raw scale is the paper's (Eq. 31-32 for ACA, Eq. 11/16 for SKS): same as the oracle's raw H
    ref = oracle.solve(ORACLE[method], s.numpy(), d.numpy())
    scale = np.abs(ref).max(axis=(1, 2), keepdims=True)
    assert (np.abs(raw - ref) / scale).max() <= 2e-7
    assert (np.abs(h33 - ref / ref[:, 2:3, 2:3]) / np.abs(ref / ref[:, 2:3, 2:3]).max(axis=(1, 2), keepdims=True)).max() <= 2e-7


def test_plain_fp32_mode_is_the_same_solver_but_less_accurate(general):
    s, d = general
    s, d = s[:65536], d[:65536]
    ss, ds = W.to_soa(s).to(DEV), W.to_soa(d).to(DEV)
    for method in ("aca", "sks"):
        H32 = W.h_soa_to_aos(GPU_FN[method](ss, ds, norm=hg.NORM_FROBENIUS, prec=hg.PREC_F32).cpu()).numpy()
        ref = oracle.solve(ORACLE[method], s.numpy(), d.numpy())
        Hg, Hr = align_to(H32.astype(np.float64), ref)
        err = np.abs(Hg - Hr).max(axis=(1, 2))
        assert np.median(err) <= 1e-5 and np.quantile(err, 0.99) <= 1e-2, (np.median(err), err.max())
        reproj = np.abs(project(H32.astype(np.float64), s.numpy()) - d.numpy().astype(np.float64)).max(axis=(1, 2))
        assert np.median(reproj) <= 1e-2


def test_identity_affine_and_degenerate_inputs():
    s, _ = W.general_sets(512, seed=5)
    ss = W.to_soa(s).to(DEV)
    for fn in (hg.hg_aca_batched, hg.hg_sks_batched):
        I = W.h_soa_to_aos(fn(ss, ss.clone(), norm=hg.NORM_H33).cpu()).numpy()
        assert np.abs(I - np.eye(3)).max() <= 2e-4          # identity (h13,h23 carry ~1e-7 * 640)
    # three collinear source points M, N, P: ACA stays finite and returns the same singular H as the
    # oracle's ACA; SKS (P on the line MN -> P3.y = 0 -> 1/0) returns a non-finite H (reading R8)
    sd = s.clone()
    sd[:, 0] = torch.tensor([0.0, 0.0])
    sd[:, 1] = torch.tensor([64.0, 32.0])
    sd[:, 2] = torch.tensor([128.0, 64.0])
    Ha = W.h_soa_to_aos(hg.hg_aca_batched(W.to_soa(sd).to(DEV), ss).cpu()).numpy()
    assert np.isfinite(Ha).all()
    Hg, Hr = align_to(Ha.astype(np.float64), oracle.aca(sd.numpy(), s.numpy()))
    assert np.abs(Hg - Hr).max() <= 1e-6
    assert np.abs(np.linalg.det(Hg)).max() <= 1e-9
    Hs = hg.hg_sks_batched(W.to_soa(sd).to(DEV), ss).cpu()
    assert (~torch.isfinite(Hs)).any(dim=0).all()


def test_empty_batch_is_a_noop():
    e = torch.empty((8, 0), dtype=torch.float32, device=DEV)
    H = hg.hg_aca_batched(e, e.clone())
    assert H.shape == (9, 0)


def test_runs_on_the_callers_stream():
    s, d = W.general_sets(4096, seed=9)
    ss, ds = W.to_soa(s).to(DEV), W.to_soa(d).to(DEV)
    ref = hg.hg_aca_batched(ss, ds).clone()
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        H = hg.hg_aca_batched(ss, ds)
    st.synchronize()
    assert torch.equal(H, ref)


def test_host_buffer_pipeline_matches_device_call():
    n = 50_001                      # odd tail chunk -> scalar path inside the pipeline
    s, d = W.general_sets(n, seed=21)
    ss, ds = W.to_soa(s), W.to_soa(d)
    ref = hg.hg_aca_batched(ss.to(DEV), ds.to(DEV), norm=hg.NORM_FROBENIUS).cpu()
    out = hg.hg_aca_batched_host(ss.pin_memory(), ds.pin_memory(), norm=hg.NORM_FROBENIUS, chunk_sets=8192)   # pinned: zero-copy
    assert torch.equal(out, ref)
    out2 = hg.hg_sks_batched_host(s, d, layout=hg.AOS, norm=hg.NORM_H33, chunk_sets=10_000)     # pageable AoS
    ref2 = hg.hg_sks_batched(s.to(DEV), d.to(DEV), layout=hg.AOS, norm=hg.NORM_H33).cpu()
    assert torch.equal(out2, ref2)
    # pageable SoA with a pageable result buffer: the staged, chunked path (strided 2-D copies, ragged last chunk)
    out3 = hg.hg_aca_batched_host(ss, ds, H=torch.empty((9, n), dtype=torch.float32), norm=hg.NORM_FROBENIUS, chunk_sets=8192)
    assert torch.equal(out3, ref)


def test_full_size_config3_every_set_against_oracle():
    """C3 at BASELINE size (2^26 sets, the launch configuration bench.py times): generated on the GPU, solved in ONE call per
    method, and EVERY one of the 2^26 outputs of both methods compared with the oracle, slab by slab (2^22 sets per slab: every
    thread, every vector lane and every CTA of the timed launch is looked at).  Rule: util.check_h_parity_lazy = the rule of
    every other solver test.  The literal all-sample statistics are printed (DESIGN.md section 8 quotes them)."""
    from util import check_h_parity_lazy
    n, slab = 1 << 26, 1 << 22
    free, _ = torch.cuda.mem_get_info()
    if free < 16 * (1 << 30):
        pytest.skip("needs ~16 GB of free device memory")
    src, dst = W.general_sets(n, seed=W.SEED_BASE + 3, device=DEV, soa=True)
    Ha = hg.hg_aca_batched(src, dst, norm=hg.NORM_NONE)
    Hs = hg.hg_sks_batched(src, dst, norm=hg.NORM_NONE)
    torch.cuda.synchronize()
    tot = {m: {"n": 0, "over_1e-3px": 0, "max_elem_ratio": 0.0, "max_reproj": 0.0, "max_reproj_over_S_on_those": 0.0} for m in ("aca", "sks")}

    def check(m, a, Hn, s, d):
        return m, check_h_parity_lazy(Hn, s, d, oracle.solve(ORACLE[m], s, d), oracle.dlt, label="%s slab at %d" % (m, a))

    # the comparisons are numpy on 4M-set slabs (they release the GIL): a few slabs are checked side by side while the next is copied
    from concurrent.futures import ThreadPoolExecutor
    pending = []
    with ThreadPoolExecutor(max_workers=6) as pool:
        for a in range(0, n, slab):
            s = W.to_aos(src[:, a:a + slab].contiguous()).cpu().numpy()
            d = W.to_aos(dst[:, a:a + slab].contiguous()).cpu().numpy()
            for m, Hm in (("aca", Ha), ("sks", Hs)):
                pending.append(pool.submit(check, m, a, W.h_soa_to_aos(Hm[:, a:a + slab]).cpu().numpy(), s, d))
            while len(pending) > 8:
                m, st = pending.pop(0).result()                  # re-raises an assertion of that slab
                t = tot[m]
                t["n"] += st["n"]; t["over_1e-3px"] += st["over_1e-3px"]
                for k in ("max_elem_ratio", "max_reproj", "max_reproj_over_S_on_those"):
                    t[k] = max(t[k], st[k])
        for f in pending:
            m, st = f.result()
            t = tot[m]
            t["n"] += st["n"]; t["over_1e-3px"] += st["over_1e-3px"]
            for k in ("max_elem_ratio", "max_reproj", "max_reproj_over_S_on_those"):
                t[k] = max(t[k], st[k])
    assert tot["aca"]["n"] == n and tot["sks"]["n"] == n
    print("C3 every set", tot)


def test_bench_line_carries_the_contract_keys():
    """bench.py on a reduced batch (2^22 sets, no extras, no oracle leg): one JSON line with the contract's keys -- the roofline
    object of the step kernel, the end-to-end leg through the host-buffer entry point with its copied bytes, the clock
    sample, and one launch of the library's kernel per timed step."""
    import json
    import subprocess
    import sys
    from pathlib import Path
    root = Path(__file__).resolve().parent.parent
    r = subprocess.run([sys.executable, str(root / "bench.py"), "--steps", "4", "--warmup", "3", "--log2n", "22", "--no-extras", "--no-cpu"],
                       capture_output=True, text=True, timeout=600, cwd=str(root))
    assert r.returncode == 0, r.stderr[-800:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["unit"] == "homographies/s" and line["higher_is_better"] is True and line["n_gpus"] == 1 and line["steps"] == 4
    assert line["gpu_launches"] == 4 and line["dtype"] == "f64" and line["scaling"] == "weak" and line["vs_baseline"] is None
    rf = line["roofline"]
    assert rf["bound"] == "hbm" and rf["unit"] == "GB/s" and rf["peak"] > 1000 and abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-9
    assert rf["algorithmic_bytes_per_launch"] == 100 * (1 << 22)
    assert abs(line["value"] - (1 << 22) / (line["ms_per_step"] * 1e-3)) <= 1e-6 * line["value"]
    e2e = line["e2e"]
    assert e2e["h2d_bytes_per_step"] == 64 * (1 << 22) and e2e["d2h_bytes_per_step"] == 36 * (1 << 22) and 0 < e2e["value"] < line["value"]
    assert e2e["matches_device_result"] is True
    assert line["clocks"]["sm_mhz"] > 0 and isinstance(line["clocks"]["reasons"], list)
