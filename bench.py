#!/usr/bin/env python
"""bench.py -- headline benchmark of libhg (BASELINE.json: "homographies/sec (ACA fp32, batch 2^26)
and % of B200 peak HBM GB/s").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A step is one pass of the hot path over one batch: one `hg_aca_batched` call (SoA fp32 in/out,
fp64-internal arithmetic) on config C3 = 2^26 general-position 4-point sets generated on the GPU by
the seeded recipe of DESIGN.md (64 B read + 36 B written per homography; 6.7 GB per step, so every
step streams from HBM: no L2 flush is needed).  Rank 0 prints ONE JSON line.

  value      whole-job homographies/s, inputs resident in HBM, CUDA events on the launch stream,
             max over ranks
  e2e        the same through `hg_aca_batched_host` (pinned HOST buffers in, HOST buffer out; the kernel
             reads and writes them directly over PCIe inside the timed region: 64 B up + 36 B down per H)
  roofline   algorithmic bytes (100 B x 2^26) / average launch duration, against MEASURED_PEAKS.json
  cpu_baseline  the fp64 oracle (oracle/) on the host cores, on a bounded sample of the same workload
  extras     the other hot-path rows at their BASELINE sizes (SKS C3, grid C5, RANSAC C4, C1 latency) and the
             SURVEY 8(f) rows (rectangle fast path, backward, affine, SK, fp64 storage, fused warp)

`--impl reference` times the oracle alone (rank 0 only), same metric/unit/config.
With N > 1 (torchrun, one rank per GPU) every rank solves its own 2^26 sets: weak scaling, no
data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import torch  # noqa: E402

METRIC = "homographies/sec (ACA fp32, batch 2^26)"
UNIT = "homographies/s"
LOG2N = 26
BYTES_PER_H = 100            # 16 fp32 read + 9 fp32 written
FALLBACK_HBM_GBS = 6650.0    # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent


def workload_config(n, world):
    return {"workload": "C3: general-position 4-point sets, batch 2^%d per GPU, fp32 SoA, ACA" % LOG2N
            if n == 1 << LOG2N else "C3-like, batch %d per GPU, fp32 SoA, ACA" % n,
            "sets_per_gpu": n, "layout": "SoA float[8][n] x2 -> float[9][n]", "arith": "fp64 internal, fp32 I/O",
            "norm": "none (raw ACA scale)", "l2": "inputs_larger_than_l2 (6.7 GB per step)",
            "parallelism": "dp%d (independent shards, no collective)" % world, "seed": 240218008 + 3}


# ---- clocks during the timed region (NVML in a thread; nvidia-smi is too coarse for a 50 ms region) ----
class ClockSampler:
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index):
        self.samples, self.reasons, self._stop, self._thr, self.max_mhz = [], set(), threading.Event(), None, None
        self.error = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = self._handle(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:      # no NVML: report that instead of a number
            self.nv, self.error = None, repr(e)

    def _handle(self, index):
        uuid = None
        try:
            uuid = str(torch.cuda.get_device_properties(index).uuid)
        except Exception:
            pass
        if uuid:
            for cand in (uuid, "GPU-" + uuid):
                try:
                    return self.nv.nvmlDeviceGetHandleByUUID(cand.encode() if isinstance(cand, str) else cand)
                except Exception:
                    continue
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
        return self.nv.nvmlDeviceGetHandleByIndex(phys)

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                bits = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for b, name in self.REASONS.items():
                    if bits & b:
                        self.reasons.add(name)
            except Exception as e:
                self.error = repr(e)
                return
            time.sleep(0.002)

    def start(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr:
            self._stop.set()
            self._thr.join()
        out = {"sm_mhz": statistics.median(self.samples) if self.samples else None, "sm_max_mhz": self.max_mhz,
               "reasons": sorted(self.reasons), "samples": len(self.samples)}
        if self.error:
            out["error"] = self.error
        return out


def measured_peak_gbs():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "B200_PROFILING.md fallback (of fallback)"


def event_time_ms(fn, reps, stream=None):
    """Total device time of `reps` back-to-back calls, CUDA events on the current stream."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def hbm_roofline(bytes_per_launch, ms, peak, peak_src, kernel, **kw):
    """The `roofline` object of an HBM-bound leg: algorithmic bytes of one launch / its average duration."""
    a = bytes_per_launch / ms / 1e6
    return dict({"bound": "hbm", "achieved": a, "peak": peak, "unit": "GB/s", "frac": a / peak, "traffic": None,
                 "kernel": kernel, "algorithmic_bytes_per_launch": bytes_per_launch, "peak_source": peak_src}, **kw)


def graph_of(fns, stream=None):
    """One CUDA graph that runs every callable of `fns` once, in order (captured on a side stream)."""
    st = stream or torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        for f in fns:
            f()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            for f in fns:
                f()
    torch.cuda.current_stream().wait_stream(st)
    g.replay()
    return g


def timed_oracle(fn, units, unit, sample, min_seconds=2.0):
    """`cpu_baseline` object: the oracle call `fn` (OpenMP over all host cores) repeated for >= min_seconds."""
    import oracle
    oracle.set_num_threads(os.cpu_count() or 1)
    fn()
    done, t0 = 0, time.perf_counter()
    while True:
        fn()
        done += 1
        dt = time.perf_counter() - t0
        if dt >= min_seconds:
            break
    return {"value": units * done / dt, "unit": unit, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": "%s; %d passes, %.1f s" % (sample, done, dt)}


# ---- the oracle on the host cores -------------------------------------------------------------------
def oracle_rate(src_aos, dst_aos, passes, warm=1, min_seconds=0.0):
    """ACA-fp64 oracle, all host cores (OpenMP): homographies/s over at least `passes` passes of the sample
    (and at least `min_seconds` of work)."""
    import oracle
    oracle.set_num_threads(os.cpu_count() or 1)      # torchrun exports OMP_NUM_THREADS=1: the baseline is "all host cores"
    for _ in range(warm):
        oracle.aca(src_aos, dst_aos)
    done = 0
    t0 = time.perf_counter()
    while True:
        oracle.aca(src_aos, dst_aos)
        done += 1
        dt = time.perf_counter() - t0
        if done >= passes and dt >= min_seconds:
            break
    return src_aos.shape[0] * done / dt, oracle.num_threads(), dt, done


def run_reference(args, rank):
    if rank != 0:
        return
    import hg_workloads as W
    n_s = 1 << 22
    src, dst = W.general_sets(n_s, seed=W.SEED_BASE + 3)
    s, d = src.numpy(), dst.numpy()
    warm = max(args.warmup, 1)
    rate, cores, dt, done = oracle_rate(s, d, passes=max(args.steps, 1), warm=warm)
    sample = "each step = the first 2^22 sets of the C3 generator (CPU stream), ACA-fp64 oracle, OpenMP over all host cores"
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": warm, "ms_per_step": dt / max(args.steps, 1) * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workload_config(1 << LOG2N, 1), sets_per_gpu=n_s, sets_per_step=n_s,
                           note="a step of this arm is a 2^22-set sample of the 2^26-set workload (rates per homography are comparable)"),
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---- parity of the TIMED buffers against the oracle (comparison arithmetic only; the rules of tests/util.py restated) ----
def h_parity(H_gpu, H_ref, src, dst, slab=1 << 21):
    """`parity` object of a solver leg.  H_gpu [n,3,3] (the GPU's result on the timed buffers, any scale) against the oracle's
    H_ref [n,3,3] on the same sets src, dst [n,4,2].  ok = every H finite and, in unit-Frobenius sign-aligned form,
    |dH_ij| <= 1e-4 |H_ij| + 1e-7 on EVERY set (north_star's element-wise rule); the 4-point reprojection error (Euclidean,
    px) is reported beside it -- sets whose own fp32-rounding sensitivity exceeds 1e-3 px (reading R12) may exceed 1e-3."""
    import numpy as np
    n = int(H_gpu.shape[0])
    worst, finite, reproj_max, n_le = 0.0, True, 0.0, 0

    def unit(h):
        h = h / np.abs(h).max(axis=1, keepdims=True)
        return h / np.sqrt((h * h).sum(axis=1, keepdims=True))

    for a in range(0, n, slab):
        g = np.asarray(H_gpu[a:a + slab], dtype=np.float64).reshape(-1, 9)
        r = np.asarray(H_ref[a:a + slab], dtype=np.float64).reshape(-1, 9)
        finite = finite and bool(np.isfinite(g).all())
        ug, ur = unit(g), unit(r)
        k, rows = np.abs(ur).argmax(axis=1), np.arange(ur.shape[0])
        sg = np.sign(ug[rows, k]) * np.sign(ur[rows, k])
        sg[sg == 0] = 1
        ug *= sg[:, None]
        worst = max(worst, float((np.abs(ug - ur) / (1e-4 * np.abs(ur) + 1e-7)).max()))
        s = np.asarray(src[a:a + slab], dtype=np.float64)
        d = np.asarray(dst[a:a + slab], dtype=np.float64)
        x = np.concatenate([s, np.ones(s.shape[:-1] + (1,))], axis=-1)
        q = np.einsum("nij,nkj->nki", g.reshape(-1, 3, 3), x)
        e = np.hypot(q[..., 0] / q[..., 2] - d[..., 0], q[..., 1] / q[..., 2] - d[..., 1]).max(axis=1)
        reproj_max = max(reproj_max, float(e.max()))
        n_le += int((e <= 1e-3).sum())
    return {"checked": n, "max_elem_ratio": worst, "max_reproj_px": reproj_max, "frac_reproj_le_1e-3px": n_le / max(n, 1),
            "against": "oracle on the timed buffers", "ok": bool(finite and worst <= 1.0)}


def soa_to_n33(H_soa, n_s):
    """float[9][n] planes -> numpy [n_s,3,3] of the first n_s sets."""
    return H_soa[:, :n_s].t().contiguous().cpu().numpy().reshape(-1, 3, 3)


def ransac_parity(counts_gpu, ref, best_index=None, best_count=None):
    """`parity` object of a RANSAC leg: counts of the timed call against the oracle's (north_star: equal except for pairs within
    1e-4 relative of the threshold, i.e. |difference| <= the oracle's band count of that hypothesis)."""
    import numpy as np
    c = np.asarray(counts_gpu).astype(np.int64)
    diff = np.abs(c - ref["counts"].astype(np.int64))
    bad = int((diff > ref["band_counts"]).sum())
    out = {"checked": int(c.shape[0]), "count_mismatches_outside_band": bad, "count_differences_inside_band": int((diff > 0).sum()) - bad,
           "against": "oracle on the timed buffers", "ok": bad == 0}
    if best_count is not None:
        out["best_count_gpu"], out["best_count_oracle"] = int(best_count), int(ref["best_count"])
        out["ok"] = out["ok"] and abs(int(best_count) - int(ref["best_count"])) <= int(ref["band_counts"].max())
    if best_index is not None:
        out["best_index_gpu"], out["best_index_oracle"] = int(best_index), int(ref["best_index"])
    return out


# ---- extras: the other rows of the hot path at BASELINE sizes -----------------------------------------
def run_extras(hg, W, dev, src, dst, H, peak, peak_src, cpu=True):
    """Every other config of BASELINE.json (and the 8(f) rows) at its full size; each leg carries its own `roofline`
    object and, with cpu=True, a `cpu_baseline` = the oracle on all host cores on a bounded sample of the same workload and a
    `parity` object = the GPU output of the timed buffers against that oracle result.  Every leg runs under its own
    try/except: a failing leg records {"error": ...} under its own name and is listed in the second return value."""
    import oracle
    n = src.shape[1]
    ex, failed = {}, []
    SOLVE_K = "hg::solve_soa_kernel<%s,double,4>"

    def attempt(name, fn):
        try:
            fn()
        except Exception as e:                       # this leg only; the others still run and report
            ex.setdefault(name, {})["error"] = repr(e)[:300]
            failed.append(name)
            try:
                torch.cuda.synchronize()
            except Exception:
                pass

    def leg_sks_c3():
        ms = event_time_ms(lambda: hg.hg_sks_batched(src, dst, H=H), 5) / 5
        ex["sks_c3"] = {"ms": ms, "homographies_per_s": n / ms * 1e3,
                        "roofline": hbm_roofline(n * BYTES_PER_H, ms, peak, peak_src, SOLVE_K % "SKS")}
        if cpu:
            n_s = min(n, 1 << 24)
            s_aos = W.to_aos(src[:, :n_s].contiguous()).cpu().numpy()
            d_aos = W.to_aos(dst[:, :n_s].contiguous()).cpu().numpy()
            Hg = soa_to_n33(H, n_s)
            ex["sks_c3"]["cpu_baseline"] = timed_oracle(lambda: oracle.sks(s_aos, d_aos), n_s, UNIT,
                                                        "first 2^%d sets of the timed workload, SKS-fp64 oracle" % (n_s.bit_length() - 1), 3.0)
            ex["sks_c3"]["parity"] = h_parity(Hg, oracle.sks(s_aos, d_aos), s_aos, d_aos)

    def leg_fp32():
        ms = event_time_ms(lambda: hg.hg_aca_batched(src, dst, H=H, prec=hg.PREC_F32), 5) / 5
        ex["aca_c3_plain_fp32"] = {"ms": ms, "GBps": n * BYTES_PER_H / ms / 1e6, "note": "HG_PREC_F32: fails the parity tolerance, measurement only"}

    # C2: 2^20 sets = 105 MB per call, smaller than the 126 MB L2.  Eight disjoint (src, dst, H) triples = 839 MB are solved in
    # turn inside one CUDA graph, so every call streams from HBM (inputs larger than L2, no flush kernel in the timed region)
    # and no Python launch path is timed; `ms_l2_warm` = the same call repeated on one triple (L2-resident).
    def leg_c2():
        n2, R = 1 << 20, 8
        trip = [(src[:, i * n2:(i + 1) * n2].contiguous(), dst[:, i * n2:(i + 1) * n2].contiguous(),
                 torch.empty((9, n2), dtype=torch.float32, device=dev)) for i in range(R)]
        s_aos = W.to_aos(trip[0][0]).cpu().numpy() if cpu else None
        d_aos = W.to_aos(trip[0][1]).cpu().numpy() if cpu else None
        for name, fn, kn, ofn in (("aca_c2", hg.hg_aca_batched, "ACA", oracle.aca), ("sks_c2", hg.hg_sks_batched, "SKS", oracle.sks)):
            def one(name=name, fn=fn, kn=kn, ofn=ofn):
                g = graph_of([(lambda a=a, b=b, c=c: fn(a, b, H=c)) for a, b, c in trip])
                ms = event_time_ms(g.replay, 20) / (20 * R)
                s2, d2, H2 = trip[0]
                Hg = soa_to_n33(H2, n2) if cpu else None           # written by the timed graph
                warm = event_time_ms(lambda: fn(s2, d2, H=H2), 20) / 20
                ex[name] = {"ms": ms, "homographies_per_s": n2 / ms * 1e3, "ms_l2_warm_python_launch": warm,
                            "l2": "inputs_larger_than_l2: 8 disjoint 105 MB triples solved in turn inside one CUDA graph",
                            "note": "ms = per call inside the graph (includes the ~2.5 us between graph kernel nodes; the kernel alone is ~16.3 us in ncu)",
                            "roofline": hbm_roofline(n2 * BYTES_PER_H, ms, peak, peak_src, SOLVE_K % kn)}
                del g
                if cpu:
                    ex[name]["cpu_baseline"] = timed_oracle(lambda: ofn(s_aos, d_aos), n2, UNIT, "all 2^20 sets of one C2 batch, %s-fp64 oracle" % kn)
                    ex[name]["parity"] = h_parity(Hg, ofn(s_aos, d_aos), s_aos, d_aos)
            attempt(name, one)

    # C5: offsets -> H -> grid, 8192 x 128 x 128 x 2 fp32 = 1.07 GB written per call (> L2)
    def leg_c5():
        import numpy as np
        off = W.offsets_workload(8192, seed=W.SEED_BASE + 5, device=dev)
        Hh = torch.empty((8192, 3, 3), dtype=torch.float32, device=dev)
        grid = torch.empty((8192, 128, 128, 2), dtype=torch.float32, device=dev)
        f5 = lambda: hg.hg_offsets_to_grid(off, 0.0, 0.0, 127.0, 127.0, 128, 128, H=Hh, grid=grid)
        f5(); f5(); f5()
        ms = event_time_ms(f5, 10) / 10
        by = grid.numel() * 4 + off.numel() * 4 + Hh.numel() * 4
        ex["grid_c5"] = {"ms": ms, "grids_per_s": 8192 / ms * 1e3, "l2": "outputs_larger_than_l2 (1.07 GB per call)",
                         "roofline": hbm_roofline(by, ms, peak, peak_src, "hg::offsets_to_grid_kernel<2>", bytes_per_item=by // 8192)}
        if cpu:
            o_np = off[:1024].cpu().numpy()
            g_np = grid[:1024].cpu().numpy()
            ex["grid_c5"]["cpu_baseline"] = timed_oracle(lambda: oracle.offsets_to_grid(o_np, 0.0, 0.0, 127.0, 127.0, 128, 128), 1024,
                                                         "grids/s", "first 1024 of the 8192 items (128 x 128 grid each), fp64 oracle")
            g_ref = oracle.offsets_to_grid(o_np, 0.0, 0.0, 127.0, 127.0, 128, 128)[1]
            mx = float(np.abs(g_np.astype(np.float64) - g_ref).max())
            ex["grid_c5"]["parity"] = {"checked": 1024, "pixels": 1024 * 128 * 128, "max_px": mx, "tolerance_px": 1e-3,
                                       "against": "oracle on the timed buffers", "ok": bool(np.isfinite(g_np).all() and mx <= 1e-3)}

    # C1: 1024 offsets -> H, launch-latency bound: us per call, plain launches and CUDA-graph replay
    def leg_c1():
        off1 = W.offsets_workload(1024, seed=W.SEED_BASE + 1, device=dev)
        H1 = torch.empty((1024, 3, 3), dtype=torch.float32, device=dev)
        c1 = {}
        for name, f1 in (("aca_rect", lambda: hg.hg_aca_rect_batched(off1, 0.0, 0.0, 127.0, 127.0, H=H1, norm=hg.NORM_H33)),
                         ("offsets_to_h", lambda: hg.hg_offsets_to_grid(off1, 0.0, 0.0, 127.0, 127.0, 128, 128, H=H1, want_grid=False))):
            for _ in range(5):
                f1()
            row = {"us_per_call_launch": event_time_ms(f1, 200) / 200 * 1e3}
            with hg.CallPlan() as plan1:              # the same call recorded once: a ctypes call per iteration, no marshalling
                f1()
            row["us_per_call_plan"] = event_time_ms(plan1, 200) / 200 * 1e3
            try:
                g = graph_of([f1] * 20)
                row["us_per_call_graph"] = event_time_ms(g.replay, 20) / (20 * 20) * 1e3
                del g
            except Exception as e:          # graph capture is a convenience measurement, never the headline
                row["graph_error"] = repr(e)[:200]
            c1[name] = row
        us = c1["offsets_to_h"].get("us_per_call_graph", c1["offsets_to_h"]["us_per_call_launch"])
        ex["c1_offsets_to_h_1024"] = dict(c1["offsets_to_h"], aca_rect_entry_point=c1["aca_rect"], homographies_per_s=1024 / us * 1e6,
                                          roofline=hbm_roofline(1024 * 68, us * 1e-3, peak, peak_src, "hg::offsets_to_h_kernel",
                                                                note="70 KB per call: bound by one kernel launch (~2 us), not by HBM"))
        if cpu:
            o1 = off1.cpu().numpy()
            ex["c1_offsets_to_h_1024"]["cpu_baseline"] = timed_oracle(
                lambda: oracle.offsets_to_grid(o1, 0.0, 0.0, 127.0, 127.0, 128, 128, want_grid=False), 1024, UNIT,
                "the 1024 offsets of C1 -> H per call, ACA-fp64 oracle", 1.0)
            s1, d1 = W.offsets_to_sets(off1.cpu())
            H_ref = oracle.offsets_to_grid(o1, 0.0, 0.0, 127.0, 127.0, 128, 128, want_grid=False)[0]
            ex["c1_offsets_to_h_1024"]["parity"] = h_parity(H1.cpu().numpy(), H_ref, s1.numpy(), d1.numpy())   # H1: last written by offsets_to_h

    # C4: fused RANSAC, 4096 correspondences x 2^20 hypotheses, 3 px
    rs = {}

    def leg_c4():
        wl = W.ransac_workload(device=dev)
        ws = torch.empty(hg.hg_ransac_workspace_bytes(4096, 1 << 20), dtype=torch.uint8, device=dev)
        cnt = torch.empty(1 << 20, dtype=torch.int32, device=dev)
        rs.update(wl=wl, ws=ws, cnt=cnt)
        f4 = lambda: hg.hg_ransac_hypothesize_score(wl["src_xy"], wl["dst_xy"], wl["hyp_idx"], 3.0, counts=cnt, workspace=ws)
        out = f4(); f4(); f4()
        cs = ClockSampler(dev.index if dev.index is not None else 0)      # the clock actually held under the FP32 load
        cs.start()
        ms = event_time_ms(f4, 50) / 50
        rclk = cs.stop()
        stats = hg.ransac_stats(ws)
        pairs = 4096 * (1 << 20)
        props = torch.cuda.get_device_properties(dev)
        # FP32 issue peak at the clock SAMPLED during this leg (falls back to the maximum clock only when NVML gave no sample)
        mhz = rclk.get("sm_mhz") or rclk.get("sm_max_mhz") or 1965.0
        alu_peak = props.multi_processor_count * 128 * mhz * 1e6
        ach = pairs * 11 / (ms * 1e-3)
        ex["ransac_c4"] = {"ms": ms, "pairs_per_s": pairs / ms * 1e3, "hypotheses_per_s": (1 << 20) / ms * 1e3,
                           "best_count": int(out["best_count"]), "hypothesis_slices_with_fp64_decisions": stats["n_fixup"],
                           "pairs_decided_in_fp64": stats["n_pairs_f64"], "pairs_in_table_wide_band": stats.get("n_band"), "clocks": rclk,
                           "roofline": {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "FP32 lane-instructions/s",
                                        "frac": ach / alu_peak, "traffic": None, "kernel": "hg::ransac_score_kernel",
                                        "lane_instr_per_pair": 11, "peak_source": "%d SMs x 128 FP32 lanes x %.0f MHz sampled during the leg"
                                                                                   % (props.multi_processor_count, mhz)},
                           "frac_of_fp32_issue_peak": ach / alu_peak}
        if cpu:
            nh = 1 << 15
            s_np, d_np, i_np = wl["src_xy"].cpu().numpy(), wl["dst_xy"].cpu().numpy(), wl["hyp_idx"][:nh].cpu().numpy()
            c_gpu = cnt[:nh].cpu().numpy()
            ex["ransac_c4"]["cpu_baseline"] = timed_oracle(lambda: oracle.ransac(s_np, d_np, i_np, 3.0), nh * 4096, "pairs/s",
                                                           "first 2^15 of the 2^20 hypotheses x all 4096 correspondences, fp64 oracle", 3.0)
            ex["ransac_c4"]["parity"] = dict(ransac_parity(c_gpu, oracle.ransac(s_np, d_np, i_np, 3.0)), pairs=nh * 4096)

    def leg_c4_reject():
        # the same call with the sample check of reading R20 (rejected hypotheses skip the sweep)
        wl, ws, cnt = rs["wl"], rs["ws"], rs["cnt"]
        f4r = lambda: hg.hg_ransac_hypothesize_score(wl["src_xy"], wl["dst_xy"], wl["hyp_idx"], 3.0, counts=cnt, workspace=ws,
                                                     reject_degenerate=True, min_area_px2=0.0)
        f4r(); f4r()
        msr = event_time_ms(f4r, 20) / 20
        str_ = hg.ransac_stats(ws)
        ex["ransac_c4_reject_degenerate"] = {"ms": msr, "hypotheses_per_s": (1 << 20) / msr * 1e3, "n_rejected": str_["n_rejected"],
                                             "pairs_swept_per_s": ((1 << 20) - str_["n_rejected"]) * 4096 / msr * 1e3}

    def leg_c4_sampled():
        # RANSAC extras: on-device sampling, rounds of one wave (296 CTAs x 512), with and without adaptive termination
        wl, ws = rs["wl"], rs["ws"]
        fa = lambda conf: hg.hg_ransac_adaptive(wl["src_xy"], wl["dst_xy"], 240218008, 1 << 20, 296 * 512, 3.0, conf,
                                                want_counts=False, workspace=ws)
        for name, conf in (("ransac_c4_sampled_all_rounds", 0.0), ("ransac_c4_sampled_adaptive_p99", 0.99)):
            o = fa(conf); fa(conf)
            ms = event_time_ms(lambda: fa(conf), 5) / 5
            ne = int(o["n_evaluated"])
            ex[name] = {"ms": ms, "n_evaluated": ne, "best_count": int(o["best_count"]), "pairs_per_s": ne * 4096 / ms * 1e3}

    # The scale of the paper's Table 6 (<= 1000 matches per image pair, a few to a few thousand loops; solver +
    # verification loops 4.5-154 us on a CPU core): us per call, plain launches and inside a CUDA graph.
    small = {}

    def leg_table6(n_pts_s, n_hyp_s):
        wls = W.ransac_workload(n_pts=n_pts_s, n_hyp=n_hyp_s, seed=W.SEED_BASE + 44, device=dev)
        wss = torch.empty(hg.hg_ransac_workspace_bytes(n_pts_s, n_hyp_s), dtype=torch.uint8, device=dev)
        o0 = hg.hg_ransac_hypothesize_score(wls["src_xy"], wls["dst_xy"], wls["hyp_idx"], 3.0, want_counts=False, workspace=wss)
        keep = (o0["best_H"], o0["best_index"], o0["best_count"])          # outputs reused: no allocation on the timed path
        fs = lambda: hg.hg_ransac_hypothesize_score(wls["src_xy"], wls["dst_xy"], wls["hyp_idx"], 3.0, want_counts=False, workspace=wss,
                                                    best=keep)
        for _ in range(5):
            fs()
        row = {"n_pts": n_pts_s, "n_hyp": n_hyp_s, "us_per_call_launch": event_time_ms(fs, 100) / 100 * 1e3}
        small["%dx%d" % (n_hyp_s, n_pts_s)] = row
        with hg.CallPlan() as plan_s:
            fs()
        row["us_per_call_plan"] = event_time_ms(plan_s, 100) / 100 * 1e3
        try:
            gs = graph_of([fs] * 10)
            row["us_per_call_graph"] = event_time_ms(gs.replay, 20) / 200 * 1e3
            del gs
        except Exception as e:
            row["graph_error"] = repr(e)[:200]
        if cpu:
            s_np, d_np, i_np = wls["src_xy"].cpu().numpy(), wls["dst_xy"].cpu().numpy(), wls["hyp_idx"].cpu().numpy()
            row["cpu_baseline"] = timed_oracle(lambda: oracle.ransac(s_np, d_np, i_np, 3.0), 1, "calls/s",
                                               "the whole call (%d hypotheses x %d correspondences), fp64 oracle" % (n_hyp_s, n_pts_s), 0.5)
            oc = hg.hg_ransac_hypothesize_score(wls["src_xy"], wls["dst_xy"], wls["hyp_idx"], 3.0, workspace=wss, best=keep)   # the timed call, with counts
            row["parity"] = ransac_parity(oc["counts"].cpu().numpy(), oracle.ransac(s_np, d_np, i_np, 3.0),
                                          best_index=int(keep[1]), best_count=int(keep[2]))
        if n_hyp_s <= 1024:           # the same call with on-device Philox sampling (adaptive entry point, one round)
            try:
                fa_s = lambda: hg.hg_ransac_adaptive(wls["src_xy"], wls["dst_xy"], 7, n_hyp_s, n_hyp_s, 3.0, 0.0, want_counts=False, workspace=wss)
                fa_s(); fa_s()
                ga = graph_of([fa_s] * 10)
                row["us_per_call_graph_sampled_on_device"] = event_time_ms(ga.replay, 20) / 200 * 1e3
                del ga
            except Exception as e:
                row["sampled_error"] = repr(e)[:200]

    attempt("sks_c3", leg_sks_c3)
    attempt("aca_c3_plain_fp32", leg_fp32)
    leg_c2()                                         # (its two legs are attempted one by one inside)
    attempt("grid_c5", leg_c5)
    attempt("c1_offsets_to_h_1024", leg_c1)
    attempt("ransac_c4", leg_c4)
    if "wl" in rs:
        attempt("ransac_c4_reject_degenerate", leg_c4_reject)
        attempt("ransac_c4_sampled", leg_c4_sampled)
    rs.clear()
    ex["ransac_table6_scale"] = small
    for n_pts_s, n_hyp_s in ((1000, 1024), (500, 256), (2000, 16384)):       # the last one: still the one-kernel path (<= 20 480 hypotheses on <= 2048 points)
        key = "%dx%d" % (n_hyp_s, n_pts_s)
        try:
            leg_table6(n_pts_s, n_hyp_s)
        except Exception as e:
            small.setdefault(key, {})["error"] = repr(e)[:300]
            failed.append("ransac_table6_scale." + key)
    run_next_rows(hg, W, dev, peak, peak_src, ex, attempt)
    return ex, failed


def run_next_rows(hg, W, dev, peak, peak_src, ex, attempt):
    """SURVEY.md 8(f) rows at 2^26 items (2^25 for fp64 storage): all streaming, HBM-bound.  Each group of legs allocates its
    own inputs and runs under `attempt`, so that one failing leg costs only itself (and the legs that share its inputs)."""
    n = 1 << 26

    def leg(name, fn, bytes_per_item, items, reps=10, **kw):
        for _ in range(3):
            fn()
        ms = event_time_ms(fn, reps) / reps
        kernel = kw.pop("kernel")
        ex[name] = dict({"ms": ms, "items_per_s": items / ms * 1e3,
                         "roofline": hbm_roofline(items * bytes_per_item, ms, peak, peak_src, kernel, bytes_per_item=bytes_per_item)}, **kw)

    def rect_aos():
        off = W.offsets_workload(n, seed=W.SEED_BASE + 6, device=dev)
        Haos = torch.empty((n, 3, 3), dtype=torch.float32, device=dev)
        leg("rect_aos_2p26", lambda: hg.hg_aca_rect_batched(off, 0.0, 0.0, 127.0, 127.0, H=Haos, layout=hg.AOS, norm=hg.NORM_H33), 68, n, kernel="hg::rect_aos_kernel<double>")

    def rect_backward_aos():
        off = W.offsets_workload(n, seed=W.SEED_BASE + 6, device=dev)
        g = torch.randn((n, 3, 3), device=dev)
        go = torch.empty((n, 4, 2), dtype=torch.float32, device=dev)
        leg("rect_backward_2p26", lambda: hg.hg_aca_rect_backward(off, 0.0, 0.0, 127.0, 127.0, g, grad_offsets=go), 100, n, kernel="hg::rect_backward_kernel")

    def rect_backward_soa():
        osoa = W.offsets_workload(n, seed=W.SEED_BASE + 6, device=dev).reshape(n, 8).t().contiguous()
        gsoa = torch.randn((9, n), device=dev)
        gosoa = torch.empty((8, n), dtype=torch.float32, device=dev)
        leg("rect_backward_soa_2p26", lambda: hg.hg_aca_rect_backward_soa(osoa, 0.0, 0.0, 127.0, 127.0, gsoa, grad_offsets=gosoa), 100, n,
            kernel="hg::rect_backward_soa_kernel<4>")

    def rect_soa():
        osoa = W.offsets_workload(n, seed=W.SEED_BASE + 6, device=dev).reshape(n, 8).t().contiguous()
        Hsoa = torch.empty((9, n), dtype=torch.float32, device=dev)
        leg("rect_soa_2p26", lambda: hg.hg_aca_rect_batched(osoa, 0.0, 0.0, 127.0, 127.0, H=Hsoa, layout=hg.SOA, norm=hg.NORM_H33), 68, n, kernel="hg::rect_soa_kernel<double,4>")

    def affine_soa():
        Hsoa = torch.empty((9, n), dtype=torch.float32, device=dev)
        a = torch.rand((6, n), device=dev) * 600.0
        b = torch.rand((6, n), device=dev) * 600.0
        leg("affine_soa_2p26", lambda: hg.hg_affine_batched(a, b, H=Hsoa), 84, n, kernel="hg::variant_soa_kernel<AffineOp>")

    def sk_soa():
        Hsoa = torch.empty((9, n), dtype=torch.float32, device=dev)
        q = W.offsets_workload(n, seed=W.SEED_BASE + 6, device=dev).reshape(n, 8).t().contiguous()
        q.mul_(10.0).add_(300.0)                                  # offsets reused as image quadruples
        leg("sk_soa_2p26", lambda: hg.hg_sk_batched((0.35, 1.6), (-0.8, -1.1), q, H=Hsoa), 68, n, kernel="hg::variant_soa_kernel<SkOp>")

    def f64_storage():
        m = 1 << 25
        s64 = torch.rand((8, m), device=dev, dtype=torch.float64) * 600.0
        d64 = torch.rand((8, m), device=dev, dtype=torch.float64) * 600.0
        H64 = torch.empty((9, m), device=dev, dtype=torch.float64)
        leg("aca_f64_soa_2p25", lambda: hg.hg_aca_batched_f64(s64, d64, H=H64), 200, m, kernel="hg::variant_soa_kernel<GeneralOp<ACA>,double>")
        leg("sks_f64_soa_2p25", lambda: hg.hg_sks_batched_f64(s64, d64, H=H64), 200, m, kernel="hg::variant_soa_kernel<GeneralOp<SKS>,double>")

    def table8():
        # The sizes of the paper's Table 8 (1 ... 1M sets, fp64 storage, RTX 3090), as context: us per call,
        # back-to-back launches (launch-bound below ~10K sets, L2-resident up to ~500K sets), and with an L2 flush at 1M.
        t8 = {}
        ex["paper_table8_sizes_f64_aos"] = t8
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
        for k8 in (1, 10, 100, 1000, 10000, 100000, 1000000):
            a8 = torch.rand((k8, 4, 2), device=dev, dtype=torch.float64) * 600.0
            b8 = torch.rand((k8, 4, 2), device=dev, dtype=torch.float64) * 600.0
            h8 = torch.empty((k8, 3, 3), device=dev, dtype=torch.float64)
            row = {}
            for nm, fn in (("aca", hg.hg_aca_batched_f64), ("sks", hg.hg_sks_batched_f64)):
                call = lambda: fn(a8, b8, H=h8, layout=hg.AOS)
                for _ in range(5):
                    call()
                row[nm + "_us"] = event_time_ms(call, 100) / 100 * 1e3
                try:
                    st8 = torch.cuda.Stream()
                    with torch.cuda.stream(st8):
                        call()
                        g8 = torch.cuda.CUDAGraph()
                        with torch.cuda.graph(g8, stream=st8):
                            for _ in range(20):
                                call()
                    torch.cuda.current_stream().wait_stream(st8)
                    g8.replay()
                    row[nm + "_us_graph"] = event_time_ms(g8.replay, 10) / 200 * 1e3
                except Exception as e:
                    row[nm + "_graph_error"] = repr(e)[:120]
                if k8 == 1000000:
                    tot = 0.0
                    for _ in range(5):
                        flush.zero_()
                        tot += event_time_ms(call, 1)
                    row[nm + "_us_l2_flushed"] = tot / 5 * 1e3
            t8[str(k8)] = row

    k = 8192

    def warp_1ch():
        # offsets -> H -> bilinear warp of 8192 single-channel 128 x 128 patches (4 B read + 4 B written per pixel)
        off5 = W.offsets_workload(k, seed=W.SEED_BASE + 5, device=dev)
        img = torch.rand((k, 1, 128, 128), device=dev)
        out = torch.empty_like(img)
        leg("warp_c5_1ch", lambda: hg.hg_offsets_to_warp(off5, 0.0, 0.0, 127.0, 127.0, 128, 128, img, warped=out), 8, k * 128 * 128,
            unit="pixels", kernel="hg::offsets_to_warp_plane_kernel")

    def warp_3ch():
        k3 = 4096
        off5 = W.offsets_workload(k, seed=W.SEED_BASE + 5, device=dev)
        img3 = torch.rand((k3, 3, 128, 128), device=dev)
        out3 = torch.empty_like(img3)
        leg("warp_c5_3ch", lambda: hg.hg_offsets_to_warp(off5[:k3], 0.0, 0.0, 127.0, 127.0, 128, 128, img3, warped=out3), 8, k3 * 3 * 128 * 128,
            unit="pixels x channels", kernel="hg::offsets_to_warp_plane_kernel (one CTA per item and channel)")

    def grid_backward():
        # backward through the grid on C5's shape: 8192 x 128 x 128 x 2 upstream gradient (1.07 GB, larger than L2) -> 8192 x 8
        off5 = W.offsets_workload(k, seed=W.SEED_BASE + 5, device=dev)
        gg = torch.randn((k, 128, 128, 2), device=dev)
        go5 = torch.empty((k, 4, 2), dtype=torch.float32, device=dev)
        leg("grid_backward_c5", lambda: hg.hg_offsets_to_grid_backward(off5, 0.0, 0.0, 127.0, 127.0, gg, grad_offsets=go5),
            128 * 128 * 8 + 64, k, unit="items (128 x 128 x 2 gradient each)", kernel="hg::grid_backward_kernel<2>")

    for name, fn in (("rect_aos_2p26", rect_aos), ("rect_backward_2p26", rect_backward_aos), ("rect_backward_soa_2p26", rect_backward_soa),
                     ("rect_soa_2p26", rect_soa), ("affine_soa_2p26", affine_soa), ("sk_soa_2p26", sk_soa), ("f64_storage_2p25", f64_storage),
                     ("paper_table8_sizes_f64_aos", table8), ("warp_c5_1ch", warp_1ch), ("warp_c5_3ch", warp_3ch), ("grid_backward_c5", grid_backward)):
        attempt(name, fn)
        torch.cuda.empty_cache()                      # each group frees its 2^26-item buffers before the next allocates


def config_summary(line):
    """The compact per-config table printed as the LAST key of the JSON line (so that a truncated tail still shows it): for each
    of C1..C5 the time, the roofline fraction and what bounds it, the oracle's rate on the host cores, and whether the GPU output
    of the timed buffers matched the oracle."""
    ex = line.get("extras", {}) if isinstance(line.get("extras"), dict) else {}

    def row(obj, t_key="ms", t_name="ms"):
        if not isinstance(obj, dict) or "error" in obj or t_key not in obj:
            return {"error": (obj or {}).get("error", "not run")[:80]} if isinstance(obj, dict) or obj is None else {"error": "not run"}
        rf, cb, pa = obj.get("roofline") or {}, obj.get("cpu_baseline") or {}, obj.get("parity") or {}
        r = {t_name: round(obj[t_key], 5), "frac": round(rf["frac"], 4) if "frac" in rf else None, "bound": rf.get("bound"),
             "cpu": float("%.4g" % cb["value"]) if "value" in cb else None, "parity_ok": pa.get("ok")}
        if "checked" in pa:
            r["checked"] = pa["checked"]
        return r

    head = {"ms": line["ms_per_step"], "roofline": line.get("roofline"), "cpu_baseline": line.get("cpu_baseline"), "parity": line.get("parity")}
    c1 = ex.get("c1_offsets_to_h_1024")
    if isinstance(c1, dict) and "us_per_call_graph" in c1:
        c1 = dict(c1, us=c1["us_per_call_graph"])
    elif isinstance(c1, dict) and "us_per_call_launch" in c1:
        c1 = dict(c1, us=c1["us_per_call_launch"])
    out = {"C1": row(c1, "us", "us_per_call"), "C2_aca": row(ex.get("aca_c2")), "C2_sks": row(ex.get("sks_c2")),
           "C3_aca": row(head), "C3_sks": row(ex.get("sks_c3")), "C4": row(ex.get("ransac_c4")), "C5": row(ex.get("grid_c5"))}
    t6 = ex.get("ransac_table6_scale")
    if isinstance(t6, dict):
        out["table6_us_graph"] = {k: (round(v["us_per_call_graph"], 2) if isinstance(v, dict) and "us_per_call_graph" in v else None) for k, v in t6.items()}
        out["table6_parity_ok"] = all(isinstance(v, dict) and (v.get("parity") or {}).get("ok", False) for v in t6.values()) if t6 else None
    return out


def launch_command(argv, n_gpus, port):
    """The command `bench.py --gpus N` (N > 1) re-executes itself as when no launcher started it: one rank per GPU on this node,
    rendezvous on 127.0.0.1 (the contract's launch line).  `argv` = this script's own arguments."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(int(n_gpus)),
            "--master-addr", "127.0.0.1", "--master-port", str(int(port)), str(Path(__file__).resolve())] + list(argv)


def self_launch_if_needed(args, argv, env=None, device_count=None):
    """`--gpus N` must mean N ranks.  Under a launcher (WORLD_SIZE set) the launcher's world is used and must equal N; without
    one, N > 1 re-executes under torch.distributed.run -- after checking that N devices exist, so that a 1-GPU box fails
    loudly instead of timing one GPU.  Returns the command to exec, or None to continue in this process."""
    env = os.environ if env is None else env
    if args.impl != "ours":
        return None
    if "WORLD_SIZE" in env:
        if int(env["WORLD_SIZE"]) != args.gpus:
            raise SystemExit("bench.py: --gpus %d but the launcher started WORLD_SIZE=%s ranks" % (args.gpus, env["WORLD_SIZE"]))
        return None
    if args.gpus <= 1:
        return None
    have = torch.cuda.device_count() if device_count is None else device_count
    if have < args.gpus:
        raise SystemExit("bench.py --gpus %d: only %d CUDA device(s) visible -- refusing to time fewer GPUs than asked for" % (args.gpus, have))
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    return launch_command(argv, args.gpus, port)


def sharded_ransac_leg(hg, W, dev, rank, world, dist):
    """N > 1 only: C4's 2^20 hypotheses split over the ranks with shard_range (every rank holds the same 4096 correspondences),
    each rank scores its range, and the one exchange the path has -- combine_best, an all-gather of 88 bytes per rank over
    NCCL -- picks the global best.  Device time of the scoring launches (max over ranks) and of the exchange."""
    from paper_2402_18008_b200.sharding import combine_best, shard_range
    wl = W.ransac_workload(device=dev)                                   # same seed on every rank: one table, one hypothesis list
    h0, h1 = shard_range(1 << 20, rank, world)
    idx = wl["hyp_idx"][h0:h1].contiguous()
    ws = torch.empty(hg.hg_ransac_workspace_bytes(4096, h1 - h0), dtype=torch.uint8, device=dev)
    cnt = torch.empty(h1 - h0, dtype=torch.int32, device=dev)
    f = lambda: hg.hg_ransac_hypothesize_score(wl["src_xy"], wl["dst_xy"], idx, 3.0, counts=cnt, workspace=ws)
    o = f(); f()
    dist.barrier()
    ms = event_time_ms(f, 20) / 20
    comb = lambda: combine_best(o["best_count"], o["best_index"] + h0, o["best_H"])
    comb(); comb()
    dist.barrier()
    us = event_time_ms(comb, 20) / 20 * 1e3
    t = torch.tensor([ms, us], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    bc, bi, _ = comb()
    return {"ms_score_max_over_ranks": float(t[0]), "us_combine_best_nccl": float(t[1]), "hypotheses_per_s": (1 << 20) / (float(t[0]) * 1e-3),
            "scaling": "strong (2^20 hypotheses over %d ranks)" % world, "best_count": int(bc), "best_index": int(bi)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--log2n", type=int, default=LOG2N, help="sets per GPU = 2^log2n (default: the BASELINE size)")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()

    cmd = self_launch_if_needed(args, sys.argv[1:])
    if cmd is not None:
        os.execv(cmd[0], cmd)

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libhg has no CPU path")
    import torch.distributed as dist
    import hg_workloads as W
    import paper_2402_18008_b200 as hg

    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    barrier = (lambda: dist.barrier()) if world > 1 else (lambda: None)

    n = 1 << args.log2n
    warm = max(args.warmup, 3)
    steps = max(args.steps, 1)
    hg.lib()
    src, dst = W.general_sets(n, seed=W.SEED_BASE + 3 + 1000 * rank, device=dev, soa=True)
    H = torch.empty((9, n), dtype=torch.float32, device=dev)
    step = lambda: hg.hg_aca_batched(src, dst, H=H, layout=hg.SOA, norm=hg.NORM_NONE, prec=hg.PREC_F64)

    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(warm):
        step()
    barrier()
    ms_total = event_time_ms(step, steps)
    barrier()
    clocks = sampler.stop()
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / steps
    value = world * n / (ms_step * 1e-3)

    # ---- end to end through the host-buffer entry point ------------------------------------------------
    e2e = None
    if not args.no_e2e:
        hs = torch.empty((8, n), dtype=torch.float32, pin_memory=True)
        hd = torch.empty((8, n), dtype=torch.float32, pin_memory=True)
        hH = torch.empty((9, n), dtype=torch.float32, pin_memory=True)
        hs.copy_(src)
        hd.copy_(dst)
        torch.cuda.synchronize()
        e_steps = min(steps, 5)
        hg.hg_aca_batched_host(hs, hd, H=hH)                  # warm-up (allocations, page faults)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e_steps):
            hg.hg_aca_batched_host(hs, hd, H=hH)              # synchronous: returns with H in host memory
        dt = time.perf_counter() - t0
        barrier()
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        same = bool(torch.equal(hH[:, :: 4097], H[:, :: 4097].cpu()))
        e2e = {"value": world * n * e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": 64 * n, "d2h_bytes_per_step": 36 * n,
               "steps": e_steps, "ms_per_step": dt / e_steps * 1e3, "api": "hg_aca_batched_host (pinned host buffers: one kernel reads and writes them over PCIe)",
               "matches_device_result": same}
        del hs, hd, hH

    sharded = None
    if world > 1:
        try:
            sharded = sharded_ransac_leg(hg, W, dev, rank, world, dist)
        except Exception as e:
            sharded = {"error": repr(e)[:300]}
    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    peak, peak_src = measured_peak_gbs()
    achieved = n * BYTES_PER_H / (ms_step * 1e-3) / 1e9
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warm,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(n, world),
            "clocks": clocks, "gpu_launches": steps,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": None, "kernel": "hg::solve_soa_kernel<ACA,double,4>", "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": n * BYTES_PER_H, "frac_of_8000_datasheet": achieved / 8000.0},
            "pct_of_peak_hbm": 100.0 * achieved / peak}
    if e2e is not None:
        line["e2e"] = e2e
    if sharded is not None:
        line["ransac_c4_sharded"] = sharded
    if world == 1 and not args.no_cpu:
        n_s = min(n, 1 << 24)
        s_aos = W.to_aos(src[:, :n_s].contiguous()).cpu().numpy()
        d_aos = W.to_aos(dst[:, :n_s].contiguous()).cpu().numpy()
        rate, cores, dt, done = oracle_rate(s_aos, d_aos, passes=3, min_seconds=10.0)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "first 2^%d sets of the timed workload, %d passes of the ACA-fp64 oracle (OpenMP, %.1f s)"
                                          % (n_s.bit_length() - 1, done, dt)}
        # the H the timed steps wrote (nothing has touched it since), against the oracle on the same sets
        try:
            import oracle
            line["parity"] = h_parity(soa_to_n33(H, n_s), oracle.aca(s_aos, d_aos), s_aos, d_aos)
        except Exception as e:
            line["parity"] = {"error": repr(e)[:200], "ok": False}
        # single-thread ns per homography on 2^20 sets (the kind of number the paper's Table 5 reports)
        try:
            import oracle
            nt = oracle.num_threads()
            oracle.set_num_threads(1)
            one = {}
            m1 = 1 << 20
            for nm, meth in (("aca", oracle.METHOD_ACA), ("sks", oracle.METHOD_SKS), ("dlt_ge", oracle.METHOD_DLT)):
                oracle.solve(meth, s_aos[: 1 << 14], d_aos[: 1 << 14])
                t0 = time.perf_counter()
                oracle.solve(meth, s_aos[:m1], d_aos[:m1])
                one[nm] = (time.perf_counter() - t0) / m1 * 1e9
            oracle.set_num_threads(nt)
            line["cpu_baseline"]["single_thread_ns_per_homography"] = one
        except Exception as e:
            line["cpu_baseline"]["single_thread_error"] = repr(e)[:200]
        del s_aos, d_aos
    if world == 1 and not args.no_extras:
        try:
            line["extras"], line["extras_failed"] = run_extras(hg, W, dev, src, dst, H, peak, peak_src, cpu=not args.no_cpu)
        except Exception as e:                   # (each leg has its own handler; this catches only the scaffolding around them)
            line["extras"], line["extras_failed"] = {"error": repr(e)[:300]}, ["run_extras"]
    # DRAM traffic: NOT measured in this run -- read from the committed ncu capture, and attached only to the sizes it was taken at
    tfile = ROOT / "profiles" / "roofline_traffic.json"
    if tfile.exists():
        try:
            tr = json.loads(tfile.read_text())
            src_note = "profiles/roofline_traffic.json (committed ncu --set full captures of rounds 2-3, dram__bytes_read.sum + dram__bytes_write.sum per launch); not measured in this run"
            if n == 1 << LOG2N:
                line["roofline"]["traffic"] = tr.get("aca_c3_dram_bytes_per_launch")
                line["roofline"]["traffic_source"] = src_note
            for leg_name, leg_obj in line.get("extras", {}).items():
                if isinstance(leg_obj, dict) and "roofline" in leg_obj and (leg_name + "_dram_bytes_per_launch") in tr \
                        and (n == 1 << LOG2N or leg_name not in ("sks_c3",)):
                    leg_obj["roofline"]["traffic"] = tr[leg_name + "_dram_bytes_per_launch"]
                    leg_obj["roofline"]["traffic_source"] = src_note
        except Exception:
            pass
    if world == 1:
        line["configs"] = config_summary(line)          # last key: the per-config table survives a truncated tail
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
