#!/usr/bin/env python
"""bench.py -- measures the hot path of arXiv 1702.08734 on B200 through the C ABI.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--skip-also] [--skip-cfg5] [--no-cpu] [--ivfpq-nb NB]

Headline (BASELINE.json configs[1], "k-select GB/s as % HBM peak"): one STEP is
fs_kselect over the whole cfg2 batch -- 10 000 rows x 16 384 fp32 ~U[0,1) (1 % of
rows with duplicated runs) at k = 1, 32, 128 and 1024, plus one row of 2^27 values at
k = 1024.  value = algorithmic bytes (4 B per input element +
8 B per output element) of all ranks / step time, inputs resident
in HBM; e2e = the same step through fs_kselect_host from pinned HOST buffers, copies
inside the timed region.  Inputs (1.19 GB per rank) are larger than the 126 MB L2.

"also" (same JSON line; compact copies under roofline.also and cpu_baseline.also):
fs_flat_l2_knn on cfg3 (nb = 10^6, nq = 10^4, d = 128, SIFT-like integers and real-valued
data, k = 1, 10, 100; rows B1-B4) in queries/s and tensor-pipe fraction, and fs_ivfpq_search
on cfg4 (10^8 vectors, nlist 65 536, M = 16) and cfg5 (10^9 vectors, nlist 262 144, M = 8) at
their stated size (rows C1-C5, D1-D3 for the build) in queries/s, whole-search and
scan-stage GB/s on code bytes; each with the oracle timed on a seeded query subset.

With N > 1 (torchrun) every rank runs the same step on its own rows (the path
partitions by row/query: no data-path collective): weak scaling, time = max
over ranks, value = sum of bytes / that time.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of
the same workload on the host cores; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "k-NN queries/s (flat L2, IVFPQ) at oracle match; k-select GB/s as % HBM peak"
N_ROWS, N_COLS, KS = 10_000, 16_384, (1, 32, 128, 1024)
BIG_N, BIG_K = 1 << 27, 1024
WORKLOAD = ("cfg2: fs_kselect on 10000x16384 fp32 U[0,1) rows (1% duplicate-run rows) at "
            "k in {1,32,128,1024} + one row of 2^27 at k=1024")


def step_bytes() -> int:
    b = 0
    for k in KS:
        b += 4 * N_ROWS * N_COLS + 8 * N_ROWS * k
    return b + 4 * BIG_N + 8 * BIG_K


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            j = json.load(f)
        return dict(hbm=float(j["hbm_gbs"]), bf16=float(j["bf16_tflops"]),
                    bf16_sustained=float(j.get("bf16_tflops_sustained", j["bf16_tflops"])),
                    sm_max_mhz=float(j.get("sm_max_mhz", 1965.0)), source="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, sm_max_mhz=1965.0,
                source="fallback (B200_PROFILING.md)")


# ----------------------------------------------------------------------------
class ClockSampler:
    """SM clock and throttle reasons sampled (NVML) while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    m = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    m = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for n, bit in names.items():
                    if m & bit:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(0.02)

    def start(self):
        if self.nv is not None:
            self._stop.clear()
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr is not None:
            self._stop.set()
            self._thr.join()
            self._thr = None

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


# ----------------------------------------------------------------------------
def run_reference(args):
    """The oracle on the host cores, same metric and config; bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    import datagen
    import oracle
    oracle.build()
    rows_per_step, big_slice = 256, 1 << 21
    rows = datagen.kselect_rows(0, rows_per_step, N_COLS)
    big = datagen.kselect_rows(10**6, 1, big_slice, duplicates=False)
    sample_bytes = sum(4 * rows.size + 8 * rows_per_step * k for k in KS) + 4 * big.size + 8 * BIG_K

    def step():
        for k in KS:
            oracle.kselect(rows, k)
        oracle.kselect(big, BIG_K)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    gbs = sample_bytes / dt / 1e9
    sample = ("per step: oracle.kselect (full sort per row) on %d of the %d rows at k in {1,32,128,1024} "
              "+ the first 2^21 of the 2^27-value row at k=1024" % (rows_per_step, N_ROWS))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic (seeded, datagen/)",
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": gbs, "unit": "GB/s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": gbs, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ----------------------------------------------------------------------------
def cpu_baseline():
    """The oracle as it stands on the host cores, bounded sample of the headline workload."""
    import datagen
    import oracle
    n_rows, big_slice = 10_000, 1 << 26
    rows = datagen.kselect_rows(0, n_rows, N_COLS)
    big = datagen.kselect_rows(10**6, 1, big_slice, duplicates=False)
    oracle.kselect(rows[:8], 32)  # load the library
    t0 = time.perf_counter()
    for k in KS:
        oracle.kselect(rows, k)
    oracle.kselect(big, BIG_K)
    dt = time.perf_counter() - t0
    b = sum(4 * rows.size + 8 * n_rows * k for k in KS) + 4 * big.size + 8 * BIG_K
    return {"value": b / dt / 1e9, "unit": "GB/s", "cores": oracle.num_threads(), "kind": "oracle",
            "seconds": dt,
            "sample": "oracle.kselect (full sort per row, OpenMP over rows) on the first %d of %d rows "
                      "at k in {1,32,128,1024} + the first 2^26 of the 2^27-value row at k=1024"
                      % (n_rows, N_ROWS)}


def event_pair():
    import torch
    return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)


def timed(fn, reps, warm=1):
    """Best and median ms over reps, CUDA events on the current stream."""
    import torch
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        a, b = event_pair()
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    ts.sort()
    return ts[0], ts[len(ts) // 2]


def also_flat(fs, gt, pk, cpu=True):
    """fs_flat_l2_knn on cfg3; per k: the call as a user makes it (database norm / operand pre-pass
    inside) and the tensor-pipe fraction; plus the oracle on a seeded query subset (cpu_baseline)."""
    import numpy as np
    import torch
    nb, nq, d = 1_000_000, 10_000, 128
    tf32_peak = pk["bf16"] / 2.0  # dense TF32 = half the measured BF16 rate (B200_PROFILING.md nominal ratio)
    out = {"workload": "cfg3: nb=1e6, nq=1e4, d=128 SIFT-like integer fp32", "engine": fs.flat_engine(),
           "flop_per_call": 2.0 * nb * nq * d, "tf32_peak_tflops": tf32_peak,
           "note": "integer data: the lo planes are zero, the checked dispatch issues 1 TF32 product per MAC (exact); "
                   "real-valued data issue 3 (3xTF32): see real_valued"}

    def run(xq, xb, k, passes):
        ws = torch.empty(fs.flat_l2_knn_ws_bytes(nq, nb, d, k), dtype=torch.uint8, device="cuda")
        od = torch.empty((nq, k), dtype=torch.float32, device="cuda")
        oi = torch.empty((nq, k), dtype=torch.int64, device="cuda")
        best, med = timed(lambda: fs.flat_l2_knn(xq, xb, k, out_dist=od, out_ids=oi, ws=ws), 3)
        tf = 2.0 * nb * nq * d / med / 1e9
        r = {"ms": med, "queries_per_s": nq / med * 1e3, "tflops": tf, "issued_tflops": passes * tf,
             "tensor_frac": passes * tf / tf32_peak}
        # the same search over a prepared database (fs_flat_prepare once, outside the timed calls: the
        # ||y||^2 pass of Eq. 2 and the database's operand split do not depend on the queries)
        od2, oi2 = torch.empty_like(od), torch.empty_like(oi)
        _, medp = timed(lambda: fs.flat_l2_knn(xq, xb, k, out_dist=od2, out_ids=oi2, ws=ws, prep=prep_of(xb)), 3)
        tfp = 2.0 * nb * nq * d / medp / 1e9
        r["prepared"] = {"ms": medp, "queries_per_s": nq / medp * 1e3, "issued_tflops": passes * tfp,
                         "tensor_frac": passes * tfp / tf32_peak,
                         "same_bits_as_plain_call": bool(torch.equal(od, od2) and torch.equal(oi, oi2))}
        return r, od, oi

    preps = {}

    def prep_of(xb):
        if xb.data_ptr() not in preps:
            preps.clear()
            t0 = time.perf_counter()
            preps[xb.data_ptr()] = fs.flat_prepare(xb)
            torch.cuda.synchronize()
            out.setdefault("prepare_ms", []).append((time.perf_counter() - t0) * 1e3)
        return preps[xb.data_ptr()]

    xb = gt.sift_like(0, nb)
    xq = gt.sift_like(nb, nq)
    res = {}
    for k in (1, 10, 100):
        out["k%d" % k], od, oi = run(xq, xb, k, 1)
        res[k] = (od, oi)
    if cpu:
        import datagen
        import oracle
        sub = datagen.unique_sample_ids(64, nq, stream=36)
        xs = xq[torch.from_numpy(sub).cuda()].cpu().numpy()
        xb_h = xb.cpu().numpy()
        oracle.flat_l2_knn(xs[:2], xb_h[:1000], 1)
        t0 = time.perf_counter()
        o = {k: oracle.flat_l2_knn(xs, xb_h, k) for k in (1, 10, 100)}
        dt = time.perf_counter() - t0
        st = torch.from_numpy(sub).cuda()
        exact = all(np.array_equal(res[k][1][st].cpu().numpy(), o[k][1]) and
                    np.array_equal(res[k][0][st].cpu().numpy(), o[k][0]) for k in (1, 10, 100))
        out["cpu_baseline"] = {"value": 3 * len(sub) / dt, "unit": "queries/s", "cores": oracle.num_threads(),
                               "kind": "oracle", "seconds": dt,
                               "sample": "oracle.flat_l2_knn (direct-difference double + full sort) on a seeded %d-query "
                                         "subset of cfg3 at k in {1,10,100}" % len(sub),
                               "gpu_matches_oracle_bit_for_bit": bool(exact)}
        del xb_h
    del xb, xq, res
    preps.clear()
    torch.cuda.empty_cache()
    xb = gt.gaussian_vectors(0, nb, d)
    xq = gt.gaussian_vectors(nb, nq, d)
    out["real_valued"] = {"workload": "same shape, i.i.d. ~N(0,1) fp32 (3xTF32 path)"}
    for k in (1, 10, 100):
        out["real_valued"]["k%d" % k] = run(xq, xb, k, 3)[0]
    del xb, xq
    return out


def also_ivfpq(fs, gt, pk, cfg, nb=None, cpu=True, graph=False):
    """fs_ivfpq_search on BASELINE.json configs[3] (cfg 4) / configs[4] (cfg 5): build the index, time
    every (nprobe, k), report the whole search and the scan stage (C2-C4: tables + list scan + pass-1
    selection, events inside the library) on code bytes, and time the oracle on the seeded query
    subset over the GPU-built lists those queries probed (cpu_baseline, with the parity it shows).
    graph: also the all-vs-all 10-NN graph of the stored vectors (f4, section 6.5) with the
    collection resident in HBM: build (train + add) and fs_ivfpq_knn_graph timed end to end."""
    import math
    import numpy as np
    import torch
    import datagen
    c = dict(datagen.IVFPQ_CONFIGS[cfg])
    full = nb is None or nb >= c["nb"]
    if not full:  # reduced run (profiling aid): same shape, fewer vectors, nlist scaled
        per_list = c["nb"] // c["nlist"]
        c["nlist"] = max(64, min(c["nlist"], int(2 ** round(math.log2(max(nb // per_list, 64))))))
        c["ntrain"] = min(nb, max(256, min(c["ntrain"], 16 * c["nlist"])))
        c["nb"] = nb
    nb, d, nlist, M, nq = c["nb"], c["d"], c["nlist"], c["M"], c["nq"]
    chunk = 1 << 22
    xall = None
    if graph:  # the collection stays in HBM (38.4 GB at 10^8 x 96): generated before anything is timed
        xall = torch.empty((nb, d), dtype=torch.float32, device="cuda")
        for b in range(0, nb, chunk):
            xall[b:b + chunk] = gt.deep_like(b, min(chunk, nb - b))
    xtrain = xall[:c["ntrain"]] if graph else gt.deep_like(0, c["ntrain"])
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ix = fs.IvfPq(d, nlist, M)
    ix.train(xtrain, niter=10, seed=0)
    torch.cuda.synchronize()
    t_train = time.perf_counter() - t0
    del xtrain
    t0 = time.perf_counter()
    for b in range(0, nb, chunk):
        ix.add(xall[b:b + chunk] if graph else gt.deep_like(b, min(chunk, nb - b)))
    xq = gt.deep_like(nb, nq)
    ix.search(xq[:8], 1, 1)  # finalise the lists
    torch.cuda.synchronize()
    t_add = time.perf_counter() - t0
    out = {"workload": "cfg%d%s: nb=%d deep-like d=96, nlist=%d, M=%d, nq=%d"
                       % (cfg, "" if full else "-shaped, REDUCED", nb, nlist, M, nq),
           "train_s": t_train, "add_s": t_add, "add_vectors_per_s": nb / t_add,
           "add_s_includes_input_generation": not graph}
    smem_lookups_peak = 148 * 32 * pk["sm_max_mhz"] * 1e6
    sub = datagen.unique_sample_ids(min(c["check_queries"], nq), nq, stream=10 * cfg + 6)
    st = torch.from_numpy(sub).cuda()
    runs = []
    for nprobe, k in c["searches"]:
        if nprobe > nlist:
            continue
        ws = torch.empty(ix.search_ws_bytes(nq, nprobe, k), dtype=torch.uint8, device="cuda")
        od = torch.empty((nq, k), dtype=torch.float32, device="cuda")
        oi = torch.empty((nq, k), dtype=torch.int64, device="cuda")
        best, med = timed(lambda: ix.search(xq, nprobe, k, out_dist=od, out_ids=oi, ws=ws), 3)
        stage = []
        for _ in range(3):  # stage times from the events the library records (read after the call ended)
            ix.search(xq, nprobe, k, out_dist=od, out_ids=oi, ws=ws)
            torch.cuda.synchronize()
            stage.append(ix.last_stage_ms)
        stage = sorted(stage, key=lambda t: t[1])[1]  # median by scan time
        codes = ix.last_scanned_codes
        key = "nprobe%d_k%d" % (nprobe, k)
        out[key] = {"ms": med, "queries_per_s": nq / med * 1e3, "code_bytes": codes,
                    "code_GBps_whole_search": codes / med / 1e6,
                    "frac_hbm_whole_search": codes / med / 1e6 / pk["hbm"],
                    "stage_ms": {"coarse_C1": stage[0], "scan_C2_C4": stage[1], "merge_C5": stage[2]},
                    "scan_stage_GBps": codes / stage[1] / 1e6,
                    "scan_stage_frac_hbm": codes / stage[1] / 1e6 / pk["hbm"],
                    "scan_stage_lookups_per_s": codes / stage[1] * 1e3,
                    "scan_stage_frac_smem_lookup_rate": codes / stage[1] * 1e3 / smem_lookups_peak}
        if cpu:
            gd, gi, gp = ix.search(xq, nprobe, k, want_probed=True)
            runs.append((nprobe, k, key, gd[st].cpu().numpy(), gi[st].cpu().numpy(), gp[st].cpu().numpy()))
        del ws, od, oi
    if cpu and runs:
        import oracle
        coarse, pq = (t.cpu().numpy() for t in ix.get_quantizers())
        xs = xq[st].cpu().numpy()
        lists = np.unique(np.concatenate([r[5].reshape(-1) for r in runs]))
        so, sc, si = ix.export_lists(lists)
        offs = np.zeros(nlist + 1, np.int64)
        lens = np.zeros(nlist, np.int64)
        lens[lists] = np.diff(so)
        np.cumsum(lens, out=offs[1:])
        codes_h, ids_h = sc.cpu().numpy(), si.cpu().numpy()
        del sc, si
        oracle.ivfpq_search(coarse, pq, offs, codes_h, ids_h, xs[:1], 1, 1)  # load the library
        for nprobe, k, key, gd, gi, gp in runs:
            t0 = time.perf_counter()
            o = oracle.ivfpq_search(coarse, pq, offs, codes_h, ids_h, xs, nprobe, k, probed_in=gp)
            dt = time.perf_counter() - t0
            fin = np.isfinite(o["dist64"]) & (gi >= 0)
            rel = np.abs(gd[fin] - o["dist64"][fin]) / np.maximum(o["dist64"][fin], 1e-30)
            out[key]["cpu_baseline"] = {
                "value": len(sub) / dt, "unit": "queries/s", "cores": oracle.num_threads(), "kind": "oracle",
                "seconds": dt,
                "sample": "oracle.ivfpq_search (Alg. 4 by explicit reconstruction in double, full sort) on the seeded "
                          "%d-query subset over the GPU-built lists those queries probed; coarse step given" % len(sub),
                "gpu_vs_oracle": {"ids_equal_frac": float((gi == o["ids"]).mean()),
                                  "queries_identical_frac": float((gi == o["ids"]).all(1).mean()),
                                  "max_rel_dist_err": float(rel.max()) if rel.size else 0.0,
                                  "within_1e-3": bool(rel.size == 0 or rel.max() <= 1e-3)}}
    if graph:
        out["knn_graph"] = knn_graph_leg(fs, ix, xall, c, cfg, t_train, t_add, cpu)
    ix.close()
    return out


def knn_graph_leg(fs, ix, xall, c, cfg, t_train, t_add, cpu):
    """All-vs-all 10-NN graph (f4): every stored vector is a query (fs_ivfpq_knn_graph, nprobe 16, k 10).
    Checked on a seeded subset of rows against the oracle over the GPU-built lists those rows probe, and
    against the exact 10-NN of those rows (fs_flat_l2_knn over the whole collection) for the graph's
    accuracy on this synthetic set (the quantity of Fig. 5; not the paper's datasets)."""
    import numpy as np
    import torch
    import datagen
    nb, d, nlist = c["nb"], c["d"], c["nlist"]
    nprobe, k = 16, 10
    gd = torch.empty((nb, k), dtype=torch.float32, device="cuda")
    gi = torch.empty((nb, k), dtype=torch.int64, device="cuda")
    warm = min(nb, 65536)
    ix.knn_graph(xall[:warm], nprobe, k, out_dist=gd[:warm], out_ids=gi[:warm])
    torch.cuda.synchronize()
    a, b = event_pair()
    a.record()
    ix.knn_graph(xall, nprobe, k, out_dist=gd, out_ids=gi)
    b.record()
    torch.cuda.synchronize()
    t_graph = a.elapsed_time(b) / 1e3
    res = {"workload": "all-vs-all: the %d stored vectors as queries, nprobe=%d, k=%d, batches of 65536" % (nb, nprobe, k),
           "graph_search_s": t_graph, "rows_per_s": nb / t_graph, "train_s": t_train, "add_s": t_add,
           "build_plus_search_s": t_train + t_add + t_graph,
           "edges": nb * k, "self_in_own_row_frac": None}
    nsub = min(c["check_queries"], nb)
    sub = datagen.unique_sample_ids(nsub, nb, stream=10 * cfg + 8)
    st = torch.from_numpy(sub).cuda()
    res["self_in_own_row_frac"] = float((gi[st] == st[:, None]).any(1).float().mean().item())
    try:  # accuracy of the graph rows against the exact neighbours
        xs_d = xall[st].contiguous()
        ed, ei = fs.flat_l2_knn(xs_d, xall, k)
        hit = (gi[st][:, :, None] == ei[:, None, :]).any(2).float().sum(1)
        res["accuracy_vs_exact_10nn"] = {"rows": int(nsub), "mean_fraction_found": float(hit.mean().item() / k),
                                         "note": "synthetic deep-like set; exact side = fs_flat_l2_knn over all vectors"}
        del ed, ei
    except Exception as e:
        res["accuracy_vs_exact_10nn"] = {"error": repr(e)}
    if cpu:
        import oracle
        sd, si, sp = ix.knn_graph(xall[st].contiguous(), nprobe, k, want_probed=True)
        torch.cuda.synchronize()
        big_d, big_i = gd[st].cpu().numpy(), gi[st].cpu().numpy()
        sp = sp.cpu().numpy()
        coarse, pq = (t.cpu().numpy() for t in ix.get_quantizers())
        lists = np.unique(sp.reshape(-1))
        so, sc, sids = ix.export_lists(lists)
        offs = np.zeros(nlist + 1, np.int64)
        lens = np.zeros(nlist, np.int64)
        lens[lists] = np.diff(so)
        np.cumsum(lens, out=offs[1:])
        xs = xall[st].cpu().numpy()
        t0 = time.perf_counter()
        o = oracle.ivfpq_search(coarse, pq, offs, sc.cpu().numpy(), sids.cpu().numpy(), xs, nprobe, k, probed_in=sp)
        dt = time.perf_counter() - t0
        fin = np.isfinite(o["dist64"]) & (big_i >= 0)
        rel = np.abs(big_d[fin] - o["dist64"][fin]) / np.maximum(o["dist64"][fin], 1e-30)
        res["cpu_baseline"] = {
            "value": nsub / dt, "unit": "rows/s", "cores": oracle.num_threads(), "kind": "oracle", "seconds": dt,
            "sample": "oracle.ivfpq_search on a seeded %d-row subset of the graph over the GPU-built lists those rows "
                      "probed (probed lists from a second run of the same rows); compared with the rows of the "
                      "full all-vs-all output" % nsub,
            "gpu_vs_oracle": {"ids_equal_frac": float((big_i == o["ids"]).mean()),
                              "rows_identical_frac": float((big_i == o["ids"]).all(1).mean()),
                              "max_rel_dist_err": float(rel.max()) if rel.size else 0.0,
                              "within_1e-3": bool(rel.size == 0 or rel.max() <= 1e-3)}}
    return res


def run_shard(args):
    """--mode shard: the database of cfg3 cut into N contiguous id shards, one per rank; every
    rank answers all 10^4 queries over its shard, one all-gather of the [nq][k] lists, then fs_merge_topk.
    Strong scaling (total work fixed): value = queries/s of the whole job, time = max over ranks."""
    import torch
    import torch.distributed as dist

    import paper_1702_08734_b200 as fs
    from paper_1702_08734_b200 import multirank as mr
    from datagen import gen_torch as gt

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    fs.lib()
    nb, nq, d, k = 1_000_000, 10_000, 128, 10
    first, n = mr.shard_range(rank, world, nb)
    xb = gt.sift_like(first, n)
    xq = gt.sift_like(nb, nq)
    ws = torch.empty(fs.flat_l2_knn_ws_bytes(nq, n, d, k), dtype=torch.uint8, device="cuda")
    od = torch.empty((nq, k), dtype=torch.float32, device="cuda")
    oi = torch.empty((nq, k), dtype=torch.int64, device="cuda")

    def step():
        return mr.sharded_search(lambda: fs.flat_l2_knn(xq, xb, k, out_dist=od, out_ids=oi, ws=ws), fs.merge_topk, first)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    sampler = ClockSampler(local)
    barrier()
    fs.reset_launch_count()
    sampler.start()
    t0, t1 = event_pair()
    t0.record()
    for _ in range(args.steps):
        step()
    t1.record()
    barrier()
    sampler.stop()
    ms = mr.max_over_ranks(t0.elapsed_time(t1), "cuda") / args.steps
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": nq / ms * 1e3, "unit": "queries/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic (seeded, datagen/)", "mode": "shard",
            "config": {"workload": "cfg3 flat L2 k-NN, nb=1e6 cut into %d id shards, nq=1e4, d=128, k=%d: local "
                                   "search + one all-gather of nq*k (dist, id) + fs_merge_topk" % (world, k),
                       "parallelism": "database shards, one NCCL all-gather per step", "l2": "database larger than L2"},
            "clocks": sampler.summary(), "gpu_launches": int(fs.launch_count()),
            "exchange_bytes_per_rank_per_step": nq * k * 12}))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_1702_08734_b200 as fs
    from paper_1702_08734_b200 import multirank as mr
    from datagen import gen_torch as gt

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    fs.lib()  # fail loudly if libfs.so is missing
    pk = peaks()

    if args.case in ("flat", "ivfpq", "ivfpq5", "graph"):  # profiling aid: only that "also" leg
        if args.case == "flat":
            out = also_flat(fs, gt, pk, cpu=not args.no_cpu)
        else:
            out = also_ivfpq(fs, gt, pk, 5 if args.case == "ivfpq5" else 4, args.ivfpq_nb, cpu=not args.no_cpu,
                             graph=args.case == "graph")
        print(json.dumps({"case": args.case, **out}))
        return

    # this rank's rows: distinct rows per rank (weak scaling)
    rows = gt.kselect_rows(mr.rank_rows(rank, N_ROWS)[0], N_ROWS, N_COLS)
    big = gt.kselect_rows(10**6 + rank, 1, BIG_N, duplicates=False)
    outs = {k: (torch.empty((N_ROWS, k), dtype=torch.float32, device="cuda"),
                torch.empty((N_ROWS, k), dtype=torch.int32, device="cuda")) for k in KS}
    bout = (torch.empty((1, BIG_K), dtype=torch.float32, device="cuda"),
            torch.empty((1, BIG_K), dtype=torch.int32, device="cuda"))
    wsb = max([fs.kselect_ws_bytes(N_ROWS, N_COLS, k) for k in KS] + [fs.kselect_ws_bytes(1, BIG_N, BIG_K), 16])
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    calls = [("k%d" % k, (lambda k=k: fs.kselect(rows, k, out_val=outs[k][0], out_idx=outs[k][1], ws=ws)),
              4 * N_ROWS * N_COLS + 8 * N_ROWS * k) for k in KS]
    calls.append(("bigrow_k1024", lambda: fs.kselect(big, BIG_K, out_val=bout[0], out_idx=bout[1], ws=ws),
                  4 * BIG_N + 8 * BIG_K))
    if args.case:  # profiling aid: only the named call(s) of the step, no e2e / also / cpu legs
        calls = [c for c in calls if c[0] in args.case.split(",")]
        for _ in range(max(args.warmup, 1)):
            for _, fn, _ in calls:
                fn()
        torch.cuda.synchronize()
        for name, fn, nbytes in calls:
            best, med = timed(fn, max(args.steps, 1), warm=0)
            print(json.dumps({"case": name, "ms": med, "GBps": nbytes / med / 1e6, "frac": nbytes / med / 1e6 / pk["hbm"]}))
        return
    per_call = {name: [] for name, _, _ in calls}

    def step(record=False):
        for name, fn, _ in calls:
            if record:
                a, b = event_pair()
                a.record()
                fn()
                b.record()
                per_call[name].append((a, b))
            else:
                fn()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    sampler = ClockSampler(local)
    barrier()
    fs.reset_launch_count()
    sampler.start()
    t0, t1 = event_pair()
    t0.record()
    for _ in range(args.steps):
        step(record=True)
    t1.record()
    barrier()
    sampler.stop()
    launches = fs.launch_count()
    ms = mr.max_over_ranks(t0.elapsed_time(t1), "cuda")
    ms_per_step = ms / args.steps
    value = mr.job_throughput(step_bytes(), ms_per_step, world) / 1e9

    # per-call device time (launch + its pass-2 launches), dominant call -> roofline
    call_ms = {n: float(np.mean([a.elapsed_time(b) for a, b in ev])) for n, ev in per_call.items()}
    call_bytes = {n: b for n, _, b in calls}
    dom = max(call_ms, key=call_ms.get)
    ach = call_bytes[dom] / call_ms[dom] / 1e6
    roofline = {"bound": "hbm", "kernel": "%s (%s call)" % ("kselect_k1_kernel" if dom == "k1" else "kselect_row_kernel", dom), "achieved": ach,
                "peak": pk["hbm"], "unit": "GB/s", "frac": ach / pk["hbm"], "traffic": None,
                "peak_source": pk["source"] + ", burst copy figure",
                "per_call": {n: {"ms": call_ms[n], "GBps": call_bytes[n] / call_ms[n] / 1e6,
                                 "frac": call_bytes[n] / call_ms[n] / 1e6 / pk["hbm"],
                                 "share_of_step": call_ms[n] / sum(call_ms.values())} for n in call_ms},
                "step_frac": value / world / pk["hbm"]}
    tr = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tr):
        try:
            with open(tr) as f:
                roofline["traffic"] = json.load(f).get(dom)
        except Exception:
            pass

    # e2e: the same step through the host entry points, pinned host buffers
    e2e_steps = max(1, min(args.steps, 2))
    h_rows = torch.empty((N_ROWS, N_COLS), dtype=torch.float32, pin_memory=True)
    h_rows.copy_(rows)
    h_big = torch.empty((1, BIG_N), dtype=torch.float32, pin_memory=True)
    h_big.copy_(big)
    h_out = {k: (torch.empty((N_ROWS, k), dtype=torch.float32, pin_memory=True),
                 torch.empty((N_ROWS, k), dtype=torch.int32, pin_memory=True)) for k in KS}
    h_bout = (torch.empty((1, BIG_K), dtype=torch.float32, pin_memory=True),
              torch.empty((1, BIG_K), dtype=torch.int32, pin_memory=True))
    torch.cuda.synchronize()

    def e2e_step():
        for k in KS:
            fs.kselect_host(h_rows, k, out_val=h_out[k][0], out_idx=h_out[k][1])
        fs.kselect_host(h_big, BIG_K, out_val=h_bout[0], out_idx=h_bout[1])

    e2e_step()
    barrier()
    w0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_s = (time.perf_counter() - w0) / e2e_steps
    e2e_s = mr.max_over_ranks(e2e_s, "cuda")
    h2d = len(KS) * 4 * N_ROWS * N_COLS + 4 * BIG_N
    d2h = sum(8 * N_ROWS * k for k in KS) + 8 * BIG_K
    e2e = {"value": world * step_bytes() / e2e_s / 1e9, "unit": "GB/s", "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3, "steps": e2e_steps,
           "api": "fs_kselect_host (pinned host buffers; per call: H2D, kernels and D2H pipelined in 8 slices on three streams, library-owned staging)"}
    # spot-check the e2e results against the device-path results
    assert torch.equal(h_out[32][1][:64], outs[32][1][:64].cpu()), "host and device paths disagree"
    del h_rows, h_big, rows, big

    line = {
        "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic (seeded counter-based generator, datagen/; stands in for the paper's random rows, P:L377)",
        "config": {"workload": WORKLOAD, "rows_per_gpu": N_ROWS, "algorithmic_bytes_per_step_per_gpu": step_bytes(),
                   "l2": "inputs (1.19 GB per GPU) larger than the 126 MB L2", "parallelism": "rows split over ranks, no collective"},
        "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
    }
    if rank == 0 and world == 1:
        if not args.skip_also:
            torch.cuda.empty_cache()
            also = {}
            for name, fn in (("flat_l2_knn", lambda: also_flat(fs, gt, pk, cpu=not args.no_cpu)),
                             ("ivfpq_search_cfg4", lambda: also_ivfpq(fs, gt, pk, 4, args.ivfpq_nb, cpu=not args.no_cpu,
                                                                  graph=not args.skip_graph)),
                             ("ivfpq_search_cfg5", lambda: also_ivfpq(fs, gt, pk, 5, None, cpu=not args.no_cpu))):
                if name == "ivfpq_search_cfg5" and args.skip_cfg5:
                    continue
                try:
                    torch.cuda.empty_cache()
                    also[name] = fn()
                except Exception as e:  # the headline stands on its own
                    also[name] = {"error": repr(e)}
            line["also"] = also
            # the other two paths' rooflines and CPU baselines, inside the keys the driver keeps
            rl = {}
            fl = also.get("flat_l2_knn", {})
            for kk in ("k1", "k10", "k100"):
                if kk in fl:
                    rl["flat_cfg3_" + kk] = {"bound": "tensor", "achieved": fl[kk]["issued_tflops"], "peak": fl["tf32_peak_tflops"],
                                             "unit": "TFLOP/s", "frac": fl[kk]["tensor_frac"], "ms": fl[kk]["ms"],
                                             "queries_per_s": fl[kk]["queries_per_s"]}
                    if "prepared" in fl[kk]:
                        pr = fl[kk]["prepared"]
                        rl["flat_cfg3_" + kk + "_prepared_database"] = {
                            "bound": "tensor", "achieved": pr["issued_tflops"], "peak": fl["tf32_peak_tflops"],
                            "unit": "TFLOP/s", "frac": pr["tensor_frac"], "ms": pr["ms"], "queries_per_s": pr["queries_per_s"]}
            for name in ("ivfpq_search_cfg4", "ivfpq_search_cfg5"):
                for kk, v in also.get(name, {}).items():
                    if isinstance(v, dict) and "scan_stage_GBps" in v:
                        rl[name[13:] + "_" + kk] = {"bound": "hbm", "achieved": v["scan_stage_GBps"], "peak": pk["hbm"],
                                                   "unit": "GB/s", "frac": v["scan_stage_frac_hbm"],
                                                   "whole_search_frac": v["frac_hbm_whole_search"], "ms": v["ms"],
                                                   "queries_per_s": v["queries_per_s"]}
            roofline["also"] = rl
        line["cpu_baseline"] = cpu_baseline()
        if not args.skip_also:
            cb = {}
            if "cpu_baseline" in line["also"].get("flat_l2_knn", {}):
                cb["flat_cfg3"] = line["also"]["flat_l2_knn"]["cpu_baseline"]
            for name in ("ivfpq_search_cfg4", "ivfpq_search_cfg5"):
                for kk, v in line["also"].get(name, {}).items():
                    if isinstance(v, dict) and "cpu_baseline" in v:
                        cb[name[13:] + "_" + kk] = v["cpu_baseline"]
            line["cpu_baseline"]["also"] = cb
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--skip-also", action="store_true")
    ap.add_argument("--mode", default="replica", choices=["replica", "shard"],
                    help="N > 1: replica = rows split over ranks (weak scaling, the headline); shard = cfg3 database "
                         "cut into id shards, all-gather + merge (strong scaling)")
    ap.add_argument("--ivfpq-nb", type=int, default=None,
                    help="cfg4 leg with fewer vectors (profiling aid; default: BASELINE.json's 10^8)")
    ap.add_argument("--skip-cfg5", action="store_true", help="leave out the 10^9-vector leg (about 5 min of index build)")
    ap.add_argument("--skip-graph", action="store_true", help="leave out the all-vs-all 10-NN graph of the cfg4 leg (about 1 min)")
    ap.add_argument("--no-cpu", action="store_true", help="leave out the oracle timings of the flat / IVFPQ legs")
    ap.add_argument("--case", default="", help="comma list of k1,k32,k128,k1024,bigrow_k1024 (time only these calls), or flat / ivfpq / ivfpq5 / graph (only that leg)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.mode == "shard":
        run_shard(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
