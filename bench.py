#!/usr/bin/env python
"""bench.py — measures the COMB link-stage hot path on B200 (contract: one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME] [--no-extras]

A *step* is one pass of the hot path over one batch of BASELINE.json configs[1] ("decode link": Llama-3-8B-
shaped layer, 128 requests x 1 query token, each linking 8 chunks of 512 tokens drawn Zipf(1.1) from a
2000-chunk pool): comb_link (block tables + the chunk-major inversion from the ordered chunk ids, one H2D copy, no
KV copy) followed by comb_cross_attn_decode over the resident chunk-KV pool.  The library's default policy sends
this batch down the chunk-major path (every distinct chunk streamed once through the tcgen05 kernel, per-request LSE
merge); the per-request split-KV path on the same batch is timed beside it.  `value` is the LOGICAL KV bytes the step
attends over (every request counts its own 8 chunks — the user-visible rate) divided by the device time (CUDA
events, max over ranks).  `roofline` is about DRAM: its `achieved` divides the bytes that must cross the HBM pins
(each distinct chunk once + Q, O, partial rows) by the dominant kernel's time; `achieved_logical` and the ncu-measured
`traffic` stand beside it.  The chunk pool itself was stored before the timed region (compile stage).
configs[2] "RAG prefill" (the metric's prefill half, TFLOP/s against the tensor roofline) is timed in the same run and
reported under the top-level key "prefill"; the other configs, the store, the link and a read-only HBM stream ceiling
are under "extras"; a compact table of all of them ends stderr.  N > 1: independent replicas, one per GPU, no
collective on the data path -> weak scaling.

`--impl reference` times the fp64 CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import re
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import comb_synth as cs  # noqa: E402  (seeded inputs only; no method arithmetic)

NOMINAL_HBM_GBS = 8000.0
NOMINAL_BF16_TFLOPS = 2250.0
FALLBACK_HBM_GBS = 6650.0
FALLBACK_BF16_TFLOPS = 1590.0
METRIC = ("decode cross-attn GB/s of linked chunk KV attended per second (logical bytes; BASELINE metric: cross-attn "
          "TFLOP/s (prefill) and HBM GB/s (decode) at 1 B200 vs roofline; the DRAM-byte roofline is under `roofline`, "
          "the prefill half under `prefill`)")


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm": float(d["hbm_gbs"]), "tf_burst": float(d["bf16_tflops"]),
                "tf_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "src": "measured"}
    return {"hbm": FALLBACK_HBM_GBS, "tf_burst": FALLBACK_BF16_TFLOPS, "tf_sustained": 1400.0, "src": "fallback"}


def ncu_traffic(kernel: str, workload: str):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of `kernel` on `workload` from the
    committed ncu --set full captures (profiles/ncu_traffic.csv), or None when that pair was not captured."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f.read().splitlines()[1:]:
            cols = line.split(",")
            if len(cols) >= 3 and cols[0] == kernel and cols[1] == workload:
                return int(cols[2])
    return None


def workload_config(name: str, w, world: int = 1) -> dict:
    """The `config` object of the JSON line — the same for both arms (the driver compares them)."""
    return {"workload": name, "requests": w.num_requests, "q_tokens_per_step": int(w.total_q),
            "kv_tokens_per_request": w.kv_len(0), "heads": "%d/%d" % (w.num_q_heads, w.num_kv_heads),
            "head_dim": "%d/%d" % (w.head_dim_qk, w.head_dim_v), "page": 16, "pool_pages": w.pool_pages,
            "distinct_chunks_linked": int(len(w.linked_chunks())),
            "chunk_links": int(sum(len(l) for l in w.links))}


# ------------------------------------------------------------------------------------------------
class L2Flush:
    """Evicts the 126 MB L2 between timed iterations: writes a 256 MB buffer, then reads a second 256 MB buffer, so
    the cache is left holding CLEAN lines of unrelated data (after the write alone it would hold ~100 MB of dirty
    lines whose write-back would be charged to the kernel under test)."""
    HOW = "flushed between iterations (256 MB written, then 256 MB read: L2 left clean)"

    def __init__(self, torch):
        self.w = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        self.r = torch.zeros(64 << 20, dtype=torch.int32, device="cuda")
        self.sink = torch.zeros((), dtype=torch.int64, device="cuda")

    def __call__(self, i: int):
        self.w.fill_(i & 0xff)
        self.sink += self.r.sum()


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons DURING the timed region (NVML, every 5 ms)."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # pragma: no cover
            log("clock sampling unavailable:", e)
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "sw_power_cap": 0x4}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.005)

    def __enter__(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}
        return {"sm_mhz": int(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def merge_clocks(a, b):
    """Clock record over two timed regions (the primary's 20 default steps last a few ms: one NVML sample)."""
    if not b or b.get("sm_mhz") is None:
        return a
    if not a or a.get("sm_mhz") is None:
        return b
    n1, n2 = a.get("samples", 1), b.get("samples", 1)
    return {"sm_mhz": int(round((a["sm_mhz"] * n1 + b["sm_mhz"] * n2) / (n1 + n2))), "sm_max_mhz": a["sm_max_mhz"],
            "reasons": sorted(set(a["reasons"]) | set(b["reasons"])), "samples": n1 + n2}


# ------------------------------------------------------------------------------------------------
def oracle_sample(w, phase: str, budget_s: float = 15.0):
    """Times the oracle (as it stands, all host cores) on a bounded prefix of the workload's requests."""
    import oracle
    oracle.build()
    ww = w.decode_phase() if phase == "decode" and int(w.lq.max()) > 1 else w
    per_req_pairs = [int(ww.lq[r]) * ww.kv_len(r) for r in range(ww.num_requests)]
    # calibrate on one request, then take as many as fit the budget
    for c in ww.links[0]:
        ww.chunk_kv(int(c))
    t0 = time.perf_counter()
    oracle.attention_for(ww, [0])
    t1 = time.perf_counter() - t0
    n = int(max(1, min(ww.num_requests, budget_s / max(t1, 1e-3))))
    reqs = list(range(n))
    t0 = time.perf_counter()
    oracle.attention_for(ww, reqs)
    dt = time.perf_counter() - t0
    pairs = sum(per_req_pairs[:n])
    flops = 2 * (ww.head_dim_qk + ww.head_dim_v) * ww.num_q_heads * pairs
    kv_bytes = 2 * ww.num_kv_heads * (ww.head_dim_qk + ww.head_dim_v) * sum(ww.kv_len(r) for r in reqs)
    return {"seconds": dt, "requests": n, "gflops": flops / dt / 1e9, "gbs": kv_bytes / dt / 1e9,
            "q_tokens_per_s": float(sum(int(ww.lq[r]) for r in reqs)) / dt, "cores": oracle.max_threads(),
            "sample": "first %d of %d requests of %s (%s phase), includes the oracle's own chunk concatenation"
                      % (n, ww.num_requests, w.name, phase)}


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the decode-link workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    w = cs.CONFIGS[args.workload]()
    phase = "decode" if args.workload == "decode_link" else "prefill"
    ww = w
    n = min(ww.num_requests, 4 if phase == "decode" else 1)
    reqs = list(range(n))
    if phase == "prefill":  # bound the sample: first 8 query tokens of request 0
        ww = cs.custom(w.name + "_sample", k=w.k, seed=w.seed, num_q_heads=w.num_q_heads, num_kv_heads=w.num_kv_heads,
                       head_dim_qk=w.head_dim_qk, head_dim_v=w.head_dim_v, chunk_len=w.chunk_len, links=w.links[:1],
                       lq=[8], scale=w.scale)
    kv_bytes = 2 * ww.num_kv_heads * (ww.head_dim_qk + ww.head_dim_v) * sum(ww.kv_len(r) for r in reqs)
    pairs = sum(int(ww.lq[r]) * ww.kv_len(r) for r in reqs)
    flops = 2 * (ww.head_dim_qk + ww.head_dim_v) * ww.num_q_heads * pairs
    for _ in range(args.warmup):
        oracle.attention_for(ww, reqs)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.attention_for(ww, reqs)
    dt = (time.perf_counter() - t0) / args.steps
    if phase == "decode":
        value, unit, metric = kv_bytes / dt / 1e9, "GB/s", METRIC
    else:
        value, unit, metric = flops / dt / 1e12, "TFLOP/s", "prefill cross-attn TFLOP/s (BASELINE metric, prefill half)"
    sample = "each step = oracle on the first %d request(s) of %s%s" % (
        n, w.name, "" if phase == "decode" else " (first 8 query tokens)")
    print(json.dumps({
        "impl": "reference", "metric": metric, "value": value, "unit": unit, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args.workload, w),
        "cpu_baseline": {"value": value, "unit": unit, "cores": oracle.max_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


KERNEL_CLASSES = (("cascade_decode_f8_kernel", "decode_cascade"), ("cascade_decode_kernel", "decode_cascade"), ("cascade_merge_kernel", "cascade_merge"),
                  ("decode_split_kernel", "decode_split"), ("decode_merge_kernel", "decode_merge"),
                  ("attn_core_kernel", "prefill"), ("prefill_merge_kernel", "prefill_merge"),
                  ("store_pages_fp8_kernel", "store_fp8"), ("dequant_pages_kernel", "dequant"), ("store_pages_kernel", "store"), ("gemm_bf16_kernel<1", "gemm_paged"), ("gemm_bf16_kernel<0", "gemm"))


def make_traffic_table(directory: str, last: int = 6):
    """profiles/ncu_traffic.csv from the ncu logs beside it: for every *traffic_<workload>.csv (the --csv log of
    `ncu --metrics gpu__time_duration.sum,dram__bytes_read.sum,dram__bytes_write.sum,lts__t_sector_hit_rate.pct ...
    python bench.py --profile-only <extras>`), the mean over the LAST `last` launches of every kernel class (the timed
    launches; earlier ones are pool fills and warm-ups)."""
    import csv
    import glob
    rows_out = []
    for path in sorted(glob.glob(os.path.join(directory, "*traffic_*.csv"))):
        if os.path.basename(path) == "ncu_traffic.csv":
            continue
        workload = os.path.basename(path).split("traffic_", 1)[1][:-4]
        with open(path) as f:
            lines = [l for l in f if l.startswith('"')]
        launches = {}  # id -> {kernel, metrics}
        for rec in csv.DictReader(lines):
            d = launches.setdefault(int(rec["ID"]), {"kernel": rec["Kernel Name"]})
            d[rec["Metric Name"]] = (float(rec["Metric Value"].replace(",", "")), rec["Metric Unit"])
        by_class = {}
        for i in sorted(launches):
            k = launches[i]["kernel"]
            for needle, cls in KERNEL_CLASSES:
                if needle in k:
                    by_class.setdefault(cls, []).append(launches[i])
                    break
        for cls, ls in by_class.items():
            if cls in ("store", "store_fp8") and not workload.endswith("_chunks"):
                continue  # pool fills of the harness
            ls = ls[-last:]
            scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1e-3, "us": 1.0, "ms": 1e3, "%": 1.0}

            def mean(metric):
                return sum(l[metric][0] * scale[l[metric][1]] for l in ls) / len(ls)
            rd, wr = mean("dram__bytes_read.sum"), mean("dram__bytes_write.sum")
            m_ = re.search(r"(\w+_kernel(<[^>]*>)?)", ls[-1]["kernel"].replace("(int)", ""))
            sym = m_.group(1) if m_ else cls
            rows_out.append((cls, workload, int(rd + wr), int(rd), int(wr), round(mean("gpu__time_duration.sum"), 1),
                             round(mean("lts__t_sector_hit_rate.pct"), 1), len(ls), sym, os.path.basename(path)))
    out = os.path.join(directory, "ncu_traffic.csv")
    with open(out, "w") as f:
        f.write("kernel,workload,dram_bytes_per_launch,dram_read,dram_write,ncu_duration_us,l2_sector_hit_pct,"
                "launches_averaged,kernel_symbol,source\n")
        for r_ in rows_out:
            f.write("%s,%s,%d,%d,%d,%.1f,%.1f,%d,\"%s\",%s\n" % r_)
    log("wrote %s (%d rows)" % (out, len(rows_out)))


def stats(x):
    x = np.asarray(x, np.float64)
    if x.size == 0:
        return {"n": 0, "mean": 0.0, "median": 0.0, "min": 0.0}
    return {"n": int(x.size), "mean": float(x.mean()), "median": float(np.median(x)), "min": float(x.min())}


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="decode_link", choices=["decode_link", "rag_prefill"])
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs, store and CPU baseline")
    ap.add_argument("--only", default="", help="comma-separated extras to run (default: all)")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--extra-launches", type=int, default=200,
                    help="timed launches behind every median/min of the extras (lower it under a profiler)")
    ap.add_argument("--profile-only", default="",
                    help="profiler driver: run ONLY these extras (comma-separated, no primary step, no JSON line) so that "
                         "an ncu capture of the command holds one workload's kernels")
    ap.add_argument("--traffic-table", default="",
                    help="no GPU: reduce DIR/*traffic_<workload>.csv (ncu --csv logs of --profile-only runs) to "
                         "DIR/ncu_traffic.csv, one row per (kernel class, workload)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    if args.traffic_table:
        make_traffic_table(args.traffic_table)
        return
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import torch.distributed as dist

    import paper_2602_01519_b200 as comb
    from paper_2602_01519_b200 import harness, replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        return replicas.max_over_ranks(x, device="cuda")

    pk = peaks()
    extras = {}
    summary = []  # compact table, printed last on stderr
    primary_prefill = args.workload == "rag_prefill"
    PATHS = {"auto": comb.DECODE_AUTO, "per_request": comb.DECODE_PER_REQUEST, "chunk_major": comb.DECODE_CHUNK_MAJOR}

    # ------------------------------------------------------------------ attention benches
    def bench_attention(w, phase, steps, warmup, *, fill, flush_l2=False, with_link=True, e2e=True, shuffle=None,
                        decode_path="auto", kv_dtype=0):
        """Timings of `steps` passes of (link +) attention on workload w. Kernel times are per launch (CUDA events
        recorded by the library on the launching stream, comb_profile_*)."""
        # free list: permuted (a chunk's pages scattered over the arena, as in a long-running server) unless told
        ld = harness.load_workload(w, fill=fill, shuffle_seed=(2024 + rank) if shuffle is None else shuffle,
                                   keep_host=False, kv_dtype=kv_dtype)
        pool = ld.pool
        pool.set_decode_path(PATHS[decode_path])
        if phase == "decode":
            wq = w.decode_phase() if int(w.lq.max()) > 1 else w
            q = harness.bits_to_device(wq.all_q(), "cuda")
            q_indptr = wq.q_indptr
        else:
            wq, q, q_indptr = w, ld.q, ld.q_indptr
        Hq = wq.num_q_heads
        out = torch.empty((q.shape[0], Hq, w.head_dim_v), dtype=torch.bfloat16, device="cuda")
        lse = torch.empty((q.shape[0], Hq), dtype=torch.float32, device="cuda")
        chunk_indptr, chunk_ids = w.chunk_indptr, w.chunk_ids_flat
        batch = ld.batch
        flush = L2Flush(torch) if flush_l2 else None

        def step():
            if with_link:
                pool.link_flat(chunk_indptr, chunk_ids, into=batch)
            if phase == "decode":
                pool.decode(batch, q, w.scale, out=out, lse=lse)
            else:
                pool.prefill(batch, q, q_indptr, w.scale, out=out, lse=lse)

        for _ in range(warmup):
            step()
        barrier()
        comb.comb_profile_enable(pool.handle, True)
        l0 = pool.launches
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * steps if flush_l2 else 2)]
        with ClockSampler(local) as clk:
            if flush_l2:
                for i in range(steps):
                    flush(i)
                    ev[2 * i].record()
                    step()
                    ev[2 * i + 1].record()
                torch.cuda.synchronize()
                total_ms = sum(ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(steps))
            else:
                ev[0].record()
                for _ in range(steps):
                    step()
                ev[1].record()
                torch.cuda.synchronize()
                total_ms = ev[0].elapsed_time(ev[1])
        barrier()
        launches = pool.launches - l0
        ks = {name: comb.comb_profile_read_samples(pool.handle, kid, cap=max(steps, 1) + 8) for name, kid in (
            ("decode_split", comb.KERNEL_DECODE_SPLIT), ("decode_merge", comb.KERNEL_DECODE_MERGE),
            ("decode_cascade", comb.KERNEL_DECODE_CASCADE), ("cascade_merge", comb.KERNEL_CASCADE_MERGE),
            ("prefill", comb.KERNEL_PREFILL), ("prefill_merge", comb.KERNEL_PREFILL_MERGE))}
        comb.comb_profile_enable(pool.handle, False)
        if phase == "decode":
            main_k = "decode_cascade" if len(ks["decode_cascade"]) else "decode_split"
            merge_k = "cascade_merge" if main_k == "decode_cascade" else "decode_merge"
        else:
            main_k, merge_k = "prefill", "prefill_merge"
        L = batch.link
        # bytes per token of K + V over all kv-heads: bf16, or e4m3 codes + one fp32 scale per (page, kv-head) block
        elt = (2 if kv_dtype == 0 else 1) * wq.num_kv_heads * (wq.head_dim_qk + wq.head_dim_v) + \
              (0 if kv_dtype == 0 else wq.num_kv_heads * 2 * 4 // 16)
        res = {"ms_per_step": max_over_ranks(total_ms / steps), "kernel": main_k, "kernel_stats": stats(ks[main_k]),
               "merge_stats": stats(ks[merge_k]), "launches": launches, "clocks": clk.summary(),
               "flops": wq.attention_flops(),
               "kv_bytes": wq.kv_bytes_logical() if kv_dtype == 0 else int(L.total_kv_tokens) * elt,
               "kv_bytes_unique": int(L.distinct_kv_tokens) * elt, "q_tokens": wq.total_q,
               "timed_seconds": total_ms / 1e3, "entries": int(L.total_entries),
               "distinct_chunks": int(L.num_distinct_chunks)}
        res["kernel_ms"] = res["kernel_stats"]["mean"]
        res["merge_ms"] = res["merge_stats"]["mean"]
        # io bytes the kernel also moves (Q in, O + LSE out); a partial-row pass writes then re-reads fp32 rows
        res["io_bytes"] = q.numel() * 2 + out.numel() * 2 + lse.numel() * 4
        res["partial_bytes"] = (int(L.total_entries) * Hq * (w.head_dim_v + 1) * 4) if main_k == "decode_cascade" else 0
        if e2e:
            # end to end through the public API with HOST buffers: pinned Q -> device, link, attention, O/LSE -> host
            qh = q.cpu().pin_memory()
            oh = torch.empty(out.shape, dtype=out.dtype).pin_memory()
            lh = torch.empty(lse.shape, dtype=lse.dtype).pin_memory()
            n_e2e = max(3, min(steps, 50))
            for i in range(3 + n_e2e):
                if i == 3:
                    barrier()
                    t0 = time.perf_counter()
                q.copy_(qh, non_blocking=True)
                pool.link_flat(chunk_indptr, chunk_ids, into=batch)
                if phase == "decode":
                    pool.decode(batch, q, w.scale, out=out, lse=lse)
                else:
                    pool.prefill(batch, q, q_indptr, w.scale, out=out, lse=lse)
                oh.copy_(out, non_blocking=True)
                lh.copy_(lse, non_blocking=True)
                torch.cuda.synchronize()
            res["e2e_serial_ms"] = max_over_ranks((time.perf_counter() - t0) * 1e3 / n_e2e)
            # the same work as a server would run it: double-buffered, the H2D copy of step i+1, the link + attention
            # of step i and the D2H copy of step i-1 overlap on three streams (every step still moves all its bytes)
            s_in, s_c, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
            qd, od, ldv = [q, torch.empty_like(q)], [out, torch.empty_like(out)], [lse, torch.empty_like(lse)]
            ohs, lhs = [oh, torch.empty_like(oh).pin_memory()], [lh, torch.empty_like(lh).pin_memory()]
            ev_in = [torch.cuda.Event() for _ in range(2)]
            ev_done = [torch.cuda.Event() for _ in range(2)]
            ev_out = [torch.cuda.Event() for _ in range(2)]
            torch.cuda.synchronize()
            for i in range(4 + n_e2e):
                b = i & 1
                if i == 4:
                    barrier()
                    t0 = time.perf_counter()
                if i >= 2:
                    s_in.wait_event(ev_done[b])   # step i-2 has consumed qd[b]
                    s_c.wait_event(ev_out[b])     # step i-2's results have left od[b]
                with torch.cuda.stream(s_in):
                    qd[b].copy_(qh, non_blocking=True)
                    ev_in[b].record(s_in)
                s_c.wait_event(ev_in[b])
                pool.link_flat(chunk_indptr, chunk_ids, into=batch, stream=s_c)
                if phase == "decode":
                    pool.decode(batch, qd[b], w.scale, out=od[b], lse=ldv[b], stream=s_c)
                else:
                    pool.prefill(batch, qd[b], q_indptr, w.scale, out=od[b], lse=ldv[b], stream=s_c)
                ev_done[b].record(s_c)
                s_out.wait_event(ev_done[b])
                with torch.cuda.stream(s_out):
                    ohs[b].copy_(od[b], non_blocking=True)
                    lhs[b].copy_(ldv[b], non_blocking=True)
                    ev_out[b].record(s_out)
            torch.cuda.synchronize()
            res["e2e_ms"] = max_over_ranks((time.perf_counter() - t0) * 1e3 / n_e2e)
            res["h2d"] = int(qh.numel() * 2 + batch.link.bytes_used)
            res["d2h"] = int(oh.numel() * 2 + lh.numel() * 4)
        pool.close()
        del ld, pool, flush
        torch.cuda.empty_cache()
        return res

    def roofline_hbm(r, wname):
        """DRAM view: the bytes that must cross the HBM pins (each distinct chunk once, Q/O/LSE, partial rows written)
        over the dominant kernel's mean launch time. The logical rate (every request counting its own chunks: what
        L2 and the chunk-major grouping serve) and ncu's measured DRAM traffic stand beside it."""
        k_ms = r["kernel_ms"]
        alg = r["kv_bytes_unique"] + r["io_bytes"] + r["partial_bytes"]
        achieved = alg / (k_ms * 1e-3) / 1e9
        logical = (r["kv_bytes"] + r["io_bytes"]) / (k_ms * 1e-3) / 1e9
        traffic = ncu_traffic(r["kernel"], wname)
        out = {"bound": "hbm", "achieved": achieved, "peak": pk["hbm"], "unit": "GB/s", "frac": achieved / pk["hbm"],
               "peak_source": pk["src"] + " copy bandwidth (MEASURED_PEAKS.json hbm_gbs)",
               "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS, "kernel": r["kernel"],
               "kernel_ms": k_ms, "kernel_ms_median": r["kernel_stats"]["median"],
               "kernel_ms_min": r["kernel_stats"]["min"], "launches_timed": r["kernel_stats"]["n"],
               "algorithmic_bytes": alg, "bytes_definition": "distinct linked chunks once + Q + O + LSE + partial rows",
               "achieved_logical": logical, "logical_bytes": r["kv_bytes"] + r["io_bytes"], "traffic": traffic,
               "merge_ms": r["merge_ms"]}
        if traffic:
            out["frac_traffic"] = traffic / (k_ms * 1e-3) / 1e9 / pk["hbm"]
        return out

    def roofline_tensor(r, wname):
        achieved = r["flops"] / (r["kernel_ms"] * 1e-3) / 1e12
        sustained = r["timed_seconds"] >= 1.0
        peak = pk["tf_sustained"] if sustained else pk["tf_burst"]
        return {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "peak_source": "%s cuBLAS bf16 %s" % (pk["src"], "sustained" if sustained else "burst"),
                "frac_of_burst": achieved / pk["tf_burst"], "frac_of_sustained": achieved / pk["tf_sustained"],
                "frac_of_nominal_2250": achieved / NOMINAL_BF16_TFLOPS, "kernel": r["kernel"],
                "kernel_ms": r["kernel_ms"], "kernel_ms_median": r["kernel_stats"]["median"],
                "kernel_ms_min": r["kernel_stats"]["min"], "launches_timed": r["kernel_stats"]["n"],
                "algorithmic_flops": r["flops"], "traffic": ncu_traffic(r["kernel"], wname), "merge_ms": r["merge_ms"]}

    def note(name, r, roof, alt=None):
        """One line of the compact table (kernel ms mean/median/min, achieved, fraction of the measured peak, clocks)."""
        c = r["clocks"]
        s = "%s k=%.4f/%.4f/%.4f step=%.4f %s=%.0f f=%.3f" % (
            name, r["kernel_stats"]["mean"], r["kernel_stats"]["median"], r["kernel_stats"]["min"], r["ms_per_step"],
            "TF" if roof["bound"] == "tensor" else "GB", roof["achieved"], roof["frac"])
        if alt:
            s += " " + alt
        s += " clk=%s%s" % (c.get("sm_mhz"), ("!" + "+".join(c["reasons"])) if c.get("reasons") else "")
        summary.append(s)

    # ------------------------------------------------------------------ primary workload
    profile_only = bool(args.profile_only)
    if profile_only:
        args.only, args.no_extras = args.profile_only, False
        r = roof = None
    elif primary_prefill:
        w = cs.rag_prefill(seed=args.seed + rank)
        r = bench_attention(w, "prefill", args.steps, args.warmup, fill="linked")
        value = world * r["flops"] / (r["ms_per_step"] * 1e-3) / 1e12
        unit, metric = "TFLOP/s", "prefill cross-attn TFLOP/s (BASELINE metric, prefill half)"
        roof = roofline_tensor(r, "rag_prefill")
        e2e_val = world * r["flops"] / (r["e2e_ms"] * 1e-3) / 1e12
    else:
        w = cs.decode_link(seed=args.seed + rank)
        r = bench_attention(w, "decode", args.steps, args.warmup, fill="linked")
        value = world * r["kv_bytes"] / (r["ms_per_step"] * 1e-3) / 1e9
        unit, metric = "GB/s", METRIC
        roof = roofline_hbm(r, "decode_link")
        e2e_val = world * r["kv_bytes"] / (r["e2e_ms"] * 1e-3) / 1e9
    dtype = "bf16"
    clocks = None
    if not profile_only:
        log("primary", json.dumps(r))
        note(args.workload, r, roof, None if primary_prefill else "log=%.0f" % roof["achieved_logical"])
        clocks = r["clocks"]

    cpu = None
    prefill_top = None
    if rank == 0 and world == 1 and not args.no_extras:
        only = set(x for x in args.only.split(",") if x)

        def want(name):
            return not only or name in only

        # ---- the other configs (not bench lines; context for the BASELINE metric's prefill half) ----
        def prefill_extra(name, wk, steps, fill, flush=False, wname=None, kv_dtype=0):
            rr = bench_attention(wk, "prefill", steps, 3, fill=fill, flush_l2=flush, e2e=False, kv_dtype=kv_dtype)
            # a prefill whose flops per logical KV byte sit under the ridge of the measured peaks is HBM-bound
            # (no GQA or few query tokens: SURVEY.md 8(d)); it is then reported against the HBM roof first
            ridge = pk["tf_burst"] * 1e12 / (pk["hbm"] * 1e9)
            intensity = rr["flops"] / (rr["kv_bytes"] + rr["io_bytes"])
            rt = roofline_tensor(rr, wname or name)
            rh = roofline_hbm(rr, wname or name) if intensity < ridge else None
            extras[name] = {"workload": name, "ms_per_step": rr["ms_per_step"], "kernel_ms": rr["kernel_ms"],
                            "tflops": rr["flops"] / (rr["ms_per_step"] * 1e-3) / 1e12,
                            "q_tokens_per_s": rr["q_tokens"] / (rr["ms_per_step"] * 1e-3),
                            "flop_per_logical_byte": intensity, "ridge_flop_per_byte": ridge,
                            "roofline_hbm": rh, "roofline": rt, "clocks": rr["clocks"], "launches": rr["launches"],
                            "l2": L2Flush.HOW if flush else "inputs larger than L2"}
            log(name, json.dumps(extras[name]))
            note(name, rr, rt, ("hbm=%.0f/%.3f" % (rh["achieved"], rh["frac"])) if rh else None)
            return rr

        def decode_extra(name, wk, steps, fill, flush=False, shuffle=None, path="auto", wname=None, kv_dtype=0):
            rr = bench_attention(wk, "decode", steps, 3, fill=fill, flush_l2=flush, e2e=False, shuffle=shuffle,
                                 decode_path=path, kv_dtype=kv_dtype)
            rh = roofline_hbm(rr, wname or name)
            extras[name] = {"workload": name, "decode_path": path, "kv_dtype": "e4m3" if kv_dtype else "bf16",
                            "ms_per_step": rr["ms_per_step"],
                            "kernel_ms": rr["kernel_ms"], "merge_ms": rr["merge_ms"],
                            "gbs_logical": rr["kv_bytes"] / (rr["ms_per_step"] * 1e-3) / 1e9,
                            "entries": rr["entries"], "distinct_chunks": rr["distinct_chunks"],
                            "roofline": rh, "clocks": rr["clocks"], "launches": rr["launches"],
                            "l2": L2Flush.HOW if flush else "inputs larger than L2"}
            log(name, json.dumps(extras[name]))
            note(name, rr, rh, "log=%.0f" % rh["achieved_logical"])
            return rr

        try:
            N = max(3, args.extra_launches)  # launches behind every median / min below
            if not primary_prefill:
                if want("rag_prefill"):
                    rp = prefill_extra("rag_prefill", cs.rag_prefill(seed=args.seed), N, "linked")
                    clocks = merge_clocks(clocks, rp["clocks"])
                    prefill_top = {"workload": "rag_prefill (BASELINE configs[2])", "unit": "TFLOP/s",
                                   "value": extras["rag_prefill"]["tflops"],
                                   "ms_per_step": extras["rag_prefill"]["ms_per_step"],
                                   "roofline": extras["rag_prefill"]["roofline"],
                                   "config": workload_config("rag_prefill", cs.rag_prefill(seed=args.seed))}
                # the same batch down the per-request path (what round 1 shipped), and the primary with a cold L2
                if want("decode_link_per_request"):
                    decode_extra("decode_link_per_request", cs.decode_link(seed=args.seed), N, "linked",
                                 path="per_request", wname="decode_link")
                if want("decode_link_cold_l2"):
                    decode_extra("decode_link_cold_l2", cs.decode_link(seed=args.seed), min(N, 50), "linked", flush=True,
                                 wname="decode_link")
                if want("decode_link_contiguous_pages"):  # ascending free list: chunks contiguous in the arena
                    decode_extra("decode_link_contiguous_pages", cs.decode_link(seed=args.seed), N, "linked", shuffle=0,
                                 wname="decode_link")
            if (primary_prefill or profile_only) and want("decode_link"):
                decode_extra("decode_link", cs.decode_link(seed=args.seed), N, "linked")
            # cfg 2 geometry with 1024 DISTINCT chunks: every linked byte has to come from HBM (2.15 GB per step)
            if want("decode_no_reuse"):
                decode_extra("decode_no_reuse_per_request", cs.decode_link(seed=args.seed, no_reuse=True), N, "linked",
                             path="per_request", wname="decode_no_reuse")
                decode_extra("decode_no_reuse_chunk_major", cs.decode_link(seed=args.seed, no_reuse=True), N, "linked",
                             path="chunk_major", wname="decode_no_reuse")
            # (f4) fp8 pools: the same batches over e4m3 pages (bytes counted as stored: codes + scales)
            if want("decode_link_fp8"):
                decode_extra("decode_link_fp8", cs.decode_link(seed=args.seed), N, "linked", wname="decode_link_fp8",
                             kv_dtype=comb.KV_E4M3)
            if want("decode_no_reuse_fp8"):
                decode_extra("decode_no_reuse_fp8", cs.decode_link(seed=args.seed, no_reuse=True), N, "linked",
                             wname="decode_no_reuse_fp8", kv_dtype=comb.KV_E4M3)
            if want("prefill_fp8"):  # fp8 pool: dequantise the batch's distinct pages into bf16 staging, then the bf16 kernel
                prefill_extra("rag_prefill_lq32_fp8", cs.rag_prefill(seed=args.seed, lq=32), min(N, 50), "linked",
                              wname="rag_prefill_lq32_fp8", kv_dtype=comb.KV_E4M3)
            if want("rag_prefill_lq32"):
                prefill_extra("rag_prefill_lq32", cs.rag_prefill(seed=args.seed, lq=32), N, "linked")
            # the paper's own regime (< 50 dynamic tokens) at a small batch: 32 work items for 148 SMs,
            # so each request's KV is cut into ranges that run on different SMs and are merged by LSE
            if want("rag_prefill_lq32_r4"):
                prefill_extra("rag_prefill_lq32_r4", cs.rag_prefill(seed=args.seed, lq=32, requests=4), N, "linked",
                              flush=True)
            if want("long_fewshot"):
                prefill_extra("long_fewshot_prefill", cs.long_fewshot(seed=args.seed), min(N, 50), "all", flush=True,
                              wname="long_fewshot")
                decode_extra("long_fewshot_decode", cs.long_fewshot(seed=args.seed), N, "all", flush=True,
                             wname="long_fewshot")
                decode_extra("long_fewshot_decode_per_request", cs.long_fewshot(seed=args.seed), N, "all", flush=True,
                             path="per_request", wname="long_fewshot")
            if want("mla_shaped"):
                prefill_extra("mla_shaped_prefill", cs.mla_shaped(seed=args.seed), N, "linked", wname="mla_shaped")
                decode_extra("mla_shaped_decode", cs.mla_shaped(seed=args.seed), N, "linked", wname="mla_shaped")
                decode_extra("mla_shaped_decode_per_request", cs.mla_shaped(seed=args.seed), N, "linked",
                             path="per_request", wname="mla_shaped")
            if want("store"):
                extras["store"] = bench_store(torch, comb, harness, cs.long_fewshot(seed=args.seed), pk, N)
                st = extras["store"]
                summary.append("store k=%.4f/%.4f/%.4f GB=%.0f f=%.3f" % (
                    st["kernel_ms"], st["kernel_ms_median"], st["kernel_ms_min"], st["roofline"]["achieved"],
                    st["roofline"]["frac"]))
            if want("project_store"):
                extras["project_store"] = bench_project_store(torch, comb, cs.long_fewshot(seed=args.seed), pk, min(N, 50))
                ps = extras["project_store"]
                summary.append("project_store k=%.4f/%.4f/%.4f TF=%.0f f=%.3f two_step=%.4f" % (
                    ps["kernel_ms"], ps["kernel_ms_median"], ps["kernel_ms_min"], ps["roofline"]["achieved"],
                    ps["roofline"]["frac"], ps["two_step_ms"]))
            if want("cross_layer"):
                extras["cross_layer_prefill"] = bench_cross_layer(torch, comb, cs.rag_prefill(seed=args.seed), pk,
                                                                 "prefill", max(3, min(N, 20)))
                extras["cross_layer_decode"] = bench_cross_layer(torch, comb, cs.decode_link(seed=args.seed), pk,
                                                                "decode", max(3, min(N, 50)))
                for nm in ("cross_layer_prefill", "cross_layer_decode"):
                    cl = extras[nm]
                    summary.append("%s L=8 step=%.3f attn=%.3f gemm=%.3f TF=%.0f us/tok=%.2f" % (
                        nm, cl["ms_per_step"], cl["attention_ms"], cl["gemm_ms"], cl["tflops"], cl["us_per_q_token"]))
            if want("link"):
                extras["link"] = bench_link(torch, comb, harness, cs.decode_link(seed=args.seed))
                summary.append("link host_p50=%.1fus resident_p50=%.1fus" % (
                    extras["link"]["host_enqueue_us_p50"], extras["link"]["resident_us_p50"]))
            if want("stream_read"):
                extras["stream_read"] = bench_stream_read(torch, comb, pk)
                summary.append("read_only_stream GB=%.0f/%.0f (mean/best) = %.3f of copy peak" % (
                    extras["stream_read"]["gbs_mean"], extras["stream_read"]["gbs_best"],
                    extras["stream_read"]["gbs_best"] / pk["hbm"]))
        except Exception as e:  # extras must never lose the primary line
            extras["error"] = repr(e)
            log("extras failed:", repr(e))
        if profile_only:
            for line_ in summary:
                log(line_[:118])
            return
        # ---- CPU baseline: the oracle on the host cores, bounded sample ----
        try:
            o = oracle_sample(w, "prefill" if primary_prefill else "decode")
            cpu = {"value": o["gflops"] / 1e3 if primary_prefill else o["gbs"], "unit": unit, "cores": o["cores"],
                   "kind": "oracle", "sample": o["sample"], "seconds": o["seconds"], "gflops_fp64": o["gflops"],
                   "q_tokens_per_s": o["q_tokens_per_s"]}
        except Exception as e:
            cpu = {"error": repr(e)}

    if rank == 0:
        cfg = workload_config(args.workload, w, world)
        cfg.update({"free_list": "permuted (scattered pages)",
                    "step": "comb_link + comb_cross_attn_%s" % ("prefill" if primary_prefill else "decode"),
                    "decode_path": None if primary_prefill else ("chunk_major" if r["kernel"] == "decode_cascade"
                                                                  else "per_request"),
                    "l2": "inputs larger than L2 (%.2f GB of distinct KV, %.2f GB logical per step)" % (
                        r["kv_bytes_unique"] / 1e9, r["kv_bytes"] / 1e9),
                    "parallelism": "replicas x%d" % world})
        line = {
            "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": dtype, "data": "synthetic", "config": cfg, "clocks": clocks,
            "e2e": {"value": e2e_val, "unit": unit, "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"],
                    "ms_per_step": r["e2e_ms"], "serial_ms_per_step": r["e2e_serial_ms"],
                    "how": "host buffers through the public API; pinned Q -> device, comb_link (tables H2D), attention, "
                           "O + LSE -> pinned host every step; double-buffered over three streams (serial_ms_per_step: "
                           "the same with a device synchronise after every step)"},
            "gpu_launches": int(r["launches"]),
            "roofline": roof,
            "q_tokens_per_s": world * r["q_tokens"] / (r["ms_per_step"] * 1e-3),
        }
        if prefill_top is not None:
            line["prefill"] = prefill_top
        if cpu is not None:
            line["cpu_baseline"] = cpu
        if extras:
            line["extras"] = extras
        print(json.dumps(line), flush=True)
        # compact table last, so that a truncated stderr tail still carries every workload's number
        log("== summary (kernel ms mean/median/min; achieved; f = fraction of the measured peak; GB = DRAM-byte rate, "
            "log = logical) ==")
        for s in summary:
            log(s[:118])
    if world > 1:
        dist.destroy_process_group()


def bench_store(torch, comb, harness, w, pk, n=200):
    """(a2) batched paged store of configs[3]'s 64 variable-length chunks, 200 times over the same page lists (a store of
    an id that exists with the same length rewrites its pages), L2 flushed clean before every launch."""
    ld = harness.load_workload(w, fill="all", shuffle_seed=77, keep_host=False)
    pool = ld.pool
    ids = list(range(w.num_chunks))
    tok = np.zeros(w.num_chunks + 1, np.int32)
    np.cumsum(w.chunk_len, out=tok[1:])
    T = int(tok[-1])
    k = torch.randn((T, w.num_kv_heads, w.head_dim_qk), device="cuda").to(torch.bfloat16)
    v = torch.randn((T, w.num_kv_heads, w.head_dim_v), device="cuda").to(torch.bfloat16)
    flush = L2Flush(torch)
    comb.comb_profile_enable(pool.handle, True)
    comb.comb_profile_read(pool.handle, comb.KERNEL_STORE)
    for i in range(n + 3):
        flush(i)
        if i == 3:
            torch.cuda.synchronize()
            comb.comb_profile_read(pool.handle, comb.KERNEL_STORE)
        pool.store_chunks(ids, tok, k, v)
    st = stats(comb.comb_profile_read_samples(pool.handle, comb.KERNEL_STORE, cap=n + 8))
    comb.comb_profile_enable(pool.handle, False)
    nbytes = 2 * T * w.num_kv_heads * (w.head_dim_qk + w.head_dim_v) * 2
    achieved = nbytes / (st["mean"] * 1e-3) / 1e9
    pool.close()
    return {"workload": "store of long_fewshot's %d chunks (%d tokens), one launch" % (w.num_chunks, T),
            "kernel_ms": st["mean"], "kernel_ms_median": st["median"], "kernel_ms_min": st["min"],
            "launches_timed": st["n"],
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": pk["hbm"], "unit": "GB/s",
                         "frac": achieved / pk["hbm"], "algorithmic_bytes": nbytes,
                         "bytes_definition": "read + write of every token's K and V",
                         "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                         "kernel": "store", "traffic": ncu_traffic("store", "long_fewshot_chunks")},
            "l2": L2Flush.HOW}


def bench_project_store(torch, comb, w, pk, n=50, d_model=4096):
    """(f2) K/V projection of configs[3]'s 64 chunks fused into the paged store (one tcgen05 GEMM launch whose epilogue
    writes the pages), L2 flushed before every launch; beside it the unfused sequence on the same data: two row-major
    GEMMs (K, V) + comb_store_chunks. Values are device-side N(0,1) (timing only; parity is tests/test_gpu_layer.py)."""
    Hkv, Dqk, Dv = w.num_kv_heads, w.head_dim_qk, w.head_dim_v
    pool = comb.Pool(Hkv, Dqk, Dv, w.pool_pages + 8, shuffle_seed=77)
    ids = list(range(w.num_chunks))
    tok = np.zeros(w.num_chunks + 1, np.int32)
    np.cumsum(w.chunk_len, out=tok[1:])
    T = int(tok[-1])
    N = Hkv * (Dqk + Dv)
    h = torch.randn((T, d_model), device="cuda").to(torch.bfloat16)
    wkv = (torch.randn((N, d_model), device="cuda") / d_model ** 0.5).to(torch.bfloat16)
    flush = L2Flush(torch)
    comb.comb_profile_enable(pool.handle, True)
    for i in range(n + 3):
        flush(i)
        if i == 3:
            torch.cuda.synchronize()
            comb.comb_profile_read(pool.handle, comb.KERNEL_GEMM)
        pool.project_store_chunks(ids, tok, h, wkv)
    st = stats(comb.comb_profile_read_samples(pool.handle, comb.KERNEL_GEMM, cap=n + 8))
    # unfused: K = H W_K^T, V = H W_V^T row-major, then the paged store
    kbuf = torch.empty((T, Hkv, Dqk), dtype=torch.bfloat16, device="cuda")
    vbuf = torch.empty((T, Hkv, Dv), dtype=torch.bfloat16, device="cuda")
    two = []
    for i in range(min(n, 20) + 3):
        flush(i)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        comb.comb_gemm_bf16(pool.handle, h, wkv[:Hkv * Dqk], kbuf, T, Hkv * Dqk, d_model)
        comb.comb_gemm_bf16(pool.handle, h, wkv[Hkv * Dqk:], vbuf, T, Hkv * Dv, d_model)
        pool.store_chunks(ids, tok, kbuf, vbuf)
        b.record()
        torch.cuda.synchronize()
        if i >= 3:
            two.append(a.elapsed_time(b))
    comb.comb_profile_enable(pool.handle, False)
    pool.close()
    flops = 2.0 * T * N * d_model
    nbytes = T * d_model * 2 + N * d_model * 2 + T * N * 2   # H and W read once, pages written once
    achieved = flops / (st["mean"] * 1e-3) / 1e12
    return {"workload": "K/V projection of long_fewshot's %d chunks (%d tokens) x d_model %d -> %d columns, written "
                        "into pages by the GEMM epilogue" % (w.num_chunks, T, d_model, N),
            "kernel_ms": st["mean"], "kernel_ms_median": st["median"], "kernel_ms_min": st["min"],
            "launches_timed": st["n"], "two_step_ms": float(np.mean(two)),
            "two_step": "2 x comb_gemm_bf16 (row-major K, V) + comb_store_chunks, CUDA events around the three launches",
            "roofline": {"bound": "tensor", "achieved": achieved, "peak": pk["tf_burst"], "unit": "TFLOP/s",
                         "frac": achieved / pk["tf_burst"], "frac_of_sustained": achieved / pk["tf_sustained"],
                         "frac_of_nominal_2250": achieved / NOMINAL_BF16_TFLOPS, "algorithmic_flops": flops,
                         "algorithmic_bytes": nbytes, "kernel": "gemm_paged",
                         "traffic": ncu_traffic("gemm_paged", "long_fewshot_chunks")},
            "l2": L2Flush.HOW}


def bench_cross_layer(torch, comb, w, pk, phase, n, d_model=4096, L=8):
    """(f3) the cross-attention sub-layer x + Attn(x W_Q) W_O over the paper's L = 8 cross layers on one
    link: 8 x (Q-projection GEMM, attention, output-projection GEMM with the residual in its epilogue). The 8-layer pool
    is filled with device-side N(0,1) (timing only); only the directory entries of the workload's chunks are made."""
    Hq, Hkv, Dqk, Dv = w.num_q_heads, w.num_kv_heads, w.head_dim_qk, w.head_dim_v
    pool = comb.Pool(Hkv, Dqk, Dv, w.pool_pages, num_layers=L, shuffle_seed=2024)
    pool.k_arena.view(torch.bfloat16).normal_()
    pool.v_arena.view(torch.bfloat16).normal_()
    for c in range(w.num_chunks):
        comb.comb_chunk_alloc(pool.handle, c, int(w.chunk_len[c]))
    lb = pool.link_flat(w.chunk_indptr, w.chunk_ids_flat)
    wq = w.decode_phase() if phase == "decode" and int(w.lq.max()) > 1 else w
    rows = int(wq.total_q)
    q_indptr = None if phase == "decode" else wq.q_indptr
    x = torch.randn((rows, d_model), device="cuda").to(torch.bfloat16)
    wqs = [(torch.randn((Hq * Dqk, d_model), device="cuda") / d_model ** 0.5).to(torch.bfloat16) for _ in range(L)]
    wos = [(torch.randn((d_model, Hq * Dv), device="cuda") * (0.1 / (Hq * Dv) ** 0.5)).to(torch.bfloat16) for _ in range(L)]

    bufs = [torch.empty_like(x), torch.empty_like(x)]

    def step():  # ping-pong between two buffers; layer 0 reads x
        src = x
        for l in range(L):
            dst = bufs[l & 1]
            pool.layer_forward(lb, src, q_indptr, wqs[l], wos[l], w.scale, layer=l, out=dst)
            src = dst

    for _ in range(3):
        step()
    torch.cuda.synchronize()
    comb.comb_profile_enable(pool.handle, True)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    with ClockSampler(torch.cuda.current_device()) as clk:
        ev[0].record()
        for _ in range(n):
            step()
        ev[1].record()
        torch.cuda.synchronize()
    ms = ev[0].elapsed_time(ev[1]) / n
    gemm_ms = comb.comb_profile_read(pool.handle, comb.KERNEL_GEMM)[0] / n
    attn_ms = sum(comb.comb_profile_read(pool.handle, k)[0] for k in (
        comb.KERNEL_PREFILL, comb.KERNEL_PREFILL_MERGE, comb.KERNEL_DECODE_SPLIT, comb.KERNEL_DECODE_MERGE,
        comb.KERNEL_DECODE_CASCADE, comb.KERNEL_CASCADE_MERGE)) / n
    comb.comb_profile_enable(pool.handle, False)
    pool.close()
    torch.cuda.empty_cache()
    gemm_flops = L * 2.0 * rows * d_model * (Hq * Dqk + Hq * Dv)
    attn_flops = L * float(wq.attention_flops())
    return {"workload": "%d cross layers (PAPER.md:78) of %s, %s phase: %d rows x d_model %d" % (
                L, w.name, phase, rows, d_model),
            "ms_per_step": ms, "gemm_ms": gemm_ms, "attention_ms": attn_ms,
            "tflops": (gemm_flops + attn_flops) / (ms * 1e-3) / 1e12, "gemm_tflops": gemm_flops / (gemm_ms * 1e-3) / 1e12,
            "us_per_q_token": ms * 1e3 / rows, "us_per_q_token_per_layer": ms * 1e3 / rows / L,
            "weight_bytes": L * 2 * d_model * (Hq * Dqk + Hq * Dv), "clocks": clk.summary(),
            "note": "Eq. 12: T_cross = O(L_cross l_query l_doc); per-layer cost = step / 8"}


def bench_link(torch, comb, harness, w):
    """(a3) link latency: host table build + enqueue of the single H2D copy; and until the tables are resident."""
    pool = comb.Pool(w.num_kv_heads, w.head_dim_qk, w.head_dim_v, w.pool_pages, shuffle_seed=5)
    for c in range(w.num_chunks):
        comb.comb_chunk_alloc(pool.handle, c, int(w.chunk_len[c]))  # directory only: link reads no KV
    ci, ids = w.chunk_indptr, w.chunk_ids_flat
    lb = pool.link_flat(ci, ids)
    host, full = [], []
    for i in range(1100):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        pool.link_flat(ci, ids, into=lb)
        t1 = time.perf_counter()
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        if i >= 100:
            host.append((t1 - t0) * 1e6)
            full.append((t2 - t0) * 1e6)
    pool.close()
    return {"workload": "decode_link: %d requests, %d table entries, %d distinct chunks, %d B copied" % (
                w.num_requests, int(lb.link.total_pages), int(lb.link.num_distinct_chunks), int(lb.link.bytes_used)),
            "host_enqueue_us_p50": float(np.percentile(host, 50)), "host_enqueue_us_p99": float(np.percentile(host, 99)),
            "resident_us_p50": float(np.percentile(full, 50)), "resident_us_p99": float(np.percentile(full, 99)),
            "kv_bytes_copied": 0}


def bench_stream_read(torch, comb, pk):
    """Read-only HBM ceiling of the day (SURVEY.md §8(d) "Denominators"): the library's streaming-read kernel over a
    4 GiB buffer (32x the L2), 20 launches after 3 warm-ups, CUDA events on the launching stream."""
    n = 4 << 30
    buf = torch.empty(n, dtype=torch.uint8, device="cuda")
    buf.random_(0, 255)
    sink = torch.zeros(1, dtype=torch.int32, device="cuda")
    ms = []
    for i in range(23):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        comb.comb_util_stream_read(buf, sink)
        b.record()
        torch.cuda.synchronize()
        if i >= 3:
            ms.append(a.elapsed_time(b))
    del buf
    torch.cuda.empty_cache()
    return {"bytes": n, "ms_mean": float(np.mean(ms)), "ms_min": float(np.min(ms)),
            "gbs_mean": n / (np.mean(ms) * 1e-3) / 1e9, "gbs_best": n / (np.min(ms) * 1e-3) / 1e9,
            "copy_peak_gbs": pk["hbm"], "how": "comb_util_stream_read, 4 GiB, 128-bit streaming loads, no stores"}


if __name__ == "__main__":
    main()
