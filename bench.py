#!/usr/bin/env python
"""bench.py — measures the COMB link-stage hot path on B200 (contract: one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME] [--no-extras]

A *step* is one pass of the hot path over one batch of BASELINE.json configs[1] ("decode link": Llama-3-8B-
shaped layer, 128 requests x 1 query token, each linking 8 chunks of 512 tokens drawn Zipf(1.1) from a
2000-chunk pool): comb_link (block tables from the ordered chunk ids, one H2D copy, no KV copy) followed by
comb_cross_attn_decode (split-KV kernel + LSE-merge kernel) over the resident chunk-KV pool.  `value` is the
logical KV bytes the step attends over divided by the device time (CUDA events, max over ranks).  The chunk pool
itself was stored before the timed region (compile stage); the paged-store kernel, the tcgen05
prefill kernel (configs[2] "RAG prefill", TFLOP/s against the tensor roofline) and configs[3]/[4] are timed in
the same run and reported under "extras".  N > 1: independent replicas, one per GPU, no collective on the data
path -> weak scaling.

`--impl reference` times the fp64 CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
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
METRIC = ("decode cross-attn HBM GB/s over block-table-linked chunk KV (BASELINE metric: cross-attn TFLOP/s "
          "(prefill) and HBM GB/s (decode) at 1 B200 vs roofline; prefill TFLOP/s is under extras.rag_prefill)")


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
    committed ncu --set full capture (profiles/ncu_traffic.csv), or None when that pair was not captured."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f.read().splitlines()[1:]:
            cols = line.split(",")
            if len(cols) >= 3 and cols[0] == kernel and cols[1] == workload:
                return int(cols[2])
    return None


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
    """Samples SM clock and throttle reasons DURING the timed region (NVML, every 10 ms)."""

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
            self._stop.wait(0.01)

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
        value, unit, metric = flops / dt / 1e12, "TFLOP/s", "prefill cross-attn TFLOP/s"
    sample = "each step = oracle on the first %d request(s) of %s%s" % (
        n, w.name, "" if phase == "decode" else " (first 8 query tokens)")
    print(json.dumps({
        "impl": "reference", "metric": metric, "value": value, "unit": unit, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "sample": sample},
        "cpu_baseline": {"value": value, "unit": unit, "cores": oracle.max_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="decode_link", choices=["decode_link", "rag_prefill"])
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs, store and CPU baseline")
    ap.add_argument("--seed", type=int, default=0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

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
    primary_prefill = args.workload == "rag_prefill"

    # ------------------------------------------------------------------ attention benches
    def bench_attention(w, phase, steps, warmup, *, fill, flush_l2=False, with_link=True, e2e=True, shuffle=None):
        """Returns a dict of timings for `steps` passes of (link +) attention on workload w."""
        # free list: permuted (a chunk's pages scattered over the arena, as in a long-running server) unless told
        ld = harness.load_workload(w, fill=fill, shuffle_seed=(2024 + rank) if shuffle is None else shuffle,
                                   keep_host=False)
        pool = ld.pool
        if phase == "decode":
            wq = w.decode_phase() if int(w.lq.max()) > 1 else w
            q = harness.bits_to_device(wq.all_q(), "cuda")
            q_indptr = wq.q_indptr
        else:
            wq, q, q_indptr = w, ld.q, ld.q_indptr
        R, Hq = wq.num_requests, wq.num_q_heads
        out = torch.empty((q.shape[0], Hq, w.head_dim_v), dtype=torch.bfloat16, device="cuda")
        lse = torch.empty((q.shape[0], Hq), dtype=torch.float32, device="cuda")
        chunk_indptr, chunk_ids = w.chunk_indptr, w.chunk_ids_flat
        batch = ld.batch
        kid = comb.KERNEL_DECODE_SPLIT if phase == "decode" else comb.KERNEL_PREFILL
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
        k_ms, k_n = comb.comb_profile_read(pool.handle, kid)
        m_ms, m_n = comb.comb_profile_read(pool.handle, comb.KERNEL_DECODE_MERGE)
        comb.comb_profile_enable(pool.handle, False)
        res = {"ms_per_step": max_over_ranks(total_ms / steps), "kernel_ms": k_ms / max(k_n, 1),
               "merge_ms": (m_ms / m_n) if m_n else 0.0, "launches": launches, "clocks": clk.summary(),
               "flops": wq.attention_flops(), "kv_bytes": wq.kv_bytes_logical(), "q_tokens": wq.total_q,
               "timed_seconds": total_ms / 1e3}
        # io bytes the kernel also moves (Q in, O + LSE out)
        res["io_bytes"] = q.numel() * 2 + out.numel() * 2 + lse.numel() * 4
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

    def roofline_hbm(r, kernel_name, wname):
        achieved = (r["kv_bytes"] + r["io_bytes"]) / (r["kernel_ms"] * 1e-3) / 1e9
        return {"bound": "hbm", "achieved": achieved, "peak": pk["hbm"], "unit": "GB/s", "frac": achieved / pk["hbm"],
                "peak_source": pk["src"] + " copy bandwidth (MEASURED_PEAKS.json hbm_gbs)",
                "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS, "kernel": kernel_name,
                "kernel_ms": r["kernel_ms"], "algorithmic_bytes": r["kv_bytes"] + r["io_bytes"],
                "traffic": ncu_traffic(kernel_name, wname)}

    def roofline_tensor(r, kernel_name, wname):
        achieved = r["flops"] / (r["kernel_ms"] * 1e-3) / 1e12
        sustained = r["timed_seconds"] >= 1.0
        peak = pk["tf_sustained"] if sustained else pk["tf_burst"]
        return {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "peak_source": "%s cuBLAS bf16 %s" % (pk["src"], "sustained" if sustained else "burst"),
                "frac_of_burst": achieved / pk["tf_burst"], "frac_of_sustained": achieved / pk["tf_sustained"],
                "frac_of_nominal_2250": achieved / NOMINAL_BF16_TFLOPS, "kernel": kernel_name,
                "kernel_ms": r["kernel_ms"], "algorithmic_flops": r["flops"], "traffic": ncu_traffic(kernel_name, wname)}

    # ------------------------------------------------------------------ primary workload
    if primary_prefill:
        w = cs.rag_prefill(seed=args.seed + rank)
        r = bench_attention(w, "prefill", args.steps, args.warmup, fill="linked")
        value = world * r["flops"] / (r["ms_per_step"] * 1e-3) / 1e12
        unit, metric = "TFLOP/s", "prefill cross-attn TFLOP/s (BASELINE metric, prefill half)"
        roof = roofline_tensor(r, "prefill", "rag_prefill")
        e2e_val = world * r["flops"] / (r["e2e_ms"] * 1e-3) / 1e12
        dtype = "bf16"
    else:
        w = cs.decode_link(seed=args.seed + rank)
        r = bench_attention(w, "decode", args.steps, args.warmup, fill="linked")
        value = world * r["kv_bytes"] / (r["ms_per_step"] * 1e-3) / 1e9
        unit, metric = "GB/s", METRIC
        roof = roofline_hbm(r, "decode_split", "decode_link")
        e2e_val = world * r["kv_bytes"] / (r["e2e_ms"] * 1e-3) / 1e9
        dtype = "bf16"
    log("primary", json.dumps(r))

    cpu = None
    if rank == 0 and world == 1 and not args.no_extras:
        # ---- the other configs (not bench lines; context for the BASELINE metric's prefill half) ----
        def prefill_extra(name, wk, steps, fill, flush=False):
            rr = bench_attention(wk, "prefill", steps, 3, fill=fill, flush_l2=flush, e2e=False)
            # a prefill whose flops per logical KV byte sit under the ridge of the measured peaks is HBM-bound
            # (no GQA or few query tokens: SURVEY.md 8(d)); it is then reported against the HBM roof first
            ridge = pk["tf_burst"] * 1e12 / (pk["hbm"] * 1e9)
            intensity = rr["flops"] / (rr["kv_bytes"] + rr["io_bytes"])
            extras[name] = {"workload": name, "ms_per_step": rr["ms_per_step"], "kernel_ms": rr["kernel_ms"],
                            "tflops": rr["flops"] / (rr["ms_per_step"] * 1e-3) / 1e12,
                            "q_tokens_per_s": rr["q_tokens"] / (rr["ms_per_step"] * 1e-3),
                            "flop_per_logical_byte": intensity, "ridge_flop_per_byte": ridge,
                            "roofline_hbm": roofline_hbm(rr, "prefill", "") if intensity < ridge else None,
                            "roofline": roofline_tensor(rr, "prefill", name.replace("_prefill", "") if name != "rag_prefill" else name), "clocks": rr["clocks"],
                            "l2": L2Flush.HOW if flush else "inputs larger than L2"}
            log(name, json.dumps(extras[name]))

        def decode_extra(name, wk, steps, fill, flush=False, shuffle=None):
            rr = bench_attention(wk, "decode", steps, 3, fill=fill, flush_l2=flush, e2e=False, shuffle=shuffle)
            extras[name] = {"workload": name, "ms_per_step": rr["ms_per_step"], "kernel_ms": rr["kernel_ms"],
                            "merge_ms": rr["merge_ms"],
                            "gbs_logical": rr["kv_bytes"] / (rr["ms_per_step"] * 1e-3) / 1e9,
                            "roofline": roofline_hbm(rr, "decode_split", name.replace("_decode", "") if name != "decode_link" else name), "clocks": rr["clocks"],
                            "l2": L2Flush.HOW if flush else "inputs larger than L2"}
            log(name, json.dumps(extras[name]))

        try:
            if not primary_prefill:
                prefill_extra("rag_prefill", cs.rag_prefill(seed=args.seed), 20, "linked")
            else:
                decode_extra("decode_link", cs.decode_link(seed=args.seed), 100, "linked")
            if not primary_prefill:  # the same primary workload with an ascending free list (contiguous chunks)
                decode_extra("decode_link_contiguous_pages", cs.decode_link(seed=args.seed), 100, "linked", shuffle=0)
            prefill_extra("rag_prefill_lq32", cs.rag_prefill(seed=args.seed, lq=32), 20, "linked")
            # the paper's own regime (< 50 dynamic tokens) at a small batch: 32 work items for 148 SMs,
            # so each request's KV is cut into ranges that run on different SMs and are merged by LSE
            prefill_extra("rag_prefill_lq32_r4", cs.rag_prefill(seed=args.seed, lq=32, requests=4), 20, "linked",
                          flush=True)
            prefill_extra("long_fewshot_prefill", cs.long_fewshot(seed=args.seed), 10, "all", flush=True)
            decode_extra("long_fewshot_decode", cs.long_fewshot(seed=args.seed), 50, "all", flush=True)
            prefill_extra("mla_shaped_prefill", cs.mla_shaped(seed=args.seed), 20, "linked")
            decode_extra("mla_shaped_decode", cs.mla_shaped(seed=args.seed), 50, "linked")
            extras["store"] = bench_store(torch, comb, harness, cs.long_fewshot(seed=args.seed), pk)
            extras["link"] = bench_link(torch, comb, harness, cs.decode_link(seed=args.seed))
        except Exception as e:  # extras must never lose the primary line
            extras["error"] = repr(e)
            log("extras failed:", repr(e))
        # ---- CPU baseline: the oracle on the host cores, bounded sample ----
        try:
            o = oracle_sample(w, "prefill" if primary_prefill else "decode")
            cpu = {"value": o["gflops"] / 1e3 if primary_prefill else o["gbs"], "unit": unit, "cores": o["cores"],
                   "kind": "oracle", "sample": o["sample"], "seconds": o["seconds"], "gflops_fp64": o["gflops"],
                   "q_tokens_per_s": o["q_tokens_per_s"]}
        except Exception as e:
            cpu = {"error": repr(e)}

    if rank == 0:
        line = {
            "metric": metric, "value": value, "unit": unit, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": dtype, "data": "synthetic",
            "config": {"workload": "rag_prefill (BASELINE configs[2])" if primary_prefill
                       else "decode_link (BASELINE configs[1])",
                       "requests": w.num_requests, "q_tokens_per_step": r["q_tokens"],
                       "kv_tokens_per_request": w.kv_len(0), "heads": "%d/%d" % (w.num_q_heads, w.num_kv_heads),
                       "head_dim": "%d/%d" % (w.head_dim_qk, w.head_dim_v), "page": 16,
                       "pool_pages": w.pool_pages, "free_list": "permuted (scattered pages)",
                       "step": "comb_link + comb_cross_attn_%s" % ("prefill" if primary_prefill else "decode"),
                       "l2": "inputs larger than L2 (logical %.2f GB KV per step)" % (r["kv_bytes"] / 1e9),
                       "parallelism": "replicas x%d" % world},
            "clocks": r["clocks"],
            "e2e": {"value": e2e_val, "unit": unit, "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"],
                    "ms_per_step": r["e2e_ms"], "serial_ms_per_step": r["e2e_serial_ms"],
                    "how": "host buffers through the public API; pinned Q -> device, comb_link (tables H2D), attention, "
                           "O + LSE -> pinned host every step; double-buffered over three streams (serial_ms_per_step: "
                           "the same with a device synchronise after every step)"},
            "gpu_launches": int(r["launches"]),
            "roofline": roof,
            "q_tokens_per_s": world * r["q_tokens"] / (r["ms_per_step"] * 1e-3),
        }
        if cpu is not None:
            line["cpu_baseline"] = cpu
        if extras:
            line["extras"] = extras
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def bench_store(torch, comb, harness, w, pk):
    """(a2) batched paged store of configs[3]'s 64 variable-length chunks: free + store again, 20 times."""
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
    n = 20
    for i in range(n + 3):
        for c in ids:
            comb.comb_chunk_free(pool.handle, c)
        flush(i)
        if i == 3:
            torch.cuda.synchronize()
            comb.comb_profile_read(pool.handle, comb.KERNEL_STORE)
        pool.store_chunks(ids, tok, k, v)
    ms, cnt = comb.comb_profile_read(pool.handle, comb.KERNEL_STORE)
    comb.comb_profile_enable(pool.handle, False)
    nbytes = 2 * T * w.num_kv_heads * (w.head_dim_qk + w.head_dim_v) * 2
    achieved = nbytes / (ms / cnt * 1e-3) / 1e9
    pool.close()
    return {"workload": "store of long_fewshot's %d chunks (%d tokens), one launch" % (w.num_chunks, T),
            "kernel_ms": ms / cnt, "roofline": {"bound": "hbm", "achieved": achieved, "peak": pk["hbm"], "unit": "GB/s",
                                                 "frac": achieved / pk["hbm"], "algorithmic_bytes": nbytes,
                                                 "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                                                 "kernel": "store", "traffic": ncu_traffic("store", "long_fewshot")},
            "l2": L2Flush.HOW}


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
    return {"workload": "decode_link: %d requests, %d table entries, %d B copied" % (
                w.num_requests, int(lb.link.total_pages), int(lb.link.bytes_used)),
            "host_enqueue_us_p50": float(np.percentile(host, 50)), "host_enqueue_us_p99": float(np.percentile(host, 99)),
            "resident_us_p50": float(np.percentile(full, 50)), "resident_us_p99": float(np.percentile(full, 99)),
            "kv_bytes_copied": 0}


if __name__ == "__main__":
    main()
