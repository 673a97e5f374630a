"""Cycle-level timeline of the prefill kernel's CTA 0 (profiling aid).

    python paper_2602_01519_b200/prefill_timeline.py [rag_prefill | rag_prefill_lq32 | rag_prefill_lq32_r4] [first tile] [tiles] [--softmax-only]

Builds libcomb_trace.so (the library's sources with -DCOMB_TRACE: clock64() stamps in one softmax thread per
warpgroup and in the tcgen05.mma issuing lane, attn_core.cuh), runs the workload's prefill call three times through
the public binding and prints, per KV tile of CTA 0's first work items, what each role waited for and for how long.
--softmax-only leaves the issuer's stamps out (they lengthen the loop by ~10 %: the issuing thread runs in step with
the tensor pipe) and is what the period should be read from.
Needs a GPU.  The product library libcomb.so carries no stamps and is not touched.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))


def main():
    argv = [x for x in sys.argv[1:] if not x.startswith("--")]
    level = 1 if "--softmax-only" in sys.argv else 2
    name = argv[0] if len(argv) > 0 else "rag_prefill"
    first = int(argv[1]) if len(argv) > 1 else 8
    count = int(argv[2]) if len(argv) > 2 else 12
    import importlib.util
    spec = importlib.util.spec_from_file_location("comb_build", os.path.join(HERE, "build.py"))
    build = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(build)
    os.environ["COMB_LIBRARY"] = build.build(trace=level)

    import numpy as np
    import torch
    import comb_synth
    from paper_2602_01519_b200 import _lib, harness

    w = {"rag_prefill": lambda: comb_synth.rag_prefill(),
         "rag_prefill_lq32": lambda: comb_synth.rag_prefill(lq=32),
         "rag_prefill_lq32_r4": lambda: comb_synth.rag_prefill(requests=4, lq=32)}[name]()
    ld = harness.load_workload(w, fill="linked", shuffle_seed=2024, keep_host=False)
    out = torch.empty((ld.q.shape[0], w.num_q_heads, w.head_dim_v), dtype=torch.bfloat16, device="cuda")
    lse = torch.empty((ld.q.shape[0], w.num_q_heads), dtype=torch.float32, device="cuda")
    for _ in range(3):
        ld.pool.prefill(ld.batch, ld.q, ld.q_indptr, w.scale, out=out, lse=lse)
    torch.cuda.synchronize()
    sm = np.zeros((2, 128, 8), np.uint64)
    mma = np.zeros((2, 128, 8), np.uint64)
    rc = C.CDLL(_lib.LIB_PATH).comb_trace_prefill_read(C.c_void_p(sm.ctypes.data), C.c_void_p(mma.ctypes.data))
    if rc != 0:
        raise SystemExit("comb_trace_prefill_read: %d" % rc)
    ctas = np.zeros((1024, 4), np.uint64)
    if C.CDLL(_lib.LIB_PATH).comb_trace_prefill_read_ctas(C.c_void_p(ctas.ctypes.data)) == 0:
        ctas = ctas.astype(np.int64)
        live = ctas[ctas[:, 3] >= ctas[:, 0].max()]  # CTAs of the last launch (older launches' stamps are smaller)
        t_first = live[:, 0].min()
        rel = live - t_first
        print("%d CTAs, %%globaltimer ns after the first CTA's entry (min / median / max): entry %d/%d/%d, set-up done "
              "%d/%d/%d, loop end %d/%d/%d, exit %d/%d/%d" % ((len(live),) + tuple(
                  int(f(rel[:, k])) for k in range(4) for f in (np.min, np.median, np.max))))
    sm = sm.astype(np.int64)
    mma = mma.astype(np.int64)
    t0 = int(sm[0, 0, 0])
    cta = sm[1, 127]
    print("workload %s: CTA 0, cycles relative to the first s_full wait of Q tile 0" % name)
    print("kernel entry %d | set-up done %d | softmax loop of thread 0 ends %d | exit %d" % (
        cta[0] - t0, cta[1] - t0, cta[2] - t0, cta[3] - t0))
    tiles = 2 if sm[1, first, 1] else 1
    for j in range(first, first + count):
        for t in range(tiles):
            y, x = sm[t, j] - t0, mma[t, j] - t0
            if sm[t, j, 1] == 0:
                continue
            line = "tile %3d Q%d softmax: waits from %7d, S seen %7d, max +%4d, P[0:64] +%4d, P[64:128] +%4d" % (
                j, t, y[0], y[1], y[3] - y[1], y[4] - y[3], y[5] - y[4])
            if level >= 2:
                line += " | issuer: at P wait %7d, first half +%4d, second half +%4d, PV issued +%4d, next S %7d..+%4d" % (
                    x[0], x[1] - x[0], x[2] - x[1], x[3] - x[2], x[5] if mma[t, j, 5] else -1,
                    (x[6] - x[5]) if mma[t, j, 5] else 0)
            print(line)
    wakes = sm[0, first:first + count, 1]
    wakes = wakes[wakes > 0]
    if len(wakes) > 1:
        print("period per KV tile (Q tile 0): %.0f cycles" % float(np.mean(np.diff(wakes))))


if __name__ == "__main__":
    main()
