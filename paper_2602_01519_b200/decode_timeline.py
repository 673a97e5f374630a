"""Cycle-level timeline of the bf16 chunk-major decode kernel's CTA 0 (profiling aid).

    python paper_2602_01519_b200/decode_timeline.py [hot | decode_link] [first tile] [tiles]

Builds libcomb_trace.so (the library's sources with -DCOMB_TRACE: clock64() stamps in softmax thread 0 and in the
tcgen05.mma issuing warp, cascade_kernel.cu), runs the decode call three times through the public binding and prints,
per KV tile of CTA 0, what each role waited for and for how long.  `hot` is cfg 2's geometry with every request linking
the same 8 chunks (full 32-row items, everything from L2); `decode_link` is cfg 2.  Needs a GPU; the product library
libcomb.so carries no stamps and is not touched.
"""
from __future__ import annotations

import ctypes as C
import importlib.util
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))


def main():
    argv = sys.argv[1:]
    name = argv[0] if argv else "hot"
    first = int(argv[1]) if len(argv) > 1 else 8
    count = int(argv[2]) if len(argv) > 2 else 12
    spec = importlib.util.spec_from_file_location("comb_build", os.path.join(HERE, "build.py"))
    build = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(build)
    os.environ["COMB_LIBRARY"] = build.build(trace=2)

    import numpy as np
    import torch
    import comb_synth
    from paper_2602_01519_b200 import _lib, harness

    w = comb_synth.decode_link(pool_chunks=8) if name == "hot" else comb_synth.decode_link()
    ld = harness.load_workload(w, fill="linked", shuffle_seed=2024, keep_host=False)
    out = torch.empty((ld.q.shape[0], w.num_q_heads, w.head_dim_v), dtype=torch.bfloat16, device="cuda")
    for _ in range(3):
        ld.pool.decode(ld.batch, ld.q, w.scale, out=out)
    torch.cuda.synchronize()
    tr = np.zeros((2, 256, 8), np.uint64)
    rc = C.CDLL(_lib.LIB_PATH).comb_trace_cascade_read(C.c_void_p(tr.ctypes.data))
    if rc != 0:
        raise SystemExit("comb_trace_cascade_read: %d" % rc)
    tr = tr.astype(np.int64)
    t0 = int(tr[0, 0, 0])
    print("workload %s: CTA 0, cycles relative to its first s_full wait" % name)
    for t in range(first, first + count):
        y, x = tr[0, t] - t0, tr[1, t] - t0
        if tr[0, t, 1] == 0:
            continue
        print("tile %3d softmax: waits from %7d, S seen +%5d, S read +%4d, vote +%4d, P buffer free +%4d, P handed over +%4d"
              " | issuer: at K/s_empty wait %7d, S issued +%5d, P seen %7d, P V issued +%4d" % (
                  t, y[0], y[1] - y[0], y[2] - y[1], y[3] - y[2], y[4] - y[3], y[5] - y[4],
                  x[0], x[1] - x[0], x[2], x[3] - x[2]))
    seen = tr[0, first:first + count, 1]
    seen = seen[seen > 0]
    if len(seen) > 1:
        print("period per KV tile: %.0f cycles" % float(np.mean(np.diff(seen))))


if __name__ == "__main__":
    main()
