"""Child process of tests/test_gpu_parity.py::test_pool_export_import_across_processes (not a test module).

    python tests/ipc_child.py <blob1> <blob2> <out.npz>

Plays the inference-engine process of PAPER.md:205: opens the pool another process exported (CUDA IPC, read-only),
links and attends over the exporter's bytes, and writes what it computed for the parent to compare with the oracle.
Calls only the public binding; the workload parameters mirror the parent's (seeded, so Q is identical)."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import comb_synth as cs  # noqa: E402
import paper_2602_01519_b200 as comb  # noqa: E402
from paper_2602_01519_b200 import harness  # noqa: E402

SPEC = dict(k=6, num_q_heads=32, num_kv_heads=8, head_dim_qk=128, head_dim_v=128, chunk_len=[300, 520, 77, 1000])
LINKS_A = [[1, 0], [2, 1, 0], [0]]
LINKS_B = [[3, 1], [2, 3, 0], [3]]


def attend(pool, links, lq):
    w = cs.custom("ipc", links=links, lq=lq, **SPEC)
    lb = pool.link([list(map(int, l)) for l in links])
    q = harness.bits_to_device(w.all_q(), "cuda")
    if max(lq) > 1:
        out, lse = pool.prefill(lb, q, w.q_indptr, w.scale)
    else:
        out, lse = pool.decode(lb, q, w.scale)
    torch.cuda.synchronize()
    return harness.device_to_bits(out), lse.cpu().numpy()


def main():
    blob1, blob2 = open(sys.argv[1], "rb").read(), open(sys.argv[2], "rb").read()
    pool = comb.Pool.from_export(blob1)
    res = {}
    res["geom"] = np.array([pool.num_layers, pool.num_kv_heads, pool.head_dim_qk, pool.head_dim_v, pool.num_pages])
    res["pages0"] = comb.comb_chunk_query(pool.handle, 0)[1]
    for path, name in ((comb.DECODE_PER_REQUEST, "dec_pr"), (comb.DECODE_CHUNK_MAJOR, "dec_cm")):
        pool.set_decode_path(path)
        res[name + "_o"], res[name + "_l"] = attend(pool, LINKS_A, [1, 1, 1])
    res["pre_o"], res["pre_l"] = attend(pool, LINKS_A, [40, 130, 7])
    status = []
    for fn in (lambda: comb.comb_chunk_alloc(pool.handle, 99, 16), lambda: comb.comb_chunk_free(pool.handle, 0),
               lambda: pool.link([[3]])):
        try:
            fn()
            status.append(0)
        except comb.CombError as e:
            status.append(e.status)
    res["status"] = np.array(status)
    pool.refresh(blob2)  # the exporter stored chunk 3 on a side stream meanwhile; the blob's event orders us after it
    pool.set_decode_path(comb.DECODE_AUTO)
    res["dec2_o"], res["dec2_l"] = attend(pool, LINKS_B, [1, 1, 1])
    res["pre2_o"], res["pre2_l"] = attend(pool, LINKS_B, [9, 200, 33])
    pool.close()
    np.savez(sys.argv[3], **res)


if __name__ == "__main__":
    main()
