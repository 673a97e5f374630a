"""GPU test of comb_cross_attn_decode_noalloc (include/comb.h): decode with its split partials in the library's fixed
device array instead of a caller workspace.  Collected last on purpose (the suite runs with pytest -x).

The new entry point runs the per-request kernels of comb_cross_attn_decode with the same split plan, so against that
path the outputs are compared bit for bit; against the default (chunk-major) path and the fp64 oracle the bars are the
ones of tests/test_gpu_parity.py (DESIGN.md §2 "Tolerances"), restated here."""
import numpy as np
import pytest

import comb_synth as cs
import oracle

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _bits(t):
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def _run_all_paths(ld, w, comb):
    """(noalloc out, lse), (per-request out, lse), (default-path out, lse) for the linked batch of `ld`."""
    pool, q = ld.pool, ld.q
    R, Hq = int(q.shape[0]), int(q.shape[1])
    out = torch.full((R, Hq, w.head_dim_v), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.full((R, Hq), float("nan"), dtype=torch.float32, device="cuda")
    pool.decode_noalloc(ld.batch, q, w.scale, out, lse)
    pool.set_decode_path(comb.DECODE_PER_REQUEST)
    out_pr, lse_pr = pool.decode(ld.batch, q, w.scale)
    pool.set_decode_path(comb.DECODE_AUTO)
    out_auto, lse_auto = pool.decode(ld.batch, q, w.scale)
    torch.cuda.synchronize()
    return (_bits(out), lse.cpu().numpy()), (_bits(out_pr), lse_pr.cpu().numpy()), (_bits(out_auto), lse_auto.cpu().numpy())


def _check(got, ref_pr, ref_auto, w, tag):
    out, lse = got
    # same kernels, same plan: bit-exact against the existing per-request path
    assert np.array_equal(out, ref_pr[0]), tag + ": output differs from comb_cross_attn_decode (per-request path)"
    assert np.array_equal(lse, ref_pr[1]), tag + ": LSE differs from comb_cross_attn_decode (per-request path)"
    # other kernel (chunk-major): |a - b| <= 2^-7 |a| + 1.5e-3, mean <= 3e-4 (close_in_ulps of test_gpu_parity.py)
    a, b = cs.bf16_bits_to_f64(out), cs.bf16_bits_to_f64(ref_auto[0])
    d = np.abs(a - b)
    assert np.all(d <= 2.0 ** -7 * np.abs(a) + 1.5e-3), "%s: vs default path max %.3e" % (tag, d.max())
    assert d.mean() <= 3e-4, "%s: vs default path mean %.3e" % (tag, d.mean())
    # fp64 oracle: BASELINE.json's bars + relative L2 and LSE
    O, L = oracle.attention_for(w)
    err = np.abs(a - O)
    assert err.max() <= 2e-2 and err.mean() <= 2e-3, "%s: vs oracle max %.3e mean %.3e" % (tag, err.max(), err.mean())
    assert np.sqrt((err ** 2).sum() / (O ** 2).sum()) <= 1e-2, tag + ": relative L2 against the oracle"
    fin = np.isfinite(L)
    assert np.array_equal(np.isneginf(lse), np.isneginf(L)), tag + ": -inf pattern of LSE"
    assert np.abs(lse[fin].astype(np.float64) - L[fin]).max() <= 2e-4, tag + ": LSE against the oracle"


def test_decode_noalloc_matches_existing_paths_on_two_calls_in_a_row():
    import paper_2602_01519_b200 as comb
    from paper_2602_01519_b200 import harness

    assert comb.comb_noalloc_scratch_bytes() == 8 << 20
    # call 1: one long request (many KV splits -> partials in the static array) beside short ones and an empty link
    w1 = cs.custom("noalloc_long", num_q_heads=8, num_kv_heads=2, head_dim_qk=128, head_dim_v=128,
                   chunk_len=[1000] * 12 + [37], links=[list(range(12)) + [12], [12], [], [3, 12, 5]], lq=[1, 1, 1, 1])
    # call 2: a Llama-shaped batch with chunk reuse and other split counts: the array still holds call 1's partials
    rng = np.random.default_rng(5)
    lens = rng.integers(100, 700, size=20).astype(np.int32)
    links = [rng.choice(20, size=int(rng.integers(2, 9)), replace=False) for _ in range(12)]
    w2 = cs.custom("noalloc_batch", k=10, num_q_heads=32, num_kv_heads=8, head_dim_qk=128, head_dim_v=128,
                   chunk_len=lens, links=links, lq=[1] * 12)
    ld1 = harness.load_workload(w1, shuffle_seed=3)
    ld2 = harness.load_workload(w2, shuffle_seed=11)
    for rep in range(2):  # 1, 2, 1, 2: every call follows one that left other contents in the array
        for name, ld, w in (("call 1", ld1, w1), ("call 2", ld2, w2)):
            got, ref_pr, ref_auto = _run_all_paths(ld, w, comb)
            _check(got, ref_pr, ref_auto, w, "%s (round %d)" % (name, rep))
    out, lse = _run_all_paths(ld1, w1, comb)[0]
    assert np.all(out[2] == 0) and np.all(np.isneginf(lse[2]))  # empty link (reading I13): O = 0, LSE = -inf

    # the call allocates nothing: torch's allocator and the device's free memory are where they were
    q, R, Hq = ld2.q, int(ld2.q.shape[0]), int(ld2.q.shape[1])
    out = torch.empty((R, Hq, w2.head_dim_v), dtype=torch.bfloat16, device="cuda")
    lse = torch.empty((R, Hq), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    alloc0, free0 = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    launches0 = ld2.pool.launches
    ld2.pool.decode_noalloc(ld2.batch, q, w2.scale, out, lse)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == alloc0
    assert torch.cuda.mem_get_info()[0] >= free0
    assert ld2.pool.launches - launches0 in (1, 2)  # split kernel (+ merge): our kernels ran

    # scope: fp8 pools have no per-request kernel
    w8 = cs.custom("noalloc_fp8", k=11, num_q_heads=8, num_kv_heads=2, head_dim_qk=128, head_dim_v=128,
                   chunk_len=[64, 40], links=[[0, 1]], lq=[1])
    ld8 = harness.load_workload(w8, kv_dtype=comb.KV_E4M3)
    o8 = torch.empty((1, 8, 128), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(comb.CombError) as e:
        ld8.pool.decode_noalloc(ld8.batch, ld8.q, w8.scale, o8)
    assert e.value.status == comb.COMB_ERR_INVALID
    for ld in (ld1, ld2, ld8):
        ld.pool.close()
