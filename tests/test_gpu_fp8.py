"""GPU parity tests (run with -m gpu on a B200) of fp8 (e4m3) pools — SURVEY.md §8(f4), include/comb.h "fp8 pools",
DESIGN.md §2 readings I31-I33 — through the C ABI against oracle/fp8.py:

  store    codes and power-of-two scales of every (page, kv-head) block BIT-EXACT (the quantisation rule is part of the
           contract); tail slots byte 0; pages owned by no chunk untouched.
  attend   attention over an fp8 pool is Eq. 7-8 over the DEQUANTISED values.  Those are exactly bf16 numbers (the scale
           is a power of two), so the expected result is the pinned fp64 C oracle run on the dequantised chunks; the
           numpy statement in oracle/fp8.py must agree with it too.

Tolerances: exactly those of bf16 pools (max abs 2e-2, mean abs 2e-3, relative L2 1e-2, |LSE error|
<= 2e-4): the kernel's hi + lo split of Q and of the weights keeps 7-8 significant bits per element, like bf16.
Measured: relative L2 1.7e-3, |LSE error| 2e-6.  What the quantisation ITSELF costs against the unquantised chunks is
recorded beside it (relative L2 3.3e-2 on N(0,1) inputs, 6.5e-2 on the peaked variants) and only sanity-checked."""
import json
import math
import os

import numpy as np
import pytest

import comb_synth as cs
import oracle
from oracle import fp8

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BYTE_SENTINEL = 0xA5


def H():
    from paper_2602_01519_b200 import harness
    return harness


def record(tag, **kw):
    try:
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, "gpurun_out", "parity_measured.jsonl"), "a") as f:
            f.write(json.dumps(dict(tag=tag, **{k: float(v) for k, v in kw.items()})) + "\n")
    except OSError:
        pass


class Dequantised:
    """The workload with every chunk replaced by its dequantised fp8 image (bf16-exact), for the C oracle."""

    def __init__(self, w):
        self._w, self._cache = w, {}

    def __getattr__(self, name):
        return getattr(self._w, name)

    def chunk_kv(self, c):
        c = int(c)
        if c not in self._cache:
            kb, vb = self._w.chunk_kv(c)
            kc, ks, vc, vs = fp8.quantise_chunk(kb, vb)
            kd = fp8.dequantise_chunk(kc, ks, kb.shape[0]).astype(np.float32)
            vd = fp8.dequantise_chunk(vc, vs, vb.shape[0]).astype(np.float32)
            kbits, vbits = cs.f32_to_bf16_bits(kd), cs.f32_to_bf16_bits(vd)
            assert np.array_equal(cs.bf16_bits_to_f64(kbits), kd.astype(np.float64))  # exact: nothing was rounded
            self._cache[c] = (kbits, vbits)
        return self._cache[c]


def check(out_bits, lse, O, L, tag, lse_tol):
    got = cs.bf16_bits_to_f64(out_bits)
    assert np.all(np.isfinite(got)), tag + ": non-finite output"
    err = np.abs(got - O)
    rel = math.sqrt(float((err ** 2).sum()) / max(float((O ** 2).sum()), 1e-300))
    excess = err - (2e-2 + 2.0 ** -8 * np.maximum(np.abs(O) - 2.0, 0.0))
    assert excess.max() <= 0, "%s: max abs %.3e" % (tag, err.max())
    assert err.mean() <= 2e-3, "%s: mean abs %.3e" % (tag, err.mean())
    assert rel <= 1e-2, "%s: rel L2 %.3e" % (tag, rel)
    fin = np.isfinite(L)
    assert np.array_equal(np.isneginf(lse), np.isneginf(L)), tag + ": -inf pattern of LSE"
    e = np.abs(lse[fin] - L[fin]).max() if fin.any() else 0.0
    assert e <= lse_tol, "%s: LSE err %.3e" % (tag, e)
    record("fp8 " + tag, max_abs=err.max(), mean_abs=err.mean(), rel_l2=rel, lse=e)


def run_decode(w, **kw):
    import paper_2602_01519_b200 as comb
    ld = H().load_workload(w, sentinel=BYTE_SENTINEL, kv_dtype=comb.KV_E4M3, **kw)
    out, lse = ld.pool.decode(ld.batch, ld.q, w.scale)
    torch.cuda.synchronize()
    return ld, H().device_to_bits(out), lse.cpu().numpy().astype(np.float64)


# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shuffle", [0, 99])
@pytest.mark.parametrize("Hkv", [2, 8])
def test_fp8_store_page_image_is_bit_exact(shuffle, Hkv):
    import paper_2602_01519_b200 as comb
    lens = [128, 1, 16, 17, 250, 33, 512, 15]
    w = cs.custom("store8", k=8, num_q_heads=Hkv, num_kv_heads=Hkv, head_dim_qk=128, head_dim_v=128, chunk_len=lens,
                  links=[[3, 0, 6], [], [7, 1, 1, 4]], lq=[1, 1, 1])
    ld = H().load_workload(w, shuffle_seed=shuffle, extra_pages=5, sentinel=BYTE_SENTINEL, batch_tokens=300,
                           kv_dtype=comb.KV_E4M3)
    num_pages = w.pool_pages + 5
    model = oracle.PoolModel(num_pages, shuffle)
    pages = {c: model.store(c, int(w.chunk_len[c])) for c in range(w.num_chunks)}
    for c in range(w.num_chunks):
        assert comb.comb_chunk_query(ld.pool.handle, c)[1].tolist() == pages[c]
    k_img, ks_img, v_img, vs_img = fp8.page_image(num_pages, (Hkv, 128, 128),
                                                  {c: w.chunk_kv(c) for c in range(w.num_chunks)}, pages,
                                                  sentinel=BYTE_SENTINEL, scale_sentinel=-7.0)
    k_got = ld.pool.k_arena.view(torch.uint8).cpu().numpy().reshape(k_img.shape)
    v_got = ld.pool.v_arena.view(torch.uint8).cpu().numpy().reshape(v_img.shape)
    assert np.array_equal(ld.pool.k_scale.cpu().numpy().reshape(ks_img.shape), ks_img), "K scales differ"
    assert np.array_equal(ld.pool.v_scale.cpu().numpy().reshape(vs_img.shape), vs_img), "V scales differ"
    assert np.array_equal(k_got, k_img), "K codes differ: %d bytes" % int((k_got != k_img).sum())
    assert np.array_equal(v_got, v_img), "V codes differ"
    ld.pool.close()


FP8_SHAPES = [(32, 8), (16, 16), (4, 2), (16, 1), (16, 2)]   # (Hq, Hkv): G = 4, 1, 2, 16, 8


@pytest.mark.parametrize("heads", FP8_SHAPES)
@pytest.mark.parametrize("peaked", [False, True])
def test_fp8_decode_matches_the_dequantised_oracle(heads, peaked):
    """Ragged chunks (partial and odd page counts: a P V k-step of the kernel spans two pages), shared chunks, an empty
    request, a duplicate link; both statements of the oracle."""
    Hq, Hkv = heads
    lens = [300, 16, 1000, 77, 512, 33, 129, 2000, 48, 5]
    links = [[0, 2, 4], [4, 0], [], [7], [1, 3, 5, 6, 8, 9], [2, 2], [9], [4, 7, 0, 2], [6, 4], [0], [4], [2, 4, 0]]
    w = cs.custom("dec8", k=8, num_q_heads=Hq, num_kv_heads=Hkv, head_dim_qk=128, head_dim_v=128, chunk_len=lens,
                  links=links, lq=[1] * len(links), q_gain=4.0 if peaked else 1.0)
    ld, out, lse = run_decode(w, shuffle_seed=5)
    wd = Dequantised(w)
    O, L = oracle.attention_for(wd)
    O2, L2 = fp8.attention_for(w)
    assert np.abs(O - O2).max() <= 1e-9 and np.abs(L[np.isfinite(L)] - L2[np.isfinite(L2)]).max() <= 1e-9
    check(out, lse, O, L, "decode %s peaked=%s" % (heads, peaked), 2e-4)
    # what the quantisation itself costs against the unquantised chunks (reported, not asserted beyond sanity)
    Ou, _ = oracle.attention_for(w)
    q_err = np.abs(cs.bf16_bits_to_f64(out) - Ou)
    record("fp8 quantisation %s peaked=%s" % (heads, peaked), max_abs=q_err.max(), mean_abs=q_err.mean(),
           rel_l2=math.sqrt(float((q_err ** 2).sum()) / float((Ou ** 2).sum())))
    assert math.sqrt(float((q_err ** 2).sum()) / float((Ou ** 2).sum())) <= 0.2
    ld.pool.close()


def test_fp8_closed_forms_on_gpu():
    """P3 single key: O = the key's V as the pool holds it (dequantised), LSE = its score; P4 equal scores (Q = 0):
    O = mean of the dequantised V, LSE = ln(kv_len); P12 empty link."""
    w = cs.custom("cf8", k=8, num_q_heads=8, num_kv_heads=2, head_dim_qk=128, head_dim_v=128, chunk_len=[1, 512, 40],
                  links=[[0], [1], [], [2, 1]], lq=[1, 1, 1, 1])
    ld, out, lse = run_decode(w)
    wd = Dequantised(w)
    O, L = oracle.attention_for(wd)
    got = cs.bf16_bits_to_f64(out)
    assert np.array_equal(got[0], O[0]), "single key: the dequantised V row, bit for bit"
    assert np.all(got[2] == 0) and np.all(np.isneginf(lse[2]))
    check(out, lse, O, L, "closed forms", 2e-4)
    # Q = 0: every weight equal
    import paper_2602_01519_b200 as comb  # noqa: F401
    q0 = torch.zeros_like(ld.q)
    out0, lse0 = ld.pool.decode(ld.batch, q0, w.scale)
    torch.cuda.synchronize()
    l0 = lse0.cpu().numpy().astype(np.float64)
    assert np.abs(l0[1] - math.log(512)).max() <= 1e-5 and np.abs(l0[3] - math.log(552)).max() <= 1e-5
    vk = cs.bf16_bits_to_f64(wd.chunk_kv(1)[1])                       # [512][Hkv][128]
    mean = vk.mean(axis=0)                                            # [Hkv][128]
    g0 = cs.bf16_bits_to_f64(H().device_to_bits(out0))[1]             # [Hq][128]
    assert np.abs(g0 - np.repeat(mean, 4, axis=0)).max() <= 2.0 ** -8 * np.abs(mean).max() + 1e-3
    ld.pool.close()


def test_fp8_full_size_decode_link_every_element():
    """BASELINE configs[1] on an fp8 pool, in the launch configuration bench.py times, every output element."""
    w = cs.decode_link(seed=0)
    ld, out, lse = run_decode(w, fill="linked", shuffle_seed=2024, keep_host=False)
    O, L = oracle.attention_for(Dequantised(w))
    check(out, lse, O, L, "cfg2 decode (every element)", 2e-4)
    ld.pool.close()


def test_fp8_pool_rejects_what_is_not_built():
    import paper_2602_01519_b200 as comb
    for dq, dv in ((64, 64), (192, 128), (128, 64)):
        with pytest.raises(comb.CombError) as e:
            comb.Pool(2, dq, dv, 16, kv_dtype=comb.KV_E4M3)
        assert e.value.status == comb.COMB_ERR_INVALID


@pytest.mark.parametrize("Hkv", [2, 8])
def test_fp8_project_store_page_image_and_attention(Hkv):
    """(f2) on an fp8 pool: K^cross = H^E W_K, V^cross = H^E W_V (Eq. 5-6) quantised by the GEMM's
    epilogue.  Expected image: fp64 projection -> bf16 RNE (what a bf16 pool would hold) -> the fp8 rule of oracle/fp8.py.
    The GPU accumulates in fp32, so a value within ~1e-6 relative of a bf16 (then e4m3) rounding boundary may land on
    the neighbouring code: at least 99 % of the codes and of the scales identical, every dequantised element within
    one e4m3 step (2^-3 relative, plus the subnormal spacing) of the expected one, tails byte 0, unowned pages
    untouched; then decode over those pages against the oracle over the EXPECTED dequantised chunks."""
    import paper_2602_01519_b200 as comb
    from oracle import layer as ol
    d_model = 320
    lens = [128, 1, 16, 17, 250, 33, 512, 15, 129]
    hs = [cs.hidden_states(3, c, int(t), d_model) for c, t in enumerate(lens)]
    tok = np.zeros(len(lens) + 1, np.int32)
    np.cumsum(lens, out=tok[1:])
    w_kv = cs.projection_weight(3, 0, 0, Hkv * 256, d_model)
    num_pages = int(sum((t + 15) // 16 for t in lens)) + 5
    pool = comb.Pool(Hkv, 128, 128, num_pages, shuffle_seed=31, sentinel=BYTE_SENTINEL, kv_dtype=comb.KV_E4M3)
    ids = list(range(len(lens)))
    hd = H().bits_to_device(np.concatenate(hs, 0), "cuda")
    wd = H().bits_to_device(w_kv, "cuda")
    pool.project_store_chunks(ids[:1], tok[:2], hd[:tok[1]], wd)
    pool.project_store_chunks(ids[1:], tok[1:] - tok[1], hd[tok[1]:], wd)
    torch.cuda.synchronize()
    model = oracle.PoolModel(num_pages, 31)
    wk64 = ol.bf16_to_f64(w_kv)
    chunks, pages = {}, {}
    for c in ids:
        pages[c] = model.store(c, lens[c])
        K, V = ol.project_kv(ol.bf16_to_f64(hs[c]), wk64, Hkv, 128, 128)
        chunks[c] = (ol.f64_to_bf16_bits(K), ol.f64_to_bf16_bits(V))
        assert comb.comb_chunk_query(pool.handle, c)[1].tolist() == pages[c]
    k_img, ks_img, v_img, vs_img = fp8.page_image(num_pages, (Hkv, 128, 128), chunks, pages, sentinel=BYTE_SENTINEL,
                                                  scale_sentinel=-7.0)
    owned = np.zeros(num_pages, bool)
    for c in ids:
        owned[pages[c]] = True
    for name, arena, sc, img, simg in (("K", pool.k_arena, pool.k_scale, k_img, ks_img),
                                       ("V", pool.v_arena, pool.v_scale, v_img, vs_img)):
        got = arena.view(torch.uint8).cpu().numpy().reshape(img.shape)
        gsc = sc.cpu().numpy().reshape(simg.shape)
        assert np.all(got[~owned] == BYTE_SENTINEL) and np.all(gsc[~owned] == -7.0), name + ": an unowned page was touched"
        assert (gsc[owned] == simg[owned]).mean() >= 0.99, name + ": scales"
        assert (got[owned] == img[owned]).mean() >= 0.99, name + ": codes"
        gv = fp8.e4m3_decode(got[owned]) * gsc[owned].astype(np.float64)[:, :, None, None]
        wv = fp8.e4m3_decode(img[owned]) * simg[owned].astype(np.float64)[:, :, None, None]
        step = np.maximum(np.abs(wv) * 2.0 ** -3, simg[owned].astype(np.float64)[:, :, None, None] * 2.0 ** -9)
        assert np.all(np.abs(gv - wv) <= step * 1.001), name + ": not a neighbouring code of the expected value"
        for c in ids:
            n = lens[c] - 16 * (len(pages[c]) - 1)
            assert np.all(got[pages[c][-1], :, n:, :] == 0), name + ": tail slots are not byte 0"
    # attend over the projected pages
    links = [[6, 0, 4], [8, 1], [2, 3, 5, 7]]
    w = cs.custom("pj8", k=8, num_q_heads=4 * Hkv, num_kv_heads=Hkv, head_dim_qk=128, head_dim_v=128, chunk_len=lens,
                  links=links, lq=[1, 1, 1])

    class Projected:
        def __getattr__(self, name):
            return getattr(w, name)

        def chunk_kv(self, c):
            kb, vb = chunks[int(c)]
            kc, ks, vc, vs = fp8.quantise_chunk(kb, vb)
            return (cs.f32_to_bf16_bits(fp8.dequantise_chunk(kc, ks, kb.shape[0]).astype(np.float32)),
                    cs.f32_to_bf16_bits(fp8.dequantise_chunk(vc, vs, vb.shape[0]).astype(np.float32)))
    lb = pool.link(links)
    out, lse = pool.decode(lb, H().bits_to_device(w.all_q(), "cuda"), w.scale)
    torch.cuda.synchronize()
    O, L = oracle.attention_for(Projected())
    check(H().device_to_bits(out), lse.cpu().numpy().astype(np.float64), O, L, "decode over projected fp8 pages", 2e-3)
    pool.close()


@pytest.mark.parametrize("heads", [(32, 8), (16, 16), (8, 1)])
def test_fp8_prefill_over_dequantised_staging(heads):
    """comb_cross_attn_prefill on an fp8 pool: the batch's distinct pages are dequantised (exactly) into bf16 staging
    in the workspace and the bf16 kernel attends over it through the link's compact page table.  Ragged chunks, shared
    chunks, an empty request, a duplicate link, query blocks of 1 .. 300 tokens (single-tile, two-tile and KV-range
    plans); and row i of the prefill equals a decode of that row on the same pool (P11)."""
    import paper_2602_01519_b200 as comb
    Hq, Hkv = heads
    lens = [300, 16, 1000, 77, 512, 33, 129, 2000]
    links = [[0, 2, 4], [4, 0], [], [7], [1, 3, 5, 6], [2, 2], [4, 7, 0, 2]]
    lq = [40, 1, 5, 300, 17, 130, 64]
    w = cs.custom("pre8", k=8, num_q_heads=Hq, num_kv_heads=Hkv, head_dim_qk=128, head_dim_v=128, chunk_len=lens,
                  links=links, lq=lq)
    ld = H().load_workload(w, sentinel=BYTE_SENTINEL, kv_dtype=comb.KV_E4M3, shuffle_seed=7)
    out, lse = ld.pool.prefill(ld.batch, ld.q, ld.q_indptr, w.scale)
    torch.cuda.synchronize()
    O, L = oracle.attention_for(Dequantised(w))
    check(H().device_to_bits(out), lse.cpu().numpy().astype(np.float64), O, L, "prefill %s" % (heads,), 2e-4)
    # the table the staging is read through: entry i of page_ids as an index into the distinct-page list
    t = ld.batch.tables()
    L_ = ld.batch.link
    off = L_.page_ids_compact - ld.batch.buf.data_ptr()
    compact = ld.batch.buf[off:off + 4 * int(L_.total_pages)].view(torch.int32).cpu().numpy()
    assert np.array_equal(t["cas_page_ids"][compact], t["page_ids"])
    # P11: the last row of request 3 as a decode over the same link list
    r = 3
    row = int(w.q_indptr[r + 1]) - 1
    wd1 = cs.custom("pre8d", k=8, num_q_heads=Hq, num_kv_heads=Hkv, head_dim_qk=128, head_dim_v=128, chunk_len=lens,
                    links=[links[r]], lq=[1])
    lb = ld.pool.link([list(map(int, links[r]))])
    o1, l1 = ld.pool.decode(lb, ld.q[row:row + 1].contiguous(), wd1.scale)
    torch.cuda.synchronize()
    a = cs.bf16_bits_to_f64(H().device_to_bits(out))[row]
    b = cs.bf16_bits_to_f64(H().device_to_bits(o1))[0]
    assert np.abs(a - b).max() <= 2.0 ** -7 * np.abs(a).max() + 1.5e-3
    assert abs(float(lse[row].max()) - float(l1.max())) <= 2e-4
    ld.pool.close()


def test_fp8_full_size_rag_prefill_lq32_whole_requests():
    """BASELINE configs[2] at lq = 32 (the paper's regime) on an fp8 pool, in bench.py's launch configuration: four
    whole requests, every element."""
    import paper_2602_01519_b200 as comb
    w = cs.rag_prefill(seed=0, lq=32)
    ld = H().load_workload(w, fill="linked", shuffle_seed=2024, keep_host=False, kv_dtype=comb.KV_E4M3)
    out, lse = ld.pool.prefill(ld.batch, ld.q, ld.q_indptr, w.scale)
    torch.cuda.synchronize()
    got_o = H().device_to_bits(out)
    got_l = lse.cpu().numpy().astype(np.float64)
    wd = Dequantised(w)
    for r in (0, 5, 17, w.num_requests - 1):
        O, L = oracle.attention_for(wd, [r])
        a, b = int(w.q_indptr[r]), int(w.q_indptr[r + 1])
        check(got_o[a:b], got_l[a:b], O, L, "rag lq32 prefill, request %d" % r, 2e-4)
    ld.pool.close()


def test_fp8_layers_and_the_sublayer():
    """L = 3 layers over one page-id space on an fp8 pool (codes AND scale tables are per layer), each layer's prefill
    and decode against the oracle over that layer's dequantised chunks; then comb_cross_layer_forward (Eq. 4, 7-8,
    PAPER.md:117) on layer 1 against the fp64 sub-layer oracle fed the dequantised K/V."""
    from dataclasses import replace
    import paper_2602_01519_b200 as comb
    from oracle import layer as ol
    base = cs.custom("lay8", k=8, num_q_heads=8, num_kv_heads=2, head_dim_qk=128, head_dim_v=128,
                     chunk_len=[130, 17, 512, 64], links=[[2, 0, 1], [3, 1], [], [1, 2]], lq=[40, 7, 3, 9])
    ws = [replace(base, seed=200 + l) for l in range(3)]
    pool = comb.Pool(2, 128, 128, base.pool_pages, num_layers=3, shuffle_seed=21, sentinel=BYTE_SENTINEL,
                     kv_dtype=comb.KV_E4M3)
    ids = list(range(base.num_chunks))
    tok = np.zeros(base.num_chunks + 1, np.int32)
    np.cumsum(base.chunk_len, out=tok[1:])
    for l in (2, 0, 1):
        kv = [ws[l].chunk_kv(c) for c in ids]
        pool.store_chunks(ids, tok, H().bits_to_device(np.concatenate([k for k, _ in kv]), "cuda"),
                          H().bits_to_device(np.concatenate([v for _, v in kv]), "cuda"), layer=l)
    batch = pool.link([list(map(int, x)) for x in base.links])
    for l in range(3):
        q = H().bits_to_device(ws[l].all_q(), "cuda")
        out, lse = pool.prefill(batch, q, base.q_indptr, base.scale, layer=l)
        torch.cuda.synchronize()
        check(H().device_to_bits(out), lse.cpu().numpy().astype(np.float64), *oracle.attention_for(Dequantised(ws[l])),
              "prefill layer %d" % l, 2e-4)
        wd = ws[l].decode_phase()
        outd, lsed = pool.decode(batch, H().bits_to_device(wd.all_q(), "cuda"), wd.scale, layer=l)
        torch.cuda.synchronize()
        check(H().device_to_bits(outd), lsed.cpu().numpy().astype(np.float64), *oracle.attention_for(Dequantised(wd)),
              "decode layer %d" % l, 2e-4)
    # the sub-layer on layer 1, prefill and decode rows
    d_model, Hq, Hkv, D = 256, 8, 2, 128
    wq = cs.projection_weight(5, 1, 1, Hq * D, d_model)
    wo = cs.projection_weight(5, 2, 1, d_model, Hq * D, gain=0.1)
    wl = Dequantised(ws[1])
    kd = [cs.bf16_bits_to_f64(wl.chunk_kv(c)[0]) for c in ids]
    vd = [cs.bf16_bits_to_f64(wl.chunk_kv(c)[1]) for c in ids]
    for q_indptr, rows in ((base.q_indptr, int(base.total_q)), (None, base.num_requests)):
        x = cs.hidden_states(9, 0 if q_indptr is not None else 1, rows, d_model)
        xd = H().bits_to_device(x, "cuda")
        y = pool.layer_forward(batch, xd, q_indptr, H().bits_to_device(wq, "cuda"), H().bits_to_device(wo, "cuda"),
                               base.scale, layer=1)
        torch.cuda.synchronize()
        ind = q_indptr if q_indptr is not None else np.arange(base.num_requests + 1, dtype=np.int32)
        want = ol.cross_layer(cs.bf16_bits_to_f64(x), ind, cs.bf16_bits_to_f64(wq), cs.bf16_bits_to_f64(wo), Hq, kd, vd,
                              [list(map(int, l)) for l in base.links], base.scale)
        got = cs.bf16_bits_to_f64(H().device_to_bits(y))
        rel = math.sqrt(float(((got - want) ** 2).sum()) / float((want ** 2).sum()))
        assert rel <= 1e-2, "sub-layer on an fp8 pool: rel L2 %.3e" % rel
        assert np.abs(got - want).max() <= 2.0 ** -6 * np.abs(want).max()
    pool.close()
