"""GPU parity tests (run with -m gpu on a B200) of the steps either side of the link-stage attention, through the C
ABI, against oracle/layer.py (fp64, nothing rounded between steps):

  (f2) comb_project_store_chunks: K^cross = H^E W_K, V^cross = H^E W_V (Eq. 5-6) written straight into
       pages by the GEMM's epilogue;
  (f3) comb_cross_layer_forward: x + Attn(x W_Q ; K, V) W_O (Eq. 4, 7-8), one layer and the L = 8 stack.

Tolerances (DESIGN.md §2 "Tolerances"): a stored K/V element is the fp32-accumulated dot product rounded to bf16, the
oracle's is the fp64 dot product rounded to bf16: they agree bit for bit unless the exact value lies within the fp32
accumulation error (~1e-6 relative) of a bf16 rounding boundary, in which case they are neighbours.  So: every element
within ONE bf16 ulp of RNE(exact), at least 99 % identical; tail slots and unowned pages bit-exact.  The sub-layer's
output rounds Q, the attention output and x to bf16 at each hand-over (unit roundoff 2^-8 each): relative L2 <= 1e-2
per layer and <= 2e-2 after the 8-layer stack, max abs <= 2^-6 max|x_out| (four bf16 roundings in sequence)."""
import json
import math
import os

import numpy as np
import pytest

import comb_synth as cs
import oracle
from oracle import layer as ol

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
SENTINEL = 0x7FC0


ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def H():
    from paper_2602_01519_b200 import harness
    return harness


def record(tag, **kw):
    """Measured worst cases, appended to gpurun_out/parity_measured.jsonl (evidence for DESIGN.md §2; not read back)."""
    try:
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, "gpurun_out", "parity_measured.jsonl"), "a") as f:
            f.write(json.dumps(dict(tag=tag, **{k: float(v) for k, v in kw.items()})) + "\n")
    except OSError:
        pass


def bf16_ulp(x):
    """Spacing of bf16 numbers around |x| (8 significant bits)."""
    ax = np.maximum(np.abs(x), 2.0 ** -126)
    return 2.0 ** (np.floor(np.log2(ax)) - 7)


def make_chunks(seed, lens, d_model):
    hs = [cs.hidden_states(seed, c, int(t), d_model) for c, t in enumerate(lens)]
    tok = np.zeros(len(lens) + 1, np.int32)
    np.cumsum(lens, out=tok[1:])
    return hs, tok


# ------------------------------------------------------------------------------------------------
# (f2) projection fused into the paged store
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shuffle", [0, 31])
@pytest.mark.parametrize("dims", [(2, 64, 64, 256), (8, 128, 128, 512), (4, 192, 128, 320), (2, 128, 64, 72)])
def test_project_store_page_image(shuffle, dims):
    import paper_2602_01519_b200 as comb
    Hkv, Dqk, Dv, d_model = dims
    lens = [128, 1, 16, 17, 250, 33, 512, 15, 129]
    hs, tok = make_chunks(3, lens, d_model)
    w_kv = cs.projection_weight(3, 0, 0, Hkv * (Dqk + Dv), d_model)
    num_pages = int(sum((t + 15) // 16 for t in lens)) + 5
    pool = comb.Pool(Hkv, Dqk, Dv, num_pages, shuffle_seed=shuffle, sentinel=SENTINEL)
    ids = list(range(len(lens)))
    # two batches (a single-chunk one and the rest), as a compile stage feeding chunks as they arrive would
    hd = H().bits_to_device(np.concatenate(hs, 0), "cuda")
    wd = H().bits_to_device(w_kv, "cuda")
    l0 = pool.launches
    pool.project_store_chunks(ids[:1], tok[:2], hd[:tok[1]], wd)
    pool.project_store_chunks(ids[1:], tok[1:] - tok[1], hd[tok[1]:], wd)
    torch.cuda.synchronize()
    assert pool.launches - l0 == 2, "one GEMM launch per batch, no separate store kernel"
    # expected image: fp64 projection -> bf16 RNE -> the oracle's page image (independent table model)
    model = oracle.PoolModel(num_pages, shuffle)
    wk64 = ol.bf16_to_f64(w_kv)
    stored_k, stored_v, exact_k, exact_v = [], [], [], []
    for c in ids:
        pages = model.store(c, lens[c])
        K, V = ol.project_kv(ol.bf16_to_f64(hs[c]), wk64, Hkv, Dqk, Dv)
        stored_k.append((ol.f64_to_bf16_bits(K), pages))
        stored_v.append((ol.f64_to_bf16_bits(V), pages))
        exact_k.append((K, pages))
        exact_v.append((V, pages))
        nt, got_pages = comb.comb_chunk_query(pool.handle, c)
        assert nt == lens[c] and got_pages.tolist() == pages
    for name, arena, D, stored, exact in (("K", pool.k_arena, Dqk, stored_k, exact_k),
                                          ("V", pool.v_arena, Dv, stored_v, exact_v)):
        img = oracle.page_image(num_pages, Hkv, D, stored, SENTINEL)
        got = arena.cpu().numpy().view(np.uint16).reshape(img.shape)
        owned = np.zeros(num_pages, bool)
        same = total = 0
        for (bits, pages), (x64, _) in zip(stored, exact):
            T = bits.shape[0]
            for i, p in enumerate(pages):
                owned[p] = True
                n = min(16, T - 16 * i)
                assert np.all(got[p, :, n:, :] == 0), "%s: tail slots of page %d are not zero bits" % (name, p)
                g = ol.bf16_to_f64(got[p, :, :n, :])
                want = np.transpose(x64[16 * i:16 * i + n], (1, 0, 2))
                assert np.all(np.abs(g - want) <= bf16_ulp(want) * 0.51 + 1e-5), name + ": not a bf16 neighbour of the exact value"
                same += int((got[p, :, :n, :] == img[p, :, :n, :]).sum())
                total += g.size
        assert same >= 0.99 * total, "%s: only %.4f of the elements equal RNE(fp64)" % (name, same / total)
        record("f2 page image %s %s" % (name, dims), identical_fraction=same / total)
        assert np.all(got[~owned] == SENTINEL), name + ": an unowned page was touched"
    pool.close()


def test_project_store_then_attend():
    """Compile (f2) -> link -> prefill and both decode paths over the projected pool, against the oracle fed with
    RNE(fp64 projection): the whole compile/link statement of the problem end to end."""
    import paper_2602_01519_b200 as comb
    Hq, Hkv, D, d_model = 8, 2, 128, 256
    lens = [300, 77, 512, 16, 129]
    links = [[2, 0, 4], [1], [], [3, 2, 1, 0]]
    lq = [33, 5, 2, 64]
    hs, tok = make_chunks(7, lens, d_model)
    w_kv = cs.projection_weight(7, 0, 0, Hkv * 2 * D, d_model)
    pool = comb.Pool(Hkv, D, D, int(sum((t + 15) // 16 for t in lens)), shuffle_seed=9, sentinel=SENTINEL)
    pool.project_store_chunks(list(range(5)), tok, H().bits_to_device(np.concatenate(hs, 0), "cuda"),
                              H().bits_to_device(w_kv, "cuda"))
    lb = pool.link(links)
    ks, vs = [], []
    for c in range(5):
        K, V = ol.project_kv(ol.bf16_to_f64(hs[c]), ol.bf16_to_f64(w_kv), Hkv, D, D)
        ks.append(ol.f64_to_bf16_bits(K))
        vs.append(ol.f64_to_bf16_bits(V))
    qs = [cs.normal_bf16(7, 3, r, (n, Hq, D)) for r, n in enumerate(lq)]
    q_indptr = np.zeros(5, np.int32)
    np.cumsum(lq, out=q_indptr[1:])
    ci = np.zeros(5, np.int32)
    np.cumsum([len(l) for l in links], out=ci[1:])
    sel = np.array([c for l in links for c in l], np.int32)
    scale = 1.0 / math.sqrt(D)
    O, L = oracle.attention(np.concatenate(qs, 0), q_indptr, ks, vs, ci, sel, scale)
    out, lse = pool.prefill(lb, H().bits_to_device(np.concatenate(qs, 0), "cuda"), q_indptr, scale)
    torch.cuda.synchronize()
    got = cs.bf16_bits_to_f64(H().device_to_bits(out))
    err = np.abs(got - O)
    rel = math.sqrt(float((err ** 2).sum()) / float((O ** 2).sum()))
    assert err.max() <= 2e-2 and err.mean() <= 2e-3 and rel <= 1e-2, (err.max(), err.mean(), rel)
    fin = np.isfinite(L)
    assert np.abs(lse.cpu().numpy()[fin] - L[fin]).max() <= 2e-4
    q1 = np.stack([q[0] for q in qs], 0)
    O1, L1 = oracle.attention(q1, np.arange(5, dtype=np.int32), ks, vs, ci, sel, scale)
    for path in (comb.DECODE_PER_REQUEST, comb.DECODE_CHUNK_MAJOR):
        pool.set_decode_path(path)
        od, ld = pool.decode(lb, H().bits_to_device(q1, "cuda"), scale)
        torch.cuda.synchronize()
        e = np.abs(cs.bf16_bits_to_f64(H().device_to_bits(od)) - O1)
        assert e.max() <= 2e-2 and e.mean() <= 2e-3, (path, e.max(), e.mean())
        assert np.abs(ld.cpu().numpy()[np.isfinite(L1)] - L1[np.isfinite(L1)]).max() <= 2e-4
    pool.close()


def test_project_store_errors_leave_the_pool_unchanged():
    import paper_2602_01519_b200 as comb
    pool = comb.Pool(2, 64, 64, 4)
    h = torch.zeros((40, 64), dtype=torch.bfloat16, device="cuda")
    w = torch.zeros((256, 64), dtype=torch.bfloat16, device="cuda")
    pool.project_store_chunks([5], [0, 40], h, w)                       # 3 pages
    with pytest.raises(comb.CombError) as e:
        pool.project_store_chunks([6], [0, 40], h, w)                   # needs 3, 1 free
    assert e.value.status == comb.COMB_ERR_NO_SPACE and pool.free_pages == 1
    with pytest.raises(comb.CombError) as e:
        pool.project_store_chunks([5], [0, 39], h[:39], w)              # same id, other length
    assert e.value.status == comb.COMB_ERR_EXISTS
    with pytest.raises(comb.CombError) as e:
        pool.project_store_chunks([7, 7], [0, 8, 16], h[:16], w)        # the same id twice in one batch
    assert e.value.status == comb.COMB_ERR_INVALID and pool.free_pages == 1
    with pytest.raises(comb.CombError) as e:
        comb.comb_project_store_chunks(pool.handle, 0, [8], [0, 8], h[:8], 60, w)   # d_model % 8 != 0
    assert e.value.status == comb.COMB_ERR_INVALID and pool.free_pages == 1
    pool.close()


# ------------------------------------------------------------------------------------------------
# the projection GEMM alone: ragged M, N and K tails, residual epilogue
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [(1, 32, 8), (129, 256, 64), (300, 288, 200), (1000, 1024, 520), (257, 4096, 1024)])
def test_gemm_rowmajor_against_fp64(shape):
    import paper_2602_01519_b200 as comb
    M, N, K = shape
    a = cs.normal_bf16(1, 20, M, (M, K))
    w = cs.normal_bf16(1, 21, N, (N, K), 1.0 / math.sqrt(K))
    r = cs.normal_bf16(1, 22, M, (M, N))
    pool = comb.Pool(2, 64, 64, 4)
    ad, wd, rd = (H().bits_to_device(x, "cuda") for x in (a, w, r))
    exact = ol.bf16_to_f64(a) @ ol.bf16_to_f64(w).T
    for res, want in ((None, exact), (rd, exact + ol.bf16_to_f64(r))):
        c = torch.full((M, N), float("nan"), dtype=torch.bfloat16, device="cuda")
        comb.comb_gemm_bf16(pool.handle, ad, wd, c, M, N, K, residual=res)
        torch.cuda.synchronize()
        got = cs.bf16_bits_to_f64(H().device_to_bits(c))
        assert np.all(np.isfinite(got))
        assert np.all(np.abs(got - want) <= 0.51 * bf16_ulp(want) + 2e-6 * math.sqrt(K)), np.abs(got - want).max()
        same = (H().device_to_bits(c) == ol.f64_to_bf16_bits(want)).mean()
        assert same >= 0.99, same
    pool.close()


# ------------------------------------------------------------------------------------------------
# (f3) the cross-attention sub-layer, one layer and the stack of 8
# ------------------------------------------------------------------------------------------------
def build_layer_case(seed, Hq, Hkv, Dqk, Dv, d_model, lens, links, lq, L=1, o_gain=1.0):
    import paper_2602_01519_b200 as comb
    pool = comb.Pool(Hkv, Dqk, Dv, int(sum((t + 15) // 16 for t in lens)), num_layers=L, shuffle_seed=seed + 1,
                     sentinel=SENTINEL)
    tok = np.zeros(len(lens) + 1, np.int32)
    np.cumsum(lens, out=tok[1:])
    ids = list(range(len(lens)))
    ck, cv, wq, wo = [], [], [], []
    for l in range(L):
        # K/V of layer l straight as pool content (bf16 N(0,1), like BASELINE's configs)
        kb = [cs.normal_bf16(seed, 4, 100 * l + c, (t, Hkv, Dqk)) for c, t in enumerate(lens)]
        vb = [cs.normal_bf16(seed, 5, 100 * l + c, (t, Hkv, Dv)) for c, t in enumerate(lens)]
        pool.store_chunks(ids, tok, H().bits_to_device(np.concatenate(kb, 0), "cuda"),
                          H().bits_to_device(np.concatenate(vb, 0), "cuda"), layer=l)
        ck.append([ol.bf16_to_f64(k) for k in kb])
        cv.append([ol.bf16_to_f64(v) for v in vb])
        wq.append(cs.projection_weight(seed, 1, l, Hq * Dqk, d_model))
        wo.append(cs.projection_weight(seed, 2, l, d_model, Hq * Dv, o_gain))
    lb = pool.link(links)
    q_indptr = np.zeros(len(lq) + 1, np.int32)
    np.cumsum(lq, out=q_indptr[1:])
    x = np.concatenate([cs.decoder_rows(seed, r, n, d_model) for r, n in enumerate(lq)], 0)
    return pool, lb, q_indptr, x, wq, wo, ck, cv


def check_rows(got_bits, want, rel_tol, tag):
    got = cs.bf16_bits_to_f64(got_bits)
    assert np.all(np.isfinite(got)), tag
    err = np.abs(got - want)
    rel = math.sqrt(float((err ** 2).sum()) / float((want ** 2).sum()))
    assert rel <= rel_tol, "%s: rel L2 %.3e" % (tag, rel)
    assert err.max() <= 2.0 ** -6 * np.abs(want).max(), "%s: max abs %.3e" % (tag, err.max())
    record(tag, rel_l2=rel, max_abs=err.max(), max_want=np.abs(want).max())
    return rel, err.max()


@pytest.mark.parametrize("shape", [(8, 2, 64, 64, 256), (32, 8, 128, 128, 512), (16, 16, 192, 128, 384)])
def test_cross_layer_prefill_and_decode(shape):
    Hq, Hkv, Dqk, Dv, d_model = shape
    lens = [130, 17, 300, 64, 1]
    links = [[2, 0, 1], [3, 1], [], [4], [0, 2, 3, 1]]
    lq = [40, 7, 3, 2, 130]
    scale = 1.0 / math.sqrt(Dqk)
    pool, lb, q_indptr, x, wq, wo, ck, cv = build_layer_case(11, Hq, Hkv, Dqk, Dv, d_model, lens, links, lq)
    want = ol.cross_layer(ol.bf16_to_f64(x), q_indptr, ol.bf16_to_f64(wq[0]), ol.bf16_to_f64(wo[0]), Hq, ck[0], cv[0],
                          links, scale)
    xd = H().bits_to_device(x, "cuda")
    wqd, wod = H().bits_to_device(wq[0], "cuda"), H().bits_to_device(wo[0], "cuda")
    l0 = pool.launches
    y = pool.layer_forward(lb, xd, q_indptr, wqd, wod, scale)
    torch.cuda.synchronize()
    assert pool.launches - l0 in (3, 4), "GEMM + attention (+ range merge) + GEMM"
    check_rows(H().device_to_bits(y), want, 1e-2, "layer prefill %s" % (shape,))
    # a request that links nothing keeps its rows bit for bit (the sub-layer only adds)
    r2 = slice(int(q_indptr[2]), int(q_indptr[3]))
    assert np.array_equal(H().device_to_bits(y)[r2], x[r2])
    # decode: one row per request, both decode paths
    import paper_2602_01519_b200 as comb
    x1 = np.stack([x[q_indptr[r]] for r in range(len(lq))], 0)
    want1 = ol.cross_layer(ol.bf16_to_f64(x1), np.arange(len(lq) + 1, dtype=np.int32), ol.bf16_to_f64(wq[0]),
                           ol.bf16_to_f64(wo[0]), Hq, ck[0], cv[0], links, scale)
    for path in (comb.DECODE_PER_REQUEST, comb.DECODE_CHUNK_MAJOR):
        pool.set_decode_path(path)
        y1 = pool.layer_forward(lb, H().bits_to_device(x1, "cuda"), None, wqd, wod, scale)
        torch.cuda.synchronize()
        check_rows(H().device_to_bits(y1), want1, 1e-2, "layer decode %s path %d" % (shape, path))
    # W_O = 0: the output IS the input, bit for bit
    y0 = pool.layer_forward(lb, xd, q_indptr, wqd, torch.zeros_like(wod), scale)
    torch.cuda.synchronize()
    assert np.array_equal(H().device_to_bits(y0), x)
    pool.close()


def test_cross_stack_of_eight_layers():
    """The paper's Llama instance has 8 cross layers sharing the decoder rows: 8 calls over ONE link
    (page ids are shared by all layers), layer l reading its own arena slice and weights; prefill and decode."""
    Hq, Hkv, D, d_model, L = 32, 8, 128, 512, 8
    lens = [200, 31, 512, 90]
    links = [[2, 0], [1, 3, 2], [3]]
    lq = [70, 9, 33]
    scale = 1.0 / math.sqrt(D)
    # output-projection gain 0.5: the residual stream grows by ~ sqrt(1 + 0.25 * attention variance) per layer
    pool, lb, q_indptr, x, wq, wo, ck, cv = build_layer_case(5, Hq, Hkv, D, D, d_model, lens, links, lq, L=L, o_gain=0.5)
    states = ol.cross_stack(ol.bf16_to_f64(x), q_indptr, [ol.bf16_to_f64(w) for w in wq], [ol.bf16_to_f64(w) for w in wo],
                            Hq, ck, cv, links, scale)
    wqd = [H().bits_to_device(w, "cuda") for w in wq]
    wod = [H().bits_to_device(w, "cuda") for w in wo]
    cur = H().bits_to_device(x, "cuda")
    rels = []
    for l in range(L):
        cur = pool.layer_forward(lb, cur, q_indptr, wqd[l], wod[l], scale, layer=l)
        torch.cuda.synchronize()
        rel, _ = check_rows(H().device_to_bits(cur), states[l], 2e-2, "stack prefill after layer %d" % l)
        rels.append(rel)
    assert rels[0] <= 1e-2
    # decode rows through the same 8 layers
    x1 = np.stack([x[q_indptr[r]] for r in range(len(lq))], 0)
    st1 = ol.cross_stack(ol.bf16_to_f64(x1), np.arange(len(lq) + 1, dtype=np.int32), [ol.bf16_to_f64(w) for w in wq],
                         [ol.bf16_to_f64(w) for w in wo], Hq, ck, cv, links, scale)
    cur = H().bits_to_device(x1, "cuda")
    for l in range(L):
        cur = pool.layer_forward(lb, cur, None, wqd[l], wod[l], scale, layer=l)
    torch.cuda.synchronize()
    check_rows(H().device_to_bits(cur), st1[-1], 2e-2, "stack decode after 8 layers")
    pool.close()
