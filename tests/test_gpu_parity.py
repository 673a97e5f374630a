"""GPU parity tests (run with -m gpu on a B200): every step of the hot path, called through the C ABI
(paper_2602_01519_b200.api -> libcomb.so), against the fp64 oracle on the same seeded inputs.

Bars (BASELINE.json north_star): block tables and page contents bit-exact; attention outputs
max abs <= 2e-2 and mean abs <= 2e-3; additionally relative L2 <= 1e-2 and |LSE error| <= 2e-3 so the claim
means something on the small outputs N(0,1) inputs give."""
import math

import numpy as np
import pytest

import comb_synth as cs
import oracle

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
SENTINEL = 0x7FC0  # bf16 NaN: any unmasked read of an unowned slot poisons the output (pin P15)


def H():
    from paper_2602_01519_b200 import harness
    return harness


def check_attention(out_bits, lse, O, L, tag=""):
    got = cs.bf16_bits_to_f64(out_bits)
    assert np.all(np.isfinite(got)), tag + ": non-finite output"
    err = np.abs(got - O)
    rel = math.sqrt(float((err ** 2).sum()) / max(float((O ** 2).sum()), 1e-300))
    assert err.max() <= 2e-2, "%s: max abs %.3e" % (tag, err.max())
    assert err.mean() <= 2e-3, "%s: mean abs %.3e" % (tag, err.mean())
    assert rel <= 1e-2, "%s: rel L2 %.3e" % (tag, rel)
    if lse is not None:
        fin = np.isfinite(L)
        assert np.array_equal(np.isneginf(lse), np.isneginf(L)), tag + ": -inf pattern of LSE"
        if fin.any():
            e = np.abs(lse[fin] - L[fin]).max()
            assert e <= 2e-3, "%s: LSE err %.3e" % (tag, e)
    return err.max(), err.mean(), rel


def close_in_ulps(a, b, tag=""):
    """Two GPU results for the same mathematical value (other tile partition, other kernel). They differ by the
    bf16 rounding of the output (<= 2^-8 relative each) and of the P weights fed to the PV contraction (each weight
    2^-9 relative, so about 2^-9 * sum_j p_j |v_j| / l ~ 2e-3 absolute for N(0,1) values), and by fp32 reassociation."""
    d = np.abs(a - b)
    assert np.all(d <= 2.0 ** -7 * np.abs(a) + 2.5e-3), "%s: worst excess %.3e" % (
        tag, (d - 2.0 ** -7 * np.abs(a)).max())
    assert d.mean() <= 3e-4, "%s: mean |a-b| = %.3e" % (tag, d.mean())


def run_prefill(w, **kw):
    ld = H().load_workload(w, sentinel=SENTINEL, **kw)
    out, lse = ld.pool.prefill(ld.batch, ld.q, ld.q_indptr, w.scale)
    torch.cuda.synchronize()
    return ld, H().device_to_bits(out), lse.cpu().numpy().astype(np.float64)


def run_decode(w, **kw):
    ld = H().load_workload(w, sentinel=SENTINEL, **kw)
    out, lse = ld.pool.decode(ld.batch, ld.q, w.scale)
    torch.cuda.synchronize()
    return ld, H().device_to_bits(out), lse.cpu().numpy().astype(np.float64)


# ------------------------------------------------------------------------------------------------
# (a2) store: page image bit-exact (O2, pin P13), (a3) link: tables bit-exact (O3), no KV copy (P14)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shuffle", [0, 99])
@pytest.mark.parametrize("dims", [(2, 64, 64), (8, 128, 128), (4, 192, 128)])
def test_store_page_image_and_link_tables(shuffle, dims):
    Hkv, Dqk, Dv = dims
    lens = [128, 1, 16, 17, 250, 33, 512, 15]
    w = cs.custom("store", num_q_heads=Hkv, num_kv_heads=Hkv, head_dim_qk=Dqk, head_dim_v=Dv, chunk_len=lens,
                  links=[[3, 0, 6], [], [7, 1, 1, 4]], lq=[1, 1, 1])
    ld = H().load_workload(w, shuffle_seed=shuffle, extra_pages=5, sentinel=SENTINEL, batch_tokens=300)
    assert ld.num_store_calls > 1  # single- and multi-chunk batches both occur
    num_pages = w.pool_pages + 5
    model = oracle.PoolModel(num_pages, shuffle)
    stored_k, stored_v = [], []
    for c in range(w.num_chunks):
        pages = model.store(c, int(w.chunk_len[c]))
        k, v = w.chunk_kv(c)
        stored_k.append((k, pages))
        stored_v.append((v, pages))
        nt, got_pages = __import__("paper_2602_01519_b200").comb_chunk_query(ld.pool.handle, c)
        assert nt == int(w.chunk_len[c]) and got_pages.tolist() == pages
    k_img = oracle.page_image(num_pages, Hkv, Dqk, stored_k, SENTINEL)
    v_img = oracle.page_image(num_pages, Hkv, Dv, stored_v, SENTINEL)
    k_before = ld.pool.k_arena.cpu().numpy().view(np.uint16).reshape(k_img.shape)
    v_before = ld.pool.v_arena.cpu().numpy().view(np.uint16).reshape(v_img.shape)
    assert np.array_equal(k_before, k_img), "K page image differs (tail zero-fill / sentinel / scatter)"
    assert np.array_equal(v_before, v_img), "V page image differs"
    # link tables, bit-exact against the independent model; order of the caller preserved
    exp = model.link([list(map(int, l)) for l in w.links])
    got = ld.batch.tables()
    for key in ("page_indptr", "page_ids", "page_ntok", "kv_len"):
        assert np.array_equal(got[key], exp[key]), key
    # policy-independent cross-check: page lists disjoint, in range, right length
    allp = np.concatenate([np.array(p) for _, p in stored_k])
    assert len(np.unique(allp)) == len(allp) and allp.min() >= 0 and allp.max() < num_pages
    # P14: link moved no K/V byte
    again = ld.pool.link([list(map(int, l)) for l in w.links])
    torch.cuda.synchronize()
    assert np.array_equal(ld.pool.k_arena.cpu().numpy().view(np.uint16).reshape(k_img.shape), k_before)
    assert np.array_equal(ld.pool.v_arena.cpu().numpy().view(np.uint16).reshape(v_img.shape), v_before)
    assert again.link.total_pages == ld.batch.link.total_pages


def test_store_errors_on_device_pool():
    import paper_2602_01519_b200 as comb
    pool = comb.Pool(2, 64, 64, 4)
    k = torch.zeros((40, 2, 64), dtype=torch.bfloat16, device="cuda")
    pool.store_chunk(5, k, k)                                 # 3 pages
    with pytest.raises(comb.CombError) as e:
        pool.store_chunk(6, k, k)                             # needs 3, 1 free
    assert e.value.status == comb.COMB_ERR_NO_SPACE and pool.free_pages == 1
    with pytest.raises(comb.CombError) as e:
        pool.store_chunk(5, k[:39], k[:39])                   # same id, other length
    assert e.value.status == comb.COMB_ERR_EXISTS
    with pytest.raises(comb.CombError) as e:
        pool.link([[5, 77]])
    assert e.value.status == comb.COMB_ERR_UNKNOWN_CHUNK
    lb = pool.link([[5]])
    q = torch.zeros((1, 2, 64), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(comb.CombError) as e:
        pool.decode(lb, q, -1.0)                              # scale must be positive and finite
    assert e.value.status == comb.COMB_ERR_INVALID
    pool.close()


# ------------------------------------------------------------------------------------------------
# (a5) decode parity
# ------------------------------------------------------------------------------------------------
def ragged_workload(name, Hq, Hkv, Dqk, Dv, lq, seed=0, k=9):
    rng = np.random.default_rng([seed, 77])
    lens = rng.integers(1, 300, size=24).astype(np.int32)
    lens[:4] = [1, 16, 17, 255]
    R = len(lq)
    links = []
    for r in range(R):
        m = int(rng.integers(1, 12))
        links.append(rng.choice(24, size=m, replace=False))
    if R > 2:
        links[1] = np.zeros(0, np.int64)           # empty link (P12)
        links[2] = np.array([0])                    # a single key in a page with 15 masked slots (P3 geometry)
    return cs.custom(name, k=k, seed=seed, num_q_heads=Hq, num_kv_heads=Hkv, head_dim_qk=Dqk, head_dim_v=Dv,
                     chunk_len=lens, links=links, lq=lq)


DECODE_SHAPES = [(8, 2, 64, 64), (32, 8, 128, 128), (16, 16, 192, 128), (4, 2, 128, 128), (4, 4, 64, 128)]


@pytest.mark.parametrize("shape", DECODE_SHAPES)
@pytest.mark.parametrize("peaked", [False, True])
def test_decode_ragged(shape, peaked):
    Hq, Hkv, Dqk, Dv = shape
    w = ragged_workload("dec", Hq, Hkv, Dqk, Dv, [1] * 9)
    if peaked:
        w = w.peaked()
    ld, out, lse = run_decode(w, shuffle_seed=7)
    O, L = oracle.attention_for(w)
    check_attention(out, lse, O, L, "decode %s peaked=%s" % (shape, peaked))
    assert np.all(out[1] == 0) and np.all(np.isneginf(lse[1]))     # empty link: O = 0, LSE = -inf
    # single key: O = V exactly (bit-exact), LSE = its score
    v0 = ld.stored_host[0][1][0]                                    # [Hkv][Dv] bits
    G = Hq // Hkv
    for h in range(Hq):
        assert np.array_equal(out[2, h], v0[h // G])


def test_decode_tiny_config_and_long_split():
    w = cs.tiny_link().decode_phase()
    _, out, lse = run_decode(w)
    check_attention(out, lse, *oracle.attention_for(w), tag="tiny decode")
    # one long request (many splits) next to short ones: split-KV + LSE merge (P8)
    w = cs.custom("long", num_q_heads=8, num_kv_heads=2, head_dim_qk=128, head_dim_v=128,
                  chunk_len=[1000] * 12 + [37], links=[list(range(12)) + [12], [12], [3, 12, 5]], lq=[1, 1, 1])
    _, out, lse = run_decode(w, shuffle_seed=3)
    check_attention(out, lse, *oracle.attention_for(w), tag="long decode")


# ------------------------------------------------------------------------------------------------
# (a4) prefill parity
# ------------------------------------------------------------------------------------------------
PREFILL_SHAPES = [(8, 2, 64, 64), (32, 8, 128, 128), (16, 16, 192, 128), (4, 2, 128, 64), (8, 1, 64, 128)]


def test_prefill_tiny_config():
    w = cs.tiny_link()
    _, out, lse = run_prefill(w)
    check_attention(out, lse, *oracle.attention_for(w), tag="tiny prefill")
    _, out, lse = run_prefill(w.peaked())
    check_attention(out, lse, *oracle.attention_for(w.peaked()), tag="tiny prefill peaked")


def test_layers_share_page_ids_but_not_data():
    """L = 3 cross-attention layers over one page-id space (the paper interleaves 8 cross layers): a
    chunk is stored once per layer with that layer's K/V, linked once, and every layer's prefill and decode read
    their own arena slice."""
    from dataclasses import replace
    from paper_2602_01519_b200 import Pool
    base = ragged_workload("layers", 8, 2, 128, 128, [9, 0, 2, 40], seed=3)
    ws = [replace(base, seed=100 + l) for l in range(3)]  # same lengths and links, different K/V/Q values
    pool = Pool(2, 128, 128, base.pool_pages, num_layers=3, shuffle_seed=21, sentinel=SENTINEL)
    ids = list(range(base.num_chunks))
    tok = np.zeros(base.num_chunks + 1, np.int32)
    np.cumsum(base.chunk_len, out=tok[1:])
    for l in (2, 0, 1):  # any layer order: the first store of a chunk allocates its page list
        kv = [ws[l].chunk_kv(c) for c in ids]
        pool.store_chunks(ids, tok, H().bits_to_device(np.concatenate([k for k, _ in kv]), "cuda"),
                          H().bits_to_device(np.concatenate([v for _, v in kv]), "cuda"), layer=l)
    assert pool.free_pages == 0
    batch = pool.link([list(map(int, x)) for x in base.links])
    for l in range(3):
        q = H().bits_to_device(ws[l].all_q(), "cuda")
        out, lse = pool.prefill(batch, q, base.q_indptr, base.scale, layer=l)
        torch.cuda.synchronize()
        check_attention(H().device_to_bits(out), lse.cpu().numpy().astype(np.float64), *oracle.attention_for(ws[l]),
                        tag="prefill layer %d" % l)
        wd = ws[l].decode_phase()
        outd, lsed = pool.decode(batch, H().bits_to_device(wd.all_q(), "cuda"), wd.scale, layer=l)
        torch.cuda.synchronize()
        check_attention(H().device_to_bits(outd), lsed.cpu().numpy().astype(np.float64), *oracle.attention_for(wd),
                        tag="decode layer %d" % l)
    pool.close()


@pytest.mark.parametrize("shape", [(32, 8, 128, 128), (16, 16, 192, 128), (8, 2, 64, 64)])
def test_prefill_kv_ranges_low_parallelism(shape):
    """Few work items for 148 SMs (the paper's regime: < 50 dynamic tokens): every request's KV is cut
    into ranges that run on different SMs and are merged by LSE (pin P8). Requests of very different lengths (one
    shorter than a range, one empty, interior partial pages) share the call."""
    Hq, Hkv, Dqk, Dv = shape
    lens = [700, 333, 512, 129, 16, 1000, 47, 800]
    w = cs.custom("ranges", num_q_heads=Hq, num_kv_heads=Hkv, head_dim_qk=Dqk, head_dim_v=Dv, chunk_len=lens,
                  links=[[0, 1, 2, 3, 5, 7, 6], [4], [], [5, 0, 7, 2, 1]], lq=[20, 7, 3, 32], seed=5)
    for ww in (w, w.peaked()):
        ld = H().load_workload(ww, sentinel=SENTINEL, shuffle_seed=13)
        l0 = ld.pool.launches
        out, lse = ld.pool.prefill(ld.batch, ld.q, ld.q_indptr, ww.scale)
        torch.cuda.synchronize()
        assert ld.pool.launches - l0 == 2, "expected the range kernel + the merge kernel"
        out, lse = H().device_to_bits(out), lse.cpu().numpy().astype(np.float64)
        check_attention(out, lse, *oracle.attention_for(ww), tag="kv ranges %s" % (shape,))
        rows2 = slice(int(ww.q_indptr[2]), int(ww.q_indptr[3]))
        assert np.all(out[rows2] == 0) and np.all(np.isneginf(lse[rows2]))
        ld.pool.close()


@pytest.mark.parametrize("shape", PREFILL_SHAPES)
@pytest.mark.parametrize("peaked", [False, True])
def test_prefill_ragged(shape, peaked):
    Hq, Hkv, Dqk, Dv = shape
    # ragged query counts: below one tile, exactly tiles, several tiles with a tail, zero rows
    w = ragged_workload("pre", Hq, Hkv, Dqk, Dv, [5, 3, 2, 70, 0, 33, 129], seed=1)
    if peaked:
        w = w.peaked()
    ld, out, lse = run_prefill(w, shuffle_seed=11)
    O, L = oracle.attention_for(w)
    check_attention(out, lse, O, L, "prefill %s peaked=%s" % (shape, peaked))
    rows1 = slice(int(w.q_indptr[1]), int(w.q_indptr[2]))
    assert np.all(out[rows1] == 0) and np.all(np.isneginf(lse[rows1]))
    rows2 = slice(int(w.q_indptr[2]), int(w.q_indptr[3]))
    v0 = ld.stored_host[0][1][0]
    G = Hq // Hkv
    for h in range(Hq):
        assert np.array_equal(out[rows2, h], np.broadcast_to(v0[h // G], out[rows2, h].shape))


def test_prefill_closed_forms():
    D = 64
    # P4: Q = 0 -> mean of V, LSE = ln(kv_len)
    w = cs.custom("p4", num_q_heads=4, num_kv_heads=2, head_dim_qk=D, head_dim_v=D, chunk_len=[128, 100, 31],
                  links=[[2, 0, 1]], lq=[3], q_gain=0.0)
    ld, out, lse = run_prefill(w)
    vs = np.concatenate([cs.bf16_bits_to_f64(ld.stored_host[c][1]) for c in (2, 0, 1)], 0).mean(0)
    got = cs.bf16_bits_to_f64(out)
    for h in range(4):
        assert np.abs(got[:, h] - vs[h // 2]).max() <= 2 ** -8 * np.abs(vs).max() + 1e-6
    assert np.abs(lse - math.log(259)).max() <= 1e-4


def test_prefill_permutation_and_split_invariance():
    # P6: any link order gives the same attention; P7: a chunk split in two == kept whole
    Hq, Hkv, D = 8, 2, 128
    base = cs.custom("perm", num_q_heads=Hq, num_kv_heads=Hkv, head_dim_qk=D, head_dim_v=D,
                     chunk_len=[53, 200, 16, 77], links=[[0, 1, 2, 3]], lq=[40])
    O, L = oracle.attention_for(base)
    outs = []
    for perm in ([0, 1, 2, 3], [3, 2, 1, 0], [2, 0, 3, 1]):
        w = cs.custom("perm", num_q_heads=Hq, num_kv_heads=Hkv, head_dim_qk=D, head_dim_v=D,
                      chunk_len=[53, 200, 16, 77], links=[perm], lq=[40])
        _, out, lse = run_prefill(w)
        check_attention(out, lse, O, L, "perm %s" % perm)
        outs.append(cs.bf16_bits_to_f64(out))
    for o in outs[1:]:
        close_in_ulps(outs[0], o, "permuted link")
    # split: store chunk 1 (200 tokens) as 21 + 179 -> interior partial page
    import paper_2602_01519_b200 as comb
    k, v = base.chunk_kv(1)
    q = H().bits_to_device(base.all_q(), "cuda")
    res = []
    for pieces in ([200], [21, 179]):
        pool = comb.Pool(Hkv, D, D, 32, sentinel=SENTINEL)
        at, ids = 0, []
        for i, n in enumerate(pieces):
            pool.store_chunk(i, H().bits_to_device(k[at:at + n], "cuda"), H().bits_to_device(v[at:at + n], "cuda"))
            ids.append(i)
            at += n
        lb = pool.link([ids])
        out, lse = pool.prefill(lb, q, base.q_indptr, base.scale)
        torch.cuda.synchronize()
        res.append((cs.bf16_bits_to_f64(H().device_to_bits(out)), lse.cpu().numpy()))
        pool.close()
    close_in_ulps(res[0][0], res[1][0], "split vs whole")
    assert np.abs(res[0][1] - res[1][1]).max() <= 1e-4


def test_prefill_row_equals_decode():
    # P11: a generated token is treated like a query token
    w = ragged_workload("p11", 32, 8, 128, 128, [6, 1, 1, 9], seed=5)
    ld, out_p, lse_p = run_prefill(w)
    out_d, lse_d = ld.pool.decode(ld.pool.link([list(map(int, w.links[0]))] * 6), ld.q[:6], w.scale)
    torch.cuda.synchronize()
    a = cs.bf16_bits_to_f64(out_p[:6])
    b = cs.bf16_bits_to_f64(H().device_to_bits(out_d))
    close_in_ulps(a, b, "prefill row vs decode")
    assert np.abs(lse_p[:6] - lse_d.cpu().numpy()).max() <= 1e-3


# ------------------------------------------------------------------------------------------------
# full BASELINE sizes, in the launch configuration bench.py times: sampled outputs against O1
# ------------------------------------------------------------------------------------------------
def sampled_check(w, ld, out_bits, lse, n_per_req=6, reqs=(0, 1, -1)):
    rng = np.random.default_rng(123)
    R = w.num_requests
    for r in [x % R for x in reqs]:
        lo, hi = int(w.q_indptr[r]), int(w.q_indptr[r + 1])
        rows = rng.integers(lo, hi, size=n_per_req).astype(np.int32)
        heads = rng.integers(0, w.num_q_heads, size=n_per_req).astype(np.int32)
        ks, vs, sel = [], [], []
        for c in w.links[r]:
            k, v = ld.stored_host[int(c)]
            sel.append(len(ks))
            ks.append(k)
            vs.append(v)
        qi = np.zeros(R + 1, np.int32)
        qi[:] = w.q_indptr
        ci = np.zeros(R + 1, np.int32)
        ci[r + 1:] = len(sel)
        q_all = H().device_to_bits(ld.q)
        O, L = oracle.attention_samples(r, q_all, qi, ks, vs, ci, np.array(sel, np.int32), w.scale, rows, heads)
        got = cs.bf16_bits_to_f64(out_bits[rows, heads])
        err = np.abs(got - O)
        assert err.max() <= 2e-2 and err.mean() <= 2e-3, (r, err.max(), err.mean())
        rel = math.sqrt(float((err ** 2).sum()) / float((O ** 2).sum()))
        assert rel <= 1e-2, (r, rel)
        assert np.abs(lse[rows, heads] - L).max() <= 2e-3


def test_full_size_decode_link_sampled():
    w = cs.decode_link()
    ld, out, lse = run_decode(w, fill="linked", shuffle_seed=2024)
    assert np.all(np.isfinite(cs.bf16_bits_to_f64(out)))
    sampled_check(w, ld, out, lse)


def test_full_size_rag_prefill_sampled():
    w = cs.rag_prefill()
    ld, out, lse = run_prefill(w, fill="linked", shuffle_seed=2024)
    assert np.all(np.isfinite(cs.bf16_bits_to_f64(out)))
    sampled_check(w, ld, out, lse)


def test_full_size_long_fewshot_sampled():
    w = cs.long_fewshot()
    ld, out, lse = run_prefill(w, shuffle_seed=2024)
    assert np.all(np.isfinite(cs.bf16_bits_to_f64(out)))
    sampled_check(w, ld, out, lse, n_per_req=4, reqs=(0, -1))
    wd = w.decode_phase()
    qd = H().bits_to_device(wd.all_q(), "cuda")
    out_d, lse_d = ld.pool.decode(ld.batch, qd, wd.scale)
    torch.cuda.synchronize()
    ld.q = qd
    sampled_check(wd, ld, H().device_to_bits(out_d), lse_d.cpu().numpy().astype(np.float64), n_per_req=4, reqs=(0, -1))


def test_full_size_mla_sampled():
    w = cs.mla_shaped()
    ld, out, lse = run_prefill(w, fill="linked", shuffle_seed=2024)
    assert np.all(np.isfinite(cs.bf16_bits_to_f64(out)))
    sampled_check(w, ld, out, lse, n_per_req=4, reqs=(0, -1))
    wd = w.decode_phase()
    qd = H().bits_to_device(wd.all_q(), "cuda")
    out_d, lse_d = ld.pool.decode(ld.batch, qd, wd.scale)
    torch.cuda.synchronize()
    ld.q = qd
    sampled_check(wd, ld, H().device_to_bits(out_d), lse_d.cpu().numpy().astype(np.float64), n_per_req=4, reqs=(0, -1))
