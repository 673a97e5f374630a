"""Pins for the fp64 oracle (run with -m "not gpu").  Each test states which mistake it would catch.
The oracle follows PAPER.md:112-119 §4.2 Eq. 7-8 + PAPER.md:149 + PAPER.md:66; see oracle/comb_oracle.c."""
import math
import os

import numpy as np
import pytest

import comb_synth as cs
import oracle
from oracle import brute

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")) as f:
    for line in f:
        if line.strip() and not line.startswith("#"):
            name, val = line.split()[:2]
            GOLD[name] = float(val)


def bits(x):
    return cs.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def run(q, ks, vs, link, scale, lq=None):
    """single request helper: q bits [lq][Hq][Dqk]"""
    q_indptr = np.array([0, q.shape[0]], np.int32)
    return oracle.attention(q, q_indptr, ks, vs, np.array([0, len(link)], np.int32), np.array(link, np.int32), scale)


def rand_case(seed, lq, Hq, Hkv, Dqk, Dv, lens):
    rng = np.random.default_rng(seed)
    q = bits(rng.standard_normal((lq, Hq, Dqk)))
    ks = [bits(rng.standard_normal((t, Hkv, Dqk))) for t in lens]
    vs = [bits(rng.standard_normal((t, Hkv, Dv))) for t in lens]
    return q, ks, vs


# ---- P1: brute force, separately written, no max subtraction ------------------------------------
@pytest.mark.parametrize("Hq,Hkv,Dqk,Dv,lens,link", [
    (4, 2, 64, 64, [5, 17, 40], [2, 0, 1]),     # GQA 2, ragged chunk lengths, shuffled link order
    (2, 2, 8, 4, [3], [0]),                       # Dqk != Dv, no GQA
    (4, 1, 16, 8, [7, 9], [1, 0, 1]),            # a chunk linked twice (taken literally, reading I14)
])
def test_p1_brute_force(Hq, Hkv, Dqk, Dv, lens, link):
    q, ks, vs = rand_case(1, 3, Hq, Hkv, Dqk, Dv, lens)
    scale = 1.0 / math.sqrt(Dqk)
    O, L = run(q, ks, vs, link, scale)
    Ob, Lb = brute.attention_brute(q, ks, vs, link, scale)
    assert np.max(np.abs(O - np.array(Ob))) <= 1e-12
    assert np.max(np.abs(L - np.array(Lb))) <= 1e-12


# ---- P2: library special case (one chunk): fp64 softmax(QK^T*scale)V with numpy matmul / torch SDPA -----
@pytest.mark.parametrize("G", [1, 4])
def test_p2_library_sdpa(G):
    torch = pytest.importorskip("torch")
    Hkv, Dqk, Dv, T, lq = 2, 64, 32, 48, 5
    Hq = Hkv * G
    q, ks, vs = rand_case(2, lq, Hq, Hkv, Dqk, Dv, [T])
    scale = 0.2  # deliberately not 1/sqrt(d): a hard-wired scale fails here
    O, L = run(q, ks, vs, [0], scale)
    qf = torch.from_numpy(cs.bf16_bits_to_f64(q)).permute(1, 0, 2)                       # [Hq][lq][Dqk]
    kf = torch.from_numpy(cs.bf16_bits_to_f64(ks[0])).permute(1, 0, 2).repeat_interleave(G, 0)   # consecutive grouping
    vf = torch.from_numpy(cs.bf16_bits_to_f64(vs[0])).permute(1, 0, 2).repeat_interleave(G, 0)
    ref = torch.nn.functional.scaled_dot_product_attention(qf, kf, vf, scale=scale).permute(1, 0, 2).numpy()
    assert np.max(np.abs(O - ref)) <= 1e-12
    s = np.einsum("hid,hjd->hij", qf.numpy(), kf.numpy()) * scale
    lse_ref = np.log(np.exp(s).sum(-1)).T
    assert np.max(np.abs(L - lse_ref)) <= 1e-12


# ---- P3: single key returns its V exactly; LSE = its score -----------------------------------------
def test_p3_single_key():
    q, ks, vs = rand_case(3, 2, 4, 2, 64, 64, [1])
    O, L = run(q, ks, vs, [0], 0.125)
    v = cs.bf16_bits_to_f64(vs[0])[0]                    # [Hkv][Dv]
    for h in range(4):
        assert np.array_equal(O[:, h, :], np.broadcast_to(v[h // 2], (2, 64)))
    s = 0.125 * np.einsum("ihd,hd->ih", cs.bf16_bits_to_f64(q), np.repeat(cs.bf16_bits_to_f64(ks[0])[0], 2, 0))
    assert np.max(np.abs(L - s)) <= 1e-12


# ---- P4: equal scores -> mean of V, LSE = ln(kv_len) ----------------------------------------------
def test_p4_equal_scores():
    _, ks, vs = rand_case(4, 1, 4, 2, 64, 64, [128, 128, 128, 128])
    q = np.zeros((3, 4, 64), np.uint16)                   # Q = 0 => every score is 0
    O, L = run(q, ks, vs, [3, 1, 0, 2], 0.125)
    mean_v = np.concatenate([cs.bf16_bits_to_f64(v) for v in vs], 0).mean(0)   # [Hkv][Dv]
    for h in range(4):
        assert np.max(np.abs(O[:, h, :] - mean_v[h // 2])) <= 1e-13
    assert np.max(np.abs(L - GOLD["ln_512"])) <= 1e-13


# ---- P5: two-level closed form sigma(1), and the unbalanced 3:1 case ------------------------------
@pytest.mark.parametrize("n1,n0,gold", [(8, 8, "sigmoid_1"), (3, 1, "two_level_3_to_1")])
def test_p5_two_level(n1, n0, gold):
    D = 16
    q = np.zeros((1, 1, D), np.float32); q[0, 0, 0] = 1.0
    k1 = np.zeros((n1, 1, D), np.float32); k1[:, 0, 0] = 1.0       # score 1, V = 1
    k0 = np.zeros((n0, 1, D), np.float32)                           # score 0, V = 0
    O, L = run(bits(q), [bits(k1), bits(k0)], [bits(np.ones((n1, 1, D))), bits(np.zeros((n0, 1, D)))], [1, 0], 1.0)
    assert np.max(np.abs(O - GOLD[gold])) <= 1e-15
    assert abs(L[0, 0] - math.log(n1 * math.e + n0)) <= 1e-14


# ---- P6: permutation invariance ("in any order/position") ---------------------------
def test_p6_permutation():
    q, ks, vs = rand_case(6, 4, 8, 2, 64, 64, [33, 16, 50, 7])
    base = run(q, ks, vs, [0, 1, 2, 3], 0.125)
    for perm in ([3, 2, 1, 0], [2, 0, 3, 1]):
        got = run(q, ks, vs, perm, 0.125)
        assert np.max(np.abs(got[0] - base[0])) <= 1e-12 and np.max(np.abs(got[1] - base[1])) <= 1e-12


# ---- P7: a chunk split in two == kept whole (l_doc = sum l_doc,i) -------------------
def test_p7_split_equals_whole():
    q, ks, vs = rand_case(7, 3, 4, 2, 64, 64, [53])
    whole = run(q, ks, vs, [0], 0.125)
    t1 = 21                                              # not a multiple of 16: interior partial page
    split = run(q, [ks[0][:t1], ks[0][t1:]], [vs[0][:t1], vs[0][t1:]], [0, 1], 0.125)
    assert np.max(np.abs(whole[0] - split[0])) <= 1e-12 and np.max(np.abs(whole[1] - split[1])) <= 1e-12


# ---- P8: merge identity over a disjoint split of the keys ------------------------------------------
def test_p8_merge_identity():
    q, ks, vs = rand_case(8, 3, 4, 2, 64, 64, [40, 25])
    OA, LA = run(q, ks, vs, [0], 0.125)
    OB, LB = run(q, ks, vs, [1], 0.125)
    O, L = run(q, ks, vs, [0, 1], 0.125)
    wa, wb = np.exp(LA)[..., None], np.exp(LB)[..., None]
    assert np.max(np.abs(O - (wa * OA + wb * OB) / (wa + wb))) <= 1e-12
    assert np.max(np.abs(L - np.log(np.exp(LA) + np.exp(LB)))) <= 1e-12
    # two identical halves: LSE shifts by exactly ln 2, O unchanged
    O2, L2 = run(q, ks, vs, [0, 0], 0.125)
    assert np.max(np.abs(O2 - OA)) <= 1e-12 and np.max(np.abs(L2 - LA - GOLD["ln_2"])) <= 1e-12


# ---- P9: shift invariance: add a vector c to every key ---------------------------------------------
def test_p9_shift_invariance():
    rng = np.random.default_rng(9)
    D, T = 8, 12
    q = rng.integers(-3, 4, (2, 2, D)).astype(np.float32)       # small integers: sums stay exact in bf16
    k = rng.integers(-3, 4, (T, 1, D)).astype(np.float32)
    v = rng.standard_normal((T, 1, D)).astype(np.float32)
    c = rng.integers(-2, 3, (D,)).astype(np.float32)
    O1, L1 = run(bits(q), [bits(k)], [bits(v)], [0], 0.25)
    O2, L2 = run(bits(q), [bits(k + c)], [bits(v)], [0], 0.25)
    assert np.max(np.abs(O1 - O2)) <= 1e-12
    assert np.max(np.abs((L2 - L1) - 0.25 * (q.astype(np.float64) @ c.astype(np.float64)))) <= 1e-12


# ---- P10: V-affinity: constant V -> that constant; O linear in V ----------------------------------
def test_p10_v_affinity():
    q, ks, vs = rand_case(10, 2, 4, 2, 64, 64, [19, 30])
    const = [bits(np.full(v.shape, 1.5)) for v in vs]
    O, _ = run(q, ks, const, [1, 0], 0.125)
    assert np.array_equal(O, np.full_like(O, 1.5)) or np.max(np.abs(O - 1.5)) <= 1e-15
    # linearity: V scaled by 2 (exact in bf16) doubles O exactly
    v2 = [bits(cs.bf16_bits_to_f32(v) * 2.0) for v in vs]
    Oa, _ = run(q, ks, vs, [1, 0], 0.125)
    Ob, _ = run(q, ks, v2, [1, 0], 0.125)
    assert np.max(np.abs(Ob - 2.0 * Oa)) <= 1e-13


# ---- P12: empty link -> O = 0, LSE = -inf (reading I13) ------------------------------------------------
def test_p12_empty_link():
    q, ks, vs = rand_case(12, 2, 4, 2, 64, 64, [16])
    q2 = np.concatenate([q, q], 0)
    O, L = oracle.attention(q2, np.array([0, 2, 4], np.int32), ks, vs, np.array([0, 0, 1], np.int32),
                            np.array([0], np.int32), 0.125)
    assert np.all(O[:2] == 0.0) and np.all(np.isneginf(L[:2]))
    assert np.all(np.isfinite(L[2:])) and np.any(O[2:] != 0.0)


# ---- multi-request bookkeeping: rows of request r only see request r's chunks ----------------------
def test_requests_are_independent():
    w = cs.custom("two", num_q_heads=4, num_kv_heads=2, head_dim_qk=64, head_dim_v=64,
                  chunk_len=[20, 33, 16], links=[[2, 0], [1]], lq=[3, 2])
    O, L = oracle.attention_for(w)
    O0, L0 = oracle.attention_for(w, [0])
    O1, L1 = oracle.attention_for(w, [1])
    assert np.array_equal(O, np.concatenate([O0, O1])) and np.array_equal(L, np.concatenate([L0, L1]))
    # sampled entry point agrees with the full one
    ks, vs = zip(*[w.chunk_kv(c) for c in range(3)])
    Os, Ls = oracle.attention_samples(1, w.all_q(), w.q_indptr, ks, vs, np.array([0, 2, 3], np.int32),
                                      np.array([2, 0, 1], np.int32), w.scale, np.array([3, 4]), np.array([1, 3]))
    assert np.array_equal(Os[0], O[3, 1]) and np.array_equal(Os[1], O[4, 3]) and Ls[1] == L[4, 3]


# ---- O3: table model ---------------------------------------------------------------------------------
def test_o3_tables_hand_example():
    m = oracle.PoolModel(10, 0)
    assert m.store(7, 20) == [0, 1]          # ceil(20/16) = 2 pages from the head
    assert m.store(9, 16) == [2]
    assert m.store(3, 33) == [3, 4, 5]
    t = m.link([[3, 7], [], [9, 7]])
    assert t["page_indptr"].tolist() == [0, 5, 5, 8]
    assert t["page_ids"].tolist() == [3, 4, 5, 0, 1, 2, 0, 1]
    assert t["page_ntok"].tolist() == [16, 16, 1, 16, 4, 16, 16, 4]   # interior partial pages keep their count
    assert t["kv_len"].tolist() == [53, 0, 36]
    m.release(7)                              # freed ids go to the TAIL
    assert m.store(11, 80) == [6, 7, 8, 9, 0]
    with pytest.raises(MemoryError):
        m.store(12, 40)


def test_o3_shuffled_free_list_is_a_permutation():
    a = oracle.initial_free_list(1000, 12345)
    assert sorted(a) == list(range(1000)) and a != list(range(1000))
    assert a == oracle.initial_free_list(1000, 12345)
    assert oracle.initial_free_list(5, 0) == [0, 1, 2, 3, 4]
    # first splitmix64 output for seed 1 is a published constant of the generator
    g = oracle._splitmix64_stream(1)
    assert next(g) == 0x910A2DEC89025CC1


# ---- O2: page image round trip -------------------------------------------------------------------------
def test_o2_page_image_round_trip():
    rng = np.random.default_rng(5)
    x = rng.integers(0, 2**16, (37, 2, 8), dtype=np.uint16)
    pages = [4, 1, 6]
    img = oracle.page_image(8, 2, 8, [(x, pages)])
    back = np.concatenate([np.transpose(img[p], (1, 0, 2)) for p in pages], 0)   # gather pages back
    assert np.array_equal(back[:37], x) and np.all(back[37:] == 0)
    assert np.all(img[[0, 2, 3, 5, 7]] == 0x7FC0)


# ---- P16: layer-count sanity of the pool byte formula ("saves 75%") -------------------
def test_p16_kv_saving():
    per_layer = 1024 * 8 * (128 + 128) * 2
    assert 1.0 - (8 * per_layer) / (32 * per_layer) == GOLD["kv_saving_llama"]


# ---- bf16 helpers used by every generator ----------------------------------------------------------------
def test_bf16_rounding_is_rne():
    x = np.array([1.0, 1.00390625, 1.01171875, -2.5, 3.0e-5], np.float32)   # 1+2^-8 ties to even (1.0); 1+3*2^-8 ties up
    b = cs.f32_to_bf16_bits(x)
    assert b[0] == 0x3F80 and b[1] == 0x3F80 and b[2] == 0x3F82 and b[3] == 0xC020
    assert np.array_equal(cs.f32_to_bf16_bits(cs.bf16_bits_to_f32(b)), b)
    torch = pytest.importorskip("torch")
    y = np.random.default_rng(0).standard_normal(4096).astype(np.float32)
    ref = torch.from_numpy(y).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(cs.f32_to_bf16_bits(y), ref)


def test_chunk_major_inversion_hand_example():
    """O3, chunk-major view (include/comb.h): worked by hand.  Requests link [5, 7], [7], [9, 7, 5]: entries in link
    order are e0=(r0,5) e1=(r0,7) e2=(r1,7) e3=(r2,9) e4=(r2,7) e5=(r2,5).  Chunk 7 is linked 3 times, 5 twice,
    9 once => slots [7, 5, 9]; slot rows in ascending entry number."""
    m = oracle.PoolModel(16)
    m.store(5, 20)   # pages 0, 1   (last page holds 4 tokens)
    m.store(7, 16)   # page  2
    m.store(9, 33)   # pages 3, 4, 5 (last page holds 1 token)
    t = m.link_chunk_major([[5, 7], [7], [9, 7, 5]])
    assert t["slot_chunks"].tolist() == [7, 5, 9]
    assert t["entry_indptr"].tolist() == [0, 2, 3, 6]
    assert t["cas_page_indptr"].tolist() == [0, 1, 3, 6]
    assert t["cas_page_ids"].tolist() == [2, 0, 1, 3, 4, 5]
    assert t["cas_page_ntok"].tolist() == [16, 16, 4, 16, 16, 1]
    assert t["cas_row_indptr"].tolist() == [0, 3, 5, 6]
    assert t["cas_row_req"].tolist() == [0, 1, 2, 0, 2, 2]
    assert t["cas_row_entry"].tolist() == [1, 2, 4, 0, 5, 3]
    # ties keep first appearance: [1, 2], [2, 1] -> both linked twice, chunk 1 appears first
    m2 = oracle.PoolModel(4)
    m2.store(1, 1)
    m2.store(2, 1)
    assert m2.link_chunk_major([[1, 2], [2, 1]])["slot_chunks"].tolist() == [1, 2]


# ------------------------------------------------------------------------------------------------
# oracle/layer.py — the projections and the sub-layer around the attention
# ------------------------------------------------------------------------------------------------
from oracle import layer as ol  # noqa: E402


def _small_layer(seed=0, Hq=4, Hkv=2, Dqk=8, Dv=4, d_model=12):
    rng = np.random.default_rng(seed)
    lens = [5, 1, 7]
    ck = [rng.standard_normal((t, Hkv, Dqk)) for t in lens]
    cv = [rng.standard_normal((t, Hkv, Dv)) for t in lens]
    links = [[2, 0], [], [1, 0, 2]]
    q_indptr = np.array([0, 3, 5, 6], np.int32)
    x = rng.standard_normal((6, d_model))
    w_q = rng.standard_normal((Hq * Dqk, d_model)) / 3.0
    w_o = rng.standard_normal((d_model, Hq * Dv)) / 3.0
    return dict(x=x, q_indptr=q_indptr, w_q=w_q, w_o=w_o, Hq=Hq, ck=ck, cv=cv, links=links, scale=0.3)


def test_project_kv_brute_force_and_identity():
    """Eq. 5-6 by explicit loops; and with W = identity blocks the projection hands the hidden state through."""
    rng = np.random.default_rng(1)
    T, d_model, Hkv, Dqk, Dv = 5, 6, 2, 3, 2
    h = rng.standard_normal((T, d_model))
    w = rng.standard_normal((Hkv * (Dqk + Dv), d_model))
    K, V = ol.project_kv(h, w, Hkv, Dqk, Dv)
    for t in range(T):
        for g in range(Hkv):
            for d in range(Dqk):
                assert abs(K[t, g, d] - sum(h[t, c] * w[g * Dqk + d, c] for c in range(d_model))) < 1e-13
            for d in range(Dv):
                assert abs(V[t, g, d] - sum(h[t, c] * w[Hkv * Dqk + g * Dv + d, c] for c in range(d_model))) < 1e-13
    eye = np.zeros((Hkv * (Dqk + Dv), 10))
    eye[np.arange(10), np.arange(10)] = 1.0
    h10 = rng.standard_normal((T, 10))
    K, V = ol.project_kv(h10, eye, Hkv, Dqk, Dv)
    assert np.array_equal(K.reshape(T, -1), h10[:, :6]) and np.array_equal(V.reshape(T, -1), h10[:, 6:])


def test_attention_f64_agrees_with_the_c_oracle_and_brute_force():
    """Two independently written statements of Eq. 7-8 (C loops over bf16 inputs; numpy matmuls over fp64 inputs) on
    bf16-exact values, plus the no-max-subtraction brute force; empty link gives O = 0, LSE = -inf."""
    w = cs.custom("pin", num_q_heads=4, num_kv_heads=2, head_dim_qk=64, head_dim_v=64, chunk_len=[20, 37, 3],
                  links=[[1, 0, 2], [], [2]], lq=[3, 2, 4])
    O, L = oracle.attention_for(w)
    for r in range(3):
        q = ol.bf16_to_f64(w.request_q(r))
        lst = [int(c) for c in w.links[r]]
        kc = np.concatenate([ol.bf16_to_f64(w.chunk_kv(c)[0]) for c in lst], 0) if lst else np.zeros((0, 2, 64))
        vc = np.concatenate([ol.bf16_to_f64(w.chunk_kv(c)[1]) for c in lst], 0) if lst else np.zeros((0, 2, 64))
        o, l = ol.attention_f64(q, kc, vc, w.scale)
        lo, hi = int(w.q_indptr[r]), int(w.q_indptr[r + 1])
        assert np.abs(o - O[lo:hi]).max() <= 1e-12
        if lst:
            assert np.abs(l - L[lo:hi]).max() <= 1e-12
            ob, lb = brute.attention_request(q, kc, vc, w.scale)
            assert np.abs(o - ob).max() <= 1e-12 and np.abs(l - lb).max() <= 1e-12
        else:
            assert np.all(o == 0) and np.all(np.isneginf(l))


def test_cross_layer_special_weights():
    """PAPER.md:117 + 30: the sub-layer only ADDS to the decoder row, so W_O = 0 recovers it exactly (the plug-in
    property); W_Q = 0 makes every score equal, so the attention is the mean of the linked V (P4) pushed through W_O;
    the result is linear in W_O; a request that links nothing keeps its rows."""
    a = _small_layer()
    y = ol.cross_layer(a["x"], a["q_indptr"], a["w_q"], a["w_o"], a["Hq"], a["ck"], a["cv"], a["links"], a["scale"])
    y0 = ol.cross_layer(a["x"], a["q_indptr"], a["w_q"], 0 * a["w_o"], a["Hq"], a["ck"], a["cv"], a["links"], a["scale"])
    assert np.array_equal(y0, a["x"])
    assert np.array_equal(y[3:5], a["x"][3:5])                       # request 1 links nothing
    y2 = ol.cross_layer(a["x"], a["q_indptr"], a["w_q"], 2 * a["w_o"], a["Hq"], a["ck"], a["cv"], a["links"], a["scale"])
    assert np.abs((y2 - a["x"]) - 2 * (y - a["x"])).max() <= 1e-13
    yq = ol.cross_layer(a["x"], a["q_indptr"], 0 * a["w_q"], a["w_o"], a["Hq"], a["ck"], a["cv"], a["links"], a["scale"])
    G = a["Hq"] // 2
    for r, rows in ((0, range(0, 3)), (2, range(5, 6))):
        vmean = np.concatenate([a["cv"][c] for c in a["links"][r]], 0).mean(0)     # [Hkv][Dv]
        heads = np.concatenate([vmean[h // G] for h in range(a["Hq"])])             # [Hq*Dv]
        for i in rows:
            assert np.abs(yq[i] - (a["x"][i] + a["w_o"] @ heads)).max() <= 1e-13


def test_cross_layer_brute_force():
    """Eq. 4 + 7-8 + output projection by explicit loops and the brute-force attention (no max subtraction)."""
    a = _small_layer(seed=3)
    y = ol.cross_layer(a["x"], a["q_indptr"], a["w_q"], a["w_o"], a["Hq"], a["ck"], a["cv"], a["links"], a["scale"])
    Hq, Dqk, Dv = a["Hq"], 8, 4
    for r, lst in enumerate(a["links"]):
        for i in range(a["q_indptr"][r], a["q_indptr"][r + 1]):
            q = np.array([[sum(a["x"][i, c] * a["w_q"][h * Dqk + d, c] for c in range(12)) for d in range(Dqk)]
                          for h in range(Hq)])
            if lst:
                kc = np.concatenate([a["ck"][c] for c in lst], 0)
                vc = np.concatenate([a["cv"][c] for c in lst], 0)
                o, _ = brute.attention_request(q[None], kc, vc, a["scale"])
                o = o[0].reshape(-1)
            else:
                o = np.zeros(Hq * Dv)
            want = a["x"][i] + np.array([sum(o[j] * a["w_o"][c, j] for j in range(Hq * Dv)) for c in range(12)])
            assert np.abs(y[i] - want).max() <= 1e-12


def test_cross_stack_is_the_layers_in_order():
    a = _small_layer(seed=5)
    wq = [a["w_q"], a["w_q"][::-1].copy()]
    wo = [a["w_o"], a["w_o"][:, ::-1].copy()]
    ck, cv = [a["ck"], [k[::-1].copy() for k in a["ck"]]], [a["cv"], [v * 0.5 for v in a["cv"]]]
    st = ol.cross_stack(a["x"], a["q_indptr"], wq, wo, a["Hq"], ck, cv, a["links"], a["scale"])
    y1 = ol.cross_layer(a["x"], a["q_indptr"], wq[0], wo[0], a["Hq"], ck[0], cv[0], a["links"], a["scale"])
    y2 = ol.cross_layer(y1, a["q_indptr"], wq[1], wo[1], a["Hq"], ck[1], cv[1], a["links"], a["scale"])
    assert np.array_equal(st[0], y1) and np.array_equal(st[1], y2)


def test_bf16_rounding_helpers():
    """bf16 keeps 8 significant bits: the spacing at 1.0 is 2^-7.  Hand-worked round-to-nearest-even cases."""
    x = np.array([1.0, 1.0 + 2.0 ** -7, 1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, 1.0 + 2.0 ** -8 + 2.0 ** -20, -2.5, 0.0])
    b = ol.f64_to_bf16_bits(x)
    assert [hex(v) for v in b] == ["0x3f80", "0x3f81", "0x3f80", "0x3f82", "0x3f81", "0xc020", "0x0"]
    #        exact     exact      tie -> even (down)  tie -> even (up)  just above the tie
    assert np.array_equal(ol.bf16_to_f64(b), [1.0, 1.0078125, 1.0, 1.015625, 1.0078125, -2.5, 0.0])


def test_lru_eviction_hand_example():
    """O3 lifecycle (include/comb.h "(f4) pool lifecycle"), worked by hand on 6 pages.
    store a(2 pages) b(2) c(2): ticks 1,2,3, pool full.  link [a] -> tick 4 stamps a.  pin b.
    store d(3 pages): needs 3; candidates in (stamp, birth) order: b is pinned; c (3) then a (4) -> evict c (2 pages,
    not enough) and a (2 more): free list tail = c's pages then a's pages = [4,5,0,1]; d takes [4,5,0]."""
    m = oracle.PoolModel(6, evict_lru=True)
    assert m.store(10, 32) == [0, 1] and m.store(11, 17) == [2, 3] and m.store(12, 20) == [4, 5]
    m.touch([[10]])
    m.pin(11)
    assert m.store(13, 40) == [4, 5, 0]
    assert m.evicted == [12, 10] and sorted(m.dir) == [11, 13] and m.free_pages() == 1
    with pytest.raises(MemoryError):          # 11 is pinned, 13 is the newest: evicting 13 alone frees 3 + 1 < 5
        m.store(14, 80)
    assert m.evicted == [] and sorted(m.dir) == [11, 13]          # all or nothing
    m.unpin(11)
    assert m.store(14, 80) == [1, 2, 3, 4, 5]                      # evicts 11 (stamp 2) then 13: tail 1 | 2,3 | 4,5,0
    assert m.evicted == [11, 13]
    no = oracle.PoolModel(2)                                       # eviction off: a full pool refuses
    no.store(1, 32)
    with pytest.raises(MemoryError):
        no.store(2, 1)


# ------------------------------------------------------------------------------------------------
# fp8 (e4m3) pages: the oracle's quantisation model (oracle/fp8.py; DESIGN.md §2 I31-I33)
# ------------------------------------------------------------------------------------------------
def test_e4m3_code_table_closed_form_and_round_trip():
    """The format's own numbers: 448 = 1.75 * 2^8 is the largest finite value, 2^-9 the smallest subnormal, 2^-6 the
    smallest normal, 0x38 is 1.0; codes ascend with their values; encode(decode(c)) = c for every finite code."""
    from oracle import fp8
    t = fp8.e4m3_value_table()
    assert t[0x7e] == 448.0 and t[0xfe] == -448.0 and np.isnan(t[0x7f]) and np.isnan(t[0xff])
    assert t[0x01] == 2.0 ** -9 and t[0x07] == 7 * 2.0 ** -9 and t[0x08] == 2.0 ** -6 and t[0x38] == 1.0
    assert t[0x39] == 1.125 and t[0x40] == 2.0 and t[0x00] == 0.0
    assert np.all(np.diff(t[:127]) > 0)
    finite = np.array([c for c in range(256) if c not in (0x7f, 0xff)], np.uint8)
    back = fp8.e4m3_encode(t[finite])
    keep = finite != 0x80                       # -0.0 encodes as the sign bit over code 0: same value
    assert np.array_equal(back[keep], finite[keep]) and fp8.e4m3_decode(back[~keep])[0] == 0.0


def test_e4m3_rounding_ties_to_even_and_saturates():
    """Hand-worked: between 1.0 (0x38, mantissa 0) and 1.125 (0x39) the midpoint 1.0625 goes to the even mantissa 1.0;
    between 1.125 (0x39) and 1.25 (0x3a) the midpoint 1.1875 goes to 1.25; just above / below a midpoint goes to the
    nearer value; beyond 448 saturates (no infinity in this format); the subnormal midpoint 1.5 * 2^-9 goes to 2^-8."""
    from oracle import fp8
    x = np.array([1.0625, 1.1875, 1.0626, 1.0624, 1000.0, -1e9, 464.0, 1.5 * 2.0 ** -9, 0.4 * 2.0 ** -9, -1.0625])
    want = np.array([1.0, 1.25, 1.125, 1.0, 448.0, -448.0, 448.0, 2.0 ** -8, 0.0, -1.0])
    assert np.array_equal(fp8.e4m3_decode(fp8.e4m3_encode(x)), want)
    # brute force: the code chosen is a nearest finite value for 20,000 random inputs
    rng = np.random.default_rng(5)
    y = rng.standard_normal(20000) * np.exp(rng.uniform(-6, 6, 20000))
    t = fp8.e4m3_value_table()
    fin = t[~np.isnan(t)]
    got = fp8.e4m3_decode(fp8.e4m3_encode(y))
    best = np.abs(np.clip(y, -448, 448)[:, None] - fin[None, :]).min(axis=1)
    assert np.allclose(np.abs(np.clip(y, -448, 448) - got), best, rtol=0, atol=0)


def test_fp8_block_quantisation_properties():
    """scale = the smallest power of two 2^e with amax <= 448 * 2^e, so the block's largest element lands in (224, 448];
    the dequantised value is within half an e4m3 step (2^-4 relative for normals) of the input and is exactly a bf16
    number; an all-zero block has scale 1 and codes 0; tail slots of a chunk's last page are byte 0 and do not
    influence the scale.  Hand-worked scales: amax 448 -> 1, 449 -> 2, 224 -> 0.5, 3.5 -> 2^-7, 3.51 -> 2^-6."""
    from oracle import fp8
    w = cs.custom("q8", k=7, num_q_heads=4, num_kv_heads=2, head_dim_qk=128, head_dim_v=128, chunk_len=[37],
                  links=[[0]], lq=[1])
    kb, vb = w.chunk_kv(0)
    kc, ks, vc, vs = fp8.quantise_chunk(kb, vb)
    assert kc.shape == (3, 2, 16, 128) and ks.shape == (3, 2)
    x = fp8.bf16_bits_to_f32(kb).astype(np.float64)
    for i in range(3):
        n = min(16, 37 - 16 * i)
        for h in range(2):
            blk = x[16 * i:16 * i + n, h]
            top = np.abs(fp8.e4m3_decode(kc[i, h, :n])).max()
            assert 224.0 < np.abs(blk).max() / float(ks[i, h]) <= 448.0 and 224.0 <= top <= 448.0
            assert float(ks[i, h]) == 2.0 ** round(np.log2(float(ks[i, h])))
            assert np.all(kc[i, h, n:] == 0)
    assert [fp8.block_scale(a) for a in (448.0, 449.0, 224.0, 3.5, 3.51, 0.0)] == [1.0, 2.0, 0.5, 2.0 ** -7, 2.0 ** -6, 1.0]
    xd = fp8.dequantise_chunk(kc, ks, 37)
    assert xd.shape == x.shape
    assert np.array_equal(cs.bf16_bits_to_f64(cs.f32_to_bf16_bits(xd.astype(np.float32))), xd)   # bf16-exact
    # half a step: 2^-4 of the value for normals, half the subnormal spacing (2^-10 * 448 / amax ...) near zero
    step = np.maximum(np.abs(x) * 2.0 ** -4, ks.max() * 2.0 ** -10)
    assert np.all(np.abs(xd - x) <= step * 1.0001)
    z = np.zeros((5, 2, 128), np.uint16)
    zc, zs, _, _ = fp8.quantise_chunk(z, z)
    assert np.all(zc == 0) and np.all(zs == 1.0)


def test_fp8_attention_reduces_to_the_bf16_oracle_on_exactly_representable_chunks():
    """When every K/V element is +-448 * 2^-j-free, i.e. a small integer multiple of the block's amax / 448 that e4m3
    holds exactly, quantisation loses nothing and attention over the fp8 pages equals the C oracle over the bf16 chunks:
    pins oracle/fp8.attention_for (concatenation order, GQA map, softmax axis) to O1."""
    from oracle import fp8
    w = cs.custom("q8exact", k=7, num_q_heads=8, num_kv_heads=2, head_dim_qk=128, head_dim_v=128,
                  chunk_len=[40, 16, 23], links=[[2, 0], [1], [0, 1, 2]], lq=[3, 1, 2])
    exact_vals = np.array([0, 1, 2, 3, 4, 6, 8, 14, 16, -1, -2, -3, -5, -7, -12, 28], np.float32)   # x 1/16: all e4m3-exact

    class Exact:  # the workload with its chunks replaced (Workload is frozen: delegate everything else)
        def __getattr__(self, name):
            return getattr(w, name)

        def chunk_kv(self, c):
            rng = np.random.default_rng([11, int(c)])
            t = int(w.chunk_len[c])

            def draw(d):
                a = exact_vals[rng.integers(0, len(exact_vals), (t, 2, d))] / np.float32(16)
                a[:, :, 0] = np.float32(28.0 / 16)  # every block's amax is 28/16 = 448 / 256: scale = 2^-8 exactly
                return cs.f32_to_bf16_bits(a)
            return draw(128), draw(128)
    we = Exact()
    O8, L8 = fp8.attention_for(we)
    O, L = oracle.attention_for(we)
    assert np.abs(O8 - O).max() <= 1e-12 and np.abs(L8 - L).max() <= 1e-12
