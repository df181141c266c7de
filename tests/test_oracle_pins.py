"""Pins for the CPU oracle (oracle/sp_oracle.c) against things OTHER than itself: values the paper
prints, closed forms, invariants, library routines and a numpy brute force on tiny inputs.
Each pin is chosen so that a plausible slip (dropped term, wrong sign/index, transposed operand,
off-by-one in the causal bound, wrong head mean) fails at least one of them.  All CPU, no GPU."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import bruteforce as bf
from oracle import oracle as orc
from paper_2606_07703_b200 import inputs as gen

HERE = os.path.dirname(os.path.abspath(__file__))


def rand_bf16(seed, shape, sigma=1.0):
    rng = np.random.Generator(np.random.Philox(seed))
    return gen.f32_to_bf16((rng.standard_normal(shape) * sigma).astype(np.float32))


def small_problem(L=48, Hq=4, Hkv=2, d=8, k=6, b=1, seed=1, **kw):
    pb = orc.Problem(L=L, Hq=Hq, Hkv=Hkv, d=d, k=k, b_sel=b, **kw)
    Q = rand_bf16(seed, (L, Hq, d))
    K = rand_bf16(seed + 1, (L, Hkv, d))
    V = rand_bf16(seed + 2, (L, Hkv, d))
    return pb, Q, K, V


# ---------------------------------------------------------------- bf16 rounding (A14)

def test_bf16_rne_known_cases():
    x = np.array([1.0, 1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, 1.0 + 2.0 ** -8 + 2.0 ** -40,
                  -1.0 - 2.0 ** -8, 0.0, 3.140625, 2.0 ** -130, 1e39])
    want = np.array([1.0, 1.0, 1.015625, 1.0078125, -1.0, 0.0, 3.140625, 2.0 ** -130, np.inf])
    got = orc.bf16_to_f64(orc.f64_to_bf16(x))
    assert np.array_equal(got, want), (got, want)


def test_bf16_roundtrip_all_finite_patterns():
    b = np.arange(0, 0x7F80, dtype=np.uint16)  # all non-negative finite bf16
    assert np.array_equal(orc.f64_to_bf16(orc.bf16_to_f64(b)), b)
    # midpoint between consecutive values goes to the even pattern
    v = orc.bf16_to_f64(b)
    mid = (v[:-1] + v[1:]) / 2
    r = orc.f64_to_bf16(mid)
    even = np.where(b[:-1] % 2 == 0, b[:-1], b[1:])
    assert np.array_equal(r, even)


# ---------------------------------------------------------------- P3: the paper's own numbers

def kept_pairs(S, k):
    return k * S - k * (k - 1) // 2


def test_paper_printed_sparsities():
    n = 0
    for line in open(os.path.join(HERE, "golden", "paper_sparsity.txt")):
        if line.startswith("#") or not line.strip():
            continue
        S, k, printed, dec = line.split()[:4]
        S, k, dec = int(S), int(k), int(dec)
        sparsity = 100.0 * (1.0 - kept_pairs(S, k) / (S * (S + 1) / 2))
        assert round(sparsity, dec) == float(printed), (S, k, sparsity, printed)
        n += 1
    assert n == 5


@pytest.mark.parametrize("L,k", [(40, 7), (33, 33), (20, 64), (64, 1)])
def test_per_query_counts_match_paper_accounting(L, k):
    """Sum over per-query rows of cnt == k*L - k(k-1)/2 under readings A1/A3."""
    R = np.random.default_rng(0).standard_normal((L, L))
    nv = np.arange(1, L + 1)
    idx, cnt = orc.topk(R, nv, k)
    kk = min(k, L)
    assert int(cnt.sum()) == kept_pairs(L, kk)
    assert int((idx >= 0).sum()) == kept_pairs(L, kk)
    assert np.array_equal(cnt, np.minimum(k, nv))


def test_config1_pair_count():
    assert kept_pairs(1024, 256) == 229504 and 1024 * 1025 // 2 == 524800


# ---------------------------------------------------------------- P7: hand-worked case

def _golden_handworked():
    rec = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "handworked_L4.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            head, vals = line.split(":")
            name, row = head.split()
            rec.setdefault(name, {})[int(row)] = [Fraction(v) for v in vals.split()]
    return rec


def test_handworked_L4():
    """tests/golden/handworked_L4.txt: L=4, Hq=2, Hkv=1, d=1, q[t,0]=1, q[t,1]=0, k_s=s, scale=ln 2, v_s=s.
    Head 0 has logits s*ln2 -> weights 2^s; head 1 is uniform.  Exact rationals derived by hand from
    PAPER.md:94, :123 (P), :127/:107 (per-query k=2) and :154/:156 (block b=2 with per-query re-mask)."""
    G = _golden_handworked()
    one = gen.f32_to_bf16(np.array([1.0], np.float32))[0]
    Q = np.zeros((4, 2, 1), np.uint16)
    Q[:, 0, 0] = one
    K = gen.f32_to_bf16(np.arange(4, dtype=np.float32)).reshape(4, 1, 1)
    V = K.copy()
    pb = orc.Problem(L=4, Hq=2, Hkv=1, d=1, k=2, b_sel=1, scale=math.log(2.0))
    P = orc.query_scores(pb, orc.MODE_ORACLE, Q, K, np.arange(4))
    for t in range(4):
        assert np.allclose(P[t, :t + 1], [float(x) for x in G["P"][t]], rtol=0, atol=1e-15)
        assert np.all(np.isneginf(P[t, t + 1:]))
    res = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V)
    assert res.idx.tolist() == [[int(x) for x in G["idx_k2"][t]] for t in range(4)]
    assert res.cnt.tolist() == [1, 2, 2, 2]
    want_o = np.array([[float(x) for x in G["o_k2"][t]] for t in range(4)])
    assert np.allclose(res.out[:, :, 0], want_o, rtol=0, atol=1e-14)
    # block-shared
    pbb = orc.Problem(L=4, Hq=2, Hkv=1, d=1, k=2, b_sel=2, scale=math.log(2.0))
    R, nv = orc.support_scores(pbb, orc.MODE_ORACLE, Q, K, [0, 1])
    assert nv.tolist() == [2, 4]
    assert np.allclose(R[1], [float(x) for x in G["R_b2"][1]], atol=1e-15)
    assert np.allclose(R[0, :2], [float(x) for x in G["R_b2"][0]], atol=1e-15) and np.all(np.isneginf(R[0, 2:]))
    resb = orc.prefill_layer(pbb, orc.MODE_ORACLE, Q, K, V)
    assert resb.idx.tolist() == [[int(x) for x in G["idx_b2"][r]] for r in range(2)]
    want_ob = np.array([[float(x) for x in G["o_b2"][t]] for t in range(4)])
    assert np.allclose(resb.out[:, :, 0], want_ob, rtol=0, atol=1e-14)
    # k=1: the mass is increasing in s for both heads, so S_t={t} and o[t]=v_t=t
    pb1 = orc.Problem(L=4, Hq=2, Hkv=1, d=1, k=1, b_sel=1, scale=math.log(2.0))
    r1 = orc.prefill_layer(pb1, orc.MODE_ORACLE, Q, K, V)
    assert r1.idx[:, 0].tolist() == [0, 1, 2, 3]
    assert np.allclose(r1.out[:, :, 0], np.arange(4)[:, None], atol=1e-15)


# ---------------------------------------------------------------- P1: mass invariants

def test_mass_rows_sum_to_one_and_nonneg():
    pb, Q, K, V = small_problem(L=96, Hq=8, Hkv=2, d=16)
    P = orc.query_scores(pb, orc.MODE_ORACLE, Q, K, np.arange(pb.L))
    for t in range(pb.L):
        assert abs(P[t, :t + 1].sum() - 1.0) < 1e-12
        assert (P[t, :t + 1] >= 0).all()
        assert np.all(np.isneginf(P[t, t + 1:]))


def test_mass_head_permutation_within_groups():
    pb, Q, K, V = small_problem(L=40, Hq=8, Hkv=2, d=8)
    P0 = orc.query_scores(pb, orc.MODE_ORACLE, Q, K, np.arange(pb.L))
    perm = [3, 1, 0, 2, 5, 7, 6, 4]                          # stays inside each KV group of 4
    P1 = orc.query_scores(pb, orc.MODE_ORACLE, Q[:, perm], K, np.arange(pb.L))
    fin = np.isfinite(P0)
    assert np.allclose(P0[fin], P1[fin], rtol=0, atol=1e-15)
    # swapping whole groups together with their KV heads
    gperm = [4, 5, 6, 7, 0, 1, 2, 3]
    P2 = orc.query_scores(pb, orc.MODE_ORACLE, Q[:, gperm], K[:, [1, 0]], np.arange(pb.L))
    assert np.allclose(P0[fin], P2[fin], rtol=0, atol=1e-15)


def test_identical_heads_give_that_heads_softmax():
    from scipy.special import softmax
    L, d = 32, 8
    q1 = rand_bf16(5, (L, 1, d))
    K = rand_bf16(6, (L, 1, d))
    Q = np.repeat(q1, 4, axis=1)
    pb = orc.Problem(L=L, Hq=4, Hkv=1, d=d, k=4)
    P = orc.query_scores(pb, orc.MODE_ORACLE, Q, K, np.arange(L))
    z = (orc.bf16_to_f64(q1)[:, 0] @ orc.bf16_to_f64(K)[:, 0].T) / math.sqrt(d)
    for t in range(L):
        assert np.allclose(P[t, :t + 1], softmax(z[t, :t + 1]), rtol=1e-13, atol=0)


def test_gqa_equals_mha_with_repeated_kv():
    pb, Q, K, V = small_problem(L=40, Hq=8, Hkv=2, d=8, k=5)
    pm = orc.Problem(L=40, Hq=8, Hkv=8, d=8, k=5)
    Kr, Vr = np.repeat(K, 4, axis=1), np.repeat(V, 4, axis=1)
    a = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V)
    b = orc.prefill_layer(pm, orc.MODE_ORACLE, Q, Kr, Vr)
    assert np.array_equal(a.idx, b.idx)
    assert np.allclose(a.out, b.out, rtol=0, atol=1e-15)
    # a WRONG group map (interleaved instead of contiguous, A5) must be visible on this input
    Ki = np.tile(K, (1, 4, 1))
    c = orc.query_scores(pm, orc.MODE_ORACLE, Q, Ki, np.arange(40))
    fin = np.isfinite(a.scores)
    assert np.abs(c[fin] - a.scores[fin]).max() > 1e-3


# ---------------------------------------------------------------- P2 / P8: top-k

@pytest.mark.parametrize("seed", range(4))
def test_topk_matches_stable_argsort(seed):
    rng = np.random.default_rng(seed)
    rows, ld, k = 17, 70, 9
    R = rng.standard_normal((rows, ld))
    R = np.round(R * 4) / 4                                   # many exact ties
    nv = rng.integers(1, ld + 1, size=rows)
    idx, cnt = orc.topk(R, nv, k)
    for r in range(rows):
        n = int(nv[r])
        want = np.sort(np.argsort(-R[r, :n], kind="stable")[:k])
        got = idx[r][idx[r] >= 0]
        assert np.array_equal(got, want)
        assert cnt[r] == min(k, n) == len(got)
        assert np.all(idx[r, cnt[r]:] == -1)
        assert np.all(np.diff(got) > 0) and (len(got) == 0 or got[-1] < n)


def test_topk_ties_go_to_lower_index():
    R = np.zeros((1, 10))
    idx, cnt = orc.topk(R, [10], 4)
    assert idx[0].tolist() == [0, 1, 2, 3]
    R[0, [7, 2]] = 1.0
    R[0, [5, 9, 1]] = 0.5
    idx, _ = orc.topk(R, [10], 3)
    assert idx[0].tolist() == [1, 2, 7]                       # 2,7 (=1.0) then the lowest of the 0.5s
    idx, _ = orc.topk(R, [10], 3, seq_start=[100])
    assert idx[0].tolist() == [101, 102, 107]


def test_duplicate_keys_resolve_to_lower_index():
    pb, Q, K, V = small_problem(L=24, Hq=4, Hkv=2, d=8, k=3)
    K[10] = K[4]
    K[17] = K[4]
    res = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V, rows=[23], pos=[23])
    P = res.scores[0]
    assert P[4] == P[10] == P[17]
    sel = res.idx[0].tolist()
    if 10 in sel:
        assert 4 in sel
    if 17 in sel:
        assert 4 in sel and 10 in sel


# ---------------------------------------------------------------- P6: closed forms

def test_q_zero_closed_form():
    L, Hq, Hkv, d, k = 20, 4, 2, 8, 5
    Q = np.zeros((L, Hq, d), np.uint16)
    K = rand_bf16(2, (L, Hkv, d))
    V = rand_bf16(3, (L, Hkv, d))
    pb = orc.Problem(L=L, Hq=Hq, Hkv=Hkv, d=d, k=k)
    res = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V)
    v = orc.bf16_to_f64(V)
    for t in range(L):
        assert np.allclose(res.scores[t, :t + 1], 1.0 / (t + 1), rtol=1e-15)
        m = min(k, t + 1)
        assert res.idx[t, :m].tolist() == list(range(m))      # all ties -> lowest indices
        for h in range(Hq):
            assert np.allclose(res.out[t, h], v[:m, h // 2].mean(axis=0), rtol=0, atol=1e-15)


def test_rank_one_logits_pick_topk_of_key_scalars():
    """d=1 effective: all q positive -> every head's softmax is increasing in the key scalar, so the
    support is the top-k of the key scalars over the prefix."""
    L, k = 30, 4
    Q = gen.f32_to_bf16(np.full((L, 2, 1), 1.5, np.float32))
    ks = np.random.default_rng(3).permutation(L).astype(np.float32) / 8
    K = gen.f32_to_bf16(ks).reshape(L, 1, 1)
    pb = orc.Problem(L=L, Hq=2, Hkv=1, d=1, k=k)
    R, nv, idx, cnt = orc.select_support(pb, orc.MODE_ORACLE, Q, K, np.arange(L))
    for t in range(L):
        want = np.sort(np.argsort(-ks[:t + 1], kind="stable")[:k])
        assert idx[t][idx[t] >= 0].tolist() == want.tolist()


# ---------------------------------------------------------------- P4: sparse == dense when k >= n; O7 vs SDPA

def test_sparse_equals_dense_when_budget_covers_prefix():
    pb, Q, K, V = small_problem(L=50, Hq=4, Hkv=2, d=8, k=50, local_window=5, local_bias=0.7)
    res = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V)
    o_d, lse_d = orc.dense_attn(pb, Q, K, V, np.arange(50), want_lse=True)
    assert np.allclose(res.out, o_d, rtol=0, atol=1e-14)
    sup = np.stack([res.idx[t] for t in range(50)])
    _, lse_s = orc.sparse_attn(pb, Q, K, V, np.arange(50), sup, want_lse=True)
    assert np.allclose(lse_s, lse_d, rtol=0, atol=1e-13)


def test_dense_matches_torch_sdpa():
    import torch
    pb, Q, K, V = small_problem(L=37, Hq=6, Hkv=2, d=16, k=4)
    o = orc.dense_attn(pb, Q, K, V, np.arange(37))
    q = torch.from_numpy(orc.bf16_to_f64(Q)).permute(1, 0, 2)[None]
    k = torch.from_numpy(np.repeat(orc.bf16_to_f64(K), 3, axis=1)).permute(1, 0, 2)[None]
    v = torch.from_numpy(np.repeat(orc.bf16_to_f64(V), 3, axis=1)).permute(1, 0, 2)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(q, k, v, is_causal=True)[0].permute(1, 0, 2).numpy()
    assert np.allclose(o, ref, rtol=0, atol=1e-13)


# ---------------------------------------------------------------- P5: block rule

def test_block_rule_properties():
    pb1, Q, K, V = small_problem(L=45, Hq=4, Hkv=2, d=8, k=6, b=1)
    pbb = orc.Problem(L=45, Hq=4, Hkv=2, d=8, k=6, b_sel=8)
    P, _ = orc.support_scores(pb1, orc.MODE_ORACLE, Q, K, np.arange(45))
    P2 = orc.query_scores(pb1, orc.MODE_ORACLE, Q, K, np.arange(45))
    assert np.array_equal(P, P2)                              # b_sel=1 block rule == per-query
    assert orc.num_rows(pbb) == 6
    R, nv = orc.support_scores(pbb, orc.MODE_ORACLE, Q, K, np.arange(6))
    assert nv.tolist() == [8, 16, 24, 32, 40, 45]             # last block ragged (A8)
    for j in range(6):
        t0, t1 = j * 8, min(44, j * 8 + 7)
        assert np.all(np.isneginf(R[j, t1 + 1:]))
        for t in range(t0, t1 + 1):
            assert np.all(R[j, :t + 1] >= P[t, :t + 1])
        want = np.max(np.where(np.isfinite(P[t0:t1 + 1]), P[t0:t1 + 1], -np.inf), axis=0)
        assert np.array_equal(R[j, :t1 + 1], want[:t1 + 1])
    res = orc.prefill_layer(pbb, orc.MODE_ORACLE, Q, K, V)
    for j in range(6):
        sel = res.idx[j][res.idx[j] >= 0]
        assert sel.max() <= min(44, j * 8 + 7)


# ---------------------------------------------------------------- brute force on tiny inputs (both modes)

@pytest.mark.parametrize("b,lw", [(1, 0), (4, 0), (1, 3), (8, 5)])
def test_oracle_mode_matches_numpy_bruteforce(b, lw):
    L, Hq, Hkv, d, k = 37, 4, 2, 8, 5
    pb, Q, K, V = small_problem(L=L, Hq=Hq, Hkv=Hkv, d=d, k=k, b=b, seed=11 + b,
                                local_window=lw, local_bias=0.9 if lw else 0.0)
    res = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V)
    kw = dict(local_window=lw, local_bias=0.9 if lw else 0.0)
    P = bf.mass(Q, K, 1 / math.sqrt(d), Hq // Hkv, **kw)
    R, nv = bf.support_rows(P, b)
    assert np.array_equal(nv, res.n_valid)
    fin = np.isfinite(res.scores)
    assert np.array_equal(fin, np.isfinite(R))
    assert np.allclose(res.scores[fin], R[fin], rtol=1e-12, atol=0)
    idx = bf.topk_rows(R, nv, k)
    assert np.array_equal(idx, res.idx)
    o = bf.sparse_attention(Q, K, V, 1 / math.sqrt(d), Hq // Hkv, idx, b, **kw)
    assert np.allclose(res.out, o, rtol=0, atol=1e-13)


@pytest.mark.parametrize("b,lw", [(1, 0), (4, 2)])
def test_indexer_mode_matches_numpy_bruteforce(b, lw):
    L, Hq, Hkv, d, k, hid, di = 33, 4, 2, 8, 6, 24, 8
    pb, Q, K, V = small_problem(L=L, Hq=Hq, Hkv=Hkv, d=d, k=k, b=b, seed=21, hidden=hid, d_idx=di,
                                local_window=lw, local_bias=-0.6 if lw else 0.0)
    X = rand_bf16(31, (L, hid))
    Wq = rand_bf16(32, (hid, di), 1 / math.sqrt(hid))
    Wk = rand_bf16(33, (hid, di), 1 / math.sqrt(hid))
    res = orc.prefill_layer(pb, orc.MODE_INDEXER, Q, K, V, X, Wq, Wk)
    # projection: fp64 matmul (library) then one RNE rounding; compare as values, allow a tie-flip nowhere
    pq = orc.bf16_to_f64(X) @ orc.bf16_to_f64(Wq)
    got = orc.bf16_to_f64(res.q_idx)
    assert np.all(np.abs(got - pq) <= np.abs(pq) * 2.0 ** -8 + 1e-300)       # within half an ulp (8 sig. bits)
    import torch
    tq = torch.from_numpy(pq).to(torch.bfloat16).to(torch.float64).numpy()
    assert (tq != got).mean() < 1e-3                                          # library cast agrees (bar double rounding)
    kw = dict(local_window=lw, local_bias=-0.6 if lw else 0.0)
    z = bf.indexer_logits(res.q_idx, res.k_idx, 1 / math.sqrt(di), **kw)
    R, nv = bf.support_rows(z, b)
    fin = np.isfinite(R)
    assert np.array_equal(fin, np.isfinite(res.scores))
    assert np.allclose(res.scores[fin], R[fin], rtol=1e-12, atol=1e-13)
    idx = bf.topk_rows(R, nv, k)
    assert np.array_equal(idx, res.idx)
    o = bf.sparse_attention(Q, K, V, 1 / math.sqrt(d), Hq // Hkv, idx, b, **kw)
    assert np.allclose(res.out, o, rtol=0, atol=1e-13)


# ---------------------------------------------------------------- P9: varlen

@pytest.mark.parametrize("mode", [orc.MODE_ORACLE, orc.MODE_INDEXER])
def test_varlen_pack_equals_separate_sequences(mode):
    lens = [19, 8, 30, 5]
    cu = np.concatenate([[0], np.cumsum(lens)])
    L, Hq, Hkv, d, k, b, hid, di = int(cu[-1]), 4, 2, 8, 6, 8, 16, 8
    Q, K, V = rand_bf16(1, (L, Hq, d)), rand_bf16(2, (L, Hkv, d)), rand_bf16(3, (L, Hkv, d))
    X = rand_bf16(4, (L, hid))
    Wq, Wk = rand_bf16(5, (hid, di), 0.25), rand_bf16(6, (hid, di), 0.25)
    kw = dict(Hq=Hq, Hkv=Hkv, d=d, k=k, b_sel=b, hidden=hid, d_idx=di, local_window=3, local_bias=0.5)
    pk = orc.Problem(L=L, cu_seqlens=cu, **kw)
    packed = orc.prefill_layer(pk, mode, Q, K, V, X, Wq, Wk)
    assert orc.num_rows(pk) == sum((n + b - 1) // b for n in lens) == len(packed.idx)
    r0 = 0
    for i, n in enumerate(lens):
        s, e = int(cu[i]), int(cu[i + 1])
        one = orc.prefill_layer(orc.Problem(L=n, **kw), mode, Q[s:e], K[s:e], V[s:e], X[s:e], Wq, Wk)
        nr = len(one.idx)
        shifted = np.where(one.idx >= 0, one.idx + s, -1)
        assert np.array_equal(packed.idx[r0:r0 + nr], shifted)
        assert np.array_equal(packed.cnt[r0:r0 + nr], one.cnt)
        assert np.allclose(packed.out[s:e], one.out, rtol=0, atol=1e-15)
        r0 += nr


def test_empty_effective_support_gives_zero_output():
    """k < b_sel: the first queries of a block may see none of the block's support (A9)."""
    pb, Q, K, V = small_problem(L=16, Hq=2, Hkv=1, d=4, k=1, b=8)
    res = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V)
    for t in range(16):
        s = res.idx[t // 8, 0]
        if s > t:
            assert np.all(res.out[t] == 0.0)
    sup = np.full((1, 1), 9, np.int32)
    o, lse = orc.sparse_attn(pb, Q, K, V, [3], sup, want_lse=True)
    assert np.all(o == 0) and np.all(np.isneginf(lse))


# ------------------------------------------------------------------ served scorer: key LayerNorm, RoPE, ReLU
# (readings A26-A28 of DESIGN.md).  Pins on the fp64 core orc_transform and on the chain.

def test_served_scorer_layernorm_closed_form():
    rng = np.random.Generator(np.random.Philox(77))
    y = rng.standard_normal(64) * 3.0 + 1.5
    z = orc.transform(y, pos_local=5, flags=orc.F_KEY_LN, key=True)
    assert abs(z.mean()) < 1e-12
    assert abs(z.var() - y.var() / (y.var() + 1e-6)) < 1e-12          # biased variance, eps = 1e-6, no affine
    assert np.allclose(z, (y - y.mean()) / np.sqrt(y.var() + 1e-6), rtol=0, atol=1e-12)
    # the query side is never normalised; a constant key row maps to 0
    assert np.array_equal(orc.transform(y, 5, orc.F_KEY_LN, key=False), y)
    assert np.allclose(orc.transform(np.full(16, 2.5), 3, orc.F_KEY_LN, key=True), 0.0, atol=1e-9)


def test_served_scorer_rope_closed_forms():
    rng = np.random.Generator(np.random.Philox(78))
    d = 32
    q, k = rng.standard_normal(d), rng.standard_normal(d)
    # position 0 is the identity; every position preserves the norm of each (i, i + d/2) pair
    assert np.array_equal(orc.transform(q, 0, orc.F_ROPE, key=False), q)
    for pos in (1, 17, 4096, 131071):
        r = orc.transform(q, pos, orc.F_ROPE, key=False)
        assert np.allclose(r[:d // 2] ** 2 + r[d // 2:] ** 2, q[:d // 2] ** 2 + q[d // 2:] ** 2, rtol=1e-12)
    # d = 2: theta_0 = pos, (1, 0) -> (cos pos, sin pos)
    for pos in (1, 2, 100):
        assert np.allclose(orc.transform(np.array([1.0, 0.0]), pos, orc.F_ROPE, key=True), [math.cos(pos), math.sin(pos)],
                           atol=1e-12)
    # frequencies: pair i turns by pos * 10000^(-2i/d)
    e = np.zeros(d); e[3] = 1.0
    r = orc.transform(e, 7, orc.F_ROPE, key=False)
    th = 7 * 10000.0 ** (-2 * 3 / d)
    assert np.allclose([r[3], r[3 + d // 2]], [math.cos(th), math.sin(th)], atol=1e-12)
    # relative-position property: <R_t q, R_s k> depends on t - s only
    a = orc.transform(q, 900, orc.F_ROPE, False) @ orc.transform(k, 650, orc.F_ROPE, True)
    b = orc.transform(q, 300, orc.F_ROPE, False) @ orc.transform(k, 50, orc.F_ROPE, True)
    assert abs(a - b) < 1e-9
    # LayerNorm is applied BEFORE the rotation on the key side
    both = orc.transform(k, 11, orc.F_KEY_LN | orc.F_ROPE, key=True)
    assert np.allclose(both, orc.transform(orc.transform(k, 11, orc.F_KEY_LN, True), 11, orc.F_ROPE, True), atol=1e-12)


def test_served_scorer_projection_uses_local_positions_and_rounds_once():
    rng = np.random.Generator(np.random.Philox(79))
    L, hid, di = 24, 32, 16
    X = orc.f64_to_bf16(rng.standard_normal((L, hid)))
    W = orc.f64_to_bf16(rng.standard_normal((hid, di)) / math.sqrt(hid))
    cu = (0, 10, 24)
    pb = orc.Problem(L=L, Hq=2, Hkv=1, d=8, k=4, hidden=hid, d_idx=di, cu_seqlens=cu,
                     flags=orc.F_KEY_LN | orc.F_ROPE)
    got = orc.project(pb, X, W, key=True)
    y = orc.bf16_to_f64(X) @ orc.bf16_to_f64(W)                        # exact products, fp64 sum
    for t in range(L):
        local = t - (0 if t < 10 else 10)
        want = orc.f64_to_bf16(orc.transform(y[t], local, pb.flags, key=True))
        assert np.array_equal(got[t], want), t
    # flags == 0 is the plain projection
    pb0 = orc.Problem(L=L, Hq=2, Hkv=1, d=8, k=4, hidden=hid, d_idx=di)
    assert np.array_equal(orc.project(pb0, X, W, key=True), orc.f64_to_bf16(y))


def test_served_scorer_relu_and_zero_ties():
    rng = np.random.Generator(np.random.Philox(80))
    L, di, k = 40, 8, 6
    q = orc.f64_to_bf16(rng.standard_normal((L, di)))
    kk = orc.f64_to_bf16(rng.standard_normal((L, di)))
    pb0 = orc.Problem(L=L, Hq=2, Hkv=1, d=8, k=k, hidden=16, d_idx=di, local_window=3, local_bias=-0.25)
    pb1 = orc.Problem(L=L, Hq=2, Hkv=1, d=8, k=k, hidden=16, d_idx=di, local_window=3, local_bias=-0.25,
                      flags=orc.F_RELU)
    pos = np.arange(L)
    z0 = orc.query_scores(pb0, orc.MODE_INDEXER, q, kk, pos)
    z1 = orc.query_scores(pb1, orc.MODE_INDEXER, q, kk, pos)
    fin = np.isfinite(z0)
    assert np.array_equal(np.isfinite(z1), fin)
    assert np.array_equal(z1[fin], np.maximum(z0[fin], 0.0))          # ReLU on the final logit (A26)
    # a query whose logits are all negative: every score is 0, ties -> the lowest indices fill the budget (A11)
    qn = q.copy(); kn = kk.copy()
    qn[:] = orc.f64_to_bf16(np.ones((L, di))); kn[:] = orc.f64_to_bf16(-np.ones((L, di)))
    pb2 = orc.Problem(L=L, Hq=2, Hkv=1, d=8, k=k, hidden=16, d_idx=di, flags=orc.F_RELU)
    R, nv = orc.support_scores(pb2, orc.MODE_INDEXER, qn, kn, np.arange(L))
    idx, cnt = orc.topk(R, nv, k)
    for t in range(k, L):
        assert np.array_equal(idx[t], np.arange(k)), t


# ------------------------------------------------------------------ support-level diagnostics

def test_support_overlap_pins():
    a = np.array([[0, 2, 5, 9], [1, 3, -1, -1], [4, 5, 6, 7]], dtype=np.int32)
    b = np.array([[2, 3, 9, 11], [0, 2, 4, -1], [4, 5, 6, 7]], dtype=np.int32)
    assert orc.support_overlap(a, b).tolist() == [2, 0, 4]
    assert orc.support_overlap(a, a).tolist() == [4, 2, 4]            # a support recovers itself; padding is ignored
    rng = np.random.Generator(np.random.Philox(5))
    x = np.sort(rng.permutation(200)[:50]); y = np.sort(rng.permutation(200)[:70])
    assert orc.support_overlap(x[None], y[None])[0] == len(np.intersect1d(x, y))


def test_row_kl_pins():
    rng = np.random.Generator(np.random.Philox(6))
    n = 37
    z = rng.standard_normal((3, 64))
    nv = np.array([n, 5, 64])
    sm = np.zeros_like(z)
    for r in range(3):
        e = np.exp(z[r, :nv[r]] - z[r, :nv[r]].max()); sm[r, :nv[r]] = e / e.sum()
    assert np.allclose(orc.row_kl(sm, z, nv), 0.0, atol=1e-12)         # KL(p || p) = 0
    assert np.allclose(orc.row_kl(sm, z + 3.25, nv), 0.0, atol=1e-12)  # softmax is shift invariant
    # uniform student: KL(P || U_n) = log n - H(P)
    P = sm[0:1]; H = -(P[0, :n] * np.log(P[0, :n])).sum()
    assert abs(orc.row_kl(P, np.zeros((1, 64)), nv[:1])[0] - (math.log(n) - H)) < 1e-12
    # one-hot teacher: KL = -log softmax(z)[j]; non-negative in general (Gibbs)
    oh = np.zeros((1, 64)); oh[0, 3] = 1.0
    assert abs(orc.row_kl(oh, z[0:1], nv[:1])[0] + math.log(sm[0, 3])) < 1e-12
    Q = rng.random((4, 64)); Q[:, 40:] = 0; Q /= Q.sum(1, keepdims=True)
    assert np.all(orc.row_kl(Q, rng.standard_normal((4, 64)), np.full(4, 40)) >= 0)


# ---------------------------------------------------------------- per-KV-group support (A29)
# the head-axis variants of the support

def _group_bruteforce(pb, Q, K, V, b):
    """Independent of oracle.py's slicing: dense [Hq, L, L] probabilities, mean over each group's heads."""
    from scipy.special import softmax
    G = pb.Hq // pb.Hkv
    z = bf.logits(Q, K, 1.0 / math.sqrt(pb.d), G)                       # [Hq, L, L]
    A = softmax(z, axis=-1)
    P = A.reshape(pb.Hkv, G, pb.L, pb.L).mean(axis=1)                   # contiguous groups (A5)
    idx = []
    for r in range(pb.Hkv):
        R, nv = bf.support_rows(P[r], b)
        idx.append(bf.topk_rows(R, nv, pb.k))
    idx = np.stack(idx)                                                 # [Hkv, rows, k]
    v = np.repeat(bf.bf16_to_f64(V), G, axis=1)
    out = np.zeros((pb.L, pb.Hq, pb.d))
    for h in range(pb.Hq):
        for t in range(pb.L):
            s = idx[h // G, t // b]
            s = s[(s >= 0) & (s <= t)]
            if len(s):
                out[t, h] = softmax(z[h, t, s]) @ v[s, h]
    return idx, out


@pytest.mark.parametrize("b", [1, 4])
def test_per_group_support_matches_bruteforce(b):
    pb, Q, K, V = small_problem(L=37, Hq=6, Hkv=3, d=8, k=5, b=b, seed=21)
    rows = np.arange(orc.num_rows(pb))
    idx, cnt = orc.select_support_per_group(pb, Q, K, rows)
    want_idx, want_out = _group_bruteforce(pb, Q, K, V, b)
    assert idx.shape == (3, len(rows), 5)
    assert np.array_equal(idx, want_idx)
    assert np.array_equal(cnt, (want_idx >= 0).sum(axis=-1))
    pos = np.arange(pb.L)
    sup = idx[:, pos // b, :]
    out = orc.sparse_attn_per_group(pb, Q, K, V, pos, sup)
    assert np.allclose(out, want_out, rtol=0, atol=1e-13)
    # the groups must really differ on this input, or the test would not see a wrong group map
    assert any(not np.array_equal(idx[0], idx[r]) for r in (1, 2))


def test_per_group_reduces_to_head_averaged_support():
    # one KV group: the group IS the head average (PAPER.md:100 third case)
    pb, Q, K, V = small_problem(L=40, Hq=4, Hkv=1, d=8, k=6, b=4, seed=31)
    rows = np.arange(orc.num_rows(pb))
    shared = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V)
    idx, cnt = orc.select_support_per_group(pb, Q, K, rows)
    assert np.array_equal(idx[0], shared.idx) and np.array_equal(cnt[0], shared.cnt)
    # identical groups: every group's mass equals the mean over all heads, so every list is the shared one
    pb2 = orc.Problem(L=40, Hq=8, Hkv=2, d=8, k=6, b_sel=4)
    Q2, K2, V2 = np.tile(Q, (1, 2, 1)), np.tile(K, (1, 2, 1)), np.tile(V, (1, 2, 1))
    shared2 = orc.prefill_layer(pb2, orc.MODE_ORACLE, Q2, K2, V2)
    idx2, _ = orc.select_support_per_group(pb2, Q2, K2, rows)
    assert np.array_equal(idx2[0], shared2.idx) and np.array_equal(idx2[1], shared2.idx)
    pos = shared2.pos
    out2 = orc.sparse_attn_per_group(pb2, Q2, K2, V2, pos, idx2[:, pos // 4, :])
    assert np.allclose(out2, shared2.out, rtol=0, atol=1e-14)


def test_per_group_equals_dense_when_budget_covers_prefix():
    pb, Q, K, V = small_problem(L=30, Hq=4, Hkv=2, d=8, k=30, seed=41)
    pos = np.arange(30)
    idx, _ = orc.select_support_per_group(pb, Q, K, pos)
    out = orc.sparse_attn_per_group(pb, Q, K, V, pos, idx)
    assert np.allclose(out, orc.dense_attn(pb, Q, K, V, pos), rtol=0, atol=1e-14)


# ---------------------------------------------------------------- per-head support ("separately per query head")

def _head_bruteforce(pb, Q, K, V, b):
    """Dense [Hq, L, L] probabilities; every head ranks ITS OWN rows (block max over the block's queries)."""
    from scipy.special import softmax
    G = pb.Hq // pb.Hkv
    z = bf.logits(Q, K, 1.0 / math.sqrt(pb.d), G)                       # [Hq, L, L]
    A = softmax(z, axis=-1)
    idx = []
    for h in range(pb.Hq):
        R, nv = bf.support_rows(A[h], b)
        idx.append(bf.topk_rows(R, nv, pb.k))
    idx = np.stack(idx)                                                 # [Hq, rows, k]
    v = np.repeat(bf.bf16_to_f64(V), G, axis=1)
    out = np.zeros((pb.L, pb.Hq, pb.d))
    for h in range(pb.Hq):
        for t in range(pb.L):
            s = idx[h, t // b]
            s = s[(s >= 0) & (s <= t)]
            if len(s):
                out[t, h] = softmax(z[h, t, s]) @ v[s, h]
    return idx, out


@pytest.mark.parametrize("b", [1, 4])
def test_per_head_support_matches_bruteforce(b):
    pb, Q, K, V = small_problem(L=37, Hq=6, Hkv=3, d=8, k=5, b=b, seed=51)
    rows = np.arange(orc.num_rows(pb))
    idx, cnt = orc.select_support_per_head(pb, Q, K, rows)
    want_idx, want_out = _head_bruteforce(pb, Q, K, V, b)
    assert idx.shape == (6, len(rows), 5)
    assert np.array_equal(idx, want_idx)
    assert np.array_equal(cnt, (want_idx >= 0).sum(axis=-1))
    pos = np.arange(pb.L)
    out = orc.sparse_attn_per_head(pb, Q, K, V, pos, idx[:, pos // b, :])
    assert np.allclose(out, want_out, rtol=0, atol=1e-13)
    # two heads of the SAME KV group must differ here, or a head -> group mix-up would go unseen
    assert not np.array_equal(idx[0], idx[1])


def test_per_head_reductions():
    # G = 1: a head is its KV group (the three granularities coincide for MHA with one head per group)
    pb, Q, K, V = small_problem(L=33, Hq=3, Hkv=3, d=8, k=6, b=2, seed=61)
    rows = np.arange(orc.num_rows(pb))
    ih, ch = orc.select_support_per_head(pb, Q, K, rows)
    ig, cg = orc.select_support_per_group(pb, Q, K, rows)
    assert np.array_equal(ih, ig) and np.array_equal(ch, cg)
    # identical heads inside a group: every head's distribution equals the group mean, so head lists == group lists
    pb2 = orc.Problem(L=33, Hq=6, Hkv=3, d=8, k=6, b_sel=2)
    Q2 = np.repeat(Q, 2, axis=1)
    ih2, _ = orc.select_support_per_head(pb2, Q2, K, rows)
    ig2, _ = orc.select_support_per_group(pb2, Q2, K, rows)
    for h in range(6):
        assert np.array_equal(ih2[h], ig2[h // 2])
    # k >= n: every list is the whole prefix, the recompute is dense attention
    pb3, Q3, K3, V3 = small_problem(L=20, Hq=4, Hkv=2, d=8, k=20, seed=71)
    pos = np.arange(20)
    i3, _ = orc.select_support_per_head(pb3, Q3, K3, pos)
    assert np.allclose(orc.sparse_attn_per_head(pb3, Q3, K3, V3, pos, i3), orc.dense_attn(pb3, Q3, K3, V3, pos), rtol=0, atol=1e-14)


# ---------------------------------------------------------------- paged KV cache / chunked prefill

def make_cache(n_ctx, ps, Hkv, d, d_idx, seed, garbage=True):
    """An empty paged cache with a random block table; unused slots hold garbage so that a wrong page shows."""
    n_blocks = (n_ctx + ps - 1) // ps
    n_pages = n_blocks + 3
    rng = np.random.Generator(np.random.Philox(seed))
    bt = rng.permutation(n_pages)[:n_blocks].astype(np.int32)
    fill = (lambda shape: rng.integers(0, 65536, size=shape, dtype=np.uint16)) if garbage else (lambda shape: np.zeros(shape, np.uint16))
    return orc.PagedCache(page_size=ps, block_table=bt, k=fill((n_pages, ps, Hkv * d)), v=fill((n_pages, ps, Hkv * d)),
                          kidx=fill((n_pages, ps, d_idx)) if d_idx else None)


@pytest.mark.parametrize("ps", [1, 16, 64])
def test_paged_gather_scatter_are_pure_indexing(ps):
    n, row = 203, 24
    rng = np.random.Generator(np.random.Philox(ps))
    n_blocks = (n + ps - 1) // ps
    bt = rng.permutation(n_blocks + 2)[:n_blocks].astype(np.int32)
    cache = rng.integers(0, 65536, size=(n_blocks + 2, ps, row), dtype=np.uint16)
    t = np.arange(37, 181)
    want = cache[bt[t // ps], t % ps]                       # numpy fancy indexing: the definition
    assert np.array_equal(orc.paged_gather(cache, bt, ps, 37, 181), want)
    rows = rng.integers(0, 65536, size=(n, row), dtype=np.uint16)
    before = cache.copy()
    orc.paged_scatter(cache, bt, ps, 50, rows[50:120])
    assert np.array_equal(orc.paged_gather(cache, bt, ps, 50, 120), rows[50:120])    # scatter then gather == identity
    untouched = np.ones(cache.shape[:2], bool)
    tt = np.arange(50, 120)
    untouched[bt[tt // ps], tt % ps] = False
    assert np.array_equal(cache[untouched], before[untouched])                       # and nothing else was written


@pytest.mark.parametrize("mode,b,ps,chunk,flags", [
    (orc.MODE_ORACLE, 1, 16, 32, 0), (orc.MODE_ORACLE, 8, 16, 40, 0),
    (orc.MODE_INDEXER, 1, 64, 48, 0), (orc.MODE_INDEXER, 8, 16, 24, 0),
    (orc.MODE_INDEXER, 8, 32, 56, orc.F_RELU | orc.F_KEY_LN | orc.F_ROPE),
])
def test_chunked_paged_prefill_equals_full_prefill(mode, b, ps, chunk, flags):
    """Chunks of `chunk` queries, each attending the paged cache of everything before it plus itself, reproduce the
    full-prefill supports and outputs BIT FOR BIT (the reconstruction is pure indexing; ragged last chunk and page)."""
    L, Hq, Hkv, d, k, hid, di = 117, 4, 2, 8, 9, 16, 8
    pb = orc.Problem(L=L, Hq=Hq, Hkv=Hkv, d=d, k=k, b_sel=b, hidden=hid, d_idx=di, local_window=5, local_bias=0.5,
                     flags=flags)
    Q, K, V = rand_bf16(11, (L, Hq, d)), rand_bf16(12, (L, Hkv, d)), rand_bf16(13, (L, Hkv, d))
    X, Wq, Wk = rand_bf16(14, (L, hid)), rand_bf16(15, (hid, di), 0.25), rand_bf16(16, (hid, di), 0.25)
    full = orc.prefill_layer(pb, mode, Q, K, V, X, Wq, Wk)
    outs = {}
    for seed in (1, 2):                                   # two different block tables: the layout must not matter
        cache = make_cache(L, ps, Hkv, d, di, seed)
        idx_rows, out_rows = [], []
        for q0 in range(0, L, chunk):
            qc = min(chunk, L - q0)
            pc = orc.Problem(L=q0 + qc, Hq=Hq, Hkv=Hkv, d=d, k=k, b_sel=b, hidden=hid, d_idx=di, local_window=5,
                             local_bias=0.5, flags=flags)
            res = orc.prefill_chunk(pc, mode, q0, qc, Q[q0:q0 + qc], K[q0:q0 + qc], V[q0:q0 + qc], cache,
                                    X[q0:q0 + qc], Wq, Wk)
            assert res.rows[0] == q0 // b and np.array_equal(res.pos, np.arange(q0, q0 + qc))
            idx_rows.append(res.idx)
            out_rows.append(res.out)
        idx = np.concatenate(idx_rows)
        out = np.concatenate(out_rows)
        assert np.array_equal(idx, full.idx)
        assert np.array_equal(out, full.out)              # bit-identical fp64
        outs[seed] = out
    assert np.array_equal(outs[1], outs[2])


def test_chunked_prefill_reads_the_cache_not_the_chunk_only():
    """Negative control: a chunk evaluated WITHOUT its prefix in the cache (garbage pages) must differ."""
    L, Hq, Hkv, d, k = 64, 2, 1, 8, 6
    pb = orc.Problem(L=L, Hq=Hq, Hkv=Hkv, d=d, k=k, b_sel=1)
    Q, K, V = rand_bf16(21, (L, Hq, d)), rand_bf16(22, (L, Hkv, d)), rand_bf16(23, (L, Hkv, d))
    full = orc.prefill_layer(pb, orc.MODE_ORACLE, Q, K, V)
    cache = make_cache(L, 16, Hkv, d, 0, 5, garbage=False)         # prefix never written: zeros
    res = orc.prefill_chunk(pb, orc.MODE_ORACLE, 32, 32, Q[32:], K[32:], V[32:], cache)
    assert not np.array_equal(res.out, full.out[32:])
