"""Pins of the CPU oracle against things other than itself (run with -m "not gpu").

Every oracle function is checked against what the paper and the mathematics fix: the paper's
counting examples (tests/golden/paper_counts.txt), closed forms, invariants, special cases that
reduce to a library routine (torch SDPA, numpy sort) and brute force written independently here
in numpy float64.  Nothing below imports the CUDA path.
"""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2605_30519_b200 import synth


def bf16(x):
    return torch.from_numpy(np.asarray(x, np.float32)).to(torch.bfloat16).to(torch.float32).numpy()


def build_cache(w, data, page_map=None, chunked=True):
    c = oracle.cache_create(w.H, w.D, w.B, w.n_hist + w.S, page_map)
    step = w.chunk if chunked else w.n_hist
    for lo in range(0, w.n_hist, step):
        hi = min(lo + step, w.n_hist)
        oracle.append_chunk(c, data["k_hist"][:, lo:hi], data["v_hist"][:, lo:hi])
    oracle.pool_keys(c)
    return c


@pytest.fixture(scope="module")
def tiny():
    w = synth.config("tiny")
    d = synth.generate(w)
    return w, d, build_cache(w, d)


# ---------------------------------------------------------------------------------- helpers
def test_bf16_round_matches_library_cast():
    rng = np.random.default_rng(0)
    xs = np.concatenate([rng.standard_normal(2000).astype(np.float32) * 10.0 ** rng.integers(-6, 6, 2000),
                         np.float32([0.0, -0.0, 1.0, 1.00390625, 1.01171875, 3.3895314e38, 1e-40])])
    got = np.float32([oracle.bf16_round(float(x)) for x in xs])
    assert np.array_equal(got.view(np.uint32), bf16(xs).view(np.uint32))


# ---------------------------------------------------------------------------------- a0 append
def test_append_pages_roundtrip_and_zero_tail():
    H, D, B = 2, 8, 16
    rng = np.random.default_rng(1)
    pm = synth.permuted_page_map(H, 8, 3)
    c = oracle.cache_create(H, D, B, 8 * B, pm)
    c.k_pages[:] = 7.0  # garbage that a fresh page must not keep
    c.v_pages[:] = 7.0
    k = bf16(rng.standard_normal((H, 40, D)))
    v = bf16(rng.standard_normal((H, 40, D)))
    oracle.append_chunk(c, k[:, :25], v[:, :25])
    oracle.append_chunk(c, k[:, 25:], v[:, 25:])
    assert c.n_hist == 40
    for h in range(H):
        for t in range(40):
            assert np.array_equal(c.k_pages[h, pm[h, t // B], t % B], k[h, t])
            assert np.array_equal(c.v_pages[h, pm[h, t // B], t % B], v[h, t])
        assert np.all(c.k_pages[h, pm[h, 2], 8:] == 0.0)  # tail of the last (fresh) page is zero
        assert np.all(c.k_pages[h, pm[h, 5]] == 7.0)  # untouched pages stay untouched


# ---------------------------------------------------------------------------------- a1 pooling
def test_pool_constant_block_is_that_row():
    H, D, B = 1, 16, 64
    row = bf16(np.linspace(-3, 3, D))
    c = oracle.cache_create(H, D, B, 2 * B)
    oracle.append_chunk(c, np.tile(row, (H, 2 * B, 1)), np.zeros((H, 2 * B, D), np.float32))
    oracle.pool_keys(c)
    assert np.array_equal(c.pooled_k[0, 0], row) and np.array_equal(c.pooled_k[0, 1], row)


@pytest.mark.parametrize("B,n", [(64, 64), (64, 32), (64, 24), (128, 88), (128, 128)])
def test_pool_ramp_closed_form_and_ragged(B, n):
    # arithmetic ramp t*2^-4 (exact in bf16 for t < 256): mean over n tokens = (n-1)/2 * 2^-4
    D = 8
    c = oracle.cache_create(1, D, B, 2 * B)
    k = np.zeros((1, B + n, D), np.float32)
    k[0, B:, :] = (np.arange(n, dtype=np.float32) / 16.0)[:, None]
    k[0, :B, 3] = 1.0
    oracle.append_chunk(c, k, k)
    oracle.pool_keys(c)
    want = bf16(np.float32((n - 1) / 2.0 / 16.0))
    assert np.all(c.pooled_k[0, 1] == want)
    assert c.pooled_k[0, 0, 3] == 1.0 and c.pooled_k[0, 0, 0] == 0.0


def test_pool_brute_force_permuted_pages_and_order_invariance():
    w = synth.config("tiny", n_hist=2048 - 40)  # ragged last block of 24
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 5)
    c = build_cache(w, d, pm)
    k = d["k_hist"].astype(np.float64)
    for h in range(w.H):
        for b in range(w.n_b):
            blk = k[h, b * w.B:min((b + 1) * w.B, w.n_hist)]
            want = bf16((np.float32(blk.sum(0)) / np.float32(len(blk))).astype(np.float32))
            assert np.array_equal(c.pooled_k[h, b], want), (h, b)
    assert len(k[0, (w.n_b - 1) * w.B:w.n_hist]) == 24
    # Cor. 1: pooling is invariant to the token order inside a block
    rng = np.random.default_rng(2)
    d2 = dict(d)
    kh = d["k_hist"].copy()
    for b in range(w.n_b):
        lo, hi = b * w.B, min((b + 1) * w.B, w.n_hist)
        kh[:, lo:hi] = kh[:, lo + rng.permutation(hi - lo)]
    d2["k_hist"] = kh
    c2 = build_cache(w, d2, pm)
    assert np.array_equal(c.pooled_k, c2.pooled_k)


def test_pool_incremental_equals_full(tiny):
    w, d, c = tiny
    c2 = oracle.cache_create(w.H, w.D, w.B, w.n_hist + w.S)
    for lo in range(0, w.n_hist, 200):  # chunks that straddle blocks: dirty block is re-pooled
        hi = min(lo + 200, w.n_hist)
        first = c2.n_hist // w.B
        oracle.append_chunk(c2, d["k_hist"][:, lo:hi], d["v_hist"][:, lo:hi])
        oracle.pool_keys(c2, first, c2.n_blocks - first)
    assert np.array_equal(c.pooled_k, c2.pooled_k)
    assert np.array_equal(c.k_pages, c2.k_pages)


# ---------------------------------------------------------------------------------- a2 scores
def test_group_count_and_last_group(golden):
    S = golden["chunk_tokens"]
    assert -(-S // 64) == 74 and S - 73 * 64 == 8  # R = ceil(S/G_q)
    q = np.ones((1, S, 4), np.float32)
    q[0, 73 * 64:] = 3.0
    qb = oracle.group_mean_q(q, 64)
    assert qb.shape == (1, 74, 4) and np.all(qb[0, 72] == 1.0) and np.all(qb[0, 73] == 3.0)
    assert oracle.group_mean_q(q, S).shape == (1, 1, 4)


def test_scores_linearity_and_exact_dot(tiny):
    w, d, c = tiny
    sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    s, qbar = sel["scores"], sel["qbar"]
    assert s.shape == (w.H, w.R, w.n_b)
    sc = np.float64(np.float32(w.softmax_scale))
    kb = c.pooled_k[:, :w.n_b].astype(np.float64)
    # (i) the stored score is the fp32 rounding of sigma * <qbar, kbar> (numpy float64 einsum)
    exact = sc * np.einsum("hrd,hbd->hrb", qbar.astype(np.float64), kb)
    assert np.max(np.abs(s - exact.astype(np.float32)) / np.spacing(np.abs(exact).astype(np.float32))) <= 1.0
    # (ii) Eq. 3: AvgPool_q of the per-query logits == sigma * <mean_q q, kbar> (linearity); the
    # only gap is the bf16 rounding of qbar (2^-9 relative per component)
    per_query = sc * np.einsum("hsd,hbd->hsb", d["q"].astype(np.float64), kb)
    avg = per_query.reshape(w.H, w.R, w.G, w.n_b).mean(2)
    bound = sc * 2.0 ** -9 * np.einsum("hrd,hbd->hrb", np.abs(qbar).astype(np.float64), np.abs(kb)) + 1e-6
    assert np.all(np.abs(avg - s) <= bound)
    assert np.max(np.abs(avg - s)) > 0  # and the rounding is really there
    # mean of a group == numpy mean, rounded
    want = bf16(np.float32(d["q"].astype(np.float64).reshape(w.H, w.R, w.G, w.D).sum(2)) / np.float32(w.G))
    assert np.array_equal(qbar, want)


def test_scores_negative_zero_canonicalised():
    c = oracle.cache_create(1, 4, 64, 128)
    k = np.zeros((1, 128, 4), np.float32)
    k[0, :, 0] = -1.0
    oracle.append_chunk(c, k, k)
    oracle.pool_keys(c)
    s = oracle.scores(c, np.zeros((1, 1, 4), np.float32), 0.5)
    assert np.all(s == 0.0) and not np.any(np.signbit(s))


# ---------------------------------------------------------------------------------- a3 AWE
def test_awe_paper_window_arithmetic(golden):
    # PAPER.md:99 fn. 3: S=4680, N_w=3, B=60 -> the window spans ceil(3*4680/60) = 234 blocks
    S, B = golden["chunk_tokens"], 60
    n_hist = 10 * S
    a = oracle.awe(n_hist, B, 3 * S, 4, 0)
    assert a["n_b"] - a["b_w"] == golden["window_blocks_S4680_Nw3_B60"] == math.ceil(3 * S / B)
    assert golden["frame_tokens"] * 3 == S
    for blk, n in ((30, "tabH1_block30_blocks_per_frame"), (60, "tabH1_block60_blocks_per_frame"),
                   (26, "tabH1_block26_blocks_per_frame"), (12, "tabH1_block12_blocks_per_frame")):
        assert synth.FRAME_TOKENS // blk == golden[n]


def test_awe_three_regimes_and_baseline_configs():
    B, K, T = 64, 16, 220
    assert oracle.awe(10 * B + 5, B, 4 * B, K, T) == {"b_w": 6, "active": False, "omega_end": 11, "n_b": 11}
    a = oracle.awe(104 * B, B, 4 * B, K, T)  # K <= b_w=100 < T_awe: inactive under App. B, active under Eq. 2
    assert a["b_w"] == 100 and not a["active"] and a["omega_end"] == 104
    assert oracle.awe(104 * B, B, 4 * B, K, K)["active"]
    a = oracle.awe(300 * B, B, 4 * B, K, T)
    assert a == {"b_w": 296, "active": True, "omega_end": 296, "n_b": 300}
    # window wider than history, and no window at all
    assert oracle.awe(3 * B, B, 10 * B, 2, 0)["omega_end"] == 3
    assert oracle.awe(300 * B, B, 0, K, T)["omega_end"] == 300
    # BASELINE configs: config 2 b_w = 1389 active; short history must NOT exclude
    w = synth.config("wan1p3b")
    a = oracle.awe(w.n_hist, w.B, w.n_wt, w.K, w.t_awe)
    assert (w.n_b, w.t_awe, a["b_w"], a["active"]) == (1463, 220, 1389, True)
    for B_ in (64, 128):
        w = synth.config("short", B=B_)
        a = oracle.awe(w.n_hist, w.B, w.n_wt, w.K, w.t_awe)
        assert not a["active"] and a["omega_end"] == w.n_b and a["b_w"] in (146, 73)
    w = synth.config("long")
    assert (w.n_b, oracle.awe(w.n_hist, w.B, w.n_wt, w.K, w.t_awe)["b_w"]) == (8775, 8701)
    w = synth.config("wan14b")
    assert (w.n_b, oracle.awe(w.n_hist, w.B, w.n_wt, w.K, w.t_awe)["b_w"]) == (2925, 2851)


def test_awe_local_bias_adversarial():
    # scores increasing with block index; K <= window blocks => without exclusion every
    # pick lies in the window, with exclusion none does
    n_b, b_w, K = 40, 30, 8
    s = np.arange(n_b, dtype=np.float32)[None, None, :]
    no_awe = oracle.topk(s, n_b, K)
    with_awe = oracle.topk(s, b_w, K)
    assert np.all(no_awe >= b_w) and np.all(with_awe < b_w)
    assert list(with_awe[0, 0]) == list(range(b_w - 1, b_w - 1 - K, -1))


# ---------------------------------------------------------------------------------- a4 top-k
def test_topk_brute_force_ties_and_padding():
    rng = np.random.default_rng(3)
    H, R, n_b, K = 3, 5, 37, 6
    s = rng.integers(-3, 4, size=(H, R, n_b)).astype(np.float32)  # many exact ties
    s[0, 0, 5] = -0.0
    for omega in (37, 20, 4, 0):
        got = oracle.topk(s, omega, K)
        for h in range(H):
            for r in range(R):
                order = np.lexsort((np.arange(omega), -s[h, r, :omega]))  # score desc, index asc
                want = list(order[:K]) + [-1] * max(0, K - omega)
                assert list(got[h, r]) == want
                valid = got[h, r][got[h, r] >= 0]
                assert len(set(valid.tolist())) == min(K, omega) and np.all(valid < max(omega, 1))
    eq = oracle.topk(np.zeros((1, 1, 9), np.float32), 9, 4)
    assert list(eq[0, 0]) == [0, 1, 2, 3]  # equal scores: lowest index wins


def test_select_invariants_tiny(tiny):
    w, d, c = tiny
    for t_awe in (4, 12):
        sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, t_awe, w.softmax_scale)
        assert sel["awe"] == {"b_w": 24, "active": True, "omega_end": 24, "n_b": 32}
        idx = sel["block_idx"]
        assert idx.shape == (w.H, w.R, w.K) and np.all((idx >= 0) & (idx < 24))
        assert all(len(set(row)) == w.K for row in idx.reshape(-1, w.K).tolist())
        sc = np.take_along_axis(sel["scores"], idx, axis=2)
        assert np.all(np.diff(sc, axis=2) <= 0)  # slots in score order
    sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, 25, w.softmax_scale)
    assert not sel["awe"]["active"] and sel["awe"]["omega_end"] == 32


# ---------------------------------------------------------------------------------- a5 table / unions
def test_ptr_table_and_union_counters(golden):
    pm = synth.permuted_page_map(2, 10, 7)
    idx = np.array([[[3, 1, -1], [9, 3, 0]], [[2, -1, -1], [2, 5, 7]]], np.int32)
    p = oracle.ptr_table(idx, pm)
    for h in range(2):
        for r in range(2):
            for t in range(3):
                assert p[h, r, t] == (-1 if idx[h, r, t] < 0 else pm[h, idx[h, r, t]])
    ident = np.tile(np.arange(10, dtype=np.int32), (2, 1))
    assert np.array_equal(oracle.ptr_table(idx, ident), idx)
    per_head, u = oracle.union_counts(idx, 10)
    assert list(per_head) == [4, 3] and u == 7 and per_head.sum() <= 2 * u  # M_scatter <= M_merge
    # PAPER.md:101 fn. 4: 4 queries, top-1 each over 4 blocks, all distinct => union = full history
    nq, nb = golden["union_toy_queries"], golden["union_toy_blocks"]
    toy = np.arange(nq, dtype=np.int32).reshape(1, nq, 1)
    per_head, u = oracle.union_counts(toy, nb)
    assert per_head[0] == nb == u and per_head[0] <= nq * 1  # |U_h| <= R*K


# ---------------------------------------------------------------------------------- a6-a8 attention
def brute_force_attention(w, d, c_pages_k, c_pages_v, token_mask_hist, h, s, scale):
    """Independent numpy float64 dense softmax attention with a boolean mask over
    [history tokens | current chunk]; history is read from the FLAT generator arrays."""
    k = np.concatenate([d["k_hist"][h][token_mask_hist], d["k_cur"][h]]).astype(np.float64)
    v = np.concatenate([d["v_hist"][h][token_mask_hist], d["v_cur"][h]]).astype(np.float64)
    u = np.float64(np.float32(scale)) * (k @ d["q"][h, s].astype(np.float64))
    p = np.exp(u - u.max())
    return (p / p.sum()) @ v, u.max() + np.log(p.sum())


@pytest.mark.parametrize("permute", [False, True])
def test_attention_joint_equals_masked_dense(permute):
    w = synth.config("tiny", n_hist=2048 - 40, n_wt=500)  # ragged last block, straddling window start
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 11) if permute else None
    c = build_cache(w, d, pm)
    sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    assert sel["awe"]["active"]
    out, lse = oracle.sparse_attn(c, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"],
                                  G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale)
    rng = np.random.default_rng(4)
    for h, s in [(0, 0), (1, 255), (0, 64), (1, 63)] + [(int(rng.integers(w.H)), int(rng.integers(w.S))) for _ in range(12)]:
        mask = np.zeros(w.n_hist, bool)
        mask[w.win_start:] = True
        for b in sel["block_idx"][h, s // w.G]:
            mask[b * w.B:(b + 1) * w.B] = True
        want, want_lse = brute_force_attention(w, d, None, None, mask, h, s, w.softmax_scale)
        assert np.allclose(out[h, s], want, rtol=0, atol=2e-6)
        assert np.isclose(np.logaddexp(lse[0, h, s], lse[1, h, s]), want_lse, atol=1e-5)


def test_attention_full_coverage_equals_dense_sdpa():
    # north_star invariant: "the selection equals dense attention when k covers all history":
    # K = b_w with AWE active and an aligned window  ==>  JOINT == dense attention over all history +
    # the current chunk, cross-checked against the library routine torch SDPA.
    w = synth.config("tiny", K=24, t_awe=24)
    d = synth.generate(w)
    c = build_cache(w, d)
    sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    assert sel["awe"]["active"] and sel["awe"]["b_w"] == 24 and w.win_start % w.B == 0
    assert all(sorted(r) == list(range(24)) for r in sel["block_idx"].reshape(-1, 24).tolist())
    out, _ = oracle.sparse_attn(c, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"],
                                G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale)
    kk = torch.from_numpy(np.concatenate([d["k_hist"], d["k_cur"]], 1)).double()
    vv = torch.from_numpy(np.concatenate([d["v_hist"], d["v_cur"]], 1)).double()
    want = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(d["q"]).double()[None], kk[None], vv[None], scale=float(np.float32(w.softmax_scale)))[0]
    assert np.allclose(out, want.numpy(), rtol=0, atol=2e-6)


def test_attention_gated_and_swa_only_sdpa(tiny):
    w, d, c = tiny
    sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    kw = dict(G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale)
    hh = np.repeat(np.arange(w.H, dtype=np.int32), 8)
    qq = np.tile(np.int32([0, 1, 63, 64, 100, 128, 200, 255]), w.H)
    args = (c, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"])
    one, zero = np.ones(w.H, np.float32), np.zeros(w.H, np.float32)
    o_swa, lse = oracle.sparse_attn_rows(*args, fuse_mode=1, g_slc=zero, g_swa=one, **kw)
    o_slc, _ = oracle.sparse_attn_rows(*args, fuse_mode=1, g_slc=one, g_swa=zero, **kw)
    # (0,1) gates == SWA-only == dense attention over a contiguous range (library SDPA)
    kk = torch.from_numpy(np.concatenate([d["k_hist"][:, w.win_start:], d["k_cur"]], 1)).double()
    vv = torch.from_numpy(np.concatenate([d["v_hist"][:, w.win_start:], d["v_cur"]], 1)).double()
    want = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(d["q"]).double()[None], kk[None], vv[None], scale=float(np.float32(w.softmax_scale)))[0].numpy()
    assert np.allclose(o_swa, want[hh, qq], rtol=0, atol=2e-6)
    # Eq. 1: gated output is linear in the gates; JOINT is the LSE-weighted mix of the same branches
    g1 = np.float32([0.25, 0.75])
    g2 = np.float32([0.5, 0.125])
    o_g, _ = oracle.sparse_attn_rows(*args, fuse_mode=1, g_slc=g1, g_swa=g2, **kw)
    assert np.allclose(o_g, g1[hh, None] * o_slc + g2[hh, None] * o_swa, atol=1e-6)
    o_j, _ = oracle.sparse_attn_rows(*args, fuse_mode=0, **kw)
    a = 1.0 / (1.0 + np.exp(np.float64(lse[1]) - np.float64(lse[0])))
    assert np.allclose(o_j, a[:, None] * o_slc + (1 - a)[:, None] * o_swa, atol=2e-6)


def test_attention_online_softmax_and_slot_semantics(tiny):
    w, d, c = tiny
    sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    kw = dict(G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale)
    hh, qq = np.int32([0, 1, 1]), np.int32([5, 70, 255])
    one, zero = np.ones(w.H, np.float32), np.zeros(w.H, np.float32)
    base, lse = oracle.sparse_attn_rows(c, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"],
                                        fuse_mode=1, g_slc=one, g_swa=zero, **kw)
    # Algorithm 1 restated here: online softmax over the K pointed blocks
    sc = np.float64(np.float32(w.softmax_scale))
    for i, (h, s) in enumerate(zip(hh, qq)):
        m, dd, a = -np.inf, 0.0, np.zeros(w.D)
        for t in range(w.K):
            p = sel["ptr_table"][h, s // w.G, t]
            if p < 0:
                continue
            Kt, Vt = c.k_pages[h, p].astype(np.float64), c.v_pages[h, p].astype(np.float64)
            u = sc * (Kt @ d["q"][h, s].astype(np.float64))
            m2 = max(m, u.max())
            wgt, alpha = np.exp(u - m2), np.exp(m - m2)
            dd = dd * alpha + wgt.sum()
            a = a * alpha + wgt @ Vt
            m = m2
        assert np.allclose(base[i], a / dd, atol=2e-6) and np.isclose(lse[0, i], m + np.log(dd), atol=1e-5)
    # slot order does not matter; masked slots contribute nothing
    perm = np.random.default_rng(5).permutation(w.K)
    o2, _ = oracle.sparse_attn_rows(c, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"][:, :, perm],
                                    sel["ptr_table"][:, :, perm], fuse_mode=1, g_slc=one, g_swa=zero, **kw)
    assert np.allclose(base, o2, atol=1e-6)
    idx2, ptr2 = sel["block_idx"].copy(), sel["ptr_table"].copy()
    idx2[:, :, 2:] = -1
    ptr2[:, :, 2:] = -1
    o3, _ = oracle.sparse_attn_rows(c, hh, qq, d["q"], d["k_cur"], d["v_cur"], idx2, ptr2,
                                    fuse_mode=1, g_slc=one, g_swa=zero, **kw)
    o4, _ = oracle.sparse_attn_rows(c, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"][:, :, :2].copy(),
                                    sel["ptr_table"][:, :, :2].copy(), fuse_mode=1, g_slc=one, g_swa=zero,
                                    **dict(kw, K=2))
    assert np.array_equal(o3, o4) and not np.allclose(o3, base, atol=1e-3)
    # every slot masked (first chunk, N_hist = 0): O_slc = 0, LSE_slc = -inf, JOINT == SWA alone (A7, A8)
    c0 = oracle.cache_create(w.H, w.D, w.B, w.S)
    sel0 = oracle.select(c0, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    assert np.all(sel0["block_idx"] == -1) and np.all(sel0["ptr_table"] == -1)
    oj, lse0 = oracle.sparse_attn_rows(c0, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel0["block_idx"], sel0["ptr_table"],
                                       fuse_mode=0, **kw)
    og, _ = oracle.sparse_attn_rows(c0, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel0["block_idx"], sel0["ptr_table"],
                                    fuse_mode=1, g_slc=one, g_swa=one, **kw)
    assert np.all(np.isneginf(lse0[0])) and np.array_equal(oj, og)
    want = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(d["q"]).double()[None], torch.from_numpy(d["k_cur"]).double()[None],
        torch.from_numpy(d["v_cur"]).double()[None], scale=float(np.float32(w.softmax_scale)))[0].numpy()
    assert np.allclose(oj, want[hh, qq], atol=2e-6)


# ---------------------------------------------------------------------------------- NEXT-1: CMP branch (Eq. 1)
def test_pool_values_closed_forms_and_brute_force():
    """Block values follow the same recipe as block keys: constant block -> that row; brute-force mean over the valid
    tokens of a ragged last block through a permuted page map."""
    w = synth.config("tiny", n_hist=2048 - 40, H=2)
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 9)
    c = build_cache(w, d, pm)
    oracle.pool_values(c)
    for h in range(w.H):
        for b in (0, 7, w.n_b - 1):
            lo, hi = b * w.B, min((b + 1) * w.B, w.n_hist)
            want = bf16((d["v_hist"][h, lo:hi].astype(np.float64).sum(0)).astype(np.float32) / np.float32(hi - lo))
            assert np.array_equal(c.pooled_v[h, b], want)
    # values pooled, keys untouched by pool_values
    k_before = c.pooled_k.copy()
    oracle.pool_values(c)
    assert np.array_equal(k_before, c.pooled_k)
    w2 = synth.config("tiny", n_hist=128, H=1)
    c2 = oracle.cache_create(1, w2.D, w2.B, 256)
    row = bf16(np.linspace(-2, 3, w2.D))
    oracle.append_chunk(c2, np.zeros((1, 128, w2.D), np.float32), np.tile(row, (1, 128, 1)))
    oracle.pool_keys(c2)
    oracle.pool_values(c2)
    assert np.array_equal(c2.pooled_v[0, 0], row) and np.array_equal(c2.pooled_v[0, 1], row)


def test_cmp_attention_brute_force_sdpa_and_degenerate(tiny):
    """Compression attention is plain softmax attention of every query over the head's N_b compressed tokens: numpy
    float64 brute force, torch SDPA on the pooled arrays (library routine), one block -> its pooled value, no history -> 0."""
    w, d, c = tiny
    oracle.pool_values(c)
    rng = np.random.default_rng(3)
    hh = rng.integers(0, w.H, 40).astype(np.int32)
    qq = rng.integers(0, w.S, 40).astype(np.int32)
    out, lse = oracle.cmp_attn_rows(c, hh, qq, d["q"], w.softmax_scale)
    for i in range(40):
        h, s = hh[i], qq[i]
        u = np.float64(w.softmax_scale) * (c.pooled_k[h, :w.n_b].astype(np.float64) @ d["q"][h, s].astype(np.float64))
        p = np.exp(u - u.max())
        want = (p[:, None] * c.pooled_v[h, :w.n_b].astype(np.float64)).sum(0) / p.sum()
        assert np.max(np.abs(out[i] - want)) < 1e-6
        assert abs(lse[i] - (u.max() + math.log(p.sum()))) < 1e-5
    ref = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(d["q"]).double(), torch.from_numpy(c.pooled_k[:, :w.n_b]).double(),
        torch.from_numpy(c.pooled_v[:, :w.n_b]).double(), scale=float(w.softmax_scale)).numpy()
    assert np.max(np.abs(out - ref[hh, qq])) < 1e-6
    # one compressed token: the softmax weight is 1
    w1 = synth.config("tiny", n_hist=40)
    d1 = synth.generate(w1)
    c1 = build_cache(w1, d1)
    oracle.pool_values(c1)
    o1, l1 = oracle.cmp_attn_rows(c1, np.zeros(3, np.int32), np.arange(3, dtype=np.int32), d1["q"], w1.softmax_scale)
    assert np.array_equal(o1, np.tile(c1.pooled_v[0, 0], (3, 1))) and np.all(np.isfinite(l1))
    # first chunk: no compressed tokens
    w0 = synth.config("tiny", n_hist=0)
    d0 = synth.generate(w0)
    c0 = build_cache(w0, d0)
    oracle.pool_values(c0)
    o0, l0 = oracle.cmp_attn_rows(c0, np.zeros(2, np.int32), np.arange(2, dtype=np.int32), d0["q"], w0.softmax_scale)
    assert not o0.any() and np.all(np.isneginf(l0))


def test_gated3_is_the_sum_of_the_three_branches(tiny):
    """Eq. 1: o = sum_c g^c Attn(Q, K^c, V^c); with one gate at 1 and the others at 0 each branch comes back alone."""
    w, d, c = tiny
    oracle.pool_values(c)
    sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    hh = np.array([0, 1, 1, 0], np.int32)
    qq = np.array([0, 17, 200, 255], np.int32)
    kw = dict(G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale)
    one, zero = np.ones(w.H, np.float32), np.zeros(w.H, np.float32)
    args = (c, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"])
    o_cmp, _ = oracle.gated3_rows(*args, **kw, g_cmp=one, g_slc=zero, g_swa=zero)
    o_slc, _ = oracle.gated3_rows(*args, **kw, g_cmp=zero, g_slc=one, g_swa=zero)
    o_swa, _ = oracle.gated3_rows(*args, **kw, g_cmp=zero, g_slc=zero, g_swa=one)
    assert np.array_equal(o_cmp, oracle.cmp_attn_rows(c, hh, qq, d["q"], w.softmax_scale)[0])
    g = (np.float32(0.3), np.float32(0.5), np.float32(0.9))
    o, lse = oracle.gated3_rows(*args, **kw, g_cmp=g[0] * one, g_slc=g[1] * one, g_swa=g[2] * one)
    assert np.max(np.abs(o - (g[0] * o_cmp + g[1] * o_slc + g[2] * o_swa))) < 1e-6 and lse.shape == (3, 4)


# ------------------------------------------------------------------- NEXT-1, second half: probability scores
def test_scores_prob_brute_force_rows_sum_to_one_and_group_of_one(tiny):
    """oracle.scores_prob (reading A1b) against (1) an independent float64 numpy softmax + group mean,
    (2) the invariant that a mean of probability distributions sums to 1, (3) the special case G_q = 1, where softmax
    is monotone per query so the probability mode must select exactly what the logit mode selects, (4) identical block
    keys => the uniform distribution 1 / N_b, and (5) the library softmax (torch) on one group."""
    w, d, c = tiny
    n_b = c.n_blocks
    sig = w.softmax_scale
    for G in (64, 48, 256):
        got = oracle.scores_prob(c, d["q"], G, sig)
        R = -(-w.S // G)
        assert got.shape == (w.H, R, n_b) and got.dtype == np.float32
        logits = sig * np.einsum("hsd,hbd->hsb", d["q"].astype(np.float64), c.pooled_k[:, :n_b].astype(np.float64))
        e = np.exp(logits - logits.max(axis=2, keepdims=True))
        p = e / e.sum(axis=2, keepdims=True)
        want = np.stack([p[:, r * G:min((r + 1) * G, w.S)].mean(axis=1) for r in range(R)], axis=1)
        assert np.max(np.abs(got - want)) <= 1e-7
        assert np.max(np.abs(got.sum(axis=2) - 1.0)) <= 1e-5
    # (5) torch's softmax, first group of head 0
    lg = torch.from_numpy(sig * (d["q"][0, :64].astype(np.float64) @ c.pooled_k[0, :n_b].astype(np.float64).T))
    assert np.max(np.abs(oracle.scores_prob(c, d["q"], 64, sig)[0, 0] - torch.softmax(lg, dim=1).mean(dim=0).numpy())) <= 1e-7
    # (3) G_q = 1: same selection as the logit mode (softmax is monotone per query)
    a = oracle.select(c, d["q"], 1, w.K, w.n_wt, w.t_awe, sig, oracle.SCORE_LOGIT)
    b = oracle.select(c, d["q"], 1, w.K, w.n_wt, w.t_awe, sig, oracle.SCORE_PROB)
    assert np.array_equal(a["block_idx"], b["block_idx"]) and np.array_equal(a["ptr_table"], b["ptr_table"])
    # with groups the two modes are different selections (otherwise the variant would be vacuous)
    a = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, sig, oracle.SCORE_LOGIT)
    b = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, sig, oracle.SCORE_PROB)
    assert a["scores"].shape == b["scores"].shape and not np.allclose(a["scores"], b["scores"])
    # (4) identical block keys => uniform
    w2 = synth.config("tiny", H=1, S=64, n_hist=640)
    d2 = synth.generate(w2)
    d2["k_hist"][:] = d2["k_hist"][:, :1]
    c2 = build_cache(w2, d2)
    u = oracle.scores_prob(c2, d2["q"], 64, sig)
    assert np.max(np.abs(u - 1.0 / c2.n_blocks)) <= 1e-7


# ------------------------------------------------------------------- NEXT-3: the paper's own geometry
def test_paper_geometry_counts_padding_and_two_level_map(golden):
    """Tab. H1 closed forms: padded tile sizes and utilisation of the pooling shapes, 52 blocks of 30
    tokens per 1560-token frame, 156 per 4680-token chunk; the two-level pointer map of Alg. 1 (lines 7-12, :366-380)
    against the flat map it stands for, a hand-computed example and -1 propagation."""
    for blk in (30, 60, 26, 104, 12, 39, 65, 130):
        assert oracle.padded_block(blk) == golden[f"tabH1_block{blk}_padded"]
    for blk in (30, 26, 65):
        assert int(1000 * blk / oracle.padded_block(blk) + 0.5) == golden[f"tabH1_util{blk}_permille"]  # the paper rounds half up
    assert golden["frame_tokens"] // 30 == golden["tabH1_block30_blocks_per_frame"]
    assert golden["chunk_tokens"] // 30 == golden["paper_blocks_per_chunk"] and golden["chunk_tokens"] % 30 == 0
    # hand example: B_pc = 4, chunk bases (head 0) 40, 8, 100: block 6 = chunk 1, offset 2 -> page 10; block 11 -> chunk 2, offset 3 -> 103
    cm = np.array([[40, 8, 100], [0, 4, 8]], np.int32)
    idx = np.array([[[6, 11, -1, 0]], [[6, 11, 3, -1]]], np.int32)
    want = np.array([[[10, 103, -1, 40]], [[6, 11, 3, -1]]], np.int32)
    assert np.array_equal(oracle.ptr_table_chunked(idx, cm, 4), want)
    # against the flat map on random selections and random chunk placements
    rng = np.random.default_rng(5)
    B_pc, n_chunks, H = 156, 7, 3
    bases = np.stack([rng.permutation(n_chunks) * B_pc for _ in range(H)]).astype(np.int32)
    flat = oracle.expand_chunk_map(bases, B_pc, n_chunks * B_pc)
    for h in range(H):
        assert sorted(flat[h].tolist()) == list(range(n_chunks * B_pc))  # a permutation of the pages
    idx = rng.integers(-1, n_chunks * B_pc, size=(H, 9, 4)).astype(np.int32)
    assert np.array_equal(oracle.ptr_table_chunked(idx, bases, B_pc), oracle.ptr_table(idx, flat))


def test_oracle_handles_blocks_of_30_tokens():
    """The oracle's pooling, AWE and attention are block-size generic: B = 30 against numpy brute force."""
    w = synth.config("tiny", H=2, D=64, S=90, n_hist=5 * 90, B=30, n_wt=180, G=15, K=4, t_awe=6, chunk=90)
    d = synth.generate(w)
    c = build_cache(w, d)
    assert c.n_blocks == 15
    want = np.stack([bf16(d["k_hist"][:, b * 30:(b + 1) * 30].astype(np.float64).sum(axis=1).astype(np.float32) / np.float32(30)) for b in range(15)], axis=1)
    assert np.array_equal(c.pooled_k[:, :15], want)
    sel = oracle.select(c, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    a = sel["awe"]
    assert (a["b_w"], a["active"], a["omega_end"]) == (9, True, 9)  # window = last 180 tokens = blocks 9..14
    hh, qq = np.meshgrid(np.arange(w.H, dtype=np.int32), np.arange(w.S, dtype=np.int32), indexing="ij")
    out, _ = oracle.sparse_attn_rows(c, hh.ravel(), qq.ravel(), d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"],
                                     G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale)
    out = out.reshape(w.H, w.S, w.D)
    for h in range(w.H):
        for s in (0, 14, 15, 89):
            toks = sorted({t for b in sel["block_idx"][h, s // 15] if b >= 0 for t in range(b * 30, b * 30 + 30)} | set(range(270, 450)))
            kk = np.concatenate([d["k_hist"][h, toks], d["k_cur"][h]]).astype(np.float64)
            vv = np.concatenate([d["v_hist"][h, toks], d["v_cur"][h]]).astype(np.float64)
            lg = w.softmax_scale * kk @ d["q"][h, s].astype(np.float64)
            p = np.exp(lg - lg.max())
            assert np.max(np.abs(out[h, s] - (p / p.sum()) @ vv)) <= 1e-5


# ------------------------------------------------------------------- NEXT-4: offload / reload policy
def test_offload_model_hand_example_and_regimes():
    """oracle.OffloadModel (PAPER.md:325 LRU hot cache, :339 skip, :374-377 wait) against a hand-worked trace and the regimes the
    paper reports: a cache too small to retain what is selected has a 0 % hit rate, one that covers the working
    set converges to 100 %; pinned (window) chunks are never evicted; a step never evicts what it needs itself."""
    m = oracle.OffloadModel(H=1, G=3, W=1)
    for c in range(3):
        m.append(c)                      # resident {0,1,2}; clocks 1,2,3
    assert set(m.res[0]) == {0, 1, 2}
    m.append(3)                          # full: LRU non-pinned = 0 goes
    assert set(m.res[0]) == {1, 2, 3} and m.evictions == 1
    before, after = m.step([{0, 2}])     # 2 hits (touched), 0 misses: victim = LRU among {1} (3 is pinned, 2 is needed) -> 1
    assert before[0] == {1, 2, 3} and after[0] == {0, 2, 3}
    assert (m.requests, m.hits, m.reloads, m.evictions) == (2, 1, 1, 2)
    before, after = m.step([{0, 1, 2}])  # 0, 2 hit; 1 misses but every non-pinned resident chunk is needed: stays on the host
    assert after[0] == {0, 2, 3} and (m.requests, m.hits, m.reloads) == (5, 3, 1)
    # G too small: two chunks alternate through one LRU slot -> never a hit ("G_LRU = 1 ... 0 % hit rate")
    m = oracle.OffloadModel(H=2, G=2, W=1)
    for c in range(5):
        m.append(c)
    for i in range(10):
        m.step([{i % 2}, {2 + i % 2}])
    assert m.hits == 0 and m.reloads == 20 and m.hit_rate == 0.0 and all(4 in r for r in m.res)
    # G covers the working set: everything hits after the first touch ("G_LRU = 4 already reaches 99.9 %")
    m = oracle.OffloadModel(H=1, G=4, W=1)
    for c in range(8):
        m.append(c)
    for i in range(100):
        m.step([{0, 1, 2}])
    assert m.reloads == 3 and m.hits == 300 - 3 and m.hit_rate > 0.98 and 7 in m.res[0]
