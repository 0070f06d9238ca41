"""GPU parity tests (-m gpu): every call goes through the C-ABI binding; expected values come from the
CPU oracle on the same seeded inputs.  Small cases are compared element by element; BASELINE.json's
full-size configs are compared on sampled rows (attention) and in full (selection)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2605_30519_b200 import binding as om
from paper_2605_30519_b200 import synth

from _parity import build_gpu, build_oracle_cache, check_attention, check_select, check_step, dev_inputs

pytestmark = pytest.mark.gpu



def bits(t):
    return t.view(torch.int16).cpu().numpy()


def as_bf16_bits(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(torch.bfloat16).view(torch.int16).numpy()


# ------------------------------------------------------------------------------------ a0 / a1
@pytest.mark.parametrize("B,D,n_hist,chunk", [(64, 64, 2048, 256), (64, 128, 1000, 333), (128, 128, 1000, 77),
                                              (128, 64, 2008, 500), (64, 128, 64, 64), (64, 128, 5, 5)])
def test_append_and_pool_bit_exact(B, D, n_hist, chunk):
    w = synth.config("tiny", B=B, D=D, n_hist=n_hist, H=3, chunk=chunk)
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 21)
    oc = build_oracle_cache(w, d, pm)
    ls = build_gpu(w, d, pm)
    torch.cuda.synchronize()
    assert ls.cache.n_hist == oc.n_hist == n_hist
    # pages: every page that holds tokens, incl. the zero-filled tail of the last one
    for h in range(w.H):
        used = pm[h, :w.n_b]
        assert np.array_equal(bits(ls.cache.k_pages[h, used]), as_bf16_bits(oc.k_pages[h, used]))
        assert np.array_equal(bits(ls.cache.v_pages[h, used]), as_bf16_bits(oc.v_pages[h, used]))
    got, want = bits(ls.cache.pooled_k[:, :w.n_b]), as_bf16_bits(oc.pooled_k[:, :w.n_b])
    assert int((got != want).sum()) == 0, "pooled keys differ"


def test_pool_explicit_range_and_errors():
    w = synth.config("tiny")
    d = synth.generate(w)
    oc = build_oracle_cache(w, d)
    ls = build_gpu(w, d)
    ls.cache.pooled_k.zero_()
    om.omnimem_pool_keys(ls.cache, 3, 7)
    torch.cuda.synchronize()
    got = ls.cache.pooled_k.float().cpu().numpy()
    assert np.array_equal(got[:, 3:10], oc.pooled_k[:, 3:10]) and not got[:, :3].any() and not got[:, 10:].any()
    with pytest.raises(om.OmniMemError) as e:
        om.omnimem_pool_keys(ls.cache, 30, 5)
    assert e.value.code == om.EINVAL
    big = torch.zeros((w.H, 10_000, w.D), dtype=torch.bfloat16, device="cuda:0")
    with pytest.raises(om.OmniMemError) as e:
        om.omnimem_append_chunk(ls.cache, big, big)
    assert e.value.code == om.ECAPACITY
    # select refuses to run on un-pooled history
    k = torch.zeros((w.H, 10, w.D), dtype=torch.bfloat16, device="cuda:0")
    om.omnimem_append_chunk(ls.cache, k, k)
    with pytest.raises(om.OmniMemError) as e:
        ls.select(dev_inputs(d)[0])
    assert e.value.code == om.ESTATE


# ------------------------------------------------------------------------------------ a2-a5
@pytest.mark.parametrize("seed", [0, 1, 2])
@pytest.mark.parametrize("t_awe", [4, 12, 25])
def test_select_tiny(seed, t_awe):
    w = synth.config("tiny", seed=seed, t_awe=t_awe)
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), seed)
    check_select(w, d, build_gpu(w, d, pm), build_oracle_cache(w, d, pm))


@pytest.mark.parametrize("over", [dict(K=64, n_hist=2048), dict(K=40, n_hist=1000, n_wt=0), dict(K=8, n_hist=300, G=48),
                                  dict(K=4, n_hist=0), dict(K=33, n_hist=5000, B=128, D=128, G=256, S=256),
                                  dict(K=16, n_hist=9000, S=200, G=15, D=128, n_wt=700, t_awe=16)])
def test_select_edges(over):
    # K > |Omega| (masked slots), no window, ragged groups, empty history, B=128, small groups
    w = synth.config("tiny", **over)
    d = synth.generate(w)
    check_select(w, d, build_gpu(w, d), build_oracle_cache(w, d))


PROB_CASES = [dict(), dict(seed=1, t_awe=12), dict(K=8, n_hist=300, G=48), dict(K=4, n_hist=0), dict(K=33, n_hist=5000, B=128, D=128, G=256, S=256),
              dict(K=16, n_hist=9000, S=200, G=15, D=128, n_wt=700, t_awe=16), dict(S=330, G=330, K=5, n_hist=1500, D=128), dict(S=1, G=1, n_hist=200),
              dict(n_hist=1, K=2)]


@pytest.mark.parametrize("case", range(len(PROB_CASES)))
def test_select_probability_scores(case):
    """OMNIMEM_SCORE_PROB (reading A1b): per-query softmax over the compressed tokens averaged over the group, then
    the same AWE / top-k / table; scores against oracle.scores_prob, selections bit-exact both ways on identical scores.  Covers
    groups of 1, 15, 48, 64 and more than 64 queries (several CTAs per group + the ordered slab reduction), both head dims, empty history."""
    w = synth.config("tiny", **PROB_CASES[case])
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), case + 60)
    ls = build_gpu(w, d, pm)
    oc = build_oracle_cache(w, d, pm)
    sel = check_select(w, d, ls, oc, expect_exact_sets=False, score_mode=om.SCORE_PROB)
    if w.n_hist > 0:
        assert np.max(np.abs(ls.scores.cpu().numpy().sum(axis=2) - 1.0)) <= 1e-4  # a mean of distributions
    # the table of this mode drives the attention like any other
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_JOINT)
    check_select(w, d, ls, oc, expect_exact_sets=False, score_mode=om.SCORE_LOGIT)  # the same handle switches back


def test_select_probability_scores_full_size():
    """Config 2 under the probability reading: selection compared in full, attention on sampled rows with the oracle's table."""
    w = FULL["wan1p3b"]
    d = synth.generate(w)
    oc = build_oracle_cache(w, d)
    ls = build_gpu(w, d, want_lse=True)
    sel = check_select(w, d, ls, oc, expect_exact_sets=False, score_mode=om.SCORE_PROB)
    assert sel["awe"]["active"] and np.all(sel["block_idx"] < sel["awe"]["b_w"])
    rows = synth.sample_rows(w, 5, 4)
    e = check_attention(w, d, ls, oc, sel, rows=rows, fuse_mode=om.FUSE_JOINT)
    print(f"wan1p3b PROB scores: near-tie rows {sel['near_tie_rows']} of {w.H * w.R}; JOINT max-abs {e[0]:.3e} mean-abs {e[1]:.3e} on {len(rows[0])} rows")


def test_select_from_scores_ties_lowest_index_first():
    w = synth.config("tiny")
    d = synth.generate(w)
    ls = build_gpu(w, d)
    rng = np.random.default_rng(0)
    s = rng.integers(-2, 3, size=(w.H, w.R, w.n_b)).astype(np.float32)  # heavy ties, some -0
    s[0, 0, :5] = -0.0
    idx = torch.empty_like(ls.block_idx)
    ptr = torch.empty_like(ls.ptr_table)
    awe = om.omnimem_select_from_scores(ls.cache, torch.from_numpy(s).cuda(), w.S, ls.sp, idx, ptr)
    torch.cuda.synchronize()
    assert np.array_equal(idx.cpu().numpy(), oracle.topk(s, awe["omega_end"], w.K))


def _topk_harness(n_b, K):
    """A cache of n_b all-zero blocks behind omnimem_select_from_scores (identity page map): the scores are the test's."""
    from paper_2605_30519_b200.runner import LayerStep
    w = synth.config("tiny", H=2, D=64, S=192, G=64, n_hist=n_b * 64, n_wt=0, K=K, t_awe=1, chunk=n_b * 64)
    ls = LayerStep(w, "cuda:0")
    z = torch.zeros((w.H, min(w.n_hist, 1 << 17), w.D), dtype=torch.bfloat16, device="cuda:0")
    left = w.n_hist
    while left > 0:
        n = min(left, z.shape[1])
        ls.append(z[:, :n], z[:, :n], pool=False)
        left -= n

    def run(sc):
        idx = torch.full_like(ls.block_idx, -9)
        ptr = torch.full_like(ls.ptr_table, -9)
        awe = om.omnimem_select_from_scores(ls.cache, torch.from_numpy(sc).cuda(), w.S, ls.sp, idx, ptr)
        torch.cuda.synchronize()
        assert awe["omega_end"] == n_b
        return idx.cpu().numpy(), ptr.cpu().numpy()
    return w, run


@pytest.mark.parametrize("n_b,K", [(300, 1), (512, 16), (513, 64), (1024, 7), (1389, 16), (1536, 64), (2048, 16), (2049, 33), (4096, 8),
                                   (8701, 32), (10240, 64), (16384, 5), (16385, 16), (20000, 64), (33, 32), (65, 64), (70, 33)])
def test_topk_rows_of_every_length(n_b, K):
    """omnimem_select_from_scores on rows of 33 .. 20000 candidates (one warp per row, two scans of the row): random scores,
    scores with heavy ties and all-equal scores (the fixed tie-break decides) -- bit-exact against the oracle."""
    w, run = _topk_harness(n_b, K)
    rng = np.random.default_rng(n_b + K)
    for kind in ("random", "ties", "all_equal"):
        if kind == "random":
            sc = rng.standard_normal((w.H, w.R, n_b)).astype(np.float32)
        elif kind == "ties":
            sc = rng.integers(-3, 4, size=(w.H, w.R, n_b)).astype(np.float32)
            sc[0, 0, :7] = -0.0
        else:
            sc = np.full((w.H, w.R, n_b), 1.5, np.float32)
        idx, ptr = run(sc)
        want = oracle.topk(sc, n_b, K)
        assert np.array_equal(idx, want), kind
        assert np.array_equal(ptr, want), kind  # identity page map


@pytest.mark.parametrize("n_b,K", [(1389, 16), (1389, 64), (4000, 33), (700, 5)])
def test_topk_scores_concentrated_in_one_lane(n_b, K):
    """The adversarial layout for the warp scan: every large score sits at a block index = 5 mod 32 (one lane), so the bound
    taken from the lane tops lets more than 64 candidates through and the exact bitwise descent over the 64-bit keys decides;
    also descending and ascending ramps.  Bit-exact against the oracle."""
    w, run = _topk_harness(n_b, K)
    rng = np.random.default_rng(7 * n_b + K)
    sc = rng.standard_normal((w.H, w.R, n_b)).astype(np.float32)
    sc[:, :, 5::32] += 50.0
    ramp = np.arange(n_b, dtype=np.float32)
    for name, x in (("one_lane", sc), ("descending", np.broadcast_to(-ramp, sc.shape).copy()), ("ascending", np.broadcast_to(ramp, sc.shape).copy())):
        idx, _ = run(x)
        assert np.array_equal(idx, oracle.topk(x, n_b, K)), name


# ------------------------------------------------------------------------------------ NEXT-2: union accounting, merged buffer
@pytest.mark.parametrize("over", [dict(H=3, D=128, K=5, n_hist=3000, n_wt=640), dict(K=4, n_hist=0), dict(G=1, S=40, K=3, n_hist=1000),
                                  dict(H=4, K=64, n_hist=2048, G=15, S=100)])
def test_union_counts_and_merged_buffer(over):
    """Eqs. 4-5 from the CUDA path: |U_h| per head, |union over heads| and the union's block list against
    oracle.union_counts / numpy on the GPU's own selection; then the Naive-Sparse merged buffer (omnimem_gather_blocks): the listed
    blocks of every head, bit for bit, in list order."""
    from paper_2605_30519_b200.runner import LayerStep
    w = synth.config("tiny", **over)
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 77)
    ls = build_gpu(w, d, pm)
    q, _, _ = dev_inputs(d)
    ls.select(q)
    n_b = ls.cache.n_blocks
    per_head = torch.full((w.H,), -1, dtype=torch.int64, device="cuda:0")
    union_all = torch.full((1,), -1, dtype=torch.int64, device="cuda:0")
    union_list = torch.full((max(n_b, 1),), -1, dtype=torch.int32, device="cuda:0")
    ws = torch.empty((w.H + 1) * max(n_b, 1), dtype=torch.uint8, device="cuda:0")
    om.omnimem_union_counts(ls.cache, ls.block_idx, per_head, union_all, union_list, ws)
    torch.cuda.synchronize()
    g_idx = ls.block_idx.cpu().numpy()
    want_ph, want_u = oracle.union_counts(g_idx, n_b)
    assert np.array_equal(per_head.cpu().numpy(), want_ph) and int(union_all.item()) == want_u
    blocks = np.unique(g_idx[g_idx >= 0])
    assert np.array_equal(union_list.cpu().numpy()[:want_u], blocks)
    assert want_ph.sum() <= w.H * want_u  # M_scatter <= M_merge
    # merged selected-KV buffer
    dst = LayerStep(w, "cuda:0", synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 78)).cache
    om.omnimem_gather_blocks(ls.cache, union_list, want_u, dst)
    torch.cuda.synchronize()
    assert dst.n_hist == want_u * w.B
    pm_d = dst.page_map.cpu().numpy()
    for h in range(w.H):
        src_pages = ls.cache.k_pages[h, torch.from_numpy(pm[h, blocks].astype(np.int64)).cuda()]
        got_pages = dst.k_pages[h, torch.from_numpy(pm_d[h, :want_u].astype(np.int64)).cuda()]
        assert torch.equal(src_pages.view(torch.int16), got_pages.view(torch.int16))
        src_v = ls.cache.v_pages[h, torch.from_numpy(pm[h, blocks].astype(np.int64)).cuda()]
        got_v = dst.v_pages[h, torch.from_numpy(pm_d[h, :want_u].astype(np.int64)).cuda()]
        assert torch.equal(src_v.view(torch.int16), got_v.view(torch.int16))
    if want_u > 0:
        with pytest.raises(om.OmniMemError) as e:  # dst is no longer empty
            om.omnimem_gather_blocks(ls.cache, union_list, want_u, dst)
        assert e.value.code == om.ESTATE


def test_union_counts_paper_footnote_example(golden):
    """PAPER.md:101 (fn. 4): four queries, top-1 each, four blocks, all distinct => the union is the whole history."""
    from paper_2605_30519_b200.runner import LayerStep
    wq = synth.config("tiny", H=1, D=64, S=4, G=1, n_hist=4 * 64, n_wt=0, K=1, t_awe=1, chunk=256)
    ls = LayerStep(wq, "cuda:0")
    z = torch.zeros((1, 256, 64), dtype=torch.bfloat16, device="cuda:0")
    ls.append(z, z, pool=False)
    sc = np.full((1, 4, 4), -1.0, np.float32)
    for qi in range(4):
        sc[0, qi, (qi * 3) % 4] = 1.0  # each query prefers a different block
    idx = torch.empty_like(ls.block_idx)
    ptr = torch.empty_like(ls.ptr_table)
    om.omnimem_select_from_scores(ls.cache, torch.from_numpy(sc).cuda(), wq.S, ls.sp, idx, ptr)
    per_head = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    union_all = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    om.omnimem_union_counts(ls.cache, idx, per_head, union_all, None, torch.empty(64, dtype=torch.uint8, device="cuda:0"))
    torch.cuda.synchronize()
    assert int(per_head.item()) == int(union_all.item()) == golden["union_toy_blocks"]


# ------------------------------------------------------------------------------------ a6-a8, small cases, every row
TINY_CASES = [
    dict(),                                              # config 1
    dict(seed=1, n_hist=2048 - 40, n_wt=500),            # ragged last block + straddling window start
    dict(seed=2, K=24, t_awe=24),                        # K covers all history outside the window
    dict(n_hist=0),                                      # first chunk: no history, all slots masked
    dict(n_wt=0, K=8),                                   # no window: SLC + current chunk only
    dict(S=200, G=48, n_hist=1000, n_wt=300),            # ragged query tile and groups that straddle tiles
    dict(S=330, G=15, K=3, n_hist=1500, n_wt=256),       # paper-like small groups (several groups per tile)
    dict(S=256, G=256, K=6),                             # one group for the whole chunk
    dict(D=128, H=3, n_hist=3000, n_wt=640, K=5),        # head_dim 128
    dict(D=128, B=128, n_hist=3000 - 70, n_wt=700, K=7, t_awe=3),  # B=128, ragged, straddle
    dict(n_hist=700, n_wt=512, K=16, t_awe=12),          # short history: AWE inactive, K > candidates
]


@pytest.mark.parametrize("case", range(len(TINY_CASES)))
def test_attention_small_all_rows(case):
    w = synth.config("tiny", **TINY_CASES[case])
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), case + 3)
    oc = build_oracle_cache(w, d, pm)
    ls = build_gpu(w, d, pm, want_lse=True)
    sel = check_select(w, d, ls, oc)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_JOINT)
    g1 = np.linspace(0.2, 0.9, w.H).astype(np.float32)
    g2 = np.linspace(0.8, 0.3, w.H).astype(np.float32)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_GATED, g_slc=g1, g_swa=g2)


def test_attention_masked_and_permuted_slots():
    w = synth.config("tiny", D=128, K=8, n_hist=4096, n_wt=512)
    d = synth.generate(w)
    oc = build_oracle_cache(w, d)
    ls = build_gpu(w, d, want_lse=True)
    sel = check_select(w, d, ls, oc)
    rng = np.random.default_rng(7)
    sel2 = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in sel.items()}
    # pointer < 0 => skip, wherever it sits in the list (Alg. 1 lines 20-22); order is free
    kill = rng.random(sel2["ptr_table"].shape) < 0.4
    sel2["ptr_table"][kill] = -1
    sel2["block_idx"][kill] = -1
    perm = rng.permutation(w.K)
    sel2["ptr_table"] = np.ascontiguousarray(sel2["ptr_table"][:, :, perm])
    sel2["block_idx"] = np.ascontiguousarray(sel2["block_idx"][:, :, perm])
    check_attention(w, d, ls, oc, sel2, fuse_mode=om.FUSE_JOINT)
    check_attention(w, d, ls, oc, sel2, fuse_mode=om.FUSE_GATED, g_slc=np.ones(w.H, np.float32), g_swa=np.ones(w.H, np.float32))


# Paired SLC tiles (attn_schedule.cuh): with G_q a multiple of 32 and at least two groups in a 128-row query tile, one KV tile holds
# slot j of an even group and slot j of the odd group behind it; each warp attends its group's 64 columns only.
PAIRED_CASES = [
    dict(S=256, G=32, K=3, n_hist=1500, n_wt=256),                  # four groups per tile, odd K
    dict(S=200, G=32, K=4, n_hist=1500 - 21, n_wt=300),             # second tile: groups 4, 5 and an 8-row group 6 (odd count, ragged)
    dict(S=300, G=96, K=5, n_hist=2048, n_wt=512),                  # group boundaries at rows 96, 192, 288: pairs of unequal height
    dict(S=400, G=160, K=2, n_hist=1000, n_wt=128),                 # tile 0 holds one group (no pairing), tiles 1-3 hold two
    dict(D=128, B=128, S=256, G=64, K=3, n_hist=3000 - 70, n_wt=700, t_awe=3),  # two slots per block, ragged last block
    dict(S=256, G=64, K=16, n_hist=700, n_wt=512, t_awe=12),       # K > candidates: masked tails in both halves of a pair
]


@pytest.mark.parametrize("case", range(len(PAIRED_CASES)))
def test_attention_paired_slc_tiles(case):
    w = synth.config("tiny", **PAIRED_CASES[case])
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), case + 41)
    oc = build_oracle_cache(w, d, pm)
    ls = build_gpu(w, d, pm, want_lse=True)
    sel = check_select(w, d, ls, oc)
    g1 = np.linspace(0.3, 0.9, w.H).astype(np.float32)
    g2 = np.linspace(0.7, 0.2, w.H).astype(np.float32)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_JOINT)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_GATED, g_slc=g1, g_swa=g2)
    # entries < 0 anywhere in a group's list: the two halves of a paired tile are then masked independently
    rng = np.random.default_rng(case)
    sel2 = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in sel.items()}
    kill = rng.random(sel2["ptr_table"].shape) < 0.5
    kill[:, 0, :] = True  # a whole group without a block: its rows see the window only
    sel2["ptr_table"][kill] = -1
    sel2["block_idx"][kill] = -1
    check_attention(w, d, ls, oc, sel2, fuse_mode=om.FUSE_JOINT)
    check_attention(w, d, ls, oc, sel2, fuse_mode=om.FUSE_GATED, g_slc=g1, g_swa=g2)


# KV-tile counts around the MMA issuer's unroll boundaries (rounds of 10 tiles, 5-slot operand ring): T = SLC tiles
# (2 groups x ceil(K / 2)) + SWA tiles (ceil((window blocks + 4 current-chunk slots) / 2)) per 128-row query tile
TILE_SWEEP = [dict(K=1, n_wt=0), dict(K=1, n_wt=37), dict(K=1, n_wt=518), dict(K=1, n_wt=629), dict(K=1, n_wt=777),   # T = 4 5 9 10 11
              dict(K=1, n_wt=888), dict(K=1, n_wt=1776), dict(K=1, n_wt=1924), dict(K=1, n_wt=2035), dict(K=3, n_wt=1924),  # 12 19 20 21 22
              dict(K=7, n_wt=2035),                                                                                        # 27
              dict(n_hist=0, S=64), dict(n_hist=0, S=200), dict(n_hist=0, S=256, G=48)]                                    # T = 1 2 2 (GATED: 0 + T)


@pytest.mark.parametrize("case", range(len(TILE_SWEEP)))
def test_attention_tile_count_sweep(case):
    w = synth.config("tiny", **{**dict(D=128, H=2, S=256, G=64, n_hist=2048 + 37, t_awe=2), **TILE_SWEEP[case]})
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), case + 11)
    oc = build_oracle_cache(w, d, pm)
    ls = build_gpu(w, d, pm, want_lse=True)
    sel = check_select(w, d, ls, oc)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_JOINT)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_GATED, g_slc=np.full(w.H, 0.7, np.float32), g_swa=np.full(w.H, 0.4, np.float32))


def test_strided_inputs():
    """q / k / v handed over as [H][n][D] views of a packed [n][H][3][D] projection output (stride_tok = 3 H D,
    stride_head = 3 D): append, select and the attention kernel must honour the caller's strides."""
    from paper_2605_30519_b200.runner import LayerStep, to_dev
    w = synth.config("tiny", D=128, H=3, S=200, G=48, n_hist=1000, n_wt=300, K=5)
    d = synth.generate(w)
    oc = build_oracle_cache(w, d)

    def packed_view(a, which):
        n = a.shape[1]
        buf = torch.full((n, w.H, 3, w.D), 7.0, dtype=torch.bfloat16, device="cuda:0")  # neighbours hold junk
        buf[:, :, which] = to_dev(a, "cuda:0").permute(1, 0, 2)
        v = buf[:, :, which].permute(1, 0, 2)
        assert v.stride() == (3 * w.D, w.H * 3 * w.D, 1)
        return v

    ls = LayerStep(w, "cuda:0", want_lse=True)
    for lo in range(0, w.n_hist, w.chunk):
        ls.append(packed_view(d["k_hist"][:, lo:lo + w.chunk], 1), packed_view(d["v_hist"][:, lo:lo + w.chunk], 2))
    inputs = (packed_view(d["q"], 0), packed_view(d["k_cur"], 1), packed_view(d["v_cur"], 2))
    sel = check_select(w, d, ls, oc, inputs=inputs)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_JOINT, inputs=inputs)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_GATED, g_slc=np.full(w.H, 0.6, np.float32), g_swa=np.full(w.H, 0.9, np.float32),
                    inputs=inputs)


def test_step_is_deterministic_and_repeatable():
    """The whole step (4 kernels chained by programmatic dependent launch) run back to back many times on the same
    buffers: tables and outputs are bit-identical every time (the per-row reference max is handed from tile to tile
    in a fixed order, so there is no run-to-run reassociation)."""
    w = synth.config("tiny", D=128, H=4, S=512, G=64, n_hist=4096 + 20, n_wt=700, K=6)
    d = synth.generate(w)
    ls = build_gpu(w, d, synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 5))
    q, k, v = dev_inputs(d)
    ref_out = ref_tab = None
    for it in range(30):
        ls.ptr_table.fill_(-7)
        ls.out.fill_(float("nan"))
        out = ls.step(q, k, v)
        if it == 0:
            torch.cuda.synchronize()
            ref_out, ref_tab = out.clone(), ls.ptr_table.clone()
            assert torch.isfinite(ref_out.float()).all()
    torch.cuda.synchronize()
    assert torch.equal(ls.ptr_table, ref_tab) and torch.equal(out.view(torch.int16), ref_out.view(torch.int16))


def test_host_pipeline_matches_serial_steps():
    """runner.HostPipeline (what bench.py's e2e figure runs): steps fed from pinned host buffers with the copies of
    neighbouring steps overlapping the kernels on three streams give, step for step, the bits of the same steps run one at
    a time -- three different inputs in rotation, so a slot that is overwritten too early or read too late shows."""
    from paper_2605_30519_b200.runner import HostPipeline
    w = synth.config("tiny", D=128, H=4, S=512, G=64, n_hist=4096 + 20, n_wt=700, K=6)
    d = synth.generate(w)
    ls = build_gpu(w, d, synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 5))
    q, k, v = dev_inputs(d)
    sets, want = [], []
    for j in range(3):
        qj, kj, vj = (torch.roll(t, shifts=17 * j, dims=1).contiguous() for t in (q, k, v))
        want.append(ls.step(qj, kj, vj).clone())
        sets.append(tuple(t.cpu().pin_memory() for t in (qj, kj, vj)))
    torch.cuda.synchronize()
    assert not torch.equal(want[0], want[1])
    pipe = HostPipeline(ls)
    n = 11
    houts = [torch.empty_like(want[0], device="cpu").pin_memory() for _ in range(n)]
    for i in range(n):
        pipe.submit(*sets[i % 3], houts[i])
    pipe.drain()
    torch.cuda.synchronize()
    for i in range(n):
        assert torch.equal(houts[i].view(torch.int16), want[i % 3].cpu().view(torch.int16)), i


def _random_configs(seed, n):
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(n):
        S = int(rng.integers(1, 700))
        G = max(1, min(int(rng.choice([1, 15, 48, 64, 100, 128, 256, S])), S))
        out.append(dict(D=128, B=int(rng.choice([64, 128])), S=S, G=G, H=int(rng.integers(1, 4)),
                        n_hist=int(rng.choice([0, int(rng.integers(1, 200)), int(rng.integers(200, 6000))])),
                        n_wt=int(rng.choice([0, int(rng.integers(1, 300)), int(rng.integers(300, 3000))])),
                        K=int(rng.choice([1, 2, 3, 5, 8, 16, 33, 64])), t_awe=int(rng.choice([1, 4, 30])),
                        chunk=max(1, int(rng.choice([S, 333, 1000])))))
    return out


RANDOM_CONFIGS = _random_configs(2605, 24)


@pytest.mark.parametrize("case", range(len(RANDOM_CONFIGS)))
def test_random_shapes_blackwell_kernel(case):
    """Seeded random geometry (chunk length 1..700, groups of 1..S queries, K 1..64, both page sizes, empty / short /
    long history, no / short / long window, AWE on and off) through the tcgen05 kernel, all rows, both fusions."""
    w = synth.config("tiny", **RANDOM_CONFIGS[case])
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), case)
    oc = build_oracle_cache(w, d, pm)
    ls = build_gpu(w, d, pm, want_lse=True)
    sel = check_select(w, d, ls, oc, expect_exact_sets=False)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_JOINT)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_GATED, g_slc=np.full(w.H, 0.7, np.float32), g_swa=np.full(w.H, 0.4, np.float32))


# ------------------------------------------------------------------------------------ NEXT-1: CMP branch, full Eq. 1
def check_attention3(w, d, ls, oc, sel, rows=None):
    """omnimem_sparse_attn3 (fed the oracle's table) against oracle.gated3_rows: output and the three LSE rows."""
    q, k_cur, v_cur = dev_inputs(d)
    ls.ptr_table.copy_(torch.from_numpy(sel["ptr_table"]))
    g = [np.linspace(a, b, w.H).astype(np.float32) for a, b in ((0.3, 0.8), (0.9, 0.2), (0.5, 0.6))]
    for t, v in zip((ls.gate_cmp, ls.gate_slc, ls.gate_swa), g):
        t.copy_(torch.from_numpy(v))
    ls.out.fill_(float("nan"))
    out = ls.attend3(q, k_cur, v_cur)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy()
    if rows is None:
        hh, qq = np.meshgrid(np.arange(w.H, dtype=np.int32), np.arange(w.S, dtype=np.int32), indexing="ij")
        hh, qq = hh.ravel(), qq.ravel()
    else:
        hh, qq = rows
    want, want_lse = oracle.gated3_rows(oc, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"], G=w.G, K=w.K,
                                        n_wt=w.n_wt, softmax_scale=w.softmax_scale, g_cmp=g[0], g_slc=g[1], g_swa=g[2])
    assert np.all(np.isfinite(out)), "non-finite or unwritten output rows"
    err = np.abs(out[hh, qq] - want)
    assert err.max() <= 2e-2 and err.mean() <= 2e-3, (err.max(), err.mean())
    got_lse = ls.lse3.cpu().numpy()[:, hh, qq]
    assert np.array_equal(np.isneginf(got_lse), np.isneginf(want_lse)), "LSE -inf pattern"
    fin = np.isfinite(want_lse)
    assert not fin.any() or np.max(np.abs(got_lse[fin] - want_lse[fin])) <= 2e-2, "LSE"
    return float(err.max()), float(err.mean())


CMP_CASES = [dict(), dict(D=64), dict(D=64, H=2, S=200, G=48, n_hist=64 * 70 + 9, n_wt=200, K=3), dict(n_hist=40), dict(n_hist=0), dict(n_hist=64 * 130 + 7, n_wt=300, K=5), dict(B=128, n_hist=3000 - 70, n_wt=700, K=7, t_awe=3),
             dict(S=200, G=48, n_hist=64 * 257, n_wt=0, K=2), dict(S=77, G=77, n_hist=64 * 64, K=1)]


@pytest.mark.parametrize("case", range(len(CMP_CASES)))
def test_cmp_branch_three_way_gated(case):
    """Pooled block values bit-exact; compression attention over 1 .. 257 compressed tokens (0: contributes nothing)
    fused with SLC and SWA by per-head gates (Eq. 1), all rows."""
    w = synth.config("tiny", **{**dict(D=128, H=3), **CMP_CASES[case]})
    d = synth.generate(w)
    pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), case + 40)
    oc = build_oracle_cache(w, d, pm)
    oracle.pool_values(oc)
    ls = build_gpu(w, d, pm, want_lse=True, cmp=True)
    torch.cuda.synchronize()
    assert np.array_equal(bits(ls.cache.pooled_v[:, :w.n_b]), as_bf16_bits(oc.pooled_v[:, :w.n_b])), "pooled values differ"
    assert np.array_equal(bits(ls.cache.pooled_k[:, :w.n_b]), as_bf16_bits(oc.pooled_k[:, :w.n_b]))
    sel = check_select(w, d, ls, oc, expect_exact_sets=False)
    check_attention3(w, d, ls, oc, sel)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_JOINT)  # the two-branch calls are untouched by the attachment


def test_cmp_branch_full_size_and_errors():
    w = synth.config("wan1p3b")
    d = synth.generate(w)
    oc = build_oracle_cache(w, d)
    oracle.pool_values(oc)
    ls = build_gpu(w, d, want_lse=True, cmp=True)
    sel = check_select(w, d, ls, oc, expect_exact_sets=False)
    e = check_attention3(w, d, ls, oc, sel, rows=synth.sample_rows(w, 5, 4))
    print(f"wan1p3b three-branch: max-abs {e[0]:.3e} mean-abs {e[1]:.3e}")
    # no pooled-value buffer -> ESTATE; JOINT is not Eq. 1 -> EINVAL
    wt = synth.config("tiny", D=128)
    dt = synth.generate(wt)
    lt = build_gpu(wt, dt)
    q, k, v = dev_inputs(dt)
    lt.select(q)
    with pytest.raises(om.OmniMemError) as ex:
        lt.attend3(q, k, v)
    assert ex.value.code == om.ESTATE
    ap = om.AttnParams(wt.G, wt.K, wt.n_wt, wt.softmax_scale, om.FUSE_JOINT, 0)
    lc = build_gpu(wt, dt, cmp=True)
    q, k, v = dev_inputs(dt)
    lc.select(q)
    with pytest.raises(om.OmniMemError) as ex:
        om.omnimem_sparse_attn3(lc.cache, q, k, v, lc.ptr_table, ap, lc.out, lc.gate_cmp, lc.gate_slc, lc.gate_swa, None, lc.ws_attn)
    assert ex.value.code == om.EINVAL


def test_attention_rejects_bad_arguments():
    w = synth.config("tiny")
    d = synth.generate(w)
    ls = build_gpu(w, d)
    q, k, v = dev_inputs(d)
    ls.select(q)
    ls.ap.fuse_mode = 5
    with pytest.raises(om.OmniMemError):
        ls.attend(q, k, v)
    ls.ap.fuse_mode = om.FUSE_JOINT
    ls.ap.reserved = 7
    with pytest.raises(om.OmniMemError) as e:
        ls.attend(q, k, v)
    assert e.value.code == om.EINVAL


# ------------------------------------------------------------------------------------ NEXT-3: the paper's own geometry
def _paper_like(**over):
    base = dict(H=2, D=128, S=150, n_hist=6 * 150, B=30, P=32, bpc=5, n_wt=3 * 150, G=15, K=4, t_awe=15, chunk=150)
    base.update(over)
    return synth.config("tiny", **base)


PAPER_CASES = [
    dict(),                                                         # 30-token blocks in 32-row pages, G_q 15, top-4, 3-chunk window, two-level map
    dict(K=3, seed=1),                                              # odd K: the last SLC slot holds one page
    dict(n_hist=6 * 150 - 40, chunk=150, bpc=0, seed=2),            # ragged last block, flat page map
    dict(n_hist=2 * 150, t_awe=15),                                 # short history: AWE inactive, selections fall into the window
    dict(D=64, H=3, S=90, n_hist=540, chunk=90, bpc=3, n_wt=200, t_awe=4),   # head_dim 64; the window starts inside a block
    dict(B=26, S=104, n_hist=8 * 104, chunk=104, bpc=4, n_wt=2 * 104, G=13, K=5, t_awe=8),   # 2 x 13 pooling block (Tab. H1), 81 % tile fit
    dict(B=60, P=64, S=240, n_hist=5 * 240, chunk=240, bpc=4, n_wt=480, G=30, K=4, t_awe=4),     # 15 x 4 block in 64-row pages
    dict(B=104, P=128, S=208, n_hist=6 * 208, chunk=208, bpc=2, n_wt=416, G=52, K=3, t_awe=4),   # 2 x 52 block in 128-row pages
    dict(n_wt=0, K=6),                                              # no window
    dict(n_hist=0),                                                 # first chunk
]


@pytest.mark.parametrize("case", range(len(PAPER_CASES)))
def test_paper_geometry_small_all_rows(case):
    """Blocks of B < P tokens in zero-padded pages, chunk-aligned blocks behind the two-level map
    (Alg. 1 lines 7-12), G_q = 15, top-4, window of 3 chunks (:319): pages and pooled keys bit-exact (pad rows zero),
    selection and pointer table, then every row of JOINT, GATED and the three-branch Eq. 1 against the oracle."""
    w = _paper_like(**PAPER_CASES[case])
    d = synth.generate(w)
    n_pages = -(-(w.n_hist + w.S) // w.B)
    pm = synth.permuted_chunk_map(w.H, -(-n_pages // w.bpc), w.bpc, case + 90) if w.bpc else synth.permuted_page_map(w.H, n_pages, case + 90)
    oc = build_oracle_cache(w, d, pm)
    oracle.pool_values(oc)
    ls = build_gpu(w, d, pm, want_lse=True, cmp=True)
    torch.cuda.synchronize()
    flat = oc.page_map
    P = w.P or w.B
    for h in range(w.H):
        used = torch.from_numpy(flat[h, :w.n_b].astype(np.int64)).cuda()
        for gp, op in ((ls.cache.k_pages, oc.k_pages), (ls.cache.v_pages, oc.v_pages)):
            assert np.array_equal(bits(gp[h, used][:, :w.B]), as_bf16_bits(op[h, flat[h, :w.n_b]]))
            assert P == w.B or not gp[h, used][:, w.B:].any()  # pad rows stay zero
    assert np.array_equal(bits(ls.cache.pooled_k[:, :w.n_b]), as_bf16_bits(oc.pooled_k[:, :w.n_b]))
    assert np.array_equal(bits(ls.cache.pooled_v[:, :w.n_b]), as_bf16_bits(oc.pooled_v[:, :w.n_b]))
    sel = check_select(w, d, ls, oc, expect_exact_sets=False)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_JOINT)
    check_attention(w, d, ls, oc, sel, fuse_mode=om.FUSE_GATED, g_slc=np.linspace(0.2, 0.9, w.H).astype(np.float32),
                    g_swa=np.linspace(0.8, 0.3, w.H).astype(np.float32))
    check_attention3(w, d, ls, oc, sel)
    check_select(w, d, ls, oc, expect_exact_sets=False, score_mode=om.SCORE_PROB)


def test_paper_geometry_full_size():
    """The paper's default configuration at full size (12 heads x 128, 4680-token chunk = 156 blocks of 30 tokens, 20 chunks of
    history, window 3 chunks, G_q 15, top-4, two-level map): selection in full, attention (JOINT and GATED) on sampled rows,
    and the benchmarked step() with the GPU-built table."""
    w = synth.config("paper")
    d = synth.generate(w)
    n_chunks = (w.n_hist + w.S) // w.chunk
    pm = synth.permuted_chunk_map(w.H, n_chunks, w.bpc, 123)
    oc = build_oracle_cache(w, d, pm)
    ls = build_gpu(w, d, pm, want_lse=True)
    sel = check_select(w, d, ls, oc, expect_exact_sets=False)
    a = sel["awe"]
    assert a["active"] and a["b_w"] == 17 * 156 and np.all(sel["block_idx"] < a["b_w"])
    rows = synth.sample_rows(w, 6, 3)
    e = check_attention(w, d, ls, oc, sel, rows=rows, fuse_mode=om.FUSE_JOINT)
    g1 = np.linspace(0.2, 0.9, w.H).astype(np.float32)
    g2 = np.linspace(0.8, 0.3, w.H).astype(np.float32)
    eg = check_attention(w, d, ls, oc, sel, rows=rows, fuse_mode=om.FUSE_GATED, g_slc=g1, g_swa=g2)
    es = check_step(w, d, ls, oc, rows, fuse_mode=om.FUSE_JOINT)
    print(f"paper geometry: JOINT max-abs {e[0]:.3e} mean-abs {e[1]:.3e}; GATED {eg[0]:.3e} / {eg[1]:.3e}; step() {es[0]:.3e} / {es[1]:.3e} on "
          f"{len(rows[0])} of {w.H * w.S} rows; near-tie rows {sel['near_tie_rows']} of {w.H * w.R}")


# ------------------------------------------------------------------------------------ NEXT-4: offload / reload
@pytest.mark.parametrize("mode,G", [(om.OFFLOAD_WAIT, 4), (om.OFFLOAD_SKIP, 4), (om.OFFLOAD_WAIT, 3), (om.OFFLOAD_SKIP, 9)])
def test_offload_rollout(mode, G):
    """A chunk-by-chunk rollout with only G chunk slots per head in HBM: every chunk is written through to pinned
    host memory, the window chunk stays pinned, selections reach back to offloaded chunks.  WAIT (Alg. 1 lines 9-11): after the
    host step the attention reads every selected block that fits -- the output equals the oracle's over the FULL history (or with
    exactly the blocks the model says stay on the host).  SKIP (:339): entries of chunks that were not resident are skipped --
    the output equals the oracle's with those entries masked.  Residency pattern, hit / reload / eviction counters and the number
    of skipped entries are compared with oracle.OffloadModel at every step."""
    from paper_2605_30519_b200.runner import LayerStep
    n_chunks, S = 8, 150
    w = _paper_like(H=2, S=S, n_hist=n_chunks * S, n_wt=S, t_awe=5, K=2, G=75)  # few blocks per step: the working set fits G slots
    d = synth.generate(w)
    ls = LayerStep(w, "cuda:0", want_lse=True, resident_chunks=G, pinned_recent=1)
    model = oracle.OffloadModel(w.H, G, 1)
    _, k_cur, v_cur = dev_inputs(d)
    hh, qq = np.meshgrid(np.arange(w.H, dtype=np.int32), np.arange(0, w.S, 7, dtype=np.int32), indexing="ij")
    hh, qq = hh.ravel(), qq.ravel()
    stats = None
    for c in range(n_chunks):
        lo = c * S
        ls.append(to_dev_chunk(d["k_hist"][:, lo:lo + S]), to_dev_chunk(d["v_hist"][:, lo:lo + S]))
        model.append(c)
        if c < 3:
            continue
        # the oracle's view of the history so far
        oc_c = oracle.cache_create(w.H, w.D, w.B, w.n_hist + w.S)
        for cc in range(c + 1):
            oracle.append_chunk(oc_c, d["k_hist"][:, cc * S:(cc + 1) * S], d["v_hist"][:, cc * S:(cc + 1) * S])
        oracle.pool_keys(oc_c)
        q_np = np.ascontiguousarray(np.roll(d["q"], 13 * c, axis=2))  # a different query chunk every step: the selections move
        q = to_dev_chunk(q_np)
        sel = oracle.select(oc_c, q_np, w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
        ls.want_scores = False
        ls.select(q)
        g_idx = ls.block_idx.cpu().numpy()
        assert np.array_equal(g_idx, sel["block_idx"])  # the selection itself does not depend on residency
        need = [set((g_idx[h][g_idx[h] >= 0] // w.bpc).tolist()) for h in range(w.H)]
        before, after = model.step(need)
        stats = om.omnimem_offload_step(ls.cache, ls.block_idx, ls.ptr_table, mode)
        g_ptr = ls.ptr_table.cpu().numpy()
        live = before if mode == om.OFFLOAD_SKIP else after
        want_on = np.zeros_like(g_idx, dtype=bool)
        for h in range(w.H):
            want_on[h] = (g_idx[h] >= 0) & np.isin(g_idx[h] // w.bpc, sorted(live[h]))
        assert np.array_equal(g_ptr >= 0, want_on), f"chunk {c}: residency pattern"
        assert (stats["requests"], stats["hits"], stats["reloads"], stats["evictions"]) == (model.requests, model.hits, model.reloads, model.evictions)
        assert stats["skipped"] == int(((g_idx >= 0) & ~want_on).sum())
        # attention through the GPU's table against the oracle with exactly the live entries
        masked = np.where(want_on, g_idx, -1).astype(np.int32)
        want, _ = oracle.sparse_attn_rows(oc_c, hh, qq, q_np, d["k_cur"], d["v_cur"], masked, oracle.ptr_table(masked, oc_c.page_map),
                                          G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale)
        ls.out.fill_(float("nan"))
        out = ls.attend(q, k_cur, v_cur)
        torch.cuda.synchronize()
        err = np.abs(out.float().cpu().numpy()[hh, qq] - want)
        assert err.max() <= 2e-2 and err.mean() <= 2e-3, (c, err.max(), err.mean())
    assert stats["requests"] > 0 and abs(stats["hit_rate"] - model.hit_rate) < 1e-12
    if G >= 9:
        assert stats["reloads"] == 0 and stats["skipped"] == 0  # everything fits: nothing is ever offloaded
    else:
        assert stats["reloads"] > 0                             # the selections did reach back to offloaded chunks
    print(f"offload mode={mode} G={G}: hit rate {stats['hit_rate']:.3f}, reloads {stats['reloads']}, evictions {stats['evictions']}")


def to_dev_chunk(a):
    from paper_2605_30519_b200.runner import to_dev
    return to_dev(a, "cuda:0")


# ------------------------------------------------------------------------------------ BASELINE full sizes
# configs 2, 3, 4 and EVERY member of config 5's grid: B {64,128} x K {8,16,32,64} x G_q {64,4680} + the two short-history cases
FULL = {w.name: w for w in [synth.config("wan1p3b"), synth.config("long"), synth.config("wan14b")] + synth.sweep_configs()}
assert len(FULL) == 21


@pytest.mark.parametrize("name", list(FULL))
def test_full_size_configs(name):
    """Full-size configs in the launch configuration bench.py times: selection compared in full
    (bit-exact on identical scores), attention on a deterministic row sample (5+ groups per head incl.
    first/last, first/last row of each group)."""
    w = FULL[name]
    d = synth.generate(w)
    oc = build_oracle_cache(w, d)
    ls = build_gpu(w, d, want_lse=True)
    sel = check_select(w, d, ls, oc, expect_exact_sets=False)
    a = sel["awe"]
    if name.startswith("short"):
        assert not a["active"] and a["omega_end"] == w.n_b  # AWE must not exclude (config 5)
    else:
        assert a["active"] and np.all(sel["block_idx"] < a["b_w"])
    per_head, union = oracle.union_counts(sel["block_idx"], w.n_b)
    assert per_head.sum() <= w.H * union and np.all(per_head <= w.R * w.K)
    n_groups = 5 if w.H <= 12 else 3
    rows = synth.sample_rows(w, n_groups, 4)
    e = check_attention(w, d, ls, oc, sel, rows=rows, fuse_mode=om.FUSE_JOINT, use_gpu_table=False)
    print(f"{name}: JOINT max-abs {e[0]:.3e} mean-abs {e[1]:.3e} on {len(rows[0])} of {w.H * w.S} rows; near-tie rows "
          f"{sel['near_tie_rows']} of {w.H * w.R}; sum|U_h|={per_head.sum()} |U|={union} H*|U|={w.H * union}")
    if name in ("wan1p3b", "short_B128", "sweep_B128_K8_G4680"):
        g1 = np.linspace(0.2, 0.9, w.H).astype(np.float32)
        g2 = np.linspace(0.8, 0.3, w.H).astype(np.float32)
        check_attention(w, d, ls, oc, sel, rows=rows, fuse_mode=om.FUSE_GATED, g_slc=g1, g_swa=g2)


@pytest.mark.parametrize("name", ["wan1p3b", "long", "wan14b", "short_B64"])
def test_full_size_step_as_benchmarked(name):
    """bench.py's timed configuration at full size: LayerStep.step() (GPU-built table, scores in the workspace, the
    launches chained by PDL), sampled rows against the oracle evaluated on the GPU's own selection; JOINT and GATED."""
    w = FULL[name]
    d = synth.generate(w)
    oc = build_oracle_cache(w, d)
    ls = build_gpu(w, d)
    rows = synth.sample_rows(w, 5 if w.H <= 12 else 3, 4)
    e = check_step(w, d, ls, oc, rows, fuse_mode=om.FUSE_JOINT)
    print(f"{name} step(): JOINT max-abs {e[0]:.3e} mean-abs {e[1]:.3e} on {len(rows[0])} of {w.H * w.S} rows; {e[2]} near-tie rows")
    g1 = np.linspace(0.2, 0.9, w.H).astype(np.float32)
    g2 = np.linspace(0.8, 0.3, w.H).astype(np.float32)
    e = check_step(w, d, ls, oc, rows, fuse_mode=om.FUSE_GATED, g_slc=g1, g_swa=g2)
    print(f"{name} step(): GATED max-abs {e[0]:.3e} mean-abs {e[1]:.3e}; {e[2]} near-tie rows")
