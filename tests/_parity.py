"""Shared helpers of the GPU parity tests: run the CUDA path (through the C-ABI binding) and the CPU
oracle on the same seeded inputs and compare.  Tolerances (north_star): block indices and pointer
tables bit-exact given the same fp32 scores; attention within max-abs 2e-2 and mean-abs 2e-3."""
import numpy as np
import torch

import oracle
from paper_2605_30519_b200 import binding as om
from paper_2605_30519_b200 import synth
from paper_2605_30519_b200.runner import LayerStep, to_dev

ATTN_MAX_ABS = 2e-2
ATTN_MEAN_ABS = 2e-3


def build_oracle_cache(w, d, page_map=None, chunk=None):
    if w.bpc > 0 and page_map is not None:  # two-level map: the oracle's storage follows the flat map it stands for
        page_map = oracle.expand_chunk_map(page_map, w.bpc, page_map.shape[1] * w.bpc)
    c = oracle.cache_create(w.H, w.D, w.B, w.n_hist + w.S, page_map)
    chunk = chunk or w.chunk
    for lo in range(0, w.n_hist, chunk):
        hi = min(lo + chunk, w.n_hist)
        oracle.append_chunk(c, d["k_hist"][:, lo:hi], d["v_hist"][:, lo:hi])
    oracle.pool_keys(c)
    return c


def gpu_page_map(w, ls):
    """The flat block -> page map of the GPU cache (expanded from the chunk bases under the two-level map)."""
    if w.bpc <= 0:
        return ls.cache.page_map.cpu().numpy()
    n_chunks = -(-ls.cache.max_blocks // w.bpc)
    cm = ls.cache.page_map.view(-1)[:w.H * n_chunks].view(w.H, n_chunks).cpu().numpy()
    return oracle.expand_chunk_map(cm, w.bpc, ls.cache.max_blocks)


def build_gpu(w, d, page_map=None, chunk=None, **kw):
    ls = LayerStep(w, "cuda:0", page_map, **kw)
    ls.load_history(d["k_hist"], d["v_hist"], chunk)
    return ls


def dev_inputs(d):
    return to_dev(d["q"], "cuda:0"), to_dev(d["k_cur"], "cuda:0"), to_dev(d["v_cur"], "cuda:0")


def check_select(w, d, ls, oc, expect_exact_sets=True, inputs=None, score_mode=0):
    """Runs omnimem_select and the oracle's select; returns the oracle selection.
    (a) GPU scores ~ oracle scores; (b) oracle top-k of the GPU's own scores == GPU block_idx bit-exact;
    (c) GPU top-k of the ORACLE's scores == oracle block_idx bit-exact; (d) ptr_table == page_map[block_idx];
    (e) end to end, selections agree except where the oracle's own K-th/(K+1)-th gap is a near-tie."""
    q, _, _ = inputs or dev_inputs(d)
    ls.want_scores = True
    ls.sp.score_mode = score_mode
    awe = ls.select(q)
    torch.cuda.synchronize()
    sel = oracle.select(oc, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale, score_mode)
    # score tolerance: logit mode 1e-5 * max|s| (fp32 accumulation of exact bf16 products); probability mode 2e-4 * max s
    # (a logit error of 1e-5 * 8 log2 units and ex2.approx's 2^-22 give a relative error near 1e-4 per probability)
    rel = 1e-5 if score_mode == 0 else 2e-4
    oa = sel["awe"]
    assert (awe["n_b"], awe["b_w"], awe["omega_end"], awe["active"], awe["n_groups"]) == \
        (oa["n_b"], oa["b_w"], oa["omega_end"], oa["active"], w.R)
    g_idx = ls.block_idx.cpu().numpy()
    g_ptr = ls.ptr_table.cpu().numpy()
    pm = gpu_page_map(w, ls)
    assert np.array_equal(pm, oc.page_map)
    if oa["n_b"] > 0:
        g_scores = ls.scores.cpu().numpy()
        smax = float(np.abs(sel["scores"]).max()) + 1e-30
        assert np.max(np.abs(g_scores - sel["scores"])) <= rel * smax + 1e-6, "scores"
        assert not np.any(np.signbit(g_scores) & (g_scores == 0))
        # (b)
        assert np.array_equal(oracle.topk(g_scores, oa["omega_end"], w.K), g_idx), "top-k of GPU scores"
        # (c)
        idx2 = torch.full_like(ls.block_idx, -2)
        ptr2 = torch.full_like(ls.ptr_table, -2)
        om.omnimem_select_from_scores(ls.cache, torch.from_numpy(sel["scores"]).cuda(), w.S, ls.sp, idx2, ptr2)
        torch.cuda.synchronize()
        assert np.array_equal(idx2.cpu().numpy(), sel["block_idx"]), "GPU top-k of oracle scores"
        assert np.array_equal(ptr2.cpu().numpy(), sel["ptr_table"]), "GPU table of oracle scores"
    # (d)
    assert np.array_equal(g_ptr, oracle.ptr_table(g_idx, pm))
    if w.bpc > 0:  # Alg. 1 lines 7-12 on the chunk bases themselves
        n_chunks = -(-ls.cache.max_blocks // w.bpc)
        cm = ls.cache.page_map.view(-1)[:w.H * n_chunks].view(w.H, n_chunks).cpu().numpy()
        assert np.array_equal(g_ptr, oracle.ptr_table_chunked(g_idx, cm, w.bpc))
    # (e)
    differ = np.argwhere(np.any(g_idx != sel["block_idx"], axis=2))
    near_tie = 0
    for h, r in differ:
        srt = np.sort(sel["scores"][h, r, :oa["omega_end"]])[::-1]
        gaps = np.abs(np.diff(srt[:w.K + 1]))
        assert gaps.size and gaps.min() <= 2 * rel * smax, (h, r, "selection differs without a near-tie")
        near_tie += 1
    if expect_exact_sets:
        assert near_tie == 0, f"{near_tie} near-tie rows (expected 0)"
    sel["near_tie_rows"] = near_tie
    return sel


def check_step(w, d, ls, oc, rows, fuse_mode=0, g_slc=None, g_swa=None):
    """The configuration bench.py times: ONE LayerStep.step() -- omnimem_select writing its scores to the workspace
    (scores_out = NULL) and omnimem_sparse_attn consuming the GPU-built pointer table, all launches chained by
    programmatic dependent launch with nothing in between.  The table must agree with the oracle's except on rows the
    oracle itself ranks as near-ties (reading A17; counted and returned), and the attention output is compared on
    `rows` with the oracle evaluated on the GPU's own block_idx (legal wherever that selection is valid)."""
    q, k_cur, v_cur = dev_inputs(d)
    ls.want_scores = False
    ls.scores = None
    ls.ap.fuse_mode = fuse_mode
    if g_slc is not None:
        ls.gate_slc.copy_(torch.from_numpy(g_slc))
        ls.gate_swa.copy_(torch.from_numpy(g_swa))
    ls.block_idx.fill_(-7)
    ls.ptr_table.fill_(-7)
    ls.out.fill_(float("nan"))
    out = ls.step(q, k_cur, v_cur)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy()
    g_idx, g_ptr = ls.block_idx.cpu().numpy(), ls.ptr_table.cpu().numpy()
    sel = oracle.select(oc, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    oa = sel["awe"]
    assert np.array_equal(g_ptr, oracle.ptr_table(g_idx, oc.page_map)), "ptr_table != page_map[block_idx]"
    # validity of the GPU selection: in range, distinct, K_eff entries, masked tail
    k_eff = min(w.K, oa["omega_end"])
    assert np.all(g_idx[:, :, :k_eff] >= 0) and np.all(g_idx[:, :, :k_eff] < max(oa["omega_end"], 1)) and np.all(g_idx[:, :, k_eff:] == -1)
    srt = np.sort(g_idx[:, :, :k_eff], axis=2)
    assert k_eff < 2 or np.all(np.diff(srt, axis=2) > 0), "duplicate block in a selection"
    differ = np.argwhere(np.any(g_idx != sel["block_idx"], axis=2))
    smax = float(np.abs(sel["scores"]).max()) + 1e-30 if oa["n_b"] > 0 else 1.0
    for h, r in differ:
        top = np.sort(sel["scores"][h, r, :oa["omega_end"]])[::-1]
        gaps = np.abs(np.diff(top[:w.K + 1]))
        assert gaps.size and gaps.min() <= 1e-5 * smax, (h, r, "selection differs without a near-tie")
    hh, qq = rows
    want, _ = oracle.sparse_attn_rows(oc, hh, qq, d["q"], d["k_cur"], d["v_cur"], g_idx, g_ptr, G=w.G, K=w.K, n_wt=w.n_wt,
                                      softmax_scale=w.softmax_scale, fuse_mode=fuse_mode, g_slc=g_slc, g_swa=g_swa)
    assert np.all(np.isfinite(out)), "non-finite or unwritten output rows"
    err = np.abs(out[hh, qq] - want)
    assert err.max() <= ATTN_MAX_ABS, f"max-abs {err.max():.4g}"
    assert err.mean() <= ATTN_MEAN_ABS, f"mean-abs {err.mean():.4g}"
    return float(err.max()), float(err.mean()), len(differ)


def check_attention(w, d, ls, oc, sel, rows=None, fuse_mode=0, g_slc=None, g_swa=None, use_gpu_table=False, inputs=None):
    """omnimem_sparse_attn (fed the ORACLE's table so that both sides attend to the same blocks) vs the
    oracle on `rows` (default: every row)."""
    q, k_cur, v_cur = inputs or dev_inputs(d)
    if not use_gpu_table:
        ls.ptr_table.copy_(torch.from_numpy(sel["ptr_table"]))
    ls.ap.fuse_mode = fuse_mode
    if g_slc is not None:
        ls.gate_slc.copy_(torch.from_numpy(g_slc))
        ls.gate_swa.copy_(torch.from_numpy(g_swa))
    if ls.lse is None:
        ls.lse = torch.empty((2, w.H, w.S), dtype=torch.float32, device="cuda:0")
    ls.out.fill_(float("nan"))
    out = ls.attend(q, k_cur, v_cur)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy()
    lse = ls.lse.cpu().numpy()
    if rows is None:
        hh, qq = np.meshgrid(np.arange(w.H, dtype=np.int32), np.arange(w.S, dtype=np.int32), indexing="ij")
        hh, qq = hh.ravel(), qq.ravel()
    else:
        hh, qq = rows
    want, want_lse = oracle.sparse_attn_rows(oc, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"],
                                             G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale, fuse_mode=fuse_mode,
                                             g_slc=g_slc, g_swa=g_swa)
    got = out[hh, qq]
    assert np.all(np.isfinite(out)), "non-finite or unwritten output rows"
    err = np.abs(got - want)
    assert err.max() <= ATTN_MAX_ABS, f"max-abs {err.max():.4g}"
    assert err.mean() <= ATTN_MEAN_ABS, f"mean-abs {err.mean():.4g}"
    got_lse = lse[:, hh, qq]
    fin = np.isfinite(want_lse)
    assert np.array_equal(np.isneginf(got_lse), np.isneginf(want_lse)), "LSE -inf pattern"
    if fin.any():
        assert np.max(np.abs(got_lse[fin] - want_lse[fin])) <= 2e-2, "LSE"
    return float(err.max()), float(err.mean())
