"""omnimem_union_counts_noalloc (include/omnimem.h): the union accounting of a selection (Eqs. 4-5) with its
scratch in a device array built into the library instead of caller memory -- for callers that cannot allocate.  Compared bit
for bit (integer work) with the existing path, omnimem_union_counts on caller scratch, and with the oracle, on two calls in a
row whose selections differ (the array keeps the first call's marks: the second result is only right if the call clears what
it uses).  This file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide other tests."""
import numpy as np
import pytest
import torch

import oracle
from paper_2605_30519_b200 import binding as om
from paper_2605_30519_b200 import synth

from _parity import build_gpu, dev_inputs

pytestmark = pytest.mark.gpu


def _both_paths(ls, block_idx, n_b, H):
    """(per_head, union_all, union_list) from the existing path and from the no-allocation entry point."""
    res = []
    for noalloc in (False, True):
        per_head = torch.full((H,), -1, dtype=torch.int64, device="cuda:0")
        union_all = torch.full((1,), -1, dtype=torch.int64, device="cuda:0")
        union_list = torch.full((max(n_b, 1),), -1, dtype=torch.int32, device="cuda:0")
        if noalloc:
            om.omnimem_union_counts_noalloc(ls.cache, block_idx, per_head, union_all, union_list)
        else:
            ws = torch.empty((H + 1) * max(n_b, 1), dtype=torch.uint8, device="cuda:0")
            om.omnimem_union_counts(ls.cache, block_idx, per_head, union_all, union_list, ws)
        torch.cuda.synchronize()
        res.append((per_head.cpu().numpy(), int(union_all.item()), union_list.cpu().numpy()))
    return res


def test_union_counts_noalloc_matches_existing_path_twice():
    # call 1: many distinct blocks marked (K = 64 of 47 blocks per group); call 2: another cache of the SAME N_b row length with a
    # sparse selection (K = 2), so every mark call 1 left behind that call 2 does not clear would be counted
    cases = [dict(H=4, K=64, n_hist=3000, G=15, S=100), dict(H=4, K=2, n_hist=3000, G=50, S=100, D=128)]
    for i, over in enumerate(cases):
        w = synth.config("tiny", **over)
        d = synth.generate(w)
        pm = synth.permuted_page_map(w.H, -(-(w.n_hist + w.S) // w.B), 5 + i)
        ls = build_gpu(w, d, pm)
        q, _, _ = dev_inputs(d)
        ls.select(q)
        torch.cuda.synchronize()
        n_b = ls.cache.n_blocks
        (ph0, u0, l0), (ph1, u1, l1) = _both_paths(ls, ls.block_idx, n_b, w.H)
        assert np.array_equal(ph0, ph1) and u0 == u1 and np.array_equal(l0, l1), f"call {i + 1}: the two paths differ"
        g_idx = ls.block_idx.cpu().numpy()
        want_ph, want_u = oracle.union_counts(g_idx, n_b)
        assert np.array_equal(ph1, want_ph) and u1 == want_u, f"call {i + 1}: differs from the oracle"
        assert np.array_equal(l1[:want_u], np.unique(g_idx[g_idx >= 0]))
    assert cases[0]["K"] > cases[1]["K"] and u1 < n_b  # the second selection really is the sparser one

    # the same call again, back to back on one stream without a synchronize in between: same answer, and the driver's free
    # memory does not move (a cudaMalloc inside the call would lower it)
    per_head = torch.full((2, w.H), -1, dtype=torch.int64, device="cuda:0")
    union_all = torch.full((2, 1), -1, dtype=torch.int64, device="cuda:0")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    om.omnimem_union_counts_noalloc(ls.cache, ls.block_idx, per_head[0], union_all[0], None)
    om.omnimem_union_counts_noalloc(ls.cache, ls.block_idx, per_head[1], union_all[1], None)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    assert np.array_equal(per_head[0].cpu().numpy(), want_ph) and np.array_equal(per_head[1].cpu().numpy(), want_ph)
    assert int(union_all[0].item()) == int(union_all[1].item()) == want_u


def test_union_counts_noalloc_rejects_sizes_beyond_the_builtin_array():
    # (H + 1) * N_b = 33 * 32800 bytes of marks > 1 MiB: a clear ECAPACITY, nothing launched.  One-token blocks in 32-row pages keep
    # the cache this needs small in tokens (it still holds H * N_b pages: 2 x 4.3 GB, released right after)
    H, n_b = 32, 32800
    assert (H + 1) * n_b > om.UNION_NOALLOC_MAX_BYTES
    cache = om.OmniMemCache(H, 64, 1, n_b, "cuda:0", page_tokens=32)
    kv = torch.zeros((H, n_b, 64), dtype=torch.bfloat16, device="cuda:0")
    om.omnimem_append_chunk(cache, kv, kv)
    assert cache.n_blocks == n_b
    idx = torch.zeros((H, 1, 1), dtype=torch.int32, device="cuda:0")
    per_head = torch.zeros(H, dtype=torch.int64, device="cuda:0")
    union_all = torch.zeros(1, dtype=torch.int64, device="cuda:0")
    before = om.launch_count()
    with pytest.raises(om.OmniMemError) as e:
        om.omnimem_union_counts_noalloc(cache, idx, per_head, union_all, None)
    assert e.value.code == om.ECAPACITY and "exceed" in str(e.value)
    assert om.launch_count() == before
    # the existing path takes the same case with caller scratch
    ws = torch.empty((H + 1) * n_b, dtype=torch.uint8, device="cuda:0")
    om.omnimem_union_counts(cache, idx, per_head, union_all, None, ws)
    torch.cuda.synchronize()
    assert int(union_all.item()) == 1 and np.all(per_head.cpu().numpy() == 1)
    del cache, kv, ws
    torch.cuda.empty_cache()
