"""Device-side plumbing for one attention layer of one AR step: allocate the buffers a workload needs,
feed history chunk by chunk through ``omnimem_append_chunk`` / ``omnimem_pool_keys`` and run
``omnimem_select`` + ``omnimem_sparse_attn``.  Used by the GPU tests, ``bench.py`` and ``smoke()``.
All arithmetic happens inside the C-ABI calls; this file only owns torch tensors.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as om
from .synth import Workload


def to_dev(a: np.ndarray, device) -> torch.Tensor:
    """float32 array holding bf16-representable values -> bf16 device tensor (exact)."""
    return torch.from_numpy(np.ascontiguousarray(a)).to(device=device, dtype=torch.bfloat16)


class LayerStep:
    def __init__(self, w: Workload, device="cuda:0", page_map: np.ndarray | None = None,
                 fuse_mode: int = om.FUSE_JOINT, want_scores: bool = False, want_lse: bool = False,
                 max_tokens: int | None = None, cmp: bool = False, resident_chunks: int = 0, pinned_recent: int = 1):
        self.w, self.device = w, torch.device(device)
        pm = None if page_map is None else torch.from_numpy(np.ascontiguousarray(page_map))
        self.cache = om.OmniMemCache(w.H, w.D, w.B, max_tokens or (w.n_hist + w.S), device, pm, page_tokens=w.P, blocks_per_chunk=w.bpc,
                                     resident_chunks=resident_chunks, pinned_recent=pinned_recent)
        self.three = False  # True: attend() runs the three-branch call (omnimem_sparse_attn3)
        if cmp:  # the compression branch of Eq. 1: the compressed cache also keeps block values
            self.cache.attach_pooled_v()
        self.sp = om.SelectParams(w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
        self.ap = om.AttnParams(w.G, w.K, w.n_wt, w.softmax_scale, fuse_mode, 0)
        sel_b, att_b = self.cache.workspace_bytes(w.S, self.sp, self.ap)
        # the tests flip fuse_mode on a live LayerStep: size the scratch for either mode
        other = om.AttnParams(w.G, w.K, w.n_wt, w.softmax_scale, 1 - fuse_mode, 0)
        att_b = max(att_b, self.cache.workspace_bytes(w.S, None, other)[1])
        sp_prob = om.SelectParams(w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale, om.SCORE_PROB)  # ... and score_mode
        sel_b = max(sel_b, self.cache.workspace_bytes(w.S, sp_prob, None)[0])
        self.ws_select = torch.empty(max(sel_b, 16), dtype=torch.uint8, device=self.device)
        self.ws_attn = torch.empty(max(att_b, 16), dtype=torch.uint8, device=self.device)
        self.block_idx = torch.full((w.H, w.R, w.K), -2, dtype=torch.int32, device=self.device)
        self.ptr_table = torch.full((w.H, w.R, w.K), -2, dtype=torch.int32, device=self.device)
        self.out = torch.empty((w.H, w.S, w.D), dtype=torch.bfloat16, device=self.device)
        self.scores = None
        self.want_scores = want_scores
        self.lse = torch.empty((2, w.H, w.S), dtype=torch.float32, device=self.device) if want_lse else None
        self.gate_slc = torch.ones(w.H, dtype=torch.float32, device=self.device)
        self.gate_swa = torch.ones(w.H, dtype=torch.float32, device=self.device)
        self.gate_cmp = torch.ones(w.H, dtype=torch.float32, device=self.device)
        self.lse3 = torch.empty((3, w.H, w.S), dtype=torch.float32, device=self.device) if (cmp and want_lse) else None
        self.awe = None

    # ---- history ------------------------------------------------------------------------------
    def append(self, k_chunk: torch.Tensor, v_chunk: torch.Tensor, pool: bool = True) -> None:
        om.omnimem_append_chunk(self.cache, k_chunk, v_chunk)
        if pool:
            om.omnimem_pool_keys(self.cache, 0, -1)

    def load_history(self, k_hist: np.ndarray, v_hist: np.ndarray, chunk: int | None = None) -> None:
        chunk = chunk or self.w.chunk
        n = k_hist.shape[1]
        for lo in range(0, n, chunk):
            hi = min(lo + chunk, n)
            self.append(to_dev(k_hist[:, lo:hi], self.device), to_dev(v_hist[:, lo:hi], self.device))

    # ---- one step -----------------------------------------------------------------------------
    def select(self, q: torch.Tensor) -> dict:
        if self.want_scores:
            n_b = self.cache.n_blocks
            if self.scores is None or self.scores.shape[2] != n_b:
                self.scores = torch.empty((self.w.H, self.w.R, n_b), dtype=torch.float32, device=self.device)
        self.awe = om.omnimem_select(self.cache, q, self.sp, self.block_idx, self.ptr_table,
                                     self.scores if self.want_scores else None, self.ws_select)
        return self.awe

    def attend(self, q: torch.Tensor, k_cur: torch.Tensor, v_cur: torch.Tensor) -> torch.Tensor:
        if self.three:
            return self.attend3(q, k_cur, v_cur)
        om.omnimem_sparse_attn(self.cache, q, k_cur, v_cur, self.ptr_table, self.ap, self.out, self.gate_slc,
                               self.gate_swa, self.lse, self.ws_attn)
        return self.out

    def attend3(self, q: torch.Tensor, k_cur: torch.Tensor, v_cur: torch.Tensor) -> torch.Tensor:
        """Full Eq. 1: gate_cmp Attn_CMP + gate_slc Attn_SLC + gate_swa Attn_SWA (needs cmp=True)."""
        ap = om.AttnParams(self.ap.group_tokens, self.ap.top_k, self.ap.window_tokens, self.ap.softmax_scale, om.FUSE_GATED, 0)
        om.omnimem_sparse_attn3(self.cache, q, k_cur, v_cur, self.ptr_table, ap, self.out, self.gate_cmp, self.gate_slc,
                                self.gate_swa, self.lse3, self.ws_attn)
        return self.out

    def step(self, q, k_cur, v_cur) -> torch.Tensor:
        self.select(q)
        return self.attend(q, k_cur, v_cur)


class HostPipeline:
    """Steps whose inputs and result live in HOST memory (pinned): the host->device copies of step i + 1, the kernels of step i
    and the device->host copy of step i - 1 run on three streams over double-buffered device tensors, so a stream of steps costs
    max(copy in, compute, copy out) per step instead of their sum.  Plumbing only: every step still runs ``LayerStep.step``.
    """

    def __init__(self, ls: LayerStep):
        self.ls = ls
        w, dev = ls.w, ls.device
        mk = lambda: torch.empty((w.H, w.S, w.D), dtype=torch.bfloat16, device=dev)
        self.q, self.k, self.v, self.o = ([mk(), mk()] for _ in range(4))
        self.s_in, self.s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        self.in_ready = [torch.cuda.Event(), torch.cuda.Event()]    # inputs of the slot have arrived
        self.in_free = [torch.cuda.Event(), torch.cuda.Event()]     # the kernels that read the slot's inputs are done
        self.out_ready = [torch.cuda.Event(), torch.cuda.Event()]   # the slot's result is complete
        self.out_free = [torch.cuda.Event(), torch.cuda.Event()]    # the slot's result has left for the host
        self.i = 0

    def submit(self, hq: torch.Tensor, hk: torch.Tensor, hv: torch.Tensor, hout: torch.Tensor) -> None:
        """Enqueue one step: copy (hq, hk, hv) in, select + attend, copy the result to ``hout``.  Returns at once; the host
        buffers may be reused after ``drain()`` (or once two more steps have been submitted)."""
        s, cur, first = self.i & 1, torch.cuda.current_stream(self.ls.device), self.i < 2
        if not first:
            self.s_in.wait_event(self.in_free[s])
        with torch.cuda.stream(self.s_in):
            self.q[s].copy_(hq, non_blocking=True)
            self.k[s].copy_(hk, non_blocking=True)
            self.v[s].copy_(hv, non_blocking=True)
            self.in_ready[s].record(self.s_in)
        cur.wait_event(self.in_ready[s])
        if not first:
            cur.wait_event(self.out_free[s])
        keep = self.ls.out
        self.ls.out = self.o[s]
        self.ls.step(self.q[s], self.k[s], self.v[s])
        self.ls.out = keep
        self.in_free[s].record(cur)
        self.out_ready[s].record(cur)
        self.s_out.wait_event(self.out_ready[s])
        with torch.cuda.stream(self.s_out):
            hout.copy_(self.o[s], non_blocking=True)
            self.out_free[s].record(self.s_out)
        self.i += 1

    def drain(self) -> None:
        cur = torch.cuda.current_stream(self.ls.device)
        cur.wait_stream(self.s_in)
        cur.wait_stream(self.s_out)
