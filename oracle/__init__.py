"""CPU oracle for the OmniMem hot path -- TEST INFRASTRUCTURE, not the product.

Thin numpy/ctypes front end of ``omnimem_oracle.c`` (plain C, double accumulation, written
from PAPER.md).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the CUDA path under
``paper_2605_30519_b200/`` never does, and this package imports nothing from it.

All arrays are C-contiguous numpy arrays.  Floating tensors are float32 holding
bf16-representable values.  Layouts are documented at the top of ``omnimem_oracle.c``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "omnimem_oracle.c")
_LIB = os.path.join(_HERE, "libomnimem_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (single translation unit, no dependencies)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_bf16_round.restype = ctypes.c_float
        _lib.oracle_bf16_round.argtypes = [ctypes.c_float]
        _lib.oracle_append_chunk.restype = ctypes.c_int64
        _lib.oracle_union_counts.restype = ctypes.c_int64
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(ctypes.c_void_p)


def _i32(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(ctypes.c_void_p)


I32, I64, F32 = ctypes.c_int32, ctypes.c_int64, ctypes.c_float


def bf16_round(x: float) -> float:
    return float(_load().oracle_bf16_round(F32(x)))


@dataclass
class OracleCache:
    """The two-level cache of PAPER.md:333-339 as plain arrays (everything resident)."""

    H: int
    D: int
    B: int
    n_pages: int
    k_pages: np.ndarray  # [H][n_pages][B][D]
    v_pages: np.ndarray
    pooled_k: np.ndarray  # [H][n_pages][D]
    page_map: np.ndarray  # [H][n_pages] int32
    n_hist: int = 0
    pooled_v: np.ndarray | None = None  # [H][n_pages][D], filled by pool_values (CMP branch)

    @property
    def n_blocks(self) -> int:
        return -(-self.n_hist // self.B)


def cache_create(H: int, D: int, B: int, max_tokens: int, page_map: np.ndarray | None = None) -> OracleCache:
    n_pages = -(-max_tokens // B)
    if page_map is None:
        page_map = np.tile(np.arange(n_pages, dtype=np.int32), (H, 1))
    page_map = np.ascontiguousarray(page_map, dtype=np.int32)
    assert page_map.shape == (H, n_pages)
    return OracleCache(
        H, D, B, n_pages,
        np.zeros((H, n_pages, B, D), np.float32), np.zeros((H, n_pages, B, D), np.float32),
        np.zeros((H, n_pages, D), np.float32), page_map, 0,
    )


def append_chunk(c: OracleCache, k_chunk: np.ndarray, v_chunk: np.ndarray) -> None:
    """a0."""
    k_chunk, kp = _f32(k_chunk)
    v_chunk, vp = _f32(v_chunk)
    H, n, D = k_chunk.shape
    assert (H, D) == (c.H, c.D) and v_chunk.shape == k_chunk.shape
    assert c.n_hist + n <= c.n_pages * c.B
    c.n_hist = int(_load().oracle_append_chunk(
        c.k_pages.ctypes.data_as(ctypes.c_void_p), c.v_pages.ctypes.data_as(ctypes.c_void_p),
        c.page_map.ctypes.data_as(ctypes.c_void_p), I32(c.H), I32(c.D), I32(c.B), I32(c.n_pages),
        I64(c.n_hist), kp, vp, I32(n)))


def pool_keys(c: OracleCache, first_block: int = 0, n_blocks: int | None = None) -> None:
    """a1."""
    if n_blocks is None:
        n_blocks = c.n_blocks - first_block
    _load().oracle_pool_keys(
        c.k_pages.ctypes.data_as(ctypes.c_void_p), c.page_map.ctypes.data_as(ctypes.c_void_p),
        I32(c.H), I32(c.D), I32(c.B), I32(c.n_pages), I64(c.n_hist), I64(first_block), I64(n_blocks),
        c.pooled_k.ctypes.data_as(ctypes.c_void_p))


def pool_values(c: OracleCache, first_block: int = 0, n_blocks: int | None = None) -> None:
    """NEXT-1: block values of the compressed cache, pooled like the keys."""
    if c.pooled_v is None:
        c.pooled_v = np.zeros((c.H, c.n_pages, c.D), np.float32)
    if n_blocks is None:
        n_blocks = c.n_blocks - first_block
    _load().oracle_pool_values(
        c.v_pages.ctypes.data_as(ctypes.c_void_p), c.page_map.ctypes.data_as(ctypes.c_void_p),
        I32(c.H), I32(c.D), I32(c.B), I32(c.n_pages), I64(c.n_hist), I64(first_block), I64(n_blocks),
        c.pooled_v.ctypes.data_as(ctypes.c_void_p))


def cmp_attn_rows(c: OracleCache, rows_h, rows_q, q, softmax_scale: float):
    """NEXT-1: compression attention Attn(Q, K^cmp, V^cmp) (Eq. 1) for a list of (head, query) rows
    over the head's N_b compressed tokens: returns (O_cmp [n][D] fp32, LSE_cmp [n] fp32).  Needs pool_keys + pool_values."""
    assert c.pooled_v is not None, "call pool_values first"
    rows_h, hp = _i32(rows_h)
    rows_q, qip = _i32(rows_q)
    q, qp = _f32(q)
    H, S, D = q.shape
    n = rows_h.shape[0]
    out = np.zeros((n, D), np.float32)
    lse = np.zeros(n, np.float32)
    _load().oracle_cmp_attn_rows(
        hp, qip, I64(n), qp, c.pooled_k.ctypes.data_as(ctypes.c_void_p), c.pooled_v.ctypes.data_as(ctypes.c_void_p),
        I32(S), I32(D), I32(c.n_pages), I64(c.n_blocks), F32(softmax_scale),
        out.ctypes.data_as(ctypes.c_void_p), lse.ctypes.data_as(ctypes.c_void_p))
    return out, lse


def gated3_rows(c: OracleCache, rows_h, rows_q, q, k_cur, v_cur, block_idx, ptr, *, G: int, K: int, n_wt: int,
                softmax_scale: float, g_cmp, g_slc, g_swa):
    """The full Eq. 1: o = g_cmp Attn_cmp + g_slc Attn_slc + g_swa Attn_swa, per-head gates.
    Returns (out [n][D], lse [3][n]) with lse rows (cmp, slc, swa)."""
    two, lse2 = sparse_attn_rows(c, rows_h, rows_q, q, k_cur, v_cur, block_idx, ptr, G=G, K=K, n_wt=n_wt,
                                 softmax_scale=softmax_scale, fuse_mode=1, g_slc=g_slc, g_swa=g_swa)
    o_cmp, lse_cmp = cmp_attn_rows(c, rows_h, rows_q, q, softmax_scale)
    gc = np.asarray(g_cmp, np.float64)[np.asarray(rows_h)][:, None]
    out = (two.astype(np.float64) + gc * o_cmp.astype(np.float64)).astype(np.float32)
    return out, np.concatenate([lse_cmp[None], lse2], axis=0)


def group_mean_q(q: np.ndarray, G: int) -> np.ndarray:
    """a2 query side."""
    q, qp = _f32(q)
    H, S, D = q.shape
    R = -(-S // G)
    out = np.zeros((H, R, D), np.float32)
    _load().oracle_group_mean_q(qp, I32(H), I32(S), I32(D), I32(G), out.ctypes.data_as(ctypes.c_void_p))
    return out


def scores(c: OracleCache, qbar: np.ndarray, score_scale: float) -> np.ndarray:
    """a2 (Eq. 3): [H][R][N_b] fp32."""
    qbar, qp = _f32(qbar)
    H, R, D = qbar.shape
    n_b = c.n_blocks
    out = np.zeros((H, R, n_b), np.float32)
    _load().oracle_scores(qp, c.pooled_k.ctypes.data_as(ctypes.c_void_p), I32(H), I32(R), I32(D),
                          I32(c.n_pages), I64(n_b), F32(score_scale), out.ctypes.data_as(ctypes.c_void_p))
    return out


def scores_prob(c: OracleCache, q: np.ndarray, G: int, score_scale: float) -> np.ndarray:
    """a2, probability reading (reading A1b): per-query softmax over the head's compressed
    tokens, averaged over the query group.  [H][R][N_b] fp32."""
    q, qp = _f32(q)
    H, S, D = q.shape
    R = -(-S // G)
    n_b = c.n_blocks
    out = np.zeros((H, R, n_b), np.float32)
    _load().oracle_scores_prob(qp, c.pooled_k.ctypes.data_as(ctypes.c_void_p), I32(H), I32(S), I32(D), I32(G),
                               I32(c.n_pages), I64(n_b), F32(score_scale), out.ctypes.data_as(ctypes.c_void_p))
    return out


def awe(n_hist: int, B: int, n_wt: int, K: int, t_awe: int) -> dict:
    """a3 (Eq. 2)."""
    out = (ctypes.c_int64 * 4)()
    _load().oracle_awe(I64(n_hist), I32(B), I64(n_wt), I32(K), I64(t_awe), out)
    return {"b_w": int(out[0]), "active": bool(out[1]), "omega_end": int(out[2]), "n_b": int(out[3])}


def topk(scores_: np.ndarray, omega_end: int, K: int) -> np.ndarray:
    """a4: [H][R][K] int32, -1 = masked."""
    scores_, sp = _f32(scores_)
    H, R, n_b = scores_.shape
    out = np.full((H, R, K), -1, np.int32)
    _load().oracle_topk(sp, I32(H), I32(R), I64(n_b), I64(omega_end), I32(K), out.ctypes.data_as(ctypes.c_void_p))
    return out


def ptr_table(block_idx: np.ndarray, page_map: np.ndarray) -> np.ndarray:
    """a5."""
    block_idx, bp = _i32(block_idx)
    page_map, pp = _i32(page_map)
    H, R, K = block_idx.shape
    out = np.full((H, R, K), -1, np.int32)
    _load().oracle_ptr_table(bp, pp, I32(H), I32(R), I32(K), I32(page_map.shape[1]), out.ctypes.data_as(ctypes.c_void_p))
    return out


def ptr_table_chunked(block_idx: np.ndarray, chunk_map: np.ndarray, B_pc: int) -> np.ndarray:
    """a5 with the paper's two-level map (Alg. 1 lines 7-12): Pi[h][I // B_pc] + I % B_pc."""
    block_idx, bp = _i32(block_idx)
    chunk_map, cp = _i32(chunk_map)
    H, R, K = block_idx.shape
    out = np.full((H, R, K), -1, np.int32)
    _load().oracle_ptr_table_chunked(bp, cp, I32(H), I32(R), I32(K), I32(chunk_map.shape[1]), I32(B_pc), out.ctypes.data_as(ctypes.c_void_p))
    return out


def expand_chunk_map(chunk_map: np.ndarray, B_pc: int, n_pages: int) -> np.ndarray:
    """The flat block -> page map a two-level map stands for: page_map[h][b] = chunk_map[h][b // B_pc] + b % B_pc."""
    b = np.arange(n_pages)
    return (np.asarray(chunk_map)[:, b // B_pc] + (b % B_pc)[None, :]).astype(np.int32)


def padded_block(block_tokens: int) -> int:
    """Tab. H1: a pooling block is padded to the next power of two inside the kernel."""
    return int(_load().oracle_padded_block(I32(block_tokens)))


def union_counts(block_idx: np.ndarray, n_b: int):
    """Eqs. 4-5: (|U_h| per head, |union over heads|)."""
    block_idx, bp = _i32(block_idx)
    H, R, K = block_idx.shape
    per_head = np.zeros(H, np.int64)
    u = _load().oracle_union_counts(bp, I32(H), I32(R), I32(K), I64(n_b), per_head.ctypes.data_as(ctypes.c_void_p))
    return per_head, int(u)


SCORE_LOGIT, SCORE_PROB = 0, 1


def select(c: OracleCache, q: np.ndarray, G: int, K: int, n_wt: int, t_awe: int, score_scale: float,
           score_mode: int = SCORE_LOGIT) -> dict:
    """a2-a5 in the paper's order: scores -> AWE -> top-k -> pointer table."""
    qbar = group_mean_q(q, G)
    s = scores(c, qbar, score_scale) if score_mode == SCORE_LOGIT else scores_prob(c, q, G, score_scale)
    a = awe(c.n_hist, c.B, n_wt, K, t_awe)
    idx = topk(s, a["omega_end"], K)
    ptr = ptr_table(idx, c.page_map)
    return {"qbar": qbar, "scores": s, "awe": a, "block_idx": idx, "ptr_table": ptr}


def sparse_attn_rows(c: OracleCache, rows_h, rows_q, q, k_cur, v_cur, block_idx, ptr, *, G: int, K: int,
                     n_wt: int, softmax_scale: float, fuse_mode: int = 0, g_slc=None, g_swa=None):
    """a6-a8 for a list of (head, query) rows: returns (out [n][D] fp32, lse [2][n] fp32)."""
    rows_h, hp = _i32(rows_h)
    rows_q, qip = _i32(rows_q)
    q, qp = _f32(q)
    k_cur, kp = _f32(k_cur)
    v_cur, vp = _f32(v_cur)
    block_idx, bp = _i32(block_idx)
    ptr, pp = _i32(ptr)
    H, S, D = q.shape
    n = rows_h.shape[0]
    g_slc = np.ones(H, np.float32) if g_slc is None else g_slc
    g_swa = np.ones(H, np.float32) if g_swa is None else g_swa
    g_slc, gsp = _f32(g_slc)
    g_swa, gwp = _f32(g_swa)
    out = np.zeros((n, D), np.float32)
    lse = np.zeros((2, n), np.float32)
    _load().oracle_sparse_attn_rows(
        hp, qip, I64(n), qp, kp, vp,
        c.k_pages.ctypes.data_as(ctypes.c_void_p), c.v_pages.ctypes.data_as(ctypes.c_void_p),
        c.page_map.ctypes.data_as(ctypes.c_void_p), bp, pp,
        I32(H), I32(S), I32(D), I32(c.B), I32(c.n_pages), I64(c.n_hist), I64(n_wt), I32(G), I32(K),
        F32(softmax_scale), I32(fuse_mode), gsp, gwp,
        out.ctypes.data_as(ctypes.c_void_p), lse.ctypes.data_as(ctypes.c_void_p))
    return out, lse


def sparse_attn(c: OracleCache, q, k_cur, v_cur, block_idx, ptr, **kw):
    """a6-a8 for every (head, query): returns (out [H][S][D], lse [2][H][S])."""
    H, S, D = np.asarray(q).shape
    hh, qq = np.meshgrid(np.arange(H, dtype=np.int32), np.arange(S, dtype=np.int32), indexing="ij")
    out, lse = sparse_attn_rows(c, hh.ravel(), qq.ravel(), q, k_cur, v_cur, block_idx, ptr, **kw)
    return out.reshape(H, S, D), lse.reshape(2, H, S)


class OffloadModel:
    """NEXT-4, the residency policy of the paper's offloading ("the GPU hot cache keeps 7 chunks resident and evicts
    cold ones with an LRU policy", :339, :374-377) written out plainly (test infrastructure): per head a set of at most
    G resident chunks with a last-use clock; the W most recent chunks are pinned (the sliding window reads them).
      append(c):  the new chunk becomes resident in every head; if the head is full, its least recently used non-pinned chunk goes.
      step(need): need[h] = chunks head h's selection touches.  Resident ones are hits (touched, ascending chunk order); then every
                  missing one, in ascending order, replaces the least recently used chunk that is neither pinned nor needed by this
                  step -- if there is none it stays on the host.  Returns (resident before, resident after) per head.
    Counters: requests, hits, reloads, evictions."""

    def __init__(self, H: int, G: int, W: int):
        self.H, self.G, self.W = H, G, W
        self.res = [dict() for _ in range(H)]  # chunk -> clock
        self.clock = 0
        self.newest = -1
        self.requests = self.hits = self.reloads = self.evictions = 0

    def _pinned(self, c):
        return c > self.newest - self.W

    def _victim(self, h, need=()):
        cands = [(t, c) for c, t in self.res[h].items() if not self._pinned(c) and c not in need]
        return min(cands)[1] if cands else None

    def append(self, c: int) -> None:
        self.newest = c
        for h in range(self.H):
            if len(self.res[h]) >= self.G:
                v = self._victim(h)
                assert v is not None, "resident_chunks must exceed pinned_recent"
                del self.res[h][v]
                self.evictions += 1
            self.clock += 1
            self.res[h][c] = self.clock

    def step(self, need):
        before = [set(r) for r in self.res]
        for h in range(self.H):
            nd = sorted(need[h])
            for c in nd:
                self.requests += 1
                if c in self.res[h]:
                    self.hits += 1
                    self.clock += 1
                    self.res[h][c] = self.clock
            for c in nd:
                if c in self.res[h]:
                    continue
                if len(self.res[h]) >= self.G:
                    v = self._victim(h, nd)
                    if v is None:
                        continue
                    del self.res[h][v]
                    self.evictions += 1
                self.clock += 1
                self.res[h][c] = self.clock
                self.reloads += 1
        return before, [set(r) for r in self.res]

    @property
    def hit_rate(self) -> float:
        return self.hits / self.requests if self.requests else 1.0
