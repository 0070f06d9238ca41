"""Thin ctypes binding of the C-ABI in ``include/omnimem.h`` -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of ``libomnimem.so``; PyTorch is used here
for device memory and streams, nothing else.  The functions carry the names of the C entry points.
There is no fallback of any kind: if the library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_float, c_int32, c_int64, c_size_t, c_void_p

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("OMNIMEM_LIB") or os.path.join(_HERE, "libomnimem.so")  # OMNIMEM_LIB: a variant build

OK, EINVAL, ECAPACITY, EUNSUPPORTED, ECUDA, ESTATE = 0, -1, -2, -3, -4, -5
DTYPE_BF16 = 1
FUSE_JOINT, FUSE_GATED = 0, 1
SCORE_LOGIT, SCORE_PROB = 0, 1

EXPORTS = [
    "omnimem_version", "omnimem_last_error", "omnimem_cache_sizes", "omnimem_cache_create",
    "omnimem_cache_identity_page_map", "omnimem_cache_reset", "omnimem_cache_destroy", "omnimem_cache_tokens",
    "omnimem_append_chunk", "omnimem_pool_keys", "omnimem_select", "omnimem_select_from_scores",
    "omnimem_sparse_attn", "omnimem_workspace_bytes", "omnimem_launch_count",
    "omnimem_cache_attach_pooled_v", "omnimem_sparse_attn3", "omnimem_union_counts", "omnimem_union_counts_noalloc", "omnimem_gather_blocks",
    "omnimem_offload_scratch_bytes", "omnimem_offload_attach", "omnimem_offload_step",
]


class CacheDesc(Structure):
    _fields_ = [("n_heads", c_int32), ("head_dim", c_int32), ("block_tokens", c_int32), ("dtype", c_int32),
                ("max_tokens", c_int64), ("page_tokens", c_int32), ("blocks_per_chunk", c_int32),
                ("resident_chunks", c_int32), ("reserved0", c_int32)]


class SelectParams(Structure):
    _fields_ = [("group_tokens", c_int32), ("top_k", c_int32), ("window_tokens", c_int64),
                ("awe_min_outside_blocks", c_int64), ("score_scale", c_float), ("score_mode", c_int32)]


class AweInfo(Structure):
    _fields_ = [("n_blocks", c_int64), ("first_window", c_int64), ("n_candidates", c_int64), ("active", c_int32),
                ("n_groups", c_int32)]


class AttnParams(Structure):
    _fields_ = [("group_tokens", c_int32), ("top_k", c_int32), ("window_tokens", c_int64), ("softmax_scale", c_float),
                ("fuse_mode", c_int32), ("reserved", c_int32)]


class OffloadStats(Structure):
    _fields_ = [("requests", c_int64), ("hits", c_int64), ("reloads", c_int64), ("evictions", c_int64), ("skipped", c_int64)]


OFFLOAD_SKIP, OFFLOAD_WAIT = 0, 1


class OmniMemError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"omnimem error {code}: {msg}")
        self.code = code


_lib = None


def load() -> ctypes.CDLL:
    """Loads libomnimem.so (built in-tree by ``python -m paper_2605_30519_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2605_30519_b200.build` "
                           "(there is no fallback path)")
    lib = ctypes.CDLL(LIB_PATH)
    lib.omnimem_version.restype = c_int32
    lib.omnimem_last_error.restype = c_char_p
    lib.omnimem_cache_tokens.restype = c_int64
    lib.omnimem_cache_tokens.argtypes = [c_void_p]
    lib.omnimem_launch_count.restype = c_int64
    lib.omnimem_cache_sizes.argtypes = [POINTER(CacheDesc)] + [POINTER(c_size_t)] * 4
    lib.omnimem_cache_create.argtypes = [POINTER(CacheDesc), c_void_p, c_void_p, c_void_p, c_void_p, POINTER(c_void_p)]
    lib.omnimem_cache_identity_page_map.argtypes = [c_void_p, c_void_p]
    lib.omnimem_cache_reset.argtypes = [c_void_p]
    lib.omnimem_cache_destroy.argtypes = [c_void_p]
    lib.omnimem_append_chunk.argtypes = [c_void_p, c_void_p, c_void_p, c_int32, c_int64, c_int64, c_void_p]
    lib.omnimem_pool_keys.argtypes = [c_void_p, c_int64, c_int64, c_void_p]
    lib.omnimem_select.argtypes = [c_void_p, c_void_p, c_int32, c_int64, c_int64, POINTER(SelectParams), c_void_p,
                                   c_void_p, c_void_p, POINTER(AweInfo), c_void_p, c_size_t, c_void_p]
    lib.omnimem_select_from_scores.argtypes = [c_void_p, c_void_p, c_int32, POINTER(SelectParams), c_void_p, c_void_p,
                                               POINTER(AweInfo), c_void_p]
    lib.omnimem_sparse_attn.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int32, c_int64, c_int64, c_void_p,
                                        POINTER(AttnParams), c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                        c_size_t, c_void_p]
    lib.omnimem_cache_attach_pooled_v.argtypes = [c_void_p, c_void_p]
    lib.omnimem_sparse_attn3.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int32, c_int64, c_int64, c_void_p,
                                         POINTER(AttnParams), c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                         c_size_t, c_void_p]
    lib.omnimem_union_counts.argtypes = [c_void_p, c_void_p, c_int32, c_int32, c_void_p, c_void_p, c_void_p, c_void_p, c_size_t, c_void_p]
    lib.omnimem_union_counts_noalloc.argtypes = [c_void_p, c_void_p, c_int32, c_int32, c_void_p, c_void_p, c_void_p, c_void_p]
    lib.omnimem_gather_blocks.argtypes = [c_void_p, c_void_p, c_int64, c_void_p, c_void_p]
    lib.omnimem_offload_scratch_bytes.argtypes = [POINTER(CacheDesc)]
    lib.omnimem_offload_scratch_bytes.restype = c_size_t
    lib.omnimem_offload_attach.argtypes = [c_void_p, c_void_p, c_void_p, c_int32, c_void_p, c_void_p, c_size_t]
    lib.omnimem_offload_step.argtypes = [c_void_p, c_void_p, c_int32, c_int32, c_int32, c_void_p, POINTER(OffloadStats), c_void_p]
    lib.omnimem_workspace_bytes.argtypes = [POINTER(CacheDesc), c_int32, POINTER(SelectParams), POINTER(AttnParams),
                                            POINTER(c_size_t), POINTER(c_size_t)]
    _lib = lib
    return lib


def _check(rc: int) -> None:
    if rc != OK:
        raise OmniMemError(rc, load().omnimem_last_error().decode())


def _stream(stream) -> c_void_p:
    s = torch.cuda.current_stream() if stream is None else stream
    return c_void_p(s.cuda_stream)


def _ptr(t) -> c_void_p:
    return c_void_p(0 if t is None else t.data_ptr())


def _hnd(t: torch.Tensor):
    """[H][n][D] bf16 CUDA tensor -> (ptr, n, stride_tok, stride_head)."""
    assert t.is_cuda and t.dtype == torch.bfloat16 and t.dim() == 3 and t.stride(2) == 1, "need [H][n][D] bf16 CUDA, D contiguous"
    return _ptr(t), t.shape[1], t.stride(1), t.stride(0)


class OmniMemCache:
    """Owns the device buffers (torch) and the library's host-side handle for one attention layer."""

    def __init__(self, n_heads: int, head_dim: int, block_tokens: int, max_tokens: int, device="cuda:0",
                 page_map: torch.Tensor | None = None, page_tokens: int = 0, blocks_per_chunk: int = 0,
                 resident_chunks: int = 0, pinned_recent: int = 1):
        """page_tokens / blocks_per_chunk: the paper's geometry (blocks of B < P tokens in zero-padded pages of P rows; two-level
        page map with one entry per chunk of B_pc blocks); page_map is then [H][ceil(max_blocks / B_pc)] chunk base pages."""
        lib = load()
        self.desc = CacheDesc(n_heads, head_dim, block_tokens, DTYPE_BF16, max_tokens, page_tokens, blocks_per_chunk, resident_chunks, 0)
        sizes = [c_size_t() for _ in range(4)]
        _check(lib.omnimem_cache_sizes(byref(self.desc), *[byref(s) for s in sizes]))
        self.H, self.D, self.B = n_heads, head_dim, block_tokens
        self.P, self.bpc = page_tokens or block_tokens, blocks_per_chunk
        self.max_blocks = -(-max_tokens // block_tokens)
        self.pool_blocks = resident_chunks * blocks_per_chunk if resident_chunks else self.max_blocks
        dev = torch.device(device)
        # zero-initialised: rows of a page that were never written must be finite (a masked column contributes P = 0 times V)
        self.k_pages = torch.zeros(sizes[0].value // 2, dtype=torch.bfloat16, device=dev).view(n_heads, self.pool_blocks, self.P, head_dim)
        self.v_pages = torch.zeros(sizes[1].value // 2, dtype=torch.bfloat16, device=dev).view(n_heads, self.pool_blocks, self.P, head_dim)
        self.pooled_k = torch.zeros(sizes[2].value // 2, dtype=torch.bfloat16, device=dev).view(n_heads, self.max_blocks, head_dim)
        self.page_map = torch.empty(sizes[3].value // 4, dtype=torch.int32, device=dev).view(n_heads, self.max_blocks)
        self._h = c_void_p()
        _check(lib.omnimem_cache_create(byref(self.desc), _ptr(self.k_pages), _ptr(self.v_pages), _ptr(self.pooled_k),
                                        _ptr(self.page_map), byref(self._h)))
        if resident_chunks:
            # offloading (NEXT-4): the full history lives in pinned host memory, HBM holds resident_chunks chunk slots per head
            assert page_map is None, "with offloading the library places the chunks"
            n_chunks = -(-self.max_blocks // blocks_per_chunk)
            chunk_el = blocks_per_chunk * self.P * head_dim
            self.host_k = torch.empty((n_heads, n_chunks, chunk_el), dtype=torch.bfloat16, pin_memory=True)
            self.host_v = torch.empty((n_heads, n_chunks, chunk_el), dtype=torch.bfloat16, pin_memory=True)
            sb = lib.omnimem_offload_scratch_bytes(byref(self.desc))
            self._scratch_host = torch.zeros(sb, dtype=torch.uint8, pin_memory=True)
            self._scratch_dev = torch.zeros(sb, dtype=torch.uint8, device=dev)
            _check(lib.omnimem_cache_identity_page_map(self._h, _stream(None)))
            _check(lib.omnimem_offload_attach(self._h, c_void_p(self.host_k.data_ptr()), c_void_p(self.host_v.data_ptr()), pinned_recent,
                                              c_void_p(self._scratch_host.data_ptr()), _ptr(self._scratch_dev), sb))
        elif page_map is None:
            _check(lib.omnimem_cache_identity_page_map(self._h, _stream(None)))
        elif blocks_per_chunk > 0:  # [H][n_chunks] chunk bases, stored at the head of the buffer
            n_chunks = -(-self.max_blocks // blocks_per_chunk)
            assert tuple(page_map.shape) == (n_heads, n_chunks)
            self.page_map.view(-1)[:n_heads * n_chunks].copy_(page_map.to(dev, torch.int32).reshape(-1))
        else:
            self.page_map.copy_(page_map.to(dev, torch.int32))

    @property
    def handle(self) -> c_void_p:
        return self._h

    @property
    def n_hist(self) -> int:
        return int(load().omnimem_cache_tokens(self._h))

    @property
    def n_blocks(self) -> int:
        return -(-self.n_hist // self.B)

    def attach_pooled_v(self) -> None:
        """Allocates the value half of the compressed cache (zeros) and hands it to the library: from now on
        omnimem_pool_keys pools values too (needed by omnimem_sparse_attn3 only).  The cache must still be empty."""
        self.pooled_v = torch.zeros_like(self.pooled_k)
        _check(load().omnimem_cache_attach_pooled_v(self._h, _ptr(self.pooled_v)))

    def reset(self) -> None:
        _check(load().omnimem_cache_reset(self._h))

    def workspace_bytes(self, n_q: int, sp: SelectParams | None, ap: AttnParams | None):
        a, b = c_size_t(), c_size_t()
        _check(load().omnimem_workspace_bytes(byref(self.desc), n_q, byref(sp) if sp else None, byref(ap) if ap else None,
                                              byref(a), byref(b)))
        return a.value, b.value

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.omnimem_cache_destroy(self._h)
            self._h = None


def omnimem_append_chunk(cache: OmniMemCache, k: torch.Tensor, v: torch.Tensor, stream=None) -> None:
    kp, n, st, sh = _hnd(k)
    vp, n2, st2, sh2 = _hnd(v)
    assert (n, st, sh) == (n2, st2, sh2), "k and v must share shape and strides"
    _check(load().omnimem_append_chunk(cache.handle, kp, vp, n, st, sh, _stream(stream)))


def omnimem_pool_keys(cache: OmniMemCache, first_block: int = 0, n_blocks: int = -1, stream=None) -> None:
    _check(load().omnimem_pool_keys(cache.handle, first_block, n_blocks, _stream(stream)))


def _awe_dict(a: AweInfo) -> dict:
    return {"n_b": a.n_blocks, "b_w": a.first_window, "omega_end": a.n_candidates, "active": bool(a.active),
            "n_groups": a.n_groups}


def omnimem_select(cache: OmniMemCache, q: torch.Tensor, params: SelectParams, block_idx: torch.Tensor | None,
                   ptr_table: torch.Tensor, scores_out: torch.Tensor | None, workspace: torch.Tensor, stream=None) -> dict:
    qp, n_q, st, sh = _hnd(q)
    awe = AweInfo()
    _check(load().omnimem_select(cache.handle, qp, n_q, st, sh, byref(params), _ptr(block_idx), _ptr(ptr_table),
                                 _ptr(scores_out), byref(awe), _ptr(workspace), workspace.numel() * workspace.element_size(),
                                 _stream(stream)))
    return _awe_dict(awe)


def omnimem_select_from_scores(cache: OmniMemCache, scores: torch.Tensor, n_q: int, params: SelectParams,
                               block_idx: torch.Tensor | None, ptr_table: torch.Tensor, stream=None) -> dict:
    assert scores.is_cuda and scores.dtype == torch.float32 and scores.is_contiguous()
    awe = AweInfo()
    _check(load().omnimem_select_from_scores(cache.handle, _ptr(scores), n_q, byref(params), _ptr(block_idx),
                                             _ptr(ptr_table), byref(awe), _stream(stream)))
    return _awe_dict(awe)


def omnimem_sparse_attn(cache: OmniMemCache, q: torch.Tensor, k_cur: torch.Tensor, v_cur: torch.Tensor,
                        ptr_table: torch.Tensor, params: AttnParams, out: torch.Tensor, gate_slc: torch.Tensor | None = None,
                        gate_swa: torch.Tensor | None = None, lse_out: torch.Tensor | None = None,
                        workspace: torch.Tensor | None = None, stream=None) -> None:
    qp, n_q, st, sh = _hnd(q)
    kp, n2, st2, sh2 = _hnd(k_cur)
    vp, n3, st3, sh3 = _hnd(v_cur)
    assert (n_q, st, sh) == (n2, st2, sh2) == (n3, st3, sh3), "q, k_cur, v_cur must share shape and strides"
    assert out.is_contiguous() and out.dtype == torch.bfloat16 and out.shape == q.shape
    wb = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(load().omnimem_sparse_attn(cache.handle, qp, kp, vp, n_q, st, sh, _ptr(ptr_table), byref(params),
                                      _ptr(gate_slc), _ptr(gate_swa), _ptr(out), _ptr(lse_out), _ptr(workspace), wb,
                                      _stream(stream)))


def omnimem_sparse_attn3(cache: OmniMemCache, q: torch.Tensor, k_cur: torch.Tensor, v_cur: torch.Tensor,
                         ptr_table: torch.Tensor, params: AttnParams, out: torch.Tensor, gate_cmp: torch.Tensor,
                         gate_slc: torch.Tensor, gate_swa: torch.Tensor, lse_out: torch.Tensor | None = None,
                         workspace: torch.Tensor | None = None, stream=None) -> None:
    qp, n_q, st, sh = _hnd(q)
    kp, n2, st2, sh2 = _hnd(k_cur)
    vp, n3, st3, sh3 = _hnd(v_cur)
    assert (n_q, st, sh) == (n2, st2, sh2) == (n3, st3, sh3), "q, k_cur, v_cur must share shape and strides"
    assert out.is_contiguous() and out.dtype == torch.bfloat16 and out.shape == q.shape
    wb = 0 if workspace is None else workspace.numel() * workspace.element_size()
    _check(load().omnimem_sparse_attn3(cache.handle, qp, kp, vp, n_q, st, sh, _ptr(ptr_table), byref(params),
                                       _ptr(gate_cmp), _ptr(gate_slc), _ptr(gate_swa), _ptr(out), _ptr(lse_out),
                                       _ptr(workspace), wb, _stream(stream)))


def omnimem_union_counts(cache: OmniMemCache, block_idx: torch.Tensor, per_head: torch.Tensor, union_all: torch.Tensor,
                         union_list: torch.Tensor | None, workspace: torch.Tensor, stream=None) -> None:
    """Eqs. 4-5 of a selection: |U_h| per head, |union over heads|, optionally the union's blocks in order."""
    assert block_idx.dtype == torch.int32 and block_idx.is_contiguous() and block_idx.dim() == 3
    assert per_head.dtype == torch.int64 and union_all.dtype == torch.int64
    _check(load().omnimem_union_counts(cache.handle, _ptr(block_idx), block_idx.shape[1], block_idx.shape[2], _ptr(per_head), _ptr(union_all),
                                       _ptr(union_list), _ptr(workspace), workspace.numel() * workspace.element_size(), _stream(stream)))


UNION_NOALLOC_MAX_BYTES = 1 << 20  # OMNIMEM_UNION_NOALLOC_MAX_BYTES (include/omnimem.h)


def omnimem_union_counts_noalloc(cache: OmniMemCache, block_idx: torch.Tensor, per_head: torch.Tensor, union_all: torch.Tensor,
                                 union_list: torch.Tensor | None, stream=None) -> None:
    """omnimem_union_counts without caller scratch and without any allocation: the marks live in a device array built into the
    library (at most UNION_NOALLOC_MAX_BYTES = (H + 1) * N_b bytes, else ECAPACITY).  All calls share that array: calls that
    overlap on the GPU race."""
    assert block_idx.dtype == torch.int32 and block_idx.is_contiguous() and block_idx.dim() == 3
    assert per_head.dtype == torch.int64 and union_all.dtype == torch.int64
    _check(load().omnimem_union_counts_noalloc(cache.handle, _ptr(block_idx), block_idx.shape[1], block_idx.shape[2], _ptr(per_head),
                                               _ptr(union_all), _ptr(union_list), _stream(stream)))


def omnimem_gather_blocks(src: OmniMemCache, block_list: torch.Tensor, n: int, dst: OmniMemCache, stream=None) -> None:
    """The Naive-Sparse baseline's merged selected-KV buffer: blocks block_list[:n] of every head of src -> blocks 0..n-1 of dst."""
    assert block_list.dtype == torch.int32 and block_list.is_contiguous()
    _check(load().omnimem_gather_blocks(src.handle, _ptr(block_list), n, dst.handle, _stream(stream)))


def omnimem_offload_step(cache: OmniMemCache, block_idx: torch.Tensor, ptr_table: torch.Tensor, mode: int, stream=None) -> dict:
    """The host step of the offloading pipeline: LRU update, reloads, and in WAIT mode the
    rebuilt pointer table.  Synchronises the stream.  Returns the cumulative counters + the hit rate."""
    st = OffloadStats()
    _check(load().omnimem_offload_step(cache.handle, _ptr(block_idx), block_idx.shape[1], block_idx.shape[2], mode, _ptr(ptr_table),
                                       byref(st), _stream(stream)))
    return {"requests": st.requests, "hits": st.hits, "reloads": st.reloads, "evictions": st.evictions, "skipped": st.skipped,
            "hit_rate": st.hits / st.requests if st.requests else 1.0}


def launch_count() -> int:
    return int(load().omnimem_launch_count())
