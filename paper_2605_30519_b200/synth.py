"""Seeded synthetic workloads shaped like the paper's (DESIGN.md section 4 states the recipe).

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench, so it holds
none of the method's arithmetic: it only draws random tensors with the shapes, value
structure and length mix of PAPER.md's workloads (480p latent 30x52 = 1560 tokens/frame,
3 latent frames per chunk => S = 4680, 12 heads x 128) and
rounds them once to bf16, so that the oracle and the GPU consume identical bits.  They stand
in for the VBench / VBench-Long rollouts the paper measures on, which
are not available here.  It imports neither ``oracle`` nor the CUDA binding.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np
import torch

FRAME_TOKENS = 1560  # 30 x 52 latent tokens per frame


@dataclass(frozen=True)
class Workload:
    name: str
    H: int
    D: int
    S: int  # tokens in the current chunk (= queries)
    n_hist: int  # cached history tokens
    B: int  # tokens per KV block
    n_wt: int  # sliding-window tokens of history
    G: int  # query-group size G_q
    K: int  # top-k blocks per (head, group)
    t_awe: int  # AWE threshold in blocks (reading A2)
    structure: str  # "block_offset" (config 1) | "frame_affinity" (configs 2-5)
    chunk: int  # tokens per appended history chunk
    seed: int = 0
    affinity_from_all_history: bool = False
    P: int = 0    # rows per page (0 = B); the paper's geometry pads a block of B = 30 tokens to 32 rows
    bpc: int = 0  # blocks per chunk of the two-level page map, 0 = one map entry per block

    @property
    def n_b(self) -> int:
        return -(-self.n_hist // self.B)

    @property
    def R(self) -> int:
        return -(-self.S // self.G)

    @property
    def win_start(self) -> int:
        return max(0, self.n_hist - self.n_wt) if self.n_wt > 0 else self.n_hist

    @property
    def softmax_scale(self) -> float:
        return float(np.float32(1.0 / np.sqrt(np.float32(self.D))))

    def flops(self) -> float:
        """4*D*S*(K*B + N_wt + S)*H  (K*B capped by the candidates that exist)."""
        k_tok = min(self.K * self.B, self.n_hist)
        n_win = self.n_hist - self.win_start
        return 4.0 * self.D * self.S * (k_tok + n_win + self.S) * self.H


def _t_awe(S: int, B: int) -> int:
    return -(-3 * S // B)  # "at least 3 chunks of history outside the window"


def config(base: str, **over) -> Workload:
    """The five BASELINE.json configs (sweep members of config 5 via keyword overrides)."""
    S = 4680
    name = base
    if name == "tiny":  # config 1
        w = Workload("tiny", H=2, D=64, S=256, n_hist=2048, B=64, n_wt=512, G=64, K=4, t_awe=4,
                     structure="block_offset", chunk=256)
    elif name == "wan1p3b":  # config 2
        w = Workload("wan1p3b", H=12, D=128, S=S, n_hist=20 * S, B=64, n_wt=S, G=64, K=16,
                     t_awe=_t_awe(S, 64), structure="frame_affinity", chunk=S)
    elif name == "long":  # config 3
        w = Workload("long", H=12, D=128, S=S, n_hist=120 * S, B=64, n_wt=S, G=64, K=32,
                     t_awe=_t_awe(S, 64), structure="frame_affinity", chunk=S)
    elif name == "wan14b":  # config 4
        w = Workload("wan14b", H=40, D=128, S=S, n_hist=40 * S, B=64, n_wt=S, G=64, K=16,
                     t_awe=_t_awe(S, 64), structure="frame_affinity", chunk=S)
    elif name == "paper":  # the paper's own geometry: pooling block 15 x 2 = 30
        # tokens in 32-row pages, groups of 15 queries, top-4, window of 3 chunks, AWE once 3 chunks lie outside the window,
        # chunk-aligned blocks (156 per chunk) behind the two-level map
        w = Workload("paper", H=12, D=128, S=S, n_hist=20 * S, B=30, n_wt=3 * S, G=15, K=4,
                     t_awe=3 * (S // 30), structure="frame_affinity", chunk=S, P=32, bpc=S // 30)
    elif name == "short":  # config 5 edge case: 3 chunks of history, AWE must not exclude
        w = Workload("short", H=12, D=128, S=S, n_hist=3 * S, B=64, n_wt=S, G=64, K=16,
                     t_awe=_t_awe(S, 64), structure="frame_affinity", chunk=S,
                     affinity_from_all_history=True)
    else:
        raise KeyError(name)
    if over:
        w = replace(w, **over)
        if "B" in over and "t_awe" not in over and w.structure == "frame_affinity":
            w = replace(w, t_awe=_t_awe(w.S, w.B))
    return w


def sweep_configs() -> list[Workload]:
    """Config 5: B in {64,128} x K in {8,16,32,64} x G_q in {64, 4680} + the short-history case."""
    out = []
    for B in (64, 128):
        for K in (8, 16, 32, 64):
            for G in (64, 4680):
                out.append(config("wan1p3b", B=B, K=K, G=G, name=f"sweep_B{B}_K{K}_G{G}"))
        out.append(config("short", B=B, name=f"short_B{B}"))
    return out


def _bf16(x: np.ndarray) -> np.ndarray:
    """Round once to bf16 (library cast), keep as float32."""
    return torch.from_numpy(x).to(torch.bfloat16).to(torch.float32).numpy()


def _randn(rng: np.random.Generator, shape) -> np.ndarray:
    return rng.standard_normal(shape, dtype=np.float32)


def generate(w: Workload) -> dict:
    """Returns float32 arrays with bf16-representable values:
    k_hist, v_hist [H][n_hist][D]; q, k_cur, v_cur [H][S][D]; plus 'frames' (the distant
    frames each head's queries correlate with, for reporting only)."""
    rng = np.random.default_rng(np.random.PCG64(1000003 * w.seed + 17))
    H, D, S, N = w.H, w.D, w.S, w.n_hist
    out = {}
    if w.structure == "block_offset":
        # config 1: N(0,1) plus a per-(head, block, dim) mean offset ~ N(0, 0.5^2)
        def with_offsets(n):
            x = _randn(rng, (H, n, D))
            nb = -(-n // w.B)
            off = 0.5 * _randn(rng, (H, nb, D))
            return x + np.repeat(off, w.B, axis=1)[:, :n]

        out["k_hist"], out["v_hist"] = with_offsets(N), with_offsets(N)
        out["q"], out["k_cur"], out["v_cur"] = with_offsets(S), with_offsets(S), with_offsets(S)
        out["frames"] = np.zeros((H, 0), np.int64)
    elif w.structure == "frame_affinity":
        # configs 2-5: per (head, frame) latent means m^K, m^V ~ N(0, I_D); tokens = mean + 0.3 eps;
        # queries = 1/2 sum of the m^K of 4 distant frames + 0.3 eps
        F = FRAME_TOKENS
        n_frames_hist = -(-N // F)
        n_frames_cur = -(-S // F)
        mk = _randn(rng, (H, n_frames_hist + n_frames_cur, D))
        mv = _randn(rng, (H, n_frames_hist + n_frames_cur, D))

        def tokens(means, first_frame, n):
            fidx = first_frame + np.arange(n) // F
            x = means[:, fidx, :]
            x = x + np.float32(0.3) * _randn(rng, (H, n, D))
            return x

        out["k_hist"] = tokens(mk, 0, N)
        out["v_hist"] = tokens(mv, 0, N)
        out["k_cur"] = tokens(mk, n_frames_hist, S)
        out["v_cur"] = tokens(mv, n_frames_hist, S)
        n_far = n_frames_hist if w.affinity_from_all_history else max(4, w.win_start // F)
        frames = np.stack([rng.permutation(n_far)[:4] for _ in range(H)])
        sig = 0.5 * mk[np.arange(H)[:, None], frames, :].sum(axis=1)  # [H][D]
        out["q"] = sig[:, None, :] + np.float32(0.3) * _randn(rng, (H, S, D))
        out["frames"] = frames
    else:
        raise ValueError(w.structure)
    for k in ("k_hist", "v_hist", "q", "k_cur", "v_cur"):
        out[k] = _bf16(np.ascontiguousarray(out[k], dtype=np.float32))
    return out


def permuted_page_map(H: int, n_pages: int, seed: int) -> np.ndarray:
    """A random per-head block -> page permutation, so a kernel that ignores the table fails."""
    rng = np.random.default_rng(seed)
    return np.stack([rng.permutation(n_pages) for _ in range(H)]).astype(np.int32)


def permuted_chunk_map(H: int, n_chunks: int, bpc: int, seed: int) -> np.ndarray:
    """Two-level map: a random per-head placement of the chunks, [H][n_chunks] base pages (multiples of B_pc)."""
    rng = np.random.default_rng(seed)
    return (np.stack([rng.permutation(n_chunks) for _ in range(H)]) * bpc).astype(np.int32)


def sample_rows(w: Workload, n_groups: int, rows_per_group: int, seed: int = 0):
    """A deterministic sample of (head, query) rows: for every head, the first, second, middle,
    next-to-last and last query groups (plus random ones up to n_groups), a few rows each,
    always including each sampled group's first and last row."""
    rng = np.random.default_rng(seed + 99)
    R = w.R
    fixed = sorted({0, min(1, R - 1), R // 2, max(R - 2, 0), R - 1})
    hs, qs = [], []
    for h in range(w.H):
        groups = list(fixed)
        extra = [g for g in rng.permutation(R).tolist() if g not in groups]
        groups = (groups + extra)[: max(n_groups, 1)]
        for r in groups:
            lo, hi = r * w.G, min((r + 1) * w.G, w.S)
            picks = {lo, hi - 1}
            picks.update(rng.integers(lo, hi, size=max(rows_per_group - 2, 0)).tolist())
            for s in sorted(picks):
                hs.append(h)
                qs.append(s)
    return np.asarray(hs, np.int32), np.asarray(qs, np.int32)
