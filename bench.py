#!/usr/bin/env python
"""bench.py -- one AR-step layer (omnimem_select + omnimem_sparse_attn) of the OmniMem hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload wan1p3b] [--impl ours|reference]

Metric (BASELINE.json): ms per AR-step layer (select + attend) on the Wan-1.3B-like config (12 heads x 128,
4680-token chunk, 93,600-token history, window 1 chunk, G_q 64, top-16), synthetic seeded data.  A "step" is
one pass of the whole per-denoising-step hot path (a2-a8) over one chunk; append_chunk / pool_keys run once per
chunk and are timed separately ("per_chunk").  Each timed step is bracketed by CUDA events on the launching
stream; L2 is flushed (256 MiB write) between steps, outside the event pairs.  Prints ONE JSON line.
With N > 1 (torchrun) every rank runs an independent replica of the layer step (heads are independent, the
path has no exchange step: DESIGN.md section 8); timing is the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            j = json.load(f)
        return {"hbm_gbs": j["hbm_gbs"], "bf16_tflops": j["bf16_tflops"], "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "source": "fallback"}


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons (every 20 ms, nvidia-smi's own timestamps); stop() keeps the
    samples that fall inside the timed region [t0, t1] (wall clock)."""

    Q = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self, t0: float, t1: float) -> dict:
        import datetime
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        self.thread.join(timeout=2)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        inside, allrows = [], []
        for r in self.rows:
            try:
                ts = datetime.datetime.strptime(r[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                rec = (float(r[1]), float(r[2]), float(r[3]), [n for n, v in zip(names, r[4:8]) if v.lower().startswith("active")])
            except (ValueError, IndexError):
                continue
            allrows.append(rec)
            if t0 - 0.02 <= ts <= t1 + 0.02:
                inside.append(rec)
        use = inside if inside else allrows
        reasons = sorted({n for rec in use for n in rec[3]})
        return {"sm_mhz": float(np.median([r[0] for r in use])) if use else None,
                "sm_max_mhz": max(r[1] for r in use) if use else None,
                "power_w_max": max(r[2] for r in use) if use else None, "reasons": reasons,
                "samples_in_timed_region": len(inside), "samples_total": len(allrows)}


def l2_ingest(w, att_ms, sm_mhz, n_sm):
    """Bytes every SM pulls from L2 into shared memory through TMA for one attention launch (128 query rows per
    CTA: a 64 KB K+V tile pair per 128 KV tokens, plus the Q tile), as bytes per SM clock, next to the measured
    ceiling of profiles/r1_microbench.md (l2_ingest.cu): the hardware ceiling this kernel sits closest to."""
    if w.D != 128 or 128 % w.G and w.G % 128:
        return None
    groups = max(1, 128 // w.G)
    slc_slots = -(-(min(w.K, w.n_b) * w.B // 64) // 2) * 2 if w.n_hist > 0 else 0
    n_win = w.n_b - w.win_start // w.B if w.n_hist > w.win_start else 0
    swa_slots = -(-(n_win * (w.B // 64) + -(-w.S // 64)) // 2) * 2
    tiles = (groups * slc_slots + swa_slots) // 2
    ctas = -(-w.S // 128) * w.H
    total = ctas * (tiles * 65536 + 32768)
    clk = sm_mhz * 1e6  # the clock sampled during the timed region
    return {"bytes_per_launch": total, "achieved_B_per_clk_per_SM": total / n_sm / (att_ms * 1e-3 * clk),
            "ceiling_B_per_clk_per_SM": {"32KB_copies": 40.5, "16KB": 37.3, "8KB": 33.6}, "sm_clock_hz": clk}


def max_over_ranks(values, device, world):
    """Replicas only: every rank times its own replica of the layer step; the job's figure is the
    slowest rank's.  The only collective of the whole program."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def union_stats(om, torch, ls, w, dev):
    """Eqs. 4-5 of the selection the step just made, counted on the device (omnimem_union_counts):
    M_scatter = sum_h |U_h| blocks (what per-head scattered access touches), M_merge = N_h * |union_h U_h| blocks (a merged
    selected-KV buffer shared by all heads), both as K+V bytes."""
    n_b = ls.cache.n_blocks
    per_head = torch.zeros(w.H, dtype=torch.int64, device=dev)
    union_all = torch.zeros(1, dtype=torch.int64, device=dev)
    union_list = torch.zeros(max(n_b, 1), dtype=torch.int32, device=dev)
    ws = torch.empty((w.H + 1) * max(n_b, 1), dtype=torch.uint8, device=dev)
    om.omnimem_union_counts(ls.cache, ls.block_idx, per_head, union_all, union_list, ws)
    torch.cuda.synchronize()
    block_bytes = 2 * w.B * w.D * 2
    s_u, u = int(per_head.sum().item()), int(union_all.item())
    return {"sum_U_h": s_u, "U_all": u, "M_scatter_bytes": s_u * block_bytes, "M_merge_bytes": w.H * u * block_bytes,
            "M_full_history_bytes": w.H * n_b * block_bytes}, union_list, u


def sweep_history(args, w0, dev):
    """The shape of the paper's scalability figure on synthetic data: ms per AR-step layer against the
    number of cached chunks, for the sparse path (window of one chunk + top-K blocks per group) and for dense attention
    over the whole history (the same kernel with the window spanning all of it and K = 1), and -- with --naive -- for the
    paper's Naive-Sparse comparison system: per-query top-K (G_q = 1, no sharing), the union of all
    heads' selections gathered into ONE merged selected-KV buffer (omnimem_gather_blocks) and dense attention of every query
    over that buffer + window + current chunk (a padded dense kernel does not skip what a query did not select).  Memory
    columns: M_scatter (per-head scattered access), M_merge (merged buffer, of the naive and of the query-shared selection)
    and the full history, Eqs. 4-5.  K/V/Q are seeded N(0,1) tensors drawn on the device (timing only: parity at these sizes
    is tests/test_gpu_parity.py's job)."""
    import torch
    from dataclasses import replace
    from paper_2605_30519_b200 import binding as om
    from paper_2605_30519_b200.runner import LayerStep

    ev = lambda: torch.cuda.Event(enable_timing=True)
    g = torch.Generator(device=dev).manual_seed(0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    q, k_cur, v_cur = (torch.randn((w0.H, w0.S, w0.D), generator=g, device=dev).to(torch.bfloat16) for _ in range(3))
    rows = []
    for n_chunks in ((4, 10, 20, 40) if args.naive else (4, 10, 20, 40, 80, 120)):
        row = {"chunks": n_chunks, "n_hist": n_chunks * w0.S}
        for mode in ("sparse", "dense") + (("naive",) if args.naive else ()):
            if mode == "naive":
                row.update(naive_sparse(args, om, torch, replace(w0, n_hist=n_chunks * w0.S), dev, g, q, k_cur, v_cur, flush))
                continue
            w = replace(w0, n_hist=n_chunks * w0.S) if mode == "sparse" else replace(w0, n_hist=n_chunks * w0.S, n_wt=n_chunks * w0.S, K=1)
            ls = LayerStep(w, dev, fuse_mode=min(args.fuse, 1), cmp=args.fuse == 2)
            ls.three = args.fuse == 2
            for _ in range(n_chunks):
                kc = torch.randn((w.H, w.S, w.D), generator=g, device=dev).to(torch.bfloat16)
                ls.append(kc, kc.flip(1))
            ts = []
            n_it = max(5, min(args.steps, 3000 // n_chunks if mode == "dense" else args.steps))
            for i in range(3 + n_it):
                flush.zero_()
                e0, e1 = ev(), ev()
                e0.record()
                ls.step(q, k_cur, v_cur)
                e1.record()
                torch.cuda.synchronize()
                if i >= 3:
                    ts.append(e0.elapsed_time(e1))
            row[mode + "_ms"] = float(np.mean(ts))
            row[mode + "_gflop"] = w.flops() / 1e9
            row[mode + "_tflops"] = w.flops() / (np.mean(ts) * 1e-3) / 1e12
            if mode == "sparse":
                u, _, _ = union_stats(om, torch, ls, w, dev)
                row.update({"M_scatter_MB": u["M_scatter_bytes"] / 1e6, "M_merge_shared_MB": u["M_merge_bytes"] / 1e6,
                            "M_full_MB": u["M_full_history_bytes"] / 1e6})
            del ls
            torch.cuda.empty_cache()
        row["speedup"] = row["dense_ms"] / row["sparse_ms"]
        rows.append(row)
    print(json.dumps({"metric": "ms per AR-step layer (select+attend) against history length", "unit": "ms", "config": {
        "workload": w0.name + " shapes, random data", "H": w0.H, "D": w0.D, "S": w0.S, "B": w0.B, "K": w0.K, "G_q": w0.G,
        "sparse": "window 1 chunk + top-K", "dense": "window = whole history, K = 1"}, "rows": rows}))


def naive_sparse(args, om, torch, w, dev, g, q, k_cur, v_cur, flush):
    """Naive Sparse on the same inputs: select with G_q = 1, merge the union of all heads' blocks, dense attention over it."""
    from dataclasses import replace
    from paper_2605_30519_b200.runner import LayerStep
    ev = lambda: torch.cuda.Event(enable_timing=True)
    w1 = replace(w, G=1)
    src = LayerStep(w1, dev)
    for _ in range(w.n_hist // w.S):
        kc = torch.randn((w.H, w.S, w.D), generator=g, device=dev).to(torch.bfloat16)
        src.append(kc, kc.flip(1))
    src.select(q)
    u, union_list, n_u = union_stats(om, torch, src, w1, dev)
    # merged buffer + the window's blocks as one history, every query attends to all of it (window = whole buffer, K = 1)
    n_tok = n_u * w.B + w.n_wt
    wd = replace(w, n_hist=n_tok, n_wt=n_tok, K=1)
    ts_sel, ts_gather, ts_att = [], [], []
    for i in range(3 + max(3, min(args.steps, 10))):
        dst = LayerStep(wd, dev, max_tokens=n_tok + w.S)
        flush.zero_()
        e0, e1, e2 = ev(), ev(), ev()
        e0.record()
        src.select(q)
        e1.record()
        om.omnimem_gather_blocks(src.cache, union_list, n_u, dst.cache)
        e2.record()
        # the window chunk follows the merged blocks (its pages are part of the buffer a dense kernel walks)
        kc = torch.randn((w.H, w.n_wt, w.D), generator=g, device=dev).to(torch.bfloat16)
        dst.append(kc, kc.flip(1))
        flush.zero_()
        e3, e4 = ev(), ev()
        e3.record()
        dst.step(q, k_cur, v_cur)
        e4.record()
        torch.cuda.synchronize()
        if i >= 3:
            ts_sel.append(e0.elapsed_time(e1)); ts_gather.append(e1.elapsed_time(e2)); ts_att.append(e3.elapsed_time(e4))
        del dst
    del src
    torch.cuda.empty_cache()
    return {"naive_ms": float(np.mean(ts_sel) + np.mean(ts_gather) + np.mean(ts_att)), "naive_select_ms": float(np.mean(ts_sel)),
            "naive_gather_ms": float(np.mean(ts_gather)), "naive_attend_ms": float(np.mean(ts_att)), "naive_union_blocks": n_u,
            "naive_M_merge_MB": u["M_merge_bytes"] / 1e6, "naive_M_scatter_MB": u["M_scatter_bytes"] / 1e6}


def sweep_lru(args, dev):
    """The shape of the paper's Fig. F1 on synthetic data: a chunk-by-chunk rollout in the paper's geometry with
    only G chunk slots per head in HBM (omnimem_offload_*), for several G: hit rate of the selections' chunk requests, reloads,
    HBM held by the full-resolution K/V pool, and the latency of a layer step including the host step (select + offload_step in
    WAIT mode + attend).  Data: seeded N(0,1) chunks plus a per-(head, chunk) offset so that heads prefer a few old chunks."""
    import torch
    from dataclasses import replace
    from paper_2605_30519_b200 import binding as om, synth
    from paper_2605_30519_b200.runner import LayerStep

    w0 = synth.config("paper")
    n_chunks = 24
    w = replace(w0, n_hist=n_chunks * w0.S, n_wt=w0.S, t_awe=w0.bpc)  # window 1 chunk (pinned), AWE once a chunk lies outside it
    g = torch.Generator(device=dev).manual_seed(0)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    rows = []
    for G in (3, 4, 6, 8, 12, n_chunks + 1):
        torch.manual_seed(0)
        g.manual_seed(0)
        ls = LayerStep(w, dev, resident_chunks=G, pinned_recent=1)
        offs = torch.randn((w.H, n_chunks, 1, w.D), generator=g, device=dev)
        k_cur = torch.randn((w.H, w.S, w.D), generator=g, device=dev).to(torch.bfloat16)
        ts, st = [], None
        for c in range(n_chunks):
            kc = (torch.randn((w.H, w.S, w.D), generator=g, device=dev) * 0.5 + offs[:, c]).to(torch.bfloat16)
            ls.append(kc, kc.flip(1))
            if c < 4:
                continue
            # the queries of this step lean towards three older chunks per head (they drift slowly along the rollout)
            tgt = [(c // 4 + j * 5) % max(c - 1, 1) for j in range(3)]
            q = (torch.randn((w.H, w.S, w.D), generator=g, device=dev) * 0.5 + offs[:, tgt].sum(dim=1)).to(torch.bfloat16)
            e0, e1 = ev(), ev()
            e0.record()
            ls.select(q)
            st = om.omnimem_offload_step(ls.cache, ls.block_idx, ls.ptr_table, om.OFFLOAD_WAIT)
            ls.attend(q, k_cur, k_cur)
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        rows.append({"G": G, "hbm_kv_pool_MB": 2 * ls.cache.k_pages.numel() * 2 / 1e6, "hit_rate": st["hit_rate"], "requests": st["requests"],
                     "reloads": st["reloads"], "evictions": st["evictions"], "skipped_last_step": st["skipped"],
                     "step_ms_mean": float(np.mean(ts)), "step_ms_median": float(np.median(ts))})
        del ls
        torch.cuda.empty_cache()
    print(json.dumps({"metric": "offload: hit rate / step latency / HBM against the number of resident chunk slots G", "unit": "ms", "config": {
        "workload": "paper geometry (B 30 in 32-row pages, G_q 15, top-4), window 1 chunk, 24-chunk rollout, random data with per-chunk offsets",
        "H": w.H, "D": w.D, "S": w.S, "mode": "WAIT (reload, then rebuild the table)", "step": "select + offload_step (one stream sync) + attend"},
        "rows": rows}))


def config_dict(w, args, world):
    """The workload description both arms print (same keys, same values: the two lines describe one configuration)."""
    return {"workload": w.name, "H": w.H, "D": w.D, "S": w.S, "n_hist": w.n_hist, "B": w.B, "K": w.K, "G_q": w.G,
            "window_tokens": w.n_wt, "fuse_mode": ["JOINT", "GATED", "GATED3 (CMP+SLC+SWA)"][args.fuse],
            "l2": "flushed with a 256 MiB write between timed steps (per_chunk kernels: write then 256 MiB read, clean lines)",
            "replicas": world}


# (head, query) rows of the bounded oracle sample: the SAME sample in the main arm's cpu_baseline and in --impl reference
ORACLE_SAMPLE = dict(n_groups=10, rows_per_group=20)


def oracle_prepare(w, d):
    """Builds the oracle's cache (append + pool, once per chunk in the method; not part of a step)."""
    import oracle

    t0 = time.perf_counter()
    oc = oracle.cache_create(w.H, w.D, w.B, w.n_hist + w.S)
    for lo in range(0, w.n_hist, w.chunk):
        oracle.append_chunk(oc, d["k_hist"][:, lo:lo + w.chunk], d["v_hist"][:, lo:lo + w.chunk])
    oracle.pool_keys(oc)
    return oc, time.perf_counter() - t0


def oracle_timed_sample(w, d, oc, n_groups=ORACLE_SAMPLE["n_groups"], rows_per_group=ORACLE_SAMPLE["rows_per_group"]):
    """One step of the oracle as it stands on the host cores: selection in full + attention on a bounded row
    sample, attention time scaled to all rows.  Returns (ms_per_step_estimate, description)."""
    import oracle
    from paper_2605_30519_b200 import synth

    t0 = time.perf_counter()
    sel = oracle.select(oc, d["q"], w.G, w.K, w.n_wt, w.t_awe, w.softmax_scale)
    t_sel = time.perf_counter() - t0
    hh, qq = synth.sample_rows(w, n_groups, rows_per_group)
    t0 = time.perf_counter()
    oracle.sparse_attn_rows(oc, hh, qq, d["q"], d["k_cur"], d["v_cur"], sel["block_idx"], sel["ptr_table"],
                            G=w.G, K=w.K, n_wt=w.n_wt, softmax_scale=w.softmax_scale)
    t_att = time.perf_counter() - t0
    ms = 1e3 * (t_sel + t_att * (w.H * w.S) / len(hh))
    desc = (f"select a2-a5 in full ({t_sel:.2f} s) + attention a6-a8 on {len(hh)} of {w.H * w.S} (head, query) rows "
            f"({t_att:.2f} s), attention time scaled by rows; single thread")
    return ms, desc


def run_reference(args, w, d):
    """--impl reference: the CPU oracle, timed as it stands on this box's host cores.  Each step is a bounded
    sample (full selection + ~2000 (head, query) rows of attention, the same sample as the main arm's cpu_baseline),
    its attention time scaled to all rows, so that the run ends within a few minutes."""
    oc, _ = oracle_prepare(w, d)
    vals = []
    desc = ""
    for i in range(args.warmup + args.steps):
        ms, desc = oracle_timed_sample(w, d, oc)
        if i >= args.warmup:
            vals.append(ms)
    v = float(np.mean(vals))
    print(json.dumps({
        "impl": "reference", "metric": "ms per AR-step layer (select+attend)", "value": v, "unit": "ms",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": v, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(w, args, 1),
        "cpu_baseline": {"value": v, "unit": "ms", "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": v, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="wan1p3b")
    ap.add_argument("--fuse", type=int, default=0, help="0 JOINT, 1 GATED (SLC + SWA), 2 GATED3 (full Eq. 1: CMP + SLC + SWA)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--naive", action="store_true", help="with --sweep-history: add the Naive-Sparse comparison (per-query top-k + merged buffer)")
    ap.add_argument("--sweep-lru", action="store_true", help="offloading: hit rate / latency / HBM against the number of resident chunk slots")
    ap.add_argument("--sweep-history", action="store_true",
                    help="latency of the step against history length, sparse (window 1 chunk + top-k) next to the same "
                         "kernel with the window spanning the whole history (dense); random device-side data")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from paper_2605_30519_b200 import synth
    w = synth.config(args.workload)

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, w, synth.generate(w))
        return

    import torch
    import torch.distributed as dist
    from paper_2605_30519_b200 import binding as om
    from paper_2605_30519_b200.runner import HostPipeline, LayerStep, to_dev

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    om.load()
    # started well before the timed region: nvidia-smi needs a few hundred ms before its first sample
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()

    if args.sweep_history:
        if rank == 0:
            sweep_history(args, w, dev)
        return
    if args.sweep_lru:
        if rank == 0:
            sweep_lru(args, dev)
        return

    d = synth.generate(w)
    ls = LayerStep(w, dev, fuse_mode=min(args.fuse, 1), cmp=args.fuse == 2)
    ls.three = args.fuse == 2
    # per-chunk work (a0, a1), timed separately: once per generated chunk, not per denoising step
    ev = lambda: torch.cuda.Event(enable_timing=True)
    t_append, t_pool = [], []
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    clean = torch.zeros(256 << 20, dtype=torch.uint8, device=dev).view(torch.int32)

    def flush_clean():
        """For the HBM-bound per-chunk kernels: write 256 MiB, then READ another 256 MiB, so that L2 ends up full of
        CLEAN foreign lines.  After a write-only flush the ~126 MB of dirty lines are written back underneath the
        next kernel and its reads share the DRAM pins with them (pool_keys: 4.5 instead of 6.1 TB/s).  The flush
        also keeps the GPU busy while the next launches are enqueued, so the events bracket kernels, not launches."""
        flush.zero_()
        return clean.sum()

    for lo in range(0, w.n_hist, w.chunk):
        kc, vc = to_dev(d["k_hist"][:, lo:lo + w.chunk], dev), to_dev(d["v_hist"][:, lo:lo + w.chunk], dev)
        flush_clean()
        e0, e1, e2 = ev(), ev(), ev()
        e0.record()
        om.omnimem_append_chunk(ls.cache, kc, vc)
        e1.record()
        om.omnimem_pool_keys(ls.cache, 0, -1)
        e2.record()
        torch.cuda.synchronize()
        t_append.append(e0.elapsed_time(e1))
        t_pool.append(e1.elapsed_time(e2))
    # full-history pooling: the bandwidth showcase of a1
    t_pool_full = []
    for _ in range(5):
        flush_clean()
        e0, e1 = ev(), ev()
        e0.record()
        om.omnimem_pool_keys(ls.cache, 0, ls.cache.n_blocks)
        e1.record()
        torch.cuda.synchronize()
        t_pool_full.append(e0.elapsed_time(e1))

    q, k_cur, v_cur = to_dev(d["q"], dev), to_dev(d["k_cur"], dev), to_dev(d["v_cur"], dev)
    hq, hk, hv = (t.cpu().pin_memory() for t in (q, k_cur, v_cur))
    hout = torch.empty_like(ls.out, device="cpu").pin_memory()

    def one_step(timed, split=False):
        """One AR-step layer.  The headline loop records no event between the two calls (the step's kernels are
        chained by programmatic dependent launch; an event in between would break the chain); the select / attend
        split is measured by a second loop with the event in place."""
        flush.zero_()
        e0, e1, e2 = ev(), ev(), ev()
        e0.record()
        ls.select(q)
        if split:
            e1.record()
        ls.attend(q, k_cur, v_cur)
        e2.record()
        if timed is not None:
            timed.append((e0, e1, e2))

    for _ in range(args.warmup):
        one_step(None)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    launches0 = om.launch_count()
    events = []
    torch.cuda.synchronize()
    t_wall0 = time.perf_counter()
    t_epoch0 = time.time()
    for _ in range(args.steps):
        one_step(events)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = om.launch_count() - launches0
    clocks = sampler.stop(t_epoch0, time.time()) if rank == 0 else None
    step_ms = [a.elapsed_time(c) for a, _, c in events]
    ms_per_step = float(np.mean(step_ms))
    split_events = []
    for _ in range(min(args.steps, 50)):
        one_step(split_events, split=True)
    torch.cuda.synchronize()
    # the warm number: the same step back to back without the L2 flush
    warm = []
    for _ in range(min(args.steps, 50)):
        e0, e2 = ev(), ev()
        e0.record()
        ls.select(q)
        ls.attend(q, k_cur, v_cur)
        e2.record()
        warm.append((e0, e2))
    torch.cuda.synchronize()
    warm_ms = float(np.mean([a.elapsed_time(b) for a, b in warm]))
    sel_ms = [a.elapsed_time(b) for a, b, _ in split_events]
    att_ms = [b.elapsed_time(c) for _, b, c in split_events]
    # the paper's own fusion, Eq. 1 without CMP (separate softmaxes + per-head gates), timed next to the headline mode
    gated = None
    if args.fuse == 0:
        ls.ap.fuse_mode = om.FUSE_GATED
        g_events, g_split = [], []
        for _ in range(3):
            one_step(None)
        for _ in range(min(args.steps, 100)):
            one_step(g_events)
        for _ in range(min(args.steps, 30)):
            one_step(g_split, split=True)
        torch.cuda.synchronize()
        ls.ap.fuse_mode = om.FUSE_JOINT
        gated = (float(np.mean([a.elapsed_time(c) for a, _, c in g_events])), float(np.mean([b.elapsed_time(c) for _, b, c in g_split])))
    union, _, _ = union_stats(om, torch, ls, w, dev)

    # end to end through the public API with HOST buffers: H2D of q/k_cur/v_cur, select+attend, D2H of out
    e2e = []
    for i in range(args.warmup + args.steps):
        flush.zero_()
        e0, e1 = ev(), ev()
        e0.record()
        q.copy_(hq, non_blocking=True)
        k_cur.copy_(hk, non_blocking=True)
        v_cur.copy_(hv, non_blocking=True)
        ls.step(q, k_cur, v_cur)
        hout.copy_(ls.out, non_blocking=True)
        e1.record()
        torch.cuda.synchronize()
        if i >= args.warmup:
            e2e.append(e0.elapsed_time(e1))
    e2e_serial_ms = float(np.mean(e2e))
    serial_out = hout.clone()
    # ... and as a stream of steps (runner.HostPipeline): the copies of neighbouring steps overlap the kernels on three streams
    # over double-buffered device tensors; every step still copies its own inputs in and its own result out
    pipe = HostPipeline(ls)
    for _ in range(args.warmup):
        flush.zero_()
        pipe.submit(hq, hk, hv, hout)
    pipe.drain()
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    e0.record()
    for _ in range(args.steps):
        flush.zero_()
        pipe.submit(hq, hk, hv, hout)
    pipe.drain()
    e1.record()
    torch.cuda.synchronize()
    e2e_ms = e0.elapsed_time(e1) / args.steps
    if not torch.equal(hout, serial_out):
        raise RuntimeError("pipelined steps disagree with the serial steps")

    ms_per_step, e2e_ms, att_mean = max_over_ranks([ms_per_step, e2e_ms, float(np.mean(att_ms))], dev, world)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = measured_peaks()
    pool_bytes = w.H * w.n_hist * w.D * 2 * (2 if args.fuse == 2 else 1)  # the compressed cache keeps block values too with the CMP branch
    flops = w.flops() + (4.0 * w.D * w.S * w.n_b * w.H if args.fuse == 2 else 0.0)  # + compression attention over N_b tokens
    tflops = flops / (att_mean * 1e-3) / 1e12
    # bytes: touched KV = selected pages per (h, r, slot) + window + current chunk
    kv_row = 2 * w.D * 2  # K and V, bf16
    touched = w.H * (w.R * min(w.K, w.n_b) * w.B + (w.n_hist - w.win_start) + w.S) * kv_row
    kv_gbs = touched / (att_mean * 1e-3) / 1e9
    t_roof_ms = max(flops / (peaks["bf16_tflops"] * 1e12), touched / (peaks["hbm_gbs"] * 1e9)) * 1e3
    out = {
        "metric": "ms per AR-step layer (select+attend)", "value": ms_per_step, "unit": "ms", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": config_dict(w, args, world),
        "warm_l2_ms_per_step": warm_ms, "select_ms": float(np.mean(sel_ms)), "attend_ms": att_mean, "min_step_ms": float(np.min(step_ms)),
        "median_step_ms": float(np.median(step_ms)),
        "attn_tflops": tflops, "kv_gbs_touched": kv_gbs,
        "step_roofline": {"t_roof_ms": t_roof_ms, "frac": t_roof_ms / ms_per_step, "peaks": peaks["source"],
                          "nominal_frac": max(flops / 2.25e15, touched / 8e12) * 1e3 / ms_per_step},
        "roofline": {"kernel": "omnimem_sparse_attn", "bound": "tensor", "achieved": tflops, "peak": peaks["bf16_tflops"] / 1.0,
                     "unit": "TFLOP/s", "frac": tflops / peaks["bf16_tflops"], "traffic": ATTN_DRAM_TRAFFIC_BYTES.get((w.name, args.fuse)),
                     "peak_source": peaks["source"] + " (burst)", "flops_per_launch": flops},
        "sm_l2_ingest": l2_ingest(w, att_mean, (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0,
                                  torch.cuda.get_device_properties(dev).multi_processor_count),
        "per_chunk": {"append_ms": float(np.median(t_append)), "pool_dirty_ms": float(np.median(t_pool)),
                      "append_gbs": 4 * w.H * w.chunk * w.D * 2 / (np.median(t_append) * 1e-3) / 1e9,
                      "pool_full_ms": float(np.min(t_pool_full)),
                      "pool_full_gbs": pool_bytes / (np.min(t_pool_full) * 1e-3) / 1e9,
                      "pool_full_frac_of_hbm": pool_bytes / (np.min(t_pool_full) * 1e-3) / 1e9 / peaks["hbm_gbs"],
                      "pool_full_pools": "K and V" if args.fuse == 2 else "K"},
        "e2e": {"value": e2e_ms, "unit": "ms", "h2d_bytes_per_step": int(3 * q.numel() * 2),
                "d2h_bytes_per_step": int(ls.out.numel() * 2), "serial_ms": e2e_serial_ms,
                "how": "value: a stream of steps through runner.HostPipeline (pinned host q / k_cur / v_cur in, result out, every step; the copies of "
                       "neighbouring steps overlap the kernels on three streams, L2 flushed every step); serial_ms: one step at a time, copies and "
                       "kernels back to back with a synchronize in between"},
        "gpu_launches": int(launches), "wall_s_timed_region": t_wall, "clocks": clocks,
        "union": union,
    }
    if gated is not None:
        out["gated"] = {"what": "Eq. 1 without CMP: g_slc * Attn_SLC + g_swa * Attn_SWA, separate softmaxes (PAPER.md:66)", "ms_per_step": gated[0],
                        "attend_ms": gated[1], "attn_tflops": flops / (gated[1] * 1e-3) / 1e12,
                        "roofline_frac": flops / (gated[1] * 1e-3) / 1e12 / peaks["bf16_tflops"], "step_roofline_frac": t_roof_ms / gated[0]}
    if world == 1 and not args.no_cpu_baseline:
        oc, _ = oracle_prepare(w, d)
        ms, desc = oracle_timed_sample(w, d, oc)
        out["cpu_baseline"] = {"value": ms, "unit": "ms", "cores": 1, "kind": "oracle", "sample": desc}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum of ONE omnimem_sparse_attn launch, from the `ncu --set full` captures summarised in
# profiles/r2_ncu_full.md (the numbers live in profiles/r2_traffic.json.txt), keyed by (workload, --fuse).  A configuration
# without a capture prints null.
def _traffic_table():
    try:
        with open(os.path.join(ROOT, "profiles", "r2_traffic.json.txt")) as f:
            t = json.load(f)
    except (OSError, ValueError):
        return {}
    return {("wan1p3b", 0): t.get("r2_attn_joint"), ("wan1p3b", 1): t.get("r2_attn_gated")}


ATTN_DRAM_TRAFFIC_BYTES = _traffic_table()

if __name__ == "__main__":
    main()
