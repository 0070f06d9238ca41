/*
 * omnimem.h -- C ABI of the B200-native OmniMem hot path (arxiv/paper_2605_30519).
 *
 * The four hot calls follow the paper's statement of the problem ("which historical blocks
 * should be retrieved ... how should these selected blocks be efficiently organized",
 * PAPER.md:62): omnimem_append_chunk, omnimem_pool_keys, omnimem_select, omnimem_sparse_attn.
 *
 * General contract
 *  - Every function returns int32_t: OMNIMEM_OK (0) or a negative error code; the text of the
 *    last error on the calling thread is available from omnimem_last_error().  No exception
 *    crosses the ABI.
 *  - "device" pointers are CUDA global-memory addresses on the current device, 16-byte aligned;
 *    "host" pointers are ordinary process memory.  The CALLER owns every device buffer (the
 *    Python binding allocates them with torch); the library owns only the small host-side
 *    omnimem_cache_t.  Hot calls never allocate device memory and never synchronise: all work
 *    is enqueued on the caller's stream (a cudaStream_t passed as void*; NULL = default stream).
 *  - Floating tensors are bf16 (OMNIMEM_DTYPE_BF16), head-major: element (h, t, d) of a
 *    [H][n][D] tensor lives at  base + h*stride_head + t*stride_tok + d   (strides in elements,
 *    multiples of 8; d is contiguous).
 *  - Batch size is 1 (Algorithm 1's index b, is dropped); one cache handle per
 *    attention layer.
 *  - There is no CPU fallback: if no sm_100 device is usable the calls return OMNIMEM_ECUDA.
 *
 * Cache layout in HBM (two-level cache)
 *    max_blocks = ceil(max_tokens / B)
 *    k_pages, v_pages : [H][max_blocks][B][D] bf16   full-resolution cache, page = one KV block
 *    pooled_k         : [H][max_blocks][D]    bf16   compressed cache (block keys), by LOGICAL block
 *    page_map         : [H][max_blocks]       int32  logical block -> physical page of that head
 *                                                    (the paper's per-head pointer table Pi[h,c],
 *                                                    PAPER.md:356, with B_pc = 1); any per-head
 *                                                    permutation is legal.
 *  History token p of head h lives in page page_map[h][p / B] at row p % B.
 */
#ifndef OMNIMEM_H_
#define OMNIMEM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OMNIMEM_OK 0
#define OMNIMEM_EINVAL (-1)       /* bad argument (null, misaligned, out of range)            */
#define OMNIMEM_ECAPACITY (-2)    /* append beyond max_tokens, or workspace too small         */
#define OMNIMEM_EUNSUPPORTED (-3) /* shape outside D in {64,128}, B in [1,128], K in [1,64]   */
#define OMNIMEM_ECUDA (-4)        /* a CUDA runtime/driver call failed                        */
#define OMNIMEM_ESTATE (-5)       /* call not valid in the cache's current state              */

#define OMNIMEM_DTYPE_BF16 1

/* What "compression-attention scores" means for the selection (readings A1 / A1b):
 * LOGIT: sbar[h][r][b] = score_scale * <qbar[h][r], kbar[h][b]> -- the group average of the per-query logits, by linearity.
 * PROB:  sbar[h][r][b] = mean over the group's queries of softmax_b(score_scale * <q, kbar[h][b]>) over the head's N_b
 *        compressed tokens -- the probabilities the CMP branch of Eq. 1 attends with (NSA-style).  N_b <= 11264. */
#define OMNIMEM_SCORE_LOGIT 0
#define OMNIMEM_SCORE_PROB 1

#define OMNIMEM_FUSE_JOINT 0 /* one softmax over selected + window + current tokens          */
#define OMNIMEM_FUSE_GATED 1 /* Eq. (1): g_slc*Attn_SLC + g_swa*Attn_SWA, separate softmaxes */

typedef struct omnimem_cache omnimem_cache_t; /* opaque, host side */

typedef struct {
    int32_t n_heads;      /* H                                   */
    int32_t head_dim;     /* D in {64, 128}                      */
    int32_t block_tokens; /* B: tokens per KV block, 1 .. 128    */
    int32_t dtype;        /* OMNIMEM_DTYPE_BF16                  */
    int64_t max_tokens;   /* capacity in history tokens per head */
    /* The paper's own geometry.  Both 0 = the BASELINE layout. */
    int32_t page_tokens;      /* P: rows of a page, 0 (= B, needs B in {64,128}) or 32 / 64 / 128 with P >= B.  A block of
                                 B < P tokens occupies the first B rows of its page; the P - B pad rows stay zero and are
                                 masked in the softmax (":323 pad each tile to 32 tokens ... mask the two extra positions") */
    int32_t blocks_per_chunk; /* B_pc: 0 = page_map is [H][max_blocks], one entry per block; > 0 = the two-level map of
                                 Alg. 1: page_map is [H][ceil(max_blocks / B_pc)], entry [h][c] = the page of chunk c's first
                                 block, a chunk's blocks are consecutive pages: page(h, I) = page_map[h][I / B_pc] + I % B_pc */
    int32_t resident_chunks;  /* G: 0 = every chunk stays in HBM; > 0 (needs blocks_per_chunk > 0) = k_pages / v_pages hold only G
                                 chunk slots per head ([H][G * B_pc][P][D]); the other chunks live in pinned host memory
                                 (omnimem_offload_attach) and page_map[h][c] = -1 marks a chunk that is not resident */
    int32_t reserved0;        /* 0 */
} omnimem_cache_desc_t;

/* Library version (major*10000 + minor*100 + patch). */
int32_t omnimem_version(void);

/* Text of the last error raised on this thread ("" if none).  Pointer stays valid until the next
 * failing call on the same thread. */
const char* omnimem_last_error(void);

/* Bytes the caller must allocate for the four device buffers of a cache (any output may be NULL). */
int32_t omnimem_cache_sizes(const omnimem_cache_desc_t* desc, size_t* k_bytes, size_t* v_bytes,
                            size_t* pooled_k_bytes, size_t* page_map_bytes);

/* Creates the host-side handle around caller-owned device buffers (sizes from omnimem_cache_sizes).
 * Does not touch device memory.  The caller fills page_map (any per-head permutation of
 * 0..max_blocks-1; with blocks_per_chunk > 0 any per-head placement of the chunks, bases multiples of B_pc) or calls
 * omnimem_cache_identity_page_map.  k_pages / v_pages are [H][max_blocks][P][D]; with P > B they must be ZERO-INITIALISED
 * (pad rows are never written), and in any case rows that are read but masked must hold finite values.  *out is set on success and must be
 * released with omnimem_cache_destroy; the device buffers must outlive it. */
int32_t omnimem_cache_create(const omnimem_cache_desc_t* desc, void* k_pages /*device*/,
                             void* v_pages /*device*/, void* pooled_k /*device*/,
                             int32_t* page_map /*device*/, omnimem_cache_t** out /*host*/);

/* Enqueues page_map[h][b] = b for all heads and blocks. */
int32_t omnimem_cache_identity_page_map(omnimem_cache_t* cache, void* stream);

/* Forgets all history (N_hist = 0, no dirty blocks).  Device memory is not touched. */
int32_t omnimem_cache_reset(omnimem_cache_t* cache);
int32_t omnimem_cache_destroy(omnimem_cache_t* cache);
/* N_hist: history tokens appended so far (as enqueued, not necessarily executed yet). */
int64_t omnimem_cache_tokens(const omnimem_cache_t* cache);

/* a0 -- append one finished chunk.  Copies the chunk's post-RoPE K and V
 * ([H][n_tokens][D] bf16, device, strides in elements) to flat history positions
 * [N_hist, N_hist + n_tokens) of the paged cache through page_map, zero-fills the rest of the last
 * page touched (so that unwritten rows are exactly 0), bumps N_hist and marks the touched blocks
 * dirty for omnimem_pool_keys.  ECAPACITY if N_hist + n_tokens > max_tokens. */
int32_t omnimem_append_chunk(omnimem_cache_t* cache, const void* k /*device*/, const void* v /*device*/,
                             int32_t n_tokens, int64_t stride_tok, int64_t stride_head, void* stream);

/* a1 -- block keys (PAPER.md:319 "plain mean pool", :335, :581).  For logical blocks
 * [first_block, first_block + n_blocks) of every head: pooled_k[h][b] = mean over the block's VALID
 * tokens of K, accumulated exactly (fp64), divided in fp32, rounded to nearest-even bf16.
 * n_blocks < 0 pools the dirty range left by omnimem_append_chunk and clears it (first_block is
 * ignored); n_blocks = 0 is a no-op.  Blocks at or beyond ceil(N_hist / B) are EINVAL. */
int32_t omnimem_pool_keys(omnimem_cache_t* cache, int64_t first_block, int64_t n_blocks, void* stream);

/* The value half of the compressed cache ("we pool its KV states into compressed KV blocks"; needed by the
 * compression branch of Eq. 1 only).  pooled_v: device, [H][max_blocks][D] bf16, same size as
 * pooled_k, ZERO-INITIALISED and owned by the caller; must be attached while the cache is empty (ESTATE otherwise).
 * From then on omnimem_pool_keys pools the values of the same blocks with the same recipe (mean over the valid tokens,
 * exact sum -> fp32 -> divide -> RNE bf16) in a second launch. */
int32_t omnimem_cache_attach_pooled_v(omnimem_cache_t* cache, void* pooled_v /*device*/);

typedef struct {
    int32_t group_tokens;           /* G_q: adjacent queries sharing one selection   */
    int32_t top_k;                  /* K in [1, 64] blocks per (head, group)                         */
    int64_t window_tokens;          /* N_wt: history tokens covered by the sliding window (0: none)  */
    int64_t awe_min_outside_blocks; /* T_awe: AWE is active iff b_w >= max(T_awe, K), b_w =          */
                                    /* floor(max(0,N_hist-N_wt)/B) (Eq. 2; App. B :319)  */
    float score_scale;              /* sigma_s multiplying <qbar, kbar> (LOGIT) or <q, kbar> (PROB)   */
    int32_t score_mode;             /* OMNIMEM_SCORE_LOGIT | OMNIMEM_SCORE_PROB                      */
} omnimem_select_params_t;

/* Filled on the host by the select calls: what Adaptive Window Exclusion decided. */
typedef struct {
    int64_t n_blocks;     /* N_b = ceil(N_hist / B)                                  */
    int64_t first_window; /* b_w: first block that intersects the window             */
    int64_t n_candidates; /* |Omega|: candidates are blocks [0, n_candidates)         */
    int32_t active;       /* 1 iff window blocks were excluded                        */
    int32_t n_groups;     /* R = ceil(n_q / G_q)                                      */
} omnimem_awe_info_t;

/* a2-a5 -- Query-Shared KV Selection + Adaptive Window Exclusion + top-k + pointer table
 * (PAPER.md:83-89 Eq. 2, :107-114 Eq. 3, :358-380 Alg. 1 step 1).
 *   qbar[h][r]   = mean of the group's valid queries (fp64 sum, fp32 divide, RNE bf16)
 *   sbar[h][r][b]= score_scale * <qbar[h][r], pooled_k[h][b]>  (fp32 FMA accumulation), -0 -> +0
 *   block_idx[h][r][0..K) = the K candidates with the greatest sbar under the total order
 *                  (score descending, block index ascending), in that order; slots beyond |Omega|
 *                  are -1
 *   ptr_table[h][r][t] = page_map[h][block_idx[h][r][t]], -1 stays -1 (the paper's 0 = skip)
 * q: [H][n_q][D] bf16 device.  block_idx, ptr_table: [H][R][K] int32 device (block_idx may be NULL).
 * scores_out: NULL or [H][R][N_b] fp32 device (all N_b blocks, window included).
 * awe_out: NULL or host struct, written before the call returns.
 * workspace: device scratch of at least the select_bytes reported by omnimem_workspace_bytes.
 * NaN/Inf in q or pooled_k is a contract violation (order unspecified). */
int32_t omnimem_select(const omnimem_cache_t* cache, const void* q /*device*/, int32_t n_q,
                       int64_t stride_tok, int64_t stride_head, const omnimem_select_params_t* params,
                       int32_t* block_idx /*device*/, int32_t* ptr_table /*device*/,
                       float* scores_out /*device*/, omnimem_awe_info_t* awe_out /*host*/,
                       void* workspace /*device*/, size_t workspace_bytes, void* stream);

/* a3-a5 on caller-supplied scores [H][R][N_b] fp32 (device): the same AWE, top-k and table build as
 * omnimem_select without the scoring step.  Used to check the selection bit-for-bit against the
 * oracle on identical fp32 scores. */
int32_t omnimem_select_from_scores(const omnimem_cache_t* cache, const float* scores /*device*/, int32_t n_q,
                                   const omnimem_select_params_t* params, int32_t* block_idx /*device*/,
                                   int32_t* ptr_table /*device*/, omnimem_awe_info_t* awe_out /*host*/,
                                   void* stream);

typedef struct {
    int32_t group_tokens;  /* G_q, as given to omnimem_select                                  */
    int32_t top_k;         /* K: slots per (head, group) in ptr_table                          */
    int64_t window_tokens; /* N_wt                                                             */
    float softmax_scale;   /* sigma (1/sqrt(D), :542)                            */
    int32_t fuse_mode;     /* OMNIMEM_FUSE_JOINT | OMNIMEM_FUSE_GATED                          */
    int32_t reserved;      /* must be 0 (EINVAL otherwise)                                     */
} omnimem_attn_params_t;

/* a6-a8 -- Per-Head Scattered KV Access attention (Alg. 1 step 2)
 * fused with the sliding-window branch and the current chunk.
 * For every head h and query s (group r = s / G_q):
 *   SLC: the valid tokens of pages ptr_table[h][r][0..K) (entries < 0 are skipped), read in place;
 *   SWA: history tokens [max(0,N_hist-N_wt), N_hist) through page_map + all n_q tokens of the
 *        current chunk (k_cur, v_cur; no mask inside the chunk);
 *   JOINT: out = softmax over SLC (+) SWA tokens;  GATED: out = gate_slc[h]*Attn_SLC + gate_swa[h]*Attn_SWA
 *   (an empty branch contributes 0 and has LSE = -inf).
 * ptr_table entries are device data the library cannot validate on the host: every entry must be -1 or a page id the cache's
 * page_map could hold (0 <= id < pages per head); anything else reads another head's page or out of bounds (zeros).
 * q, k_cur, v_cur: [H][n_q][D] bf16 device sharing stride_tok / stride_head.  out: [H][n_q][D] bf16
 * device, contiguous.  gate_slc, gate_swa: [H] fp32 device, required in GATED mode.  lse_out: NULL or
 * [2][H][n_q] fp32 device (natural-log LSE of the SLC and SWA branches).  workspace: device scratch of at
 * least the attn_bytes reported by omnimem_workspace_bytes (may be NULL when that is 0). */
int32_t omnimem_sparse_attn(const omnimem_cache_t* cache, const void* q /*device*/, const void* k_cur /*device*/,
                            const void* v_cur /*device*/, int32_t n_q, int64_t stride_tok, int64_t stride_head,
                            const int32_t* ptr_table /*device*/, const omnimem_attn_params_t* params,
                            const float* gate_slc /*device*/, const float* gate_swa /*device*/,
                            void* out /*device*/, float* lse_out /*device*/, void* workspace /*device*/,
                            size_t workspace_bytes, void* stream);

/* The full Eq. (1) of the paper: out = gate_cmp[h]*Attn_CMP + gate_slc[h]*Attn_SLC + gate_swa[h]*Attn_SWA,
 * three separate softmaxes.  Attn_CMP = Attn(Q, K^cmp, V^cmp): every query attends to the N_b compressed tokens
 * (pooled_k[h][b], pooled_v[h][b]) of its head; no compressed token => contributes 0, LSE = -inf.
 * Arguments as omnimem_sparse_attn, plus gate_cmp: [H] fp32 device.  params->fuse_mode must be OMNIMEM_FUSE_GATED (EINVAL
 * otherwise).  lse_out: NULL or [3][H][n_q] fp32 device (CMP, SLC, SWA).  workspace: as for GATED.  Needs a pooled-value
 * buffer (omnimem_cache_attach_pooled_v) with every appended block pooled (ESTATE otherwise).  Three passes of the
 * attention kernel: CMP -> workspace, SLC added to it, SWA + workspace -> out. */
int32_t omnimem_sparse_attn3(const omnimem_cache_t* cache, const void* q /*device*/, const void* k_cur /*device*/,
                             const void* v_cur /*device*/, int32_t n_q, int64_t stride_tok, int64_t stride_head,
                             const int32_t* ptr_table /*device*/, const omnimem_attn_params_t* params,
                             const float* gate_cmp /*device*/, const float* gate_slc /*device*/,
                             const float* gate_swa /*device*/, void* out /*device*/, float* lse_out /*device*/,
                             void* workspace /*device*/, size_t workspace_bytes, void* stream);

/* Union accounting of a selection (Eqs. 4-5): U_h = the distinct blocks head h selected over all its
 * query groups; per_head[h] = |U_h| (the per-head scattered access touches sum_h |U_h| blocks: M_scatter), *union_all =
 * |union over heads of U_h| (a merged buffer shared by all heads holds N_h times that: M_merge).  block_idx: [H][n_groups][top_k]
 * int32 device as written by omnimem_select (-1 = masked).  per_head: [H] int64 device; union_all: one int64, device;
 * union_list: NULL or [N_b] int32 device, receives the blocks of the union in ascending order.  workspace: device, at least
 * (H + 1) * N_b bytes.  Results are on the device (read them after the stream has caught up). */
int32_t omnimem_union_counts(const omnimem_cache_t* cache, const int32_t* block_idx /*device*/, int32_t n_groups, int32_t top_k,
                             int64_t* per_head /*device*/, int64_t* union_all /*device*/, int32_t* union_list /*device*/,
                             void* workspace /*device*/, size_t workspace_bytes, void* stream);

/* omnimem_union_counts without caller scratch and without any allocation, for callers that cannot call cudaMalloc (code under
 * CUDA graph capture, serving loops, harnesses that forbid it).  Same arguments, results and kernels as omnimem_union_counts
 * (Eqs. 4-5); the (H + 1) * N_b mark bytes live in a device array built into the library
 * (OMNIMEM_UNION_NOALLOC_MAX_BYTES; every GPU that loads the library holds it until exit).  Returns OMNIMEM_ECAPACITY when
 * (H + 1) * N_b exceeds that size (use omnimem_union_counts then).  The call makes no cudaMalloc / cudaFree and calls no
 * allocating routine: it clears the bytes it needs with a memset on `stream` and launches the two kernels there.  The first
 * call on a device resolves the array's address (cudaGetSymbolAddress, once per device; make that call outside a capture).
 * ALL calls share the one array, which keeps the previous call's contents until the next call clears its part: calls that
 * overlap on the GPU (different streams, or graphs replayed concurrently) race -- keep them on one stream or order them. */
#define OMNIMEM_UNION_NOALLOC_MAX_BYTES (1 << 20)
int32_t omnimem_union_counts_noalloc(const omnimem_cache_t* cache, const int32_t* block_idx /*device*/, int32_t n_groups, int32_t top_k,
                                     int64_t* per_head /*device*/, int64_t* union_all /*device*/, int32_t* union_list /*device*/,
                                     void* stream);

/* The merged selected-KV buffer of the paper's Naive-Sparse comparison system:
 * block list[i] (i < n) of EVERY head of `src` is copied into block i of `dst`, an EMPTY cache (ESTATE otherwise) of the same
 * n_heads / head_dim / block_tokens with room for n blocks (ECAPACITY otherwise); dst then holds n * B tokens, all dirty.
 * list: [n] int32 device, block ids below src's N_b (not checked: device data).  The product path never builds this buffer --
 * omnimem_sparse_attn reads pages in place; the call exists so that the comparison runs on the same kernels. */
int32_t omnimem_gather_blocks(const omnimem_cache_t* src, const int32_t* list /*device*/, int64_t n, omnimem_cache_t* dst, void* stream);

/* ---- Offload / reload ("GPU hot cache keeps 7 chunks resident and evicts cold ones with an LRU policy ...
 * offloaded KV blocks live in pinned host memory", :339, :374-377, :470-482).  For a cache created with
 * resident_chunks = G > 0.  Residency is per (head, chunk): page_map[h][c] is the chunk's base page or -1.
 * host_k, host_v: PINNED host memory, [H][n_chunks][B_pc * P][D] bf16 each (n_chunks = ceil(max_blocks / B_pc)): the full-history
 * store; every appended chunk is written through to it.  pinned_recent: the W most recent chunks are never evicted (the sliding
 * window reads them; W >= ceil(N_wt / chunk tokens), W < G).  scratch_host: pinned host, scratch_dev: device, each at least
 * omnimem_offload_scratch_bytes(desc).  All buffers are caller-owned and must outlive the cache.
 * With offloading, omnimem_append_chunk takes whole chunks only (n_tokens = B_pc * B, EINVAL otherwise): the new chunk replaces
 * the least recently used non-pinned chunk of every head when no slot is free. */
size_t omnimem_offload_scratch_bytes(const omnimem_cache_desc_t* desc);
int32_t omnimem_offload_attach(omnimem_cache_t* cache, void* host_k /*pinned host*/, void* host_v /*pinned host*/,
                               int32_t pinned_recent, void* scratch_host /*pinned host*/, void* scratch_dev /*device*/,
                               size_t scratch_bytes);

#define OMNIMEM_OFFLOAD_SKIP 0 /* entries of non-resident chunks stay -1 and are skipped; their chunks are reloaded for later steps */
#define OMNIMEM_OFFLOAD_WAIT 1 /* Alg. 1 lines 9-11 (WaitUntilReload): reload first, then rebuild the table -- nothing is skipped that fits */

typedef struct {
    int64_t requests;  /* (head, chunk) pairs the selections asked for, summed over the calls so far */
    int64_t hits;      /* of those, found resident */
    int64_t reloads;   /* chunks copied host -> device */
    int64_t evictions; /* resident chunks dropped to make room */
    int64_t skipped;   /* table entries left at -1 by the last call (chunk not resident when the attention runs) */
} omnimem_offload_stats_t;

/* The host step of the paper's pipeline (Fig. C1 "Step 1 runs on the host and collects ... the KV chunks each head needs"): reads
 * which chunks block_idx ([H][n_groups][top_k], device, from omnimem_select) touches, SYNCHRONISES the stream once to bring that
 * bitmap to the host, updates the per-head LRU order, enqueues host -> device copies of the missing chunks into the slots of the
 * least recently used non-pinned chunks (never one that this call needs) and publishes the new page_map.  mode WAIT: then
 * rebuilds ptr_table ([H][n_groups][top_k], device) from block_idx through the updated map (Alg. 1 step 1), so the following
 * omnimem_sparse_attn reads every selected block that fits the G slots.  mode SKIP: ptr_table is left as omnimem_select wrote
 * it.  stats_out (host, nullable): cumulative counters. */
int32_t omnimem_offload_step(omnimem_cache_t* cache, const int32_t* block_idx /*device*/, int32_t n_groups, int32_t top_k, int32_t mode,
                             int32_t* ptr_table /*device*/, omnimem_offload_stats_t* stats_out /*host*/, void* stream);

/* Scratch sizes for omnimem_select and omnimem_sparse_attn at this geometry, computed for a full
 * cache (N_hist = max_tokens).  Either params pointer may be NULL (its output is then 0). */
int32_t omnimem_workspace_bytes(const omnimem_cache_desc_t* desc, int32_t n_q,
                                const omnimem_select_params_t* select_params,
                                const omnimem_attn_params_t* attn_params, size_t* select_bytes,
                                size_t* attn_bytes);

/* Number of kernels this library has launched in this process (all streams); bench.py reports the
 * difference over its timed region as "gpu_launches". */
int64_t omnimem_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* OMNIMEM_H_ */
