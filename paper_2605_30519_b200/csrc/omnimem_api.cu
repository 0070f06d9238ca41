// C-ABI boundary of the OmniMem hot path (include/omnimem.h): argument validation, host-side cache
// state and kernel launches.  No device allocation and no synchronisation happens here.
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <atomic>
#include <new>

#include "common.cuh"

namespace omnimem {

static thread_local char g_err[512] = "";
static std::atomic<int64_t> g_launches{0};

int32_t fail(int32_t code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int32_t check_launch(const char* what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "%s: launch failed: %s", what, cudaGetErrorString(e));
    return OMNIMEM_OK;
}

void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

Awe awe_decide(const Cache* c, int64_t window_tokens, int32_t top_k, int64_t t_awe)
{
    Awe a;
    a.n_b = ceil_div64(c->n_hist, c->B);
    a.win_start = c->n_hist - window_tokens;
    if (a.win_start < 0) a.win_start = 0;
    a.b_w = (window_tokens == 0) ? a.n_b : a.win_start / c->B;
    const int64_t need = t_awe > top_k ? t_awe : (int64_t)top_k;
    a.active = a.b_w >= need ? 1 : 0;
    a.n_cand = a.active ? a.b_w : a.n_b;
    return a;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int32_t check_desc(const omnimem_cache_desc_t* d)
{
    if (!d) return fail(OMNIMEM_EINVAL, "desc is NULL");
    if (d->n_heads < 1 || d->max_tokens < 1) return fail(OMNIMEM_EINVAL, "n_heads and max_tokens must be >= 1");
    if (d->dtype != OMNIMEM_DTYPE_BF16) return fail(OMNIMEM_EUNSUPPORTED, "dtype %d: only bf16 is supported", d->dtype);
    if (d->head_dim != 64 && d->head_dim != 128) return fail(OMNIMEM_EUNSUPPORTED, "head_dim %d not in {64,128}", d->head_dim);
    if (d->block_tokens < 1 || d->block_tokens > 128) return fail(OMNIMEM_EUNSUPPORTED, "block_tokens %d not in [1, 128]", d->block_tokens);
    const int32_t P = d->page_tokens ? d->page_tokens : d->block_tokens;
    if (P != 32 && P != 64 && P != 128)
        return fail(OMNIMEM_EUNSUPPORTED, "page rows %d not in {32,64,128} (block_tokens outside {64,128} needs page_tokens)", P);
    if (P < d->block_tokens) return fail(OMNIMEM_EINVAL, "page_tokens %d < block_tokens %d", P, d->block_tokens);
    if (d->blocks_per_chunk < 0) return fail(OMNIMEM_EINVAL, "blocks_per_chunk < 0");
    if (d->resident_chunks < 0 || d->reserved0 != 0) return fail(OMNIMEM_EINVAL, "resident_chunks < 0 or reserved0 != 0");
    if (d->resident_chunks > 0 && d->blocks_per_chunk <= 0) return fail(OMNIMEM_EINVAL, "resident_chunks needs the two-level map (blocks_per_chunk > 0)");
    const int64_t max_blocks = ceil_div64(d->max_tokens, d->block_tokens);
    if ((int64_t)d->n_heads * max_blocks * P >= (int64_t)1 << 31)
        return fail(OMNIMEM_EUNSUPPORTED, "H * max_blocks * P must stay below 2^31 rows");
    return OMNIMEM_OK;
}

static int32_t check_select_params(const omnimem_select_params_t* p, int32_t n_q)
{
    if (!p) return fail(OMNIMEM_EINVAL, "select params is NULL");
    if (n_q < 1) return fail(OMNIMEM_EINVAL, "n_q must be >= 1");
    if (p->group_tokens < 1 || p->group_tokens > n_q) return fail(OMNIMEM_EINVAL, "group_tokens %d not in [1, n_q]", p->group_tokens);
    if (p->top_k < 1 || p->top_k > 64) return fail(OMNIMEM_EUNSUPPORTED, "top_k %d not in [1, 64]", p->top_k);
    if (p->window_tokens < 0 || p->awe_min_outside_blocks < 0) return fail(OMNIMEM_EINVAL, "negative window or threshold");
    if (p->score_mode != OMNIMEM_SCORE_LOGIT && p->score_mode != OMNIMEM_SCORE_PROB) return fail(OMNIMEM_EINVAL, "score_mode %d", p->score_mode);
    return OMNIMEM_OK;
}

static void fill_awe(const Cache* c, const Awe& a, int32_t n_q, int32_t G, omnimem_awe_info_t* out)
{
    if (!out) return;
    out->n_blocks = a.n_b;
    out->first_window = a.b_w;
    out->n_candidates = a.n_cand;
    out->active = a.active;
    out->n_groups = (int32_t)ceil_div64(n_q, G);
    (void)c;
}

}  // namespace omnimem

using namespace omnimem;

extern "C" {

int32_t omnimem_version(void) { return 100; }

const char* omnimem_last_error(void) { return g_err; }

int64_t omnimem_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int32_t omnimem_cache_sizes(const omnimem_cache_desc_t* desc, size_t* k_bytes, size_t* v_bytes,
                            size_t* pooled_k_bytes, size_t* page_map_bytes)
{
    if (int32_t rc = check_desc(desc)) return rc;
    const size_t max_blocks = (size_t)ceil_div64(desc->max_tokens, desc->block_tokens);
    const size_t page = (size_t)(desc->page_tokens ? desc->page_tokens : desc->block_tokens) * desc->head_dim * 2;
    const size_t pool_blocks = desc->resident_chunks > 0 ? (size_t)desc->resident_chunks * desc->blocks_per_chunk : max_blocks;
    if (k_bytes) *k_bytes = (size_t)desc->n_heads * pool_blocks * page;
    if (v_bytes) *v_bytes = (size_t)desc->n_heads * pool_blocks * page;
    if (pooled_k_bytes) *pooled_k_bytes = (size_t)desc->n_heads * max_blocks * desc->head_dim * 2;
    if (page_map_bytes) *page_map_bytes = (size_t)desc->n_heads * max_blocks * 4;
    return OMNIMEM_OK;
}

int32_t omnimem_cache_create(const omnimem_cache_desc_t* desc, void* k_pages, void* v_pages, void* pooled_k,
                             int32_t* page_map, omnimem_cache_t** out)
{
    if (int32_t rc = check_desc(desc)) return rc;
    if (!k_pages || !v_pages || !pooled_k || !page_map || !out) return fail(OMNIMEM_EINVAL, "NULL buffer or out pointer");
    if (!aligned16(k_pages) || !aligned16(v_pages) || !aligned16(pooled_k) || !aligned16(page_map))
        return fail(OMNIMEM_EINVAL, "cache buffers must be 16-byte aligned");
    Cache* c = new (std::nothrow) Cache();
    if (!c) return fail(OMNIMEM_ECAPACITY, "out of host memory");
    c->H = desc->n_heads;
    c->D = desc->head_dim;
    c->B = desc->block_tokens;
    c->P = desc->page_tokens ? desc->page_tokens : desc->block_tokens;
    c->bpc = desc->blocks_per_chunk;
    c->resident_chunks = desc->resident_chunks;
    c->off = nullptr;
    c->max_tokens = desc->max_tokens;
    c->max_blocks = (int32_t)ceil_div64(desc->max_tokens, desc->block_tokens);
    c->k_pages = (__nv_bfloat16*)k_pages;
    c->v_pages = (__nv_bfloat16*)v_pages;
    c->pooled_k = (__nv_bfloat16*)pooled_k;
    c->pooled_v = nullptr;
    c->page_map = page_map;
    c->pool_blocks = c->resident_chunks > 0 ? c->resident_chunks * c->bpc : c->max_blocks;
    c->n_hist = 0;
    c->dirty_first = c->dirty_end = 0;
    c->tmaps_ready = false;
    c->tmaps_cmp_ready = false;
    c->call_q = c->call_k = c->call_v = nullptr;
    c->call_n = 0;
    c->call_st = c->call_sh = 0;
    *out = reinterpret_cast<omnimem_cache_t*>(c);
    return OMNIMEM_OK;
}

int32_t omnimem_cache_identity_page_map(omnimem_cache_t* cache, void* stream)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    return launch_identity_page_map(reinterpret_cast<Cache*>(cache), (cudaStream_t)stream);
}

int32_t omnimem_cache_reset(omnimem_cache_t* cache)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    Cache* c = reinterpret_cast<Cache*>(cache);
    if (c->off) return fail(OMNIMEM_ESTATE, "a cache with offloading attached cannot be reset: create a new one");
    c->n_hist = 0;
    c->dirty_first = c->dirty_end = 0;
    return OMNIMEM_OK;
}

int32_t omnimem_cache_destroy(omnimem_cache_t* cache)
{
    if (cache) offload_destroy(reinterpret_cast<Cache*>(cache)->off);
    delete reinterpret_cast<Cache*>(cache);
    return OMNIMEM_OK;
}

int64_t omnimem_cache_tokens(const omnimem_cache_t* cache)
{
    return cache ? reinterpret_cast<const Cache*>(cache)->n_hist : (int64_t)OMNIMEM_EINVAL;
}

int32_t omnimem_append_chunk(omnimem_cache_t* cache, const void* k, const void* v, int32_t n_tokens,
                             int64_t stride_tok, int64_t stride_head, void* stream)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    Cache* c = reinterpret_cast<Cache*>(cache);
    if (n_tokens < 0) return fail(OMNIMEM_EINVAL, "n_tokens < 0");
    if (n_tokens == 0) return OMNIMEM_OK;
    if (!k || !v || !aligned16(k) || !aligned16(v)) return fail(OMNIMEM_EINVAL, "k/v NULL or not 16-byte aligned");
    if (stride_tok < c->D || stride_tok % 8 || stride_head % 8) return fail(OMNIMEM_EINVAL, "strides must be multiples of 8 elements, stride_tok >= D");
    if (c->n_hist + n_tokens > c->max_tokens)
        return fail(OMNIMEM_ECAPACITY, "append of %d tokens exceeds max_tokens (%lld + %d > %lld)", n_tokens,
                    (long long)c->n_hist, n_tokens, (long long)c->max_tokens);
    if (c->resident_chunks > 0)
        if (int32_t rc = offload_on_append(c, n_tokens, (cudaStream_t)stream)) return rc;
    if (int32_t rc = launch_append(c, k, v, n_tokens, stride_tok, stride_head, (cudaStream_t)stream)) return rc;
    if (c->resident_chunks > 0)
        if (int32_t rc = offload_after_append(c, c->n_hist / ((int64_t)c->bpc * c->B), (cudaStream_t)stream)) return rc;
    const int64_t first = c->n_hist / c->B;
    c->n_hist += n_tokens;
    const int64_t end = ceil_div64(c->n_hist, c->B);
    if (c->dirty_first == c->dirty_end) {
        c->dirty_first = first;
        c->dirty_end = end;
    } else {
        if (first < c->dirty_first) c->dirty_first = first;
        if (end > c->dirty_end) c->dirty_end = end;
    }
    return OMNIMEM_OK;
}

int32_t omnimem_cache_attach_pooled_v(omnimem_cache_t* cache, void* pooled_v)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    Cache* c = reinterpret_cast<Cache*>(cache);
    if (!pooled_v || !aligned16(pooled_v)) return fail(OMNIMEM_EINVAL, "pooled_v NULL or not 16-byte aligned");
    if (c->n_hist != 0) return fail(OMNIMEM_ESTATE, "attach the pooled-value buffer before the first append (N_hist = %lld)", (long long)c->n_hist);
    c->pooled_v = (__nv_bfloat16*)pooled_v;
    c->tmaps_cmp_ready = false;
    return OMNIMEM_OK;
}

// keys, and values too once the value half of the compressed cache is attached
static int32_t pool_range(const Cache* c, int64_t first, int64_t n, cudaStream_t s)
{
    if (int32_t rc = launch_pool(c, c->k_pages, c->pooled_k, first, n, s)) return rc;
    if (c->pooled_v)
        if (int32_t rc = launch_pool(c, c->v_pages, c->pooled_v, first, n, s)) return rc;
    return OMNIMEM_OK;
}

int32_t omnimem_pool_keys(omnimem_cache_t* cache, int64_t first_block, int64_t n_blocks, void* stream)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    Cache* c = reinterpret_cast<Cache*>(cache);
    if (n_blocks < 0) {
        const int64_t f = c->dirty_first, n = c->dirty_end - c->dirty_first;
        if (int32_t rc = pool_range(c, f, n, (cudaStream_t)stream)) return rc;
        c->dirty_first = c->dirty_end = 0;
        return OMNIMEM_OK;
    }
    if (n_blocks == 0) return OMNIMEM_OK;
    const int64_t n_b = ceil_div64(c->n_hist, c->B);
    if (first_block < 0 || first_block + n_blocks > n_b)
        return fail(OMNIMEM_EINVAL, "blocks [%lld, %lld) outside the %lld blocks that hold tokens", (long long)first_block,
                    (long long)(first_block + n_blocks), (long long)n_b);
    return pool_range(c, first_block, n_blocks, (cudaStream_t)stream);
}

int32_t omnimem_workspace_bytes(const omnimem_cache_desc_t* desc, int32_t n_q, const omnimem_select_params_t* sp,
                                const omnimem_attn_params_t* ap, size_t* select_bytes, size_t* attn_bytes)
{
    if (int32_t rc = check_desc(desc)) return rc;
    if (n_q < 1) return fail(OMNIMEM_EINVAL, "n_q must be >= 1");
    if (select_bytes) {
        *select_bytes = 0;
        if (sp) {
            if (int32_t rc = check_select_params(sp, n_q)) return rc;
            const size_t R = (size_t)ceil_div64(n_q, sp->group_tokens);
            const size_t max_blocks = (size_t)ceil_div64(desc->max_tokens, desc->block_tokens);
            size_t qbar = (size_t)desc->n_heads * R * desc->head_dim * 2;
            qbar = (qbar + 255) / 256 * 256;
            *select_bytes = qbar + (size_t)desc->n_heads * R * max_blocks * 4;
            if (sp->score_mode == OMNIMEM_SCORE_PROB)
                *select_bytes += scores_prob_partial_floats(desc->n_heads, n_q, sp->group_tokens, (int64_t)max_blocks) * 4 + 256;
        }
    }
    if (attn_bytes) {
        *attn_bytes = 0;
        if (ap) {
            *attn_bytes = attn_tcgen05_workspace_bytes(desc->n_heads, n_q, desc->head_dim, ap->fuse_mode);
        }
    }
    return OMNIMEM_OK;
}

int32_t omnimem_select(const omnimem_cache_t* cache, const void* q, int32_t n_q, int64_t stride_tok,
                       int64_t stride_head, const omnimem_select_params_t* p, int32_t* block_idx, int32_t* ptr_table,
                       float* scores_out, omnimem_awe_info_t* awe_out, void* workspace, size_t workspace_bytes,
                       void* stream)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    const Cache* c = reinterpret_cast<const Cache*>(cache);
    if (int32_t rc = check_select_params(p, n_q)) return rc;
    if (!q || !aligned16(q) || !ptr_table) return fail(OMNIMEM_EINVAL, "q/ptr_table NULL or q misaligned");
    if (stride_tok < c->D || stride_tok % 8 || stride_head % 8) return fail(OMNIMEM_EINVAL, "strides must be multiples of 8 elements, stride_tok >= D");
    if (c->dirty_first != c->dirty_end) return fail(OMNIMEM_ESTATE, "blocks [%lld, %lld) were appended but not pooled; call omnimem_pool_keys first",
                                                    (long long)c->dirty_first, (long long)c->dirty_end);
    const Awe a = awe_decide(c, p->window_tokens, p->top_k, p->awe_min_outside_blocks);
    const int32_t R = (int32_t)ceil_div64(n_q, p->group_tokens);
    cudaStream_t s = (cudaStream_t)stream;
    if (p->score_mode == OMNIMEM_SCORE_PROB) {
        // per-query softmax over the compressed tokens, averaged over the group; then the same top-k
        if (!scores_prob_fits(a.n_b)) return fail(OMNIMEM_EUNSUPPORTED, "OMNIMEM_SCORE_PROB: N_b = %lld exceeds the supported 11264", (long long)a.n_b);
        const size_t sc_bytes = scores_out ? 0 : ((size_t)c->H * R * (size_t)a.n_b * 4 + 255) / 256 * 256;
        const size_t part_bytes = scores_prob_partial_floats(c->H, n_q, p->group_tokens, a.n_b) * 4;
        if (a.n_b > 0 && (!workspace || !aligned16(workspace) || workspace_bytes < sc_bytes + part_bytes))
            return fail(OMNIMEM_ECAPACITY, "select workspace: need %zu bytes, got %zu", sc_bytes + part_bytes, workspace_bytes);
        float* scores = scores_out ? scores_out : (float*)workspace;
        float* partial = (float*)((char*)workspace + sc_bytes);
        if (int32_t rc = launch_scores_prob(c, q, n_q, stride_tok, stride_head, p->group_tokens, a.n_b, p->score_scale, scores, partial, s)) return rc;
        if (int32_t rc = launch_topk(c, scores, R, a.n_b, a.n_cand, p->top_k, block_idx, ptr_table, s)) return rc;
        fill_awe(c, a, n_q, p->group_tokens, awe_out);
        return OMNIMEM_OK;
    }
    if (select_fused_fits(a.n_b)) {
        // one launch: the groups' scores stay in shared memory (no workspace needed)
        if (int32_t rc = launch_select_fused(c, q, n_q, stride_tok, stride_head, p->group_tokens, a.n_b, a.n_cand, p->top_k, p->score_scale,
                                             scores_out, block_idx, ptr_table, s))
            return rc;
        fill_awe(c, a, n_q, p->group_tokens, awe_out);
        return OMNIMEM_OK;
    }
    size_t qbar_bytes = (size_t)c->H * R * c->D * 2;
    qbar_bytes = (qbar_bytes + 255) / 256 * 256;
    const size_t need = qbar_bytes + (scores_out ? 0 : (size_t)c->H * R * (size_t)a.n_b * 4);
    if (a.n_b > 0 && (!workspace || !aligned16(workspace) || workspace_bytes < need))
        return fail(OMNIMEM_ECAPACITY, "select workspace: need %zu bytes, got %zu", need, workspace_bytes);
    __nv_bfloat16* qbar = (__nv_bfloat16*)workspace;
    float* scores = scores_out ? scores_out : (float*)((char*)workspace + qbar_bytes);
    if (a.n_b > 0) {
        if (int32_t rc = launch_group_mean(c, q, n_q, stride_tok, stride_head, p->group_tokens, qbar, s)) return rc;
        if (int32_t rc = launch_scores(c, qbar, R, a.n_b, p->score_scale, scores, s)) return rc;
    }
    if (int32_t rc = launch_topk(c, scores, R, a.n_b, a.n_cand, p->top_k, block_idx, ptr_table, s)) return rc;
    fill_awe(c, a, n_q, p->group_tokens, awe_out);
    return OMNIMEM_OK;
}

int32_t omnimem_select_from_scores(const omnimem_cache_t* cache, const float* scores, int32_t n_q,
                                   const omnimem_select_params_t* p, int32_t* block_idx, int32_t* ptr_table,
                                   omnimem_awe_info_t* awe_out, void* stream)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    const Cache* c = reinterpret_cast<const Cache*>(cache);
    if (int32_t rc = check_select_params(p, n_q)) return rc;
    if (!ptr_table) return fail(OMNIMEM_EINVAL, "ptr_table is NULL");
    const Awe a = awe_decide(c, p->window_tokens, p->top_k, p->awe_min_outside_blocks);
    if (a.n_b > 0 && !scores) return fail(OMNIMEM_EINVAL, "scores is NULL");
    const int32_t R = (int32_t)ceil_div64(n_q, p->group_tokens);
    if (int32_t rc = launch_topk(c, scores, R, a.n_b, a.n_cand, p->top_k, block_idx, ptr_table, (cudaStream_t)stream)) return rc;
    fill_awe(c, a, n_q, p->group_tokens, awe_out);
    return OMNIMEM_OK;
}

int32_t omnimem_union_counts(const omnimem_cache_t* cache, const int32_t* block_idx, int32_t n_groups, int32_t top_k, int64_t* per_head,
                             int64_t* union_all, int32_t* union_list, void* workspace, size_t workspace_bytes, void* stream)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    const Cache* c = reinterpret_cast<const Cache*>(cache);
    if (!block_idx || !per_head || !union_all) return fail(OMNIMEM_EINVAL, "NULL argument");
    if (n_groups < 1 || top_k < 1) return fail(OMNIMEM_EINVAL, "n_groups and top_k must be >= 1");
    const int64_t n_b = ceil_div64(c->n_hist, c->B);
    const size_t need = (size_t)(c->H + 1) * (size_t)(n_b > 0 ? n_b : 1);
    if (!workspace || workspace_bytes < need) return fail(OMNIMEM_ECAPACITY, "union workspace: need %zu bytes, got %zu", need, workspace_bytes);
    return launch_union_counts(c, block_idx, n_groups, top_k, n_b, (long long*)per_head, (long long*)union_all, union_list,
                               (unsigned char*)workspace, (cudaStream_t)stream);
}

int32_t omnimem_gather_blocks(const omnimem_cache_t* src, const int32_t* list, int64_t n, omnimem_cache_t* dst, void* stream)
{
    if (!src || !dst) return fail(OMNIMEM_EINVAL, "cache is NULL");
    const Cache* a = reinterpret_cast<const Cache*>(src);
    Cache* b = reinterpret_cast<Cache*>(dst);
    if (n < 0 || (n > 0 && !list)) return fail(OMNIMEM_EINVAL, "bad list");
    if (a->H != b->H || a->D != b->D || a->B != b->B || a->P != b->P) return fail(OMNIMEM_EINVAL, "src and dst geometries differ");
    if (b->n_hist != 0) return fail(OMNIMEM_ESTATE, "dst must be empty (N_hist = %lld)", (long long)b->n_hist);
    if (n > b->max_blocks) return fail(OMNIMEM_ECAPACITY, "dst holds %d blocks, %lld asked for", b->max_blocks, (long long)n);
    if (int32_t rc = launch_gather_blocks(a, list, n, b, (cudaStream_t)stream)) return rc;
    b->n_hist = n * b->B;
    b->dirty_first = 0;
    b->dirty_end = n;
    return OMNIMEM_OK;
}

static int32_t sparse_attn_impl(const omnimem_cache_t* cache, const void* q, const void* k_cur, const void* v_cur,
                                int32_t n_q, int64_t stride_tok, int64_t stride_head, const int32_t* ptr_table,
                                const omnimem_attn_params_t* p, const float* gate_cmp, const float* gate_slc, const float* gate_swa,
                                void* out, float* lse_out, void* workspace, size_t workspace_bytes, void* stream, bool three)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    const Cache* c = reinterpret_cast<const Cache*>(cache);
    if (!p) return fail(OMNIMEM_EINVAL, "attn params is NULL");
    if (n_q < 1) return fail(OMNIMEM_EINVAL, "n_q must be >= 1");
    if (!q || !k_cur || !v_cur || !out || !ptr_table) return fail(OMNIMEM_EINVAL, "NULL tensor argument");
    if (!aligned16(q) || !aligned16(k_cur) || !aligned16(v_cur) || !aligned16(out)) return fail(OMNIMEM_EINVAL, "tensors must be 16-byte aligned");
    if (stride_tok < c->D || stride_tok % 8 || stride_head % 8) return fail(OMNIMEM_EINVAL, "strides must be multiples of 8 elements, stride_tok >= D");
    if (p->group_tokens < 1 || p->group_tokens > n_q) return fail(OMNIMEM_EINVAL, "group_tokens %d not in [1, n_q]", p->group_tokens);
    if (p->top_k < 1 || p->top_k > 64) return fail(OMNIMEM_EUNSUPPORTED, "top_k %d not in [1, 64]", p->top_k);
    if (p->window_tokens < 0) return fail(OMNIMEM_EINVAL, "window_tokens < 0");
    if (p->fuse_mode != OMNIMEM_FUSE_JOINT && p->fuse_mode != OMNIMEM_FUSE_GATED) return fail(OMNIMEM_EINVAL, "fuse_mode %d", p->fuse_mode);
    if (p->fuse_mode == OMNIMEM_FUSE_GATED && (!gate_slc || !gate_swa)) return fail(OMNIMEM_EINVAL, "GATED mode needs gate_slc and gate_swa");
    if (!(p->softmax_scale > 0.f)) return fail(OMNIMEM_EINVAL, "softmax_scale must be > 0");
    if (p->reserved != 0) return fail(OMNIMEM_EINVAL, "attn params: reserved must be 0");
    if (three) {
        if (p->fuse_mode != OMNIMEM_FUSE_GATED) return fail(OMNIMEM_EINVAL, "the three-branch call is Eq. (1): fuse_mode must be OMNIMEM_FUSE_GATED");
        if (!gate_cmp) return fail(OMNIMEM_EINVAL, "gate_cmp is NULL");
        if (!c->pooled_v) return fail(OMNIMEM_ESTATE, "no pooled-value buffer: call omnimem_cache_attach_pooled_v before appending");
        if (c->dirty_first != c->dirty_end) return fail(OMNIMEM_ESTATE, "blocks [%lld, %lld) were appended but not pooled; call omnimem_pool_keys first",
                                                        (long long)c->dirty_first, (long long)c->dirty_end);
    }
    AttnArgs a;
    a.cache = c;
    a.q = q;
    a.k_cur = k_cur;
    a.v_cur = v_cur;
    a.n_q = n_q;
    a.stride_tok = stride_tok;
    a.stride_head = stride_head;
    a.ptr_table = ptr_table;
    a.p = *p;
    a.gate_slc = gate_slc;
    a.gate_swa = gate_swa;
    a.gate_cmp = three ? gate_cmp : nullptr;
    a.out = out;
    a.lse_out = lse_out;
    a.workspace = workspace;
    a.workspace_bytes = workspace_bytes;
    a.stream = (cudaStream_t)stream;
    return launch_attn_tcgen05(a);  // ONE kernel for every supported shape: TMA + tcgen05 / TMEM
}

int32_t omnimem_sparse_attn(const omnimem_cache_t* cache, const void* q, const void* k_cur, const void* v_cur,
                            int32_t n_q, int64_t stride_tok, int64_t stride_head, const int32_t* ptr_table,
                            const omnimem_attn_params_t* p, const float* gate_slc, const float* gate_swa, void* out,
                            float* lse_out, void* workspace, size_t workspace_bytes, void* stream)
{
    return sparse_attn_impl(cache, q, k_cur, v_cur, n_q, stride_tok, stride_head, ptr_table, p, nullptr, gate_slc, gate_swa, out, lse_out,
                            workspace, workspace_bytes, stream, false);
}

int32_t omnimem_sparse_attn3(const omnimem_cache_t* cache, const void* q, const void* k_cur, const void* v_cur,
                             int32_t n_q, int64_t stride_tok, int64_t stride_head, const int32_t* ptr_table,
                             const omnimem_attn_params_t* p, const float* gate_cmp, const float* gate_slc, const float* gate_swa,
                             void* out, float* lse_out, void* workspace, size_t workspace_bytes, void* stream)
{
    return sparse_attn_impl(cache, q, k_cur, v_cur, n_q, stride_tok, stride_head, ptr_table, p, gate_cmp, gate_slc, gate_swa, out, lse_out,
                            workspace, workspace_bytes, stream, true);
}

}  // extern "C"
