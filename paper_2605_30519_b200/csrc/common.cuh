// Shared host/device helpers of the CUDA path (sm_100a).  No code here is shared with oracle/.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/omnimem.h"

namespace omnimem {

// Host-side cache handle: geometry, caller-owned device buffers, token counter, dirty block range.
struct Cache {
    int32_t H, D, B;
    int32_t P;    // rows per page (>= B; pad rows stay zero)
    int32_t bpc;  // blocks per chunk of the two-level page map, 0 = one map entry per block
    int32_t pool_blocks;      // pages per head of k_pages / v_pages: max_blocks, or resident_chunks * bpc with offloading
    int32_t resident_chunks;  // > 0: only this many chunks per head live in HBM (NEXT-4), the rest in pinned host memory
    struct Offload* off;      // host-side residency manager (offload.cu), nullptr until omnimem_offload_attach
    int64_t max_tokens;
    int32_t max_blocks;
    __nv_bfloat16* k_pages;
    __nv_bfloat16* v_pages;
    __nv_bfloat16* pooled_k;
    __nv_bfloat16* pooled_v;  // nullptr until omnimem_cache_attach_pooled_v (CMP branch)
    int32_t* page_map;
    int64_t n_hist;
    int64_t dirty_first, dirty_end;  // logical blocks [dirty_first, dirty_end) need re-pooling
    // cached TMA descriptors of the page pools (built lazily by the tcgen05 attention path)
    bool tmaps_ready;
    alignas(64) unsigned char tmap_k[128];
    alignas(64) unsigned char tmap_v[128];
    alignas(64) unsigned char tmap_k32[128];  // the same pools, 32-row boxes (page_tokens = 32)
    alignas(64) unsigned char tmap_v32[128];
    bool tmaps_cmp_ready;     // the same for the compressed cache (pooled_k, pooled_v)
    alignas(64) unsigned char tmap_kc[128];
    alignas(64) unsigned char tmap_vc[128];
    // per-call tensors of omnimem_sparse_attn (q, k_cur, v_cur): descriptors are re-encoded only when the call's
    // pointers / strides / length differ from the previous call's
    const void *call_q, *call_k, *call_v;
    int32_t call_n;
    int64_t call_st, call_sh;
    alignas(64) unsigned char tmap_q[128];
    alignas(64) unsigned char tmap_kcur[128];
    alignas(64) unsigned char tmap_kcur128[128];
    alignas(64) unsigned char tmap_vcur[128];
};

int32_t fail(int32_t code, const char* fmt, ...);
int32_t check_launch(const char* what);
void count_launch(int n = 1);

// Programmatic dependent launch (PDL): the kernels of one step are launched back to back with the
// "programmatic stream serialization" attribute; each calls pdl_launch_dependents() at its start (the next kernel's
// CTAs may then be scheduled as soon as resources free up, so its prologue overlaps this kernel's tail) and
// pdl_wait() before it touches anything an earlier kernel of the stream wrote (blocks until that grid has completed
// and its writes are visible).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// the same launch in plain stream order (no programmatic attribute): griddepcontrol.wait inside the kernel is then a no-op
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_plain(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cfg.attrs = nullptr;
    cfg.numAttrs = 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

__host__ __device__ static inline int64_t ceil_div64(int64_t a, int64_t b) { return (a + b - 1) / b; }

// Physical page of logical block b of head h: one map entry per block, or the paper's two-level map (Alg. 1 lines 7-12,
// PAPER.md:366-380): the chunk's base page + the block's offset inside the chunk.
__device__ __forceinline__ int32_t page_of(const int32_t* __restrict__ map, int64_t h, int64_t b, int32_t max_blocks, int32_t bpc)
{
    if (bpc <= 0) return __ldg(map + h * max_blocks + b);
    const int32_t n_chunks = (max_blocks + bpc - 1) / bpc;
    const int32_t base = __ldg(map + h * n_chunks + b / bpc);
    return base < 0 ? -1 : base + (int32_t)(b % bpc);  // base < 0: the chunk is not resident (the paper's Pi[h][c] = 0)
}

// AWE decision (Eq. 2; threshold PAPER.md:319) from host-known scalars.
struct Awe {
    int64_t n_b, win_start, b_w, n_cand;
    int32_t active;
};
Awe awe_decide(const Cache* c, int64_t window_tokens, int32_t top_k, int64_t t_awe);

// launchers (defined in the kernel translation units)
int32_t launch_identity_page_map(const Cache* c, cudaStream_t s);
int32_t launch_append(const Cache* c, const void* k, const void* v, int32_t n_tokens, int64_t stride_tok,
                      int64_t stride_head, cudaStream_t s);
int32_t launch_pool(const Cache* c, const __nv_bfloat16* pages, __nv_bfloat16* pooled, int64_t first_block, int64_t n_blocks,
                    cudaStream_t s);
int32_t launch_union_counts(const Cache* c, const int32_t* block_idx, int32_t R, int32_t K, int64_t n_b, long long* per_head,
                            long long* union_all, int32_t* union_list, unsigned char* marks, cudaStream_t s);
int32_t launch_gather_blocks(const Cache* src, const int32_t* list, int64_t n, const Cache* dst, cudaStream_t s);
struct Offload;
void offload_destroy(Offload* o);
int32_t offload_on_append(Cache* c, int32_t n_tokens, cudaStream_t s);       // before the append kernel: place the new chunk
int32_t offload_after_append(Cache* c, int64_t chunk, cudaStream_t s);        // after it: write the chunk through to the host store
int32_t launch_group_mean(const Cache* c, const void* q, int32_t n_q, int64_t stride_tok, int64_t stride_head,
                          int32_t G, __nv_bfloat16* qbar, cudaStream_t s);
int32_t launch_scores(const Cache* c, const __nv_bfloat16* qbar, int32_t R, int64_t n_b, float scale,
                      float* scores, cudaStream_t s);
int32_t launch_topk(const Cache* c, const float* scores, int32_t R, int64_t n_b, int64_t n_cand, int32_t K,
                    int32_t* block_idx, int32_t* ptr_table, cudaStream_t s);
bool scores_prob_fits(int64_t n_b);
size_t scores_prob_partial_floats(int32_t H, int32_t n_q, int32_t G, int64_t n_b);
int32_t launch_scores_prob(const Cache* c, const void* q, int32_t n_q, int64_t stride_tok, int64_t stride_head, int32_t G, int64_t n_b,
                           float scale, float* scores, float* partial, cudaStream_t s);
bool select_fused_fits(int64_t n_b);
// CTAs of the kernel omnimem_select (logit scores) runs last for this geometry when that is ONE kernel; INT64_MAX when the selection
// takes several kernels, 0 when there is nothing to select
int64_t select_launch_ctas(int32_t H, int32_t n_q, int32_t G, int64_t n_b);
int32_t launch_select_fused(const Cache* c, const void* q, int32_t n_q, int64_t stride_tok, int64_t stride_head, int32_t G, int64_t n_b,
                            int64_t n_cand, int32_t K, float scale, float* scores_out, int32_t* block_idx, int32_t* ptr_table, cudaStream_t s);

struct AttnArgs {
    const Cache* cache;
    const void *q, *k_cur, *v_cur;
    int32_t n_q;
    int64_t stride_tok, stride_head;
    const int32_t* ptr_table;
    omnimem_attn_params_t p;
    const float *gate_slc, *gate_swa;
    const float* gate_cmp;  // non-null: the three-branch call (omnimem_sparse_attn3)
    void* out;
    float* lse_out;
    void* workspace;
    size_t workspace_bytes;
    cudaStream_t stream;
};
int32_t launch_attn_tcgen05(const AttnArgs& a);
size_t attn_tcgen05_workspace_bytes(int32_t H, int32_t n_q, int32_t D, int32_t fuse_mode);

}  // namespace omnimem
