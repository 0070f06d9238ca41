// a0 append_chunk and a1 pool_keys: HBM-bound kernels of the paged cache.
#include <mutex>

#include "common.cuh"

namespace omnimem {

// ---------------------------------------------------------------------------------------------
__global__ void identity_page_map_kernel(int32_t* __restrict__ page_map, int32_t per_head, int32_t step, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) page_map[i] = (int32_t)(i % per_head) * step;  // two-level map: chunk c starts at page c * B_pc
}

int32_t launch_identity_page_map(const Cache* c, cudaStream_t s)
{
    const int32_t per_head = c->bpc > 0 ? (int32_t)ceil_div64(c->max_blocks, c->bpc) : c->max_blocks;
    int64_t n = (int64_t)c->H * per_head;
    if (c->resident_chunks > 0) {  // offloading: nothing is resident until a chunk is appended (entry -1 = not in HBM)
        cudaError_t e = cudaMemsetAsync(c->page_map, 0xff, (size_t)n * 4, s);
        return e == cudaSuccess ? OMNIMEM_OK : fail(OMNIMEM_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
    }
    identity_page_map_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, s>>>(c->page_map, per_head, c->bpc > 0 ? c->bpc : 1, n);
    count_launch();
    return check_launch("identity_page_map");
}

// ---------------------------------------------------------------------------------------------
// a0: one thread moves one 16-byte piece (8 bf16) of K and of V.  Token index t runs over the
// chunk [0, n_tokens) and then over the zero-filled tail of the last page touched.  Consecutive
// threads touch consecutive 16-byte pieces of a row, so both the loads and the stores are fully
// coalesced 128-bit accesses; the only indirection is one page_map read per row (L1/L2 hit).
template <int D>
__global__ void __launch_bounds__(256)
append_chunk_kernel(const uint4* __restrict__ k_src, const uint4* __restrict__ v_src,
                    uint4* __restrict__ k_pages, uint4* __restrict__ v_pages,
                    const int32_t* __restrict__ page_map, int32_t B, int32_t P, int32_t bpc, int32_t max_blocks, int32_t pool_blocks,
                    int64_t n_hist, int32_t n_tokens, int32_t n_total, int64_t stride_tok16, int64_t stride_head16)
{
    constexpr int PIECES = D / 8;
    const int h = blockIdx.y;
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)n_total * PIECES) return;
    const int32_t t = (int32_t)(i / PIECES);
    const int32_t c = (int32_t)(i % PIECES);
    const int64_t pos = n_hist + t;
    const int64_t b = pos / B;
    const int32_t page = page_of(page_map, h, b, max_blocks, bpc);
    const int64_t dst = (((int64_t)h * pool_blocks + page) * P + (pos % B)) * PIECES + c;
    uint4 kv = make_uint4(0, 0, 0, 0), vv = make_uint4(0, 0, 0, 0);
    if (t < n_tokens) {
        const int64_t src = (int64_t)h * stride_head16 + (int64_t)t * stride_tok16 + c;
        kv = __ldg(k_src + src);
        vv = __ldg(v_src + src);
    }
    k_pages[dst] = kv;
    v_pages[dst] = vv;
}

int32_t launch_append(const Cache* c, const void* k, const void* v, int32_t n_tokens, int64_t stride_tok,
                      int64_t stride_head, cudaStream_t s)
{
    const int64_t new_hist = c->n_hist + n_tokens;
    const int32_t tail = (int32_t)((c->B - new_hist % c->B) % c->B);
    const int32_t n_total = n_tokens + tail;
    const int pieces = c->D / 8;
    dim3 grid((unsigned)ceil_div64((int64_t)n_total * pieces, 256), (unsigned)c->H);
    if (c->D == 128)
        append_chunk_kernel<128><<<grid, 256, 0, s>>>((const uint4*)k, (const uint4*)v, (uint4*)c->k_pages,
                                                      (uint4*)c->v_pages, c->page_map, c->B, c->P, c->bpc, c->max_blocks, c->pool_blocks, c->n_hist,
                                                      n_tokens, n_total, stride_tok / 8, stride_head / 8);
    else
        append_chunk_kernel<64><<<grid, 256, 0, s>>>((const uint4*)k, (const uint4*)v, (uint4*)c->k_pages,
                                                     (uint4*)c->v_pages, c->page_map, c->B, c->P, c->bpc, c->max_blocks, c->pool_blocks, c->n_hist,
                                                     n_tokens, n_total, stride_tok / 8, stride_head / 8);
    count_launch();
    return check_launch("append_chunk");
}

// ---------------------------------------------------------------------------------------------
// a1: one warp per (head, block).  A block is one contiguous page of B rows x D bf16 (16 KB at
// B=64, D=128).  Lane l owns the 16-byte piece (l % PIECES) of rows (l / PIECES) + j*ROWS, so a warp
// load instruction reads 512 contiguous bytes.  Sums are carried in fp64 so that they are exact
// (order-independent) and the result matches the oracle's definition bit for bit; the pipe that
// matters is still HBM.  Warp-shuffle reduction across the row groups.
__device__ __forceinline__ void add_piece(double (&acc)[8], const uint4& u)
{
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        acc[2 * i] += (double)__uint_as_float(w[i] << 16);
        acc[2 * i + 1] += (double)__uint_as_float(w[i] & 0xffff0000u);
    }
}

template <int D>
__global__ void __launch_bounds__(128)
pool_keys_kernel(const uint4* __restrict__ k_pages, const int32_t* __restrict__ page_map,
                 __nv_bfloat16* __restrict__ pooled_k, int32_t B, int32_t P, int32_t bpc, int32_t max_blocks, int32_t pool_blocks,
                 int64_t n_hist, int64_t first_block, int64_t n_blocks)
{
    constexpr int PIECES = D / 8;       // 16-byte pieces per row
    constexpr int ROWS = 32 / PIECES;   // rows per warp load
    const int lane = threadIdx.x & 31;
    const int64_t wb = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (wb >= n_blocks) return;
    const int h = blockIdx.y;
    const int64_t b = first_block + wb;
    int64_t len64 = n_hist - b * B;
    const int len = (int)(len64 < B ? len64 : B);
    const int32_t page = page_of(page_map, h, b, max_blocks, bpc);
    const uint4* src = k_pages + (((int64_t)h * pool_blocks + page) * P) * PIECES;
    const int piece = lane % PIECES, row0 = lane / PIECES;

    double acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = 0.0;
    if (len == B && B % (8 * ROWS) == 0) {
        // full block: B/ROWS independent 128-bit loads per lane, issued 8 at a time
        for (int j0 = 0; j0 < B / ROWS; j0 += 8) {
            uint4 u[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) u[j] = __ldg(src + (int64_t)(row0 + (j0 + j) * ROWS) * PIECES + piece);
#pragma unroll
            for (int j = 0; j < 8; ++j) add_piece(acc, u[j]);
        }
    } else {
        for (int r = row0; r < len; r += ROWS) add_piece(acc, __ldg(src + (int64_t)r * PIECES + piece));
    }
#pragma unroll
    for (int off = 16; off >= PIECES; off >>= 1)
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], off);
    if (lane < PIECES) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            float lo = __fdiv_rn((float)acc[2 * i], (float)len);
            float hi = __fdiv_rn((float)acc[2 * i + 1], (float)len);
            w[i] = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(lo)) |
                   ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(hi)) << 16);
        }
        uint4* dst = (uint4*)(pooled_k + ((int64_t)h * max_blocks + b) * D) + piece;
        *dst = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

int32_t launch_pool(const Cache* c, const __nv_bfloat16* pages, __nv_bfloat16* pooled, int64_t first_block, int64_t n_blocks,
                    cudaStream_t s)
{
    if (n_blocks <= 0) return OMNIMEM_OK;
    dim3 grid((unsigned)ceil_div64(n_blocks, 4), (unsigned)c->H);
    if (c->D == 128)
        pool_keys_kernel<128><<<grid, 128, 0, s>>>((const uint4*)pages, c->page_map, pooled, c->B, c->P, c->bpc,
                                                   c->max_blocks, c->pool_blocks, c->n_hist, first_block, n_blocks);
    else
        pool_keys_kernel<64><<<grid, 128, 0, s>>>((const uint4*)pages, c->page_map, pooled, c->B, c->P, c->bpc,
                                                  c->max_blocks, c->pool_blocks, c->n_hist, first_block, n_blocks);
    count_launch();
    return check_launch("pool_keys");
}

// ---------------------------------------------------------------------------------------------
// Union accounting of a selection (Eqs. 4-5): U_h = union over the head's groups of its selected
// blocks, per_head[h] = |U_h|, union_all = |union over heads of U_h|; union_list = the blocks of that union in
// ascending order.  marks: [H + 1][n_b] bytes of scratch (row H is the union over heads).
__global__ void __launch_bounds__(256)
union_mark_kernel(const int32_t* __restrict__ block_idx, int64_t per_head_entries, int64_t n_entries, int64_t n_b, int32_t H,
                  unsigned char* __restrict__ marks)
{
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n_entries) return;
    const int32_t b = block_idx[i];
    if (b < 0 || b >= n_b) return;  // masked slot
    const int64_t h = i / per_head_entries;
    marks[h * n_b + b] = 1;        // every writer stores the same value
    marks[(int64_t)H * n_b + b] = 1;
}
// one CTA per row of marks (H heads + the union row): count, and for the union row the ordered list
__global__ void __launch_bounds__(1024)
union_count_kernel(const unsigned char* __restrict__ marks, int64_t n_b, int32_t H, long long* __restrict__ per_head,
                   long long* __restrict__ union_all, int32_t* __restrict__ union_list)
{
    __shared__ int warp_tot[32];
    __shared__ long long base_s;
    const int row = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned char* m = marks + (int64_t)row * n_b;
    if (tid == 0) base_s = 0;
    __syncthreads();
    for (int64_t b0 = 0; b0 < n_b; b0 += 1024) {  // ordered scan, 1024 blocks per trip
        const int64_t b = b0 + tid;
        const int v = (b < n_b && m[b]) ? 1 : 0;
        const unsigned bal = __ballot_sync(0xffffffffu, v);
        if (lane == 0) warp_tot[warp] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
        for (int w = 0; w < 32; ++w) { const int t = warp_tot[w]; if (w < warp) before += t; total += t; }
        const long long base = base_s;
        if (v && row == H && union_list) union_list[base + before + __popc(bal & ((1u << lane) - 1u))] = (int32_t)b;
        __syncthreads();
        if (tid == 0) base_s = base + total;
        __syncthreads();
    }
    if (tid == 0) {
        if (row < H) per_head[row] = base_s;
        else *union_all = base_s;
    }
}

int32_t launch_union_counts(const Cache* c, const int32_t* block_idx, int32_t R, int32_t K, int64_t n_b, long long* per_head,
                            long long* union_all, int32_t* union_list, unsigned char* marks, cudaStream_t s)
{
    const int64_t n_entries = (int64_t)c->H * R * K;
    cudaError_t e = cudaMemsetAsync(marks, 0, (size_t)(c->H + 1) * (size_t)(n_b > 0 ? n_b : 1), s);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
    if (n_entries > 0 && n_b > 0) {
        union_mark_kernel<<<(unsigned)ceil_div64(n_entries, 256), 256, 0, s>>>(block_idx, (int64_t)R * K, n_entries, n_b, c->H, marks);
        count_launch();
    }
    union_count_kernel<<<(unsigned)(c->H + 1), 1024, 0, s>>>(marks, n_b, c->H, per_head, union_all, union_list);
    count_launch();
    return check_launch("union_counts");
}

// ---------------------------------------------------------------------------------------------
// omnimem_union_counts_noalloc: the same two kernels, marks in a file-scope device array instead of caller scratch, for
// callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Every GPU that loads
// the library holds the array (OMNIMEM_UNION_NOALLOC_MAX_BYTES) until exit.  In HOST code `g_union_marks` is only a
// stand-in for the symbol, not a device address: the kernels get the pointer cudaGetSymbolAddress returns, looked up once
// per device with that device current.
static __device__ __align__(256) unsigned char g_union_marks[OMNIMEM_UNION_NOALLOC_MAX_BYTES];

static int32_t union_marks_device_ptr(unsigned char** out)
{
    constexpr int MAX_DEV = 64;
    static unsigned char* ptr_of[MAX_DEV];  // zero-initialised; one slot per device ordinal
    static std::mutex mu;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEV) return fail(OMNIMEM_EUNSUPPORTED, "device ordinal %d outside the %d the no-alloc path tracks", dev, MAX_DEV);
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of[dev]) {
        unsigned char* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_union_marks);  // the CURRENT device's copy of the array
        if (e != cudaSuccess || !p) return fail(OMNIMEM_ECUDA, "cudaGetSymbolAddress(g_union_marks): %s", cudaGetErrorString(e));
        ptr_of[dev] = p;
    }
    *out = ptr_of[dev];
    return OMNIMEM_OK;
}

// ---------------------------------------------------------------------------------------------
// The merged selected-KV buffer of the Naive-Sparse baseline: block list[i] of EVERY head of
// `src` becomes block i of `dst`.  One CTA row per (list entry, head); 16-byte pieces, coalesced.
__global__ void __launch_bounds__(256)
gather_blocks_kernel(const uint4* __restrict__ k_src, const uint4* __restrict__ v_src, const int32_t* __restrict__ map_src, int32_t mb_src,
                     int32_t bpc_src, int32_t pool_src, uint4* __restrict__ k_dst, uint4* __restrict__ v_dst, const int32_t* __restrict__ map_dst,
                     int32_t mb_dst, int32_t bpc_dst, int32_t pool_dst, const int32_t* __restrict__ list, int32_t page_pieces)
{
    const int i = blockIdx.x, h = blockIdx.y;
    const int32_t b = __ldg(list + i);
    const int64_t ps = (int64_t)h * pool_src + page_of(map_src, h, b, mb_src, bpc_src);
    const int64_t pd = (int64_t)h * pool_dst + page_of(map_dst, h, i, mb_dst, bpc_dst);
    for (int p = threadIdx.x; p < page_pieces; p += 256) {
        k_dst[pd * page_pieces + p] = __ldg(k_src + ps * page_pieces + p);
        v_dst[pd * page_pieces + p] = __ldg(v_src + ps * page_pieces + p);
    }
}

int32_t launch_gather_blocks(const Cache* src, const int32_t* list, int64_t n, const Cache* dst, cudaStream_t s)
{
    if (n <= 0) return OMNIMEM_OK;
    const int32_t pieces = src->P * src->D / 8;
    gather_blocks_kernel<<<dim3((unsigned)n, (unsigned)src->H), 256, 0, s>>>((const uint4*)src->k_pages, (const uint4*)src->v_pages, src->page_map,
                                                                           src->max_blocks, src->bpc, src->pool_blocks, (uint4*)dst->k_pages, (uint4*)dst->v_pages,
                                                                           dst->page_map, dst->max_blocks, dst->bpc, dst->pool_blocks, list, pieces);
    count_launch();
    return check_launch("gather_blocks");
}

}  // namespace omnimem

// The no-allocation entry point lives in this file, next to its device array: the symbol lookup, the clear and both launches
// use the pointer resolved above (include/omnimem.h states the contract).
extern "C" int32_t omnimem_union_counts_noalloc(const omnimem_cache_t* cache, const int32_t* block_idx, int32_t n_groups, int32_t top_k,
                                                int64_t* per_head, int64_t* union_all, int32_t* union_list, void* stream)
{
    using namespace omnimem;
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    const Cache* c = reinterpret_cast<const Cache*>(cache);
    if (!block_idx || !per_head || !union_all) return fail(OMNIMEM_EINVAL, "NULL argument");
    if (n_groups < 1 || top_k < 1) return fail(OMNIMEM_EINVAL, "n_groups and top_k must be >= 1");
    const int64_t n_b = ceil_div64(c->n_hist, c->B);
    const size_t need = (size_t)(c->H + 1) * (size_t)(n_b > 0 ? n_b : 1);
    if (need > (size_t)OMNIMEM_UNION_NOALLOC_MAX_BYTES)
        return fail(OMNIMEM_ECAPACITY, "union_counts_noalloc: (H + 1) * N_b = %zu bytes of marks exceed the built-in %zu; use omnimem_union_counts with caller scratch",
                    need, (size_t)OMNIMEM_UNION_NOALLOC_MAX_BYTES);
    unsigned char* marks = nullptr;
    if (int32_t rc = union_marks_device_ptr(&marks)) return rc;
    // launch_union_counts clears the (H + 1) * N_b bytes it uses first (the array keeps the previous call's marks)
    return launch_union_counts(c, block_idx, n_groups, top_k, n_b, (long long*)per_head, (long long*)union_all, union_list, marks,
                               (cudaStream_t)stream);
}
