// a0 append_chunk and a1 pool_keys: HBM-bound kernels of the paged cache.
#include "common.cuh"

namespace omnimem {

// ---------------------------------------------------------------------------------------------
__global__ void identity_page_map_kernel(int32_t* __restrict__ page_map, int32_t max_blocks, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) page_map[i] = (int32_t)(i % max_blocks);
}

int32_t launch_identity_page_map(const Cache* c, cudaStream_t s)
{
    int64_t n = (int64_t)c->H * c->max_blocks;
    identity_page_map_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, s>>>(c->page_map, c->max_blocks, n);
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
                    const int32_t* __restrict__ page_map, int32_t B, int32_t max_blocks, int64_t n_hist,
                    int32_t n_tokens, int32_t n_total, int64_t stride_tok16, int64_t stride_head16)
{
    constexpr int PIECES = D / 8;
    const int h = blockIdx.y;
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (int64_t)n_total * PIECES) return;
    const int32_t t = (int32_t)(i / PIECES);
    const int32_t c = (int32_t)(i % PIECES);
    const int64_t pos = n_hist + t;
    const int64_t b = pos / B;
    const int32_t page = __ldg(page_map + (int64_t)h * max_blocks + b);
    const int64_t dst = (((int64_t)h * max_blocks + page) * B + (pos % B)) * PIECES + c;
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
                                                      (uint4*)c->v_pages, c->page_map, c->B, c->max_blocks, c->n_hist,
                                                      n_tokens, n_total, stride_tok / 8, stride_head / 8);
    else
        append_chunk_kernel<64><<<grid, 256, 0, s>>>((const uint4*)k, (const uint4*)v, (uint4*)c->k_pages,
                                                     (uint4*)c->v_pages, c->page_map, c->B, c->max_blocks, c->n_hist,
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
                 __nv_bfloat16* __restrict__ pooled_k, int32_t B, int32_t max_blocks, int64_t n_hist,
                 int64_t first_block, int64_t n_blocks)
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
    const int32_t page = __ldg(page_map + (int64_t)h * max_blocks + b);
    const uint4* src = k_pages + (((int64_t)h * max_blocks + page) * B) * PIECES;
    const int piece = lane % PIECES, row0 = lane / PIECES;

    double acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = 0.0;
    if (len == B) {
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
        pool_keys_kernel<128><<<grid, 128, 0, s>>>((const uint4*)pages, c->page_map, pooled, c->B,
                                                   c->max_blocks, c->n_hist, first_block, n_blocks);
    else
        pool_keys_kernel<64><<<grid, 128, 0, s>>>((const uint4*)pages, c->page_map, pooled, c->B,
                                                  c->max_blocks, c->n_hist, first_block, n_blocks);
    count_launch();
    return check_launch("pool_keys");
}

}  // namespace omnimem
