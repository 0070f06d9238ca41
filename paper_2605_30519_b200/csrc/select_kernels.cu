// a2-a5: Query-Shared KV Selection scores, Adaptive Window Exclusion, top-k, pointer table
// (PAPER.md:83-89 Eq. 2, :107-114 Eq. 3, :358-380).  DESIGN.md section 6.3.
#include "common.cuh"

namespace omnimem {

// ---------------------------------------------------------------------------------------------
// qbar[h][r][:] = mean over the group's valid queries.  One CTA per (group, head); thread t owns
// the 16-byte piece (t % PIECES) of rows (t / PIECES) + j*ROWS; fp64 sums (exact), smem reduction.
template <int D>
__global__ void __launch_bounds__(256)
group_mean_kernel(const uint4* __restrict__ q, int32_t n_q, int64_t stride_tok16, int64_t stride_head16,
                  int32_t G, int32_t R, __nv_bfloat16* __restrict__ qbar)
{
    constexpr int PIECES = D / 8;
    constexpr int ROWS = 256 / PIECES;
    __shared__ double red[ROWS][PIECES][8 + 1];
    const int r = blockIdx.x, h = blockIdx.y;
    const int lo = r * G, hi = min(lo + G, n_q);
    const int piece = threadIdx.x % PIECES, row0 = threadIdx.x / PIECES;
    double acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = 0.0;
    const uint4* base = q + (int64_t)h * stride_head16 + piece;
    for (int s = lo + row0; s < hi; s += ROWS) {
        const uint4 u = __ldg(base + (int64_t)s * stride_tok16);
        const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            acc[2 * i] += (double)__uint_as_float(w[i] << 16);
            acc[2 * i + 1] += (double)__uint_as_float(w[i] & 0xffff0000u);
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) red[row0][piece][i] = acc[i];
    __syncthreads();
    if (threadIdx.x < D) {
        const int p = threadIdx.x / 8, i = threadIdx.x % 8;
        double sum = 0.0;
        for (int rr = 0; rr < ROWS; ++rr) sum += red[rr][p][i];
        const float f = __fdiv_rn((float)sum, (float)(hi - lo));
        qbar[((int64_t)h * R + r) * D + threadIdx.x] = __float2bfloat16_rn(f);
    }
}

int32_t launch_group_mean(const Cache* c, const void* q, int32_t n_q, int64_t stride_tok, int64_t stride_head,
                          int32_t G, __nv_bfloat16* qbar, cudaStream_t s)
{
    const int32_t R = (int32_t)ceil_div64(n_q, G);
    dim3 grid((unsigned)R, (unsigned)c->H);
    if (c->D == 128)
        group_mean_kernel<128><<<grid, 256, 0, s>>>((const uint4*)q, n_q, stride_tok / 8, stride_head / 8, G, R, qbar);
    else
        group_mean_kernel<64><<<grid, 256, 0, s>>>((const uint4*)q, n_q, stride_tok / 8, stride_head / 8, G, R, qbar);
    count_launch();
    return check_launch("group_mean");
}

// ---------------------------------------------------------------------------------------------
// sbar[h][r][b] = scale * <qbar[h][r], pooled_k[h][b]>: per head a (R x D) x (D x N_b) product.
// 64 x 64 output tile per CTA, 256 threads x (4 x 4) outputs, D consumed in slabs of 32 staged in
// padded shared memory (conflict-free: thread (tx,ty) owns rows ty+16i and columns tx+16j).
// fp32 FMA accumulation in a fixed order (d ascending).
template <int D>
__global__ void __launch_bounds__(256)
scores_kernel(const __nv_bfloat16* __restrict__ qbar, const __nv_bfloat16* __restrict__ pooled_k, int32_t R,
              int32_t max_blocks, int64_t n_b, float scale, float* __restrict__ scores)
{
    __shared__ float qs[64][33];
    __shared__ float ks[64][33];
    const int h = blockIdx.z;
    const int r0 = blockIdx.y * 64;
    const int64_t b0 = (int64_t)blockIdx.x * 64;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    float acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

    for (int d0 = 0; d0 < D; d0 += 32) {
        // 64 rows x 32 d per operand = 2048 elements: each thread loads 8 (one 16-byte piece)
        {
            const int row = threadIdx.x >> 2, pc = threadIdx.x & 3;
            uint4 u = make_uint4(0, 0, 0, 0), v = make_uint4(0, 0, 0, 0);
            if (r0 + row < R) u = __ldg((const uint4*)(qbar + ((int64_t)h * R + r0 + row) * D + d0) + pc);
            if (b0 + row < n_b) v = __ldg((const uint4*)(pooled_k + ((int64_t)h * max_blocks + b0 + row) * D + d0) + pc);
            const uint32_t uw[4] = {u.x, u.y, u.z, u.w}, vw[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                qs[row][pc * 8 + 2 * i] = __uint_as_float(uw[i] << 16);
                qs[row][pc * 8 + 2 * i + 1] = __uint_as_float(uw[i] & 0xffff0000u);
                ks[row][pc * 8 + 2 * i] = __uint_as_float(vw[i] << 16);
                ks[row][pc * 8 + 2 * i + 1] = __uint_as_float(vw[i] & 0xffff0000u);
            }
        }
        __syncthreads();
#pragma unroll 8
        for (int d = 0; d < 32; ++d) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = qs[ty + 16 * i][d];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = ks[tx + 16 * j][d];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = r0 + ty + 16 * i;
        if (r >= R) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int64_t b = b0 + tx + 16 * j;
            if (b < n_b) scores[((int64_t)h * R + r) * n_b + b] = scale * acc[i][j] + 0.0f;
        }
    }
}

int32_t launch_scores(const Cache* c, const __nv_bfloat16* qbar, int32_t R, int64_t n_b, float scale,
                      float* scores, cudaStream_t s)
{
    if (n_b <= 0) return OMNIMEM_OK;
    dim3 grid((unsigned)ceil_div64(n_b, 64), (unsigned)ceil_div64(R, 64), (unsigned)c->H);
    if (c->D == 128)
        scores_kernel<128><<<grid, 256, 0, s>>>(qbar, c->pooled_k, R, c->max_blocks, n_b, scale, scores);
    else
        scores_kernel<64><<<grid, 256, 0, s>>>(qbar, c->pooled_k, R, c->max_blocks, n_b, scale, scores);
    count_launch();
    return check_launch("scores");
}

// ---------------------------------------------------------------------------------------------
// Warp-level top-k with a fixed tie-break.  A candidate is the 64-bit key
//     (order-preserving bits of the fp32 score) << 32 | (0xFFFFFFFF - block index)
// so that "greater key" == (score descending, block index ascending); 0 is the empty key.
// A warp keeps its current best 64 keys sorted in two registers per lane (position p lives in
// register p/32 of lane p%32) and streams candidates 32 at a time: a ballot finds those that beat
// the current K-th key, each is inserted with two shuffles.  Eight warps scan disjoint slices of
// the row; warp 0 then merges the eight sorted lists and writes block ids and table entries.
__device__ __forceinline__ unsigned long long make_key(float s, uint32_t b)
{
    s += 0.0f;  // -0 -> +0
    uint32_t u = __float_as_uint(s);
    u = (u & 0x80000000u) ? ~u : (u | 0x80000000u);
    return ((unsigned long long)u << 32) | (unsigned long long)(0xFFFFFFFFu - b);
}

struct WarpTopK {
    unsigned long long k0, k1;  // positions lane and lane+32
    unsigned long long thr;     // key at position K-1
    int K, lane;

    __device__ __forceinline__ void init(int K_, int lane_)
    {
        k0 = k1 = thr = 0ull;
        K = K_;
        lane = lane_;
    }
    __device__ __forceinline__ void insert(unsigned long long c)
    {
        const int p = __popc(__ballot_sync(0xffffffffu, k0 > c)) + __popc(__ballot_sync(0xffffffffu, k1 > c));
        unsigned long long up0 = __shfl_up_sync(0xffffffffu, k0, 1);
        unsigned long long up1 = __shfl_up_sync(0xffffffffu, k1, 1);
        const unsigned long long last0 = __shfl_sync(0xffffffffu, k0, 31);
        if (lane == 0) up1 = last0;
        const int i0 = lane, i1 = lane + 32;
        k0 = (i0 < p) ? k0 : (i0 == p ? c : up0);
        k1 = (i1 < p) ? k1 : (i1 == p ? c : up1);
        const unsigned long long src = (K - 1 < 32) ? k0 : k1;
        thr = __shfl_sync(0xffffffffu, src, (K - 1) & 31);
    }
    // offer one candidate per lane (0 = none)
    __device__ __forceinline__ void offer(unsigned long long key)
    {
        unsigned mask = __ballot_sync(0xffffffffu, key > thr);
        while (mask) {
            const int src = __ffs(mask) - 1;
            mask &= mask - 1;
            const unsigned long long c = __shfl_sync(0xffffffffu, key, src);
            if (c > thr) insert(c);  // warp-uniform: c and thr are uniform
        }
    }
};

constexpr int TOPK_WARPS = 8;

__global__ void __launch_bounds__(TOPK_WARPS * 32)
topk_kernel(const float* __restrict__ scores, const int32_t* __restrict__ page_map, int32_t R, int64_t n_b,
            int64_t n_cand, int32_t K, int32_t max_blocks, int32_t* __restrict__ block_idx,
            int32_t* __restrict__ ptr_table)
{
    __shared__ unsigned long long lists[TOPK_WARPS][64];
    const int r = blockIdx.x, h = blockIdx.y;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const float* row = scores + ((int64_t)h * R + r) * n_b;

    WarpTopK tk;
    tk.init(K, lane);
    // slice of this warp, in multiples of 32 candidates
    const int64_t per = ceil_div64(ceil_div64(n_cand, TOPK_WARPS), 32) * 32;
    const int64_t lo = (int64_t)warp * per;
    const int64_t hi = (lo + per < n_cand) ? lo + per : n_cand;
    for (int64_t base = lo; base < hi; base += 128) {
        float sv[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int64_t b = base + j * 32 + lane;
            sv[j] = (b < hi) ? __ldg(row + b) : 0.f;
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int64_t b = base + j * 32 + lane;
            tk.offer((b < hi) ? make_key(sv[j], (uint32_t)b) : 0ull);
        }
    }
    lists[warp][lane] = tk.k0;
    lists[warp][lane + 32] = tk.k1;
    __syncthreads();
    if (warp != 0) return;
    for (int w = 1; w < TOPK_WARPS; ++w) {
        tk.offer(lists[w][lane]);
        if (K > 32) tk.offer(lists[w][lane + 32]);
    }
    // positions [0, K) hold the selection in (score desc, index asc) order; empty keys -> -1
    for (int half = 0; half < 2; ++half) {
        const int t = lane + 32 * half;
        if (t >= K) break;
        const unsigned long long key = half ? tk.k1 : tk.k0;
        const int32_t b = key ? (int32_t)(0xFFFFFFFFu - (uint32_t)key) : -1;
        const int64_t o = ((int64_t)h * R + r) * K + t;
        if (block_idx) block_idx[o] = b;
        ptr_table[o] = (b < 0) ? -1 : __ldg(page_map + (int64_t)h * max_blocks + b);
    }
}

int32_t launch_topk(const Cache* c, const float* scores, int32_t R, int64_t n_b, int64_t n_cand, int32_t K,
                    int32_t* block_idx, int32_t* ptr_table, cudaStream_t s)
{
    dim3 grid((unsigned)R, (unsigned)c->H);
    topk_kernel<<<grid, TOPK_WARPS * 32, 0, s>>>(scores, c->page_map, R, n_b, n_cand, K, c->max_blocks, block_idx,
                                                 ptr_table);
    count_launch();
    return check_launch("topk");
}

}  // namespace omnimem
