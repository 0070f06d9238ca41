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
    pdl_launch_dependents();
    pdl_wait();
    double acc[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i] = 0.0;
    const uint4* base = q + (int64_t)h * stride_head16 + piece;
    // four rows per trip: the loads of a trip are in flight together (G = 64, D = 128: one trip per thread)
    for (int s0 = lo + row0; s0 < hi; s0 += 4 * ROWS) {
        uint4 u[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int s = s0 + j * ROWS;
            u[j] = s < hi ? __ldg(base + (int64_t)s * stride_tok16) : make_uint4(0, 0, 0, 0);  // +0.0 terms change nothing
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t w[4] = {u[j].x, u[j].y, u[j].z, u[j].w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                acc[2 * i] += (double)__uint_as_float(w[i] << 16);
                acc[2 * i + 1] += (double)__uint_as_float(w[i] & 0xffff0000u);
            }
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
        launch_pdl(group_mean_kernel<128>, grid, dim3(256), 0, s, (const uint4*)q, n_q, stride_tok / 8, stride_head / 8, G, R, qbar);
    else
        launch_pdl(group_mean_kernel<64>, grid, dim3(256), 0, s, (const uint4*)q, n_q, stride_tok / 8, stride_head / 8, G, R, qbar);
    count_launch();
    return check_launch("group_mean");
}

// ---------------------------------------------------------------------------------------------
// sbar[h][r][b] = scale * <qbar[h][r], pooled_k[h][b]>: per head a (R x D) x (D x N_b) product on the
// tensor cores (warp-level mma.sync m16n8k16, bf16 x bf16 -> fp32: the contraction is 0.1 % of the
// step's FLOPs, so a TMEM pipeline would buy nothing; what matters is that pooled_k is read once).
// CTA tile = 32 groups x 128 blocks, 4 warps of 16 x 64; operands staged with cp.async into
// XOR-swizzled shared memory and read with ldmatrix.
__device__ __forceinline__ uint32_t sel_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sel_cp16(uint32_t dst, const void* src, bool ok)
{
    const int sz = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(sz));
}
__device__ __forceinline__ void sel_ldsm4(uint32_t (&r)[4], uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void sel_mma(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

template <int D>
__global__ void __launch_bounds__(128)
scores_kernel(const __nv_bfloat16* __restrict__ qbar, const __nv_bfloat16* __restrict__ pooled_k, int32_t R,
              int32_t max_blocks, int64_t n_b, float scale, float* __restrict__ scores)
{
    constexpr int CH = D / 8;  // 16-byte chunks per row
    __shared__ __align__(128) unsigned char sq[32 * D * 2];
    __shared__ __align__(128) unsigned char sk[128 * D * 2];
    const int h = blockIdx.z, r0 = blockIdx.y * 32;
    const int64_t b0 = (int64_t)blockIdx.x * 128;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    auto off = [](int row, int ch) { return (uint32_t)(row * (D * 2) + ((ch ^ (row & 7)) << 4)); };
    const uint32_t sq_a = sel_smem_u32(sq), sk_a = sel_smem_u32(sk);
    pdl_launch_dependents();
    pdl_wait();  // qbar comes from group_mean_kernel
    for (int i = tid; i < 32 * CH; i += 128) {
        const int row = i / CH, ch = i % CH;
        const bool ok = r0 + row < R;
        sel_cp16(sq_a + off(row, ch), ok ? (const void*)(qbar + ((int64_t)h * R + r0 + row) * D + ch * 8) : (const void*)qbar, ok);
    }
    for (int i = tid; i < 128 * CH; i += 128) {
        const int row = i / CH, ch = i % CH;
        const bool ok = b0 + row < n_b;
        sel_cp16(sk_a + off(row, ch), ok ? (const void*)(pooled_k + ((int64_t)h * max_blocks + b0 + row) * D + ch * 8) : (const void*)pooled_k, ok);
    }
    asm volatile("cp.async.commit_group;\n" ::);
    asm volatile("cp.async.wait_group 0;\n" ::);
    __syncthreads();
    const int wr = (warp >> 1) * 16, wc = (warp & 1) * 64;  // warp tile origin
    float acc[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.f;
#pragma unroll
    for (int ks = 0; ks < D / 16; ++ks) {
        uint32_t af[4];
        sel_ldsm4(af, sq_a + off(wr + (lane & 7) + ((lane >> 3) & 1) * 8, ks * 2 + (lane >> 4)));
#pragma unroll
        for (int nb2 = 0; nb2 < 4; ++nb2) {
            uint32_t bf[4];
            sel_ldsm4(bf, sk_a + off(wc + (nb2 * 2 + (lane >> 4)) * 8 + (lane & 7), ks * 2 + ((lane >> 3) & 1)));
            sel_mma(acc[nb2 * 2], af, bf[0], bf[1]);
            sel_mma(acc[nb2 * 2 + 1], af, bf[2], bf[3]);
        }
    }
    const int gq = lane >> 2, tq = lane & 3;
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const int r = r0 + wr + gq + e * 8;
        if (r >= R) continue;
        float* dst = scores + ((int64_t)h * R + r) * n_b;
#pragma unroll
        for (int nb = 0; nb < 8; ++nb) {
            const int64_t b = b0 + wc + nb * 8 + 2 * tq;
            if (b < n_b) dst[b] = scale * acc[nb][2 * e] + 0.0f;
            if (b + 1 < n_b) dst[b + 1] = scale * acc[nb][2 * e + 1] + 0.0f;
        }
    }
}

int32_t launch_scores(const Cache* c, const __nv_bfloat16* qbar, int32_t R, int64_t n_b, float scale,
                      float* scores, cudaStream_t s)
{
    if (n_b <= 0) return OMNIMEM_OK;
    dim3 grid((unsigned)ceil_div64(n_b, 128), (unsigned)ceil_div64(R, 32), (unsigned)c->H);
    if (c->D == 128)
        launch_pdl(scores_kernel<128>, grid, dim3(128), 0, s, qbar, (const __nv_bfloat16*)c->pooled_k, R, c->max_blocks, n_b, scale, scores);
    else
        launch_pdl(scores_kernel<64>, grid, dim3(128), 0, s, qbar, (const __nv_bfloat16*)c->pooled_k, R, c->max_blocks, n_b, scale, scores);
    count_launch();
    return check_launch("scores");
}

// ---------------------------------------------------------------------------------------------
// Top-k with a fixed tie-break (a4) + pointer table (a5).  One CTA per (head, group).
// A candidate's order is the 64-bit key  (order-preserving bits of the fp32 score) << 32 | ~block,
// so "greater key" == (score descending, block index ascending).
//  1. the row's score keys are staged in shared memory (-0 canonicalised to +0);
//  2. a most-significant-byte-first radix select (shared-memory histograms, warp-shuffle suffix scan) narrows
//     the key of the K-th best score one byte per pass; as soon as everything at or above the threshold bin fits
//     the 64-entry sorter (typically after two passes) the remaining passes are skipped, otherwise all four passes
//     give the exact 32-bit key T and how many candidates equal to T are needed (ties go to the lowest block
//     index: an ordered block scan ranks the equal candidates);
//  3. the <= 64 survivors are sorted by their 64-bit key with a warp-level bitonic network and written
//     in (score desc, index asc) order; slots beyond |Omega| are -1.
__device__ __forceinline__ uint32_t score_key(float s)
{
    s += 0.0f;  // -0 -> +0
    const uint32_t u = __float_as_uint(s);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

constexpr int TOPK_THREADS = 256;

__global__ void __launch_bounds__(TOPK_THREADS)
topk_kernel(const float* __restrict__ scores, const int32_t* __restrict__ page_map, int32_t R, int64_t n_b,
            int32_t n_cand, int32_t K, int32_t max_blocks, int32_t keys_in_smem, int32_t* __restrict__ block_idx,
            int32_t* __restrict__ ptr_table)
{
    extern __shared__ uint32_t skeys[];  // [n_cand] when keys_in_smem
    __shared__ uint32_t hist[256];
    __shared__ uint32_t s_prefix, s_want, s_super;
    __shared__ uint32_t scan_buf[TOPK_THREADS / 32];
    __shared__ unsigned long long sel[64];
    __shared__ uint32_t n_sel;
    const int r = blockIdx.x, h = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float* row = scores + ((int64_t)h * R + r) * n_b;
    const int64_t out0 = ((int64_t)h * R + r) * K;
    auto key_at = [&](int b) -> uint32_t { return keys_in_smem ? skeys[b] : score_key(__ldg(row + b)); };

    if (tid < 64) sel[tid] = 0ull;
    if (tid == 0) { n_sel = 0; s_prefix = 0; s_want = (uint32_t)K; s_super = 0xffffffffu; }
    int t_shift = 0;
    pdl_launch_dependents();
    pdl_wait();  // the scores come from scores_kernel (or from the caller's previous kernel)
    if (keys_in_smem)
        for (int b = tid; b < n_cand; b += TOPK_THREADS) skeys[b] = score_key(__ldg(row + b));
    __syncthreads();

    if (n_cand > K) {
        for (int pass = 3; pass >= 0; --pass) {
            hist[tid] = 0;
            __syncthreads();
            const uint32_t prefix = s_prefix;
            const int sh = 8 * pass;
            for (int b = tid; b < n_cand; b += TOPK_THREADS) {
                const uint32_t k = key_at(b);
                if (pass == 3 || (k >> (sh + 8)) == prefix) atomicAdd(&hist[(k >> sh) & 255u], 1u);
            }
            __syncthreads();
            if (warp == 0) {
                // suffix sums over the 256 bins, 8 bins per lane (lane 31 owns the top bins)
                uint32_t c[8], tot = 0;
#pragma unroll
                for (int i = 0; i < 8; ++i) { c[i] = hist[lane * 8 + i]; tot += c[i]; }
                uint32_t above = tot;  // inclusive suffix over lanes
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t v = __shfl_down_sync(0xffffffffu, above, o);
                    if (lane + o < 32) above += v;
                }
                above -= tot;  // candidates in bins strictly above this lane's bins
                const uint32_t want = s_want;
                if (above < want && above + tot >= want) {  // the K-th best lies in this lane's bins
                    uint32_t acc = above;
                    int d = 7;
                    for (; d >= 0; --d) {
                        if (acc + c[d] >= want) break;
                        acc += c[d];
                    }
                    s_prefix = (prefix << 8) | (uint32_t)(lane * 8 + d);
                    s_want = want - acc;
                    // candidates at or above the threshold bin: K - (want - acc) strictly above + c[d] inside it
                    s_super = (uint32_t)K - (want - acc) + c[d];
                }
            }
            __syncthreads();
            // early exit: once everything at or above the threshold bin fits the 64-entry sorter, the sorter's
            // 64-bit key (score, then lowest index) settles the rest exactly; remaining digits are not needed
            if (s_super <= 64u && pass > 0) {
                t_shift = 8 * pass;
                break;
            }
        }
    }
    // T: key (or key prefix, shifted down by t_shift) of the K-th best score; a candidate is taken when its key
    // (prefix) is greater than T, or equal to T and among the first want_eq such candidates in index order.  After
    // an early exit every candidate equal to T is taken (want_eq unbounded): at most 64 candidates qualify.
    const uint32_t T = s_prefix;
    const uint32_t want_eq = (n_cand > K && t_shift == 0) ? s_want : 0xffffffffu;
    // ordered pass: thread t owns the contiguous candidates [t*per, (t+1)*per)
    const int per = (n_cand + TOPK_THREADS - 1) / TOPK_THREADS;
    const int lo = tid * per, hi = min(lo + per, (int)n_cand);
    uint32_t n_eq = 0;
    if (n_cand > K && t_shift == 0)
        for (int b = lo; b < hi; ++b) n_eq += (key_at(b) == T);
    // exclusive block scan of n_eq
    uint32_t incl = n_eq;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) scan_buf[warp] = incl;
    __syncthreads();
    uint32_t base = 0;
    for (int wv = 0; wv < warp; ++wv) base += scan_buf[wv];
    uint32_t rank = base + incl - n_eq;
    for (int b = lo; b < hi; ++b) {
        const uint32_t k = key_at(b);
        const uint32_t kp = k >> t_shift;
        bool take;
        if (n_cand <= K) take = true;
        else if (kp > T) take = true;
        else if (kp == T) take = (rank++ < want_eq);
        else take = false;
        if (take) {
            const uint32_t slot = atomicAdd(&n_sel, 1u);
            if (slot < 64) sel[slot] = ((unsigned long long)k << 32) | (unsigned long long)(0xFFFFFFFFu - (uint32_t)b);
        }
    }
    __syncthreads();
    if (warp != 0) return;
    // bitonic sort of 64 keys, descending, two per lane (element i = lane + 32*j)
    unsigned long long v0 = sel[lane], v1 = sel[lane + 32];
    for (int size = 2; size <= 64; size <<= 1) {
        for (int stride = size >> 1; stride >= 1; stride >>= 1) {
            if (stride == 32) {
                // partner of element lane is lane+32 (same lane); direction: descending for the final merge
                const bool desc = true;
                const unsigned long long a = v0, b2 = v1;
                const bool sw = desc ? (a < b2) : (a > b2);
                v0 = sw ? b2 : a;
                v1 = sw ? a : b2;
            } else {
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    unsigned long long& v = j ? v1 : v0;
                    const int i = lane + 32 * j;
                    const unsigned long long o = __shfl_xor_sync(0xffffffffu, v, stride);
                    const bool desc = ((i & size) == 0) || size == 64;
                    const bool lower = (i & stride) == 0;  // the element that should hold the "first" of the pair
                    const bool keep_max = desc ? lower : !lower;
                    v = keep_max ? (v > o ? v : o) : (v < o ? v : o);
                }
            }
        }
    }
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const int t = lane + 32 * j;
        if (t >= K) continue;
        const unsigned long long key = j ? v1 : v0;
        const int32_t b = key ? (int32_t)(0xFFFFFFFFu - (uint32_t)key) : -1;
        if (block_idx) block_idx[out0 + t] = b;
        ptr_table[out0 + t] = (b < 0) ? -1 : __ldg(page_map + (int64_t)h * max_blocks + b);
    }
}

int32_t launch_topk(const Cache* c, const float* scores, int32_t R, int64_t n_b, int64_t n_cand, int32_t K,
                    int32_t* block_idx, int32_t* ptr_table, cudaStream_t s)
{
    dim3 grid((unsigned)R, (unsigned)c->H);
    const size_t key_bytes = (size_t)n_cand * 4;
    const int in_smem = key_bytes <= 200 * 1024;
    const size_t smem = in_smem ? key_bytes : 0;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(topk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaFuncSetAttribute(topk): %s", cudaGetErrorString(e));
    }
    launch_pdl(topk_kernel, grid, dim3(TOPK_THREADS), smem, s, scores, (const int32_t*)c->page_map, R, n_b, (int32_t)n_cand, K, c->max_blocks,
               (int32_t)in_smem, block_idx, ptr_table);
    count_launch();
    return check_launch("topk");
}

}  // namespace omnimem
