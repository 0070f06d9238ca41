// a2-a5: Query-Shared KV Selection scores, Adaptive Window Exclusion, top-k, pointer table
// (PAPER.md:83-89 Eq. 2, :107-114 Eq. 3, :358-380).  DESIGN.md section 6.3.
#include <atomic>
#include <stdint.h>

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
// Top-k with a fixed tie-break (a4) + pointer table (a5): one WARP per (head, group) row.
// A candidate's order is the 64-bit key  (order-preserving bits of the fp32 score) << 32 | ~block,
// so "greater key" == (score descending, block index ascending) and no two candidates compare equal.
//  1. every lane scans its share of the row (candidate e at lane e % 32) and keeps its greatest key (its two
//     greatest when K > 32).  The K-th greatest of these 32 (64) lane tops -- one warp-level bitonic sort -- is
//     a LOWER BOUND of the row's K-th greatest key, because the lane tops are K distinct candidates.
//  2. a second scan compacts every candidate at or above that bound (warp ballots, no atomics).  With scores
//     spread over the lanes these are a few dozen; if they fit the 64-entry sorter, sorting them settles the K
//     best exactly -- keys are distinct, so there is nothing left to break ties on.
//  3. when more than 64 candidates pass (K close to the number of lane tops, or a row whose large scores sit in one
//     lane) the exact K-th greatest key is found by a bitwise descent over the 64-bit keys of the buffered candidates
//     (up to 256, eight per lane in registers; over the whole row only if even that buffer overflowed) and the scan is
//     repeated with it: exactly K candidates pass.
//  4. the survivors are sorted by key and written in (score desc, index asc) order with their page_map entries;
//     slots beyond |Omega| are -1.
// The row is read from wherever the caller keeps it: shared memory in the fused selection kernel, global memory
// (L2-resident behind scores_kernel) in topk_kernel.
__device__ __forceinline__ uint32_t score_key(float s)
{
    s += 0.0f;  // -0 -> +0
    const uint32_t u = __float_as_uint(s);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);  // never 0 for a non-NaN score: 0 marks "no candidate"
}
__device__ __forceinline__ unsigned long long cand_key(float s, int e)
{
    return ((unsigned long long)score_key(s) << 32) | (unsigned long long)(~(uint32_t)e);
}

// 64 keys, two per lane (element i at lane i % 32, register i / 32), sorted descending by a bitonic network
__device__ __forceinline__ void bitonic64_desc(unsigned long long& v0, unsigned long long& v1, int lane)
{
    for (int size = 2; size <= 64; size <<= 1) {
        for (int stride = size >> 1; stride >= 1; stride >>= 1) {
            if (stride == 32) {
                const unsigned long long a = v0, b2 = v1;  // partner of element lane is lane + 32: same lane
                const bool sw = a < b2;
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
}

// One warp: the K best of row[0 .. n) under the key order, written to block_idx / ptr_table (K entries each).
// sel: TOPK_CAND entries of shared memory owned by this warp.
constexpr int TOPK_CAND = 256;

// UNR: entries a lane reads per trip (x 32 per warp), every load in flight before the first use: 16 for a row in global memory
// (topk_kernel, six warps per SM: one L2 round trip per 32 entries otherwise), 1 for a row in shared memory.
template <int UNR>
__device__ __forceinline__ void warp_topk_row(const float* row, int n, int K, unsigned long long* sel, int lane,
                                              const int32_t* __restrict__ page_map, int32_t h, int32_t max_blocks, int32_t bpc,
                                              int32_t* block_idx_row, int32_t* ptr_row)
{
    // compaction of the candidates with key >= bound into sel[0 .. cap); returns how many passed (only the first cap are stored)
    auto gather = [&](unsigned long long bound, int cap) -> int {
        int cnt = 0;
        for (int e0 = 0; e0 < n; e0 += 32 * UNR) {
            float v[UNR];
#pragma unroll
            for (int j = 0; j < UNR; ++j) { const int e = e0 + 32 * j + lane; v[j] = e < n ? row[e] : 0.f; }
#pragma unroll
            for (int j = 0; j < UNR; ++j) {
                const int e = e0 + 32 * j + lane;
                const unsigned long long k = e < n ? cand_key(v[j], e) : 0ull;
                const bool take = e < n && k >= bound;
                const uint32_t m = __ballot_sync(0xffffffffu, take);
                const int slot = cnt + __popc(m & ((1u << lane) - 1u));
                if (take && slot < cap) sel[slot] = k;
                cnt += __popc(m);
            }
        }
        return cnt;
    };
    int cnt;
    if (n > K) {
        unsigned long long t1 = 0ull, t2 = 0ull;  // this lane's greatest and second greatest key
        for (int e0 = lane; e0 < n; e0 += 32 * UNR) {
            float v[UNR];
#pragma unroll
            for (int j = 0; j < UNR; ++j) { const int e = e0 + 32 * j; v[j] = e < n ? row[e] : 0.f; }
#pragma unroll
            for (int j = 0; j < UNR; ++j) {
                const int e = e0 + 32 * j;
                const unsigned long long k = e < n ? cand_key(v[j], e) : 0ull;
                if (k > t1) { t2 = t1; t1 = k; }
                else if (k > t2) t2 = k;
            }
        }
        if (K <= 16) t2 = 0ull;  // 32 lane tops bound the 16 best tightly; beyond that the second greatest of every lane joins
        bitonic64_desc(t1, t2, lane);
        // at least K tops exist: n > K, and 32 (64) lane tops cover K <= 16 (K <= 64)
        const unsigned long long kth = __shfl_sync(0xffffffffu, (K - 1) < 32 ? t1 : t2, (K - 1) & 31);
        cnt = gather(kth, TOPK_CAND);
        if (cnt > 64) {
            // more candidates than the sorter takes: the exact K-th greatest key by a bitwise descent -- over the buffered
            // candidates, TOPK_CAND / 32 per lane in registers (the usual case: a few dozen too many), or, when even the
            // buffer overflowed (large scores piled up in one lane), over the whole row
            unsigned long long T = 0ull;
            if (cnt <= TOPK_CAND) {
                __syncwarp();
                unsigned long long c8[TOPK_CAND / 32];
#pragma unroll
                for (int j = 0; j < TOPK_CAND / 32; ++j) c8[j] = (j * 32 + lane) < cnt ? sel[j * 32 + lane] : 0ull;
                for (int bit = 63; bit >= 0; --bit) {
                    const unsigned long long cand = T | (1ull << bit);
                    int c = 0;
#pragma unroll
                    for (int j = 0; j < TOPK_CAND / 32; ++j) c += c8[j] >= cand;
                    if (__reduce_add_sync(0xffffffffu, c) >= K) T = cand;
                }
            } else {
                for (int bit = 63; bit >= 0; --bit) {
                    const unsigned long long cand = T | (1ull << bit);
                    int c = 0;
                    for (int e0 = lane; e0 < n; e0 += 32 * UNR) {
                        float v[UNR];
#pragma unroll
                        for (int j = 0; j < UNR; ++j) { const int e = e0 + 32 * j; v[j] = e < n ? row[e] : 0.f; }
#pragma unroll
                        for (int j = 0; j < UNR; ++j) { const int e = e0 + 32 * j; c += e < n && cand_key(v[j], e) >= cand; }
                    }
                    if (__reduce_add_sync(0xffffffffu, c) >= K) T = cand;
                }
            }
            __syncwarp();
            cnt = gather(T, 64);  // exactly K
        }
    } else {
        cnt = gather(1ull, 64);  // at most K candidates: every one of them is taken
    }
    __syncwarp();
    unsigned long long v0 = lane < cnt ? sel[lane] : 0ull, v1 = lane + 32 < cnt ? sel[lane + 32] : 0ull;
    bitonic64_desc(v0, v1, lane);
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const int s = lane + 32 * j;
        if (s >= K) continue;
        const unsigned long long kv = j ? v1 : v0;
        const int32_t b = kv ? (int32_t)(~(uint32_t)kv) : -1;
        if (block_idx_row) block_idx_row[s] = b;
        ptr_row[s] = (b < 0) ? -1 : page_of(page_map, h, b, max_blocks, bpc);
    }
}

// Two warps (half = 0, 1) share one row: each scans half of it (a lane of the pair sees every 64th candidate), the 64 lane tops
// bound the K-th greatest key from below, each warp compacts the candidates of its half at or above the bound into its half of
// sel_row, and warp 0 finishes (sort, or the exact descent when more than 64 passed) and writes.  bar_id: a named barrier of the
// pair (64 threads).  sel_row: TOPK_CAND entries, tops_row: 64 entries, cnt_row: 2 ints of shared memory owned by the pair.
template <int UNR>
__device__ __forceinline__ void pair_topk_row(const float* row, int n_cand, int K, unsigned long long* sel_row, unsigned long long* tops_row,
                                              int* cnt_row, int bar_id, int half, int lane, const int32_t* __restrict__ page_map, int32_t h,
                                              int32_t max_blocks, int32_t bpc, int32_t* block_idx_row, int32_t* ptr_row)
{
    unsigned long long* mine = sel_row + half * (TOPK_CAND / 2);  // this warp's half of the candidate buffer
    if (n_cand <= K || n_cand < 128) {
        // short rows: one warp does it all
        if (half == 0) warp_topk_row<UNR>(row, n_cand, K, sel_row, lane, page_map, h, max_blocks, bpc, block_idx_row, ptr_row);
    } else {
        unsigned long long top = 0ull;
        for (int e0 = half * 32 + lane; e0 < n_cand; e0 += 64 * UNR) {
            float v[UNR];
#pragma unroll
            for (int j = 0; j < UNR; ++j) { const int e = e0 + 64 * j; v[j] = e < n_cand ? row[e] : 0.f; }
#pragma unroll
            for (int j = 0; j < UNR; ++j) {
                const int e = e0 + 64 * j;
                const unsigned long long k = e < n_cand ? cand_key(v[j], e) : 0ull;
                top = k > top ? k : top;
            }
        }
        tops_row[half * 32 + lane] = top;
        asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory");
        unsigned long long t1 = tops_row[lane], t2 = tops_row[32 + lane];
        bitonic64_desc(t1, t2, lane);  // both warps sort the 64 tops: no second hand-over
        const unsigned long long kth = __shfl_sync(0xffffffffu, (K - 1) < 32 ? t1 : t2, (K - 1) & 31);
        int cnt = 0;
        for (int e0 = half * 32; e0 < n_cand; e0 += 64 * UNR) {
            float v[UNR];
#pragma unroll
            for (int j = 0; j < UNR; ++j) { const int e = e0 + 64 * j + lane; v[j] = e < n_cand ? row[e] : 0.f; }
#pragma unroll
            for (int j = 0; j < UNR; ++j) {
                const int e = e0 + 64 * j + lane;
                const unsigned long long k = e < n_cand ? cand_key(v[j], e) : 0ull;
                const bool take = e < n_cand && k >= kth;
                const uint32_t m = __ballot_sync(0xffffffffu, take);
                const int slot = cnt + __popc(m & ((1u << lane) - 1u));
                if (take && slot < TOPK_CAND / 2) mine[slot] = k;
                cnt += __popc(m);
            }
        }
        if (lane == 0) cnt_row[half] = cnt;
        asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory");
        if (half == 0) {
            const int c0 = cnt_row[0], c1 = cnt_row[1];
            if (c0 > TOPK_CAND / 2 || c1 > TOPK_CAND / 2) {
                // a half overflowed its buffer (large scores piled up in a few lanes): the one-warp routine, from scratch
                warp_topk_row<UNR>(row, n_cand, K, sel_row, lane, page_map, h, max_blocks, bpc, block_idx_row, ptr_row);
            } else {
                // candidate i of the pair: the first c0 sit in this warp's half of the buffer, the next c1 in the other
                auto cand_at = [&](int i) -> unsigned long long {
                    return i < c0 ? sel_row[i] : (i < c0 + c1 ? sel_row[TOPK_CAND / 2 + i - c0] : 0ull);
                };
                unsigned long long T = 0ull;
                if (c0 + c1 > 64) {  // exact K-th greatest key: bitwise descent over the buffered candidates, in registers
                    unsigned long long c8[TOPK_CAND / 32];
#pragma unroll
                    for (int j = 0; j < TOPK_CAND / 32; ++j) c8[j] = cand_at(j * 32 + lane);
                    for (int bit = 63; bit >= 0; --bit) {
                        const unsigned long long cd = T | (1ull << bit);
                        int c = 0;
#pragma unroll
                        for (int j = 0; j < TOPK_CAND / 32; ++j) c += c8[j] >= cd;
                        if (__reduce_add_sync(0xffffffffu, c) >= K) T = cd;
                    }
                }
                // the survivors (all of them, or those at or above T: exactly K), two per lane, sorted
                unsigned long long v0 = 0ull, v1 = 0ull;
                int kept = 0;
                for (int i0 = 0; i0 < c0 + c1; i0 += 32) {
                    const unsigned long long k = cand_at(i0 + lane);
                    const bool take = k != 0ull && k >= T;
                    const uint32_t m = __ballot_sync(0xffffffffu, take);
                    const int slot = kept + __popc(m & ((1u << lane) - 1u));
                    if (take) tops_row[slot & 63] = k;  // the tops are done with: reuse their 64 entries
                    kept += __popc(m);
                }
                __syncwarp();
                v0 = lane < kept ? tops_row[lane] : 0ull;
                v1 = lane + 32 < kept ? tops_row[lane + 32] : 0ull;
                bitonic64_desc(v0, v1, lane);
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int sl = lane + 32 * j;
                    if (sl >= K) continue;
                    const unsigned long long kv = j ? v1 : v0;
                    const int32_t b = kv ? (int32_t)(~(uint32_t)kv) : -1;
                    if (block_idx_row) block_idx_row[sl] = b;
                    ptr_row[sl] = (b < 0) ? -1 : page_of(page_map, h, b, max_blocks, bpc);
                }
            }
        }
    }
}

constexpr int TOPK_ROWS = 4, TOPK_THREADS = TOPK_ROWS * 64;  // two warps per row, 222 CTAs at config 3: every SM has rows

__global__ void __launch_bounds__(TOPK_THREADS)
topk_kernel(const float* __restrict__ scores, const int32_t* __restrict__ page_map, int32_t n_rows, int32_t R, int64_t n_b,
            int32_t n_cand, int32_t K, int32_t max_blocks, int32_t bpc, int32_t* __restrict__ block_idx, int32_t* __restrict__ ptr_table)
{
    __shared__ unsigned long long sel[TOPK_ROWS][TOPK_CAND];
    __shared__ unsigned long long pair_tops[TOPK_ROWS][64];
    __shared__ int pair_cnt[TOPK_ROWS][2];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rowi = warp % TOPK_ROWS, half = warp / TOPK_ROWS;  // warps w and w + TOPK_ROWS share row w
    const int row_id = blockIdx.x * TOPK_ROWS + rowi;
    pdl_launch_dependents();
    pdl_wait();  // the scores come from scores_kernel (or from the caller's previous kernel)
    if (row_id >= n_rows) return;  // both warps of the pair leave: nobody is left waiting at the pair's barrier
    const int h = row_id / R;
    // 16 entries per lane and trip in flight (8: 77 us of selection on config 3, 16: 64.5, 32: 87 -- the registers cost residency)
    pair_topk_row<16>(scores + (int64_t)row_id * n_b, n_cand, K, sel[rowi], pair_tops[rowi], pair_cnt[rowi], 1 + rowi, half, lane, page_map, h,
                     max_blocks, bpc, block_idx ? block_idx + (int64_t)row_id * K : nullptr, ptr_table + (int64_t)row_id * K);
}

int32_t launch_topk(const Cache* c, const float* scores, int32_t R, int64_t n_b, int64_t n_cand, int32_t K,
                    int32_t* block_idx, int32_t* ptr_table, cudaStream_t s)
{
    const int32_t n_rows = c->H * R;
    cudaError_t e = launch_pdl(topk_kernel, dim3((unsigned)ceil_div64(n_rows, TOPK_ROWS)), dim3(TOPK_THREADS), 0, s, scores,
                               (const int32_t*)c->page_map, n_rows, R, n_b, (int32_t)n_cand, K, c->max_blocks, c->bpc, block_idx, ptr_table);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "topk launch: %s", cudaGetErrorString(e));
    count_launch();
    return check_launch("topk");
}

// ---------------------------------------------------------------------------------------------
// a2-a5 in ONE launch: group means, score tiles, top-k and pointer table for RPC = 8 query groups of one head per
// CTA; the groups' scores never leave shared memory (scores_out, when the caller asks for it, is a copy).
//   phase 1  qbar: warps take (group, 32-query chunk) items; a lane owns a 16-byte piece of the rows it reads, sums
//            in fp64 (exact, so the order does not matter) and adds its share into shared-memory doubles.
//   phase 2  scores: one m16n8k16 tile = 8 groups (rows 8-15 of A are zero) x 8 blocks.  The MMA's k index is a free
//            permutation of the head dimension as long as A and B use the same one: it is chosen so that a lane's B
//            registers of all k-steps are D/64 aligned 16-byte loads straight from pooled_k (a quad covers a 64-byte
//            segment of its block's row per load) -- no staging, no ldmatrix.
//   phase 3  top-k: warp w owns group w's row in shared memory (warp_topk_row above).
// Used while 8 rows of N_b scores fit in shared memory (N_b <= SEL_FUSED_MAX_NB); longer histories take the three
// kernels above, whose score tiles go through global memory.
constexpr int SEL_RPC = 8;
constexpr int SEL_FUSED_MAX_NB = 5120;  // 8 rows x 5120 x 4 B = 160 KB

constexpr int SEL_THREADS = 512, SEL_WARPS = SEL_THREADS / 32;

template <int D>
__global__ void __launch_bounds__(SEL_THREADS)
select_fused_kernel(const uint4* __restrict__ q, int32_t n_q, int64_t stride_tok16, int64_t stride_head16, int32_t G, int32_t R,
                    const __nv_bfloat16* __restrict__ pooled_k, const int32_t* __restrict__ page_map, int32_t max_blocks, int32_t bpc, int32_t n_b,
                    int32_t n_score /* blocks scored: n_b if the scores are exported, else n_cand */, int32_t n_cand, int32_t K, float scale,
                    float* __restrict__ scores_out, int32_t* __restrict__ block_idx, int32_t* __restrict__ ptr_table)
{
    constexpr int PIECES = D / 8;      // 16-byte pieces per row
    constexpr int RL = 32 / PIECES;    // rows a warp reads per load instruction
    constexpr int NL = D / 32;         // 16-byte loads per lane and block row in phase 2 (a quad covers 64 bytes per load)
    extern __shared__ __align__(16) unsigned char sel_smem[];
    __shared__ double qsum[SEL_RPC][D];
    __shared__ __align__(16) __nv_bfloat16 qbar_s[SEL_RPC][D];
    __shared__ unsigned long long sel[SEL_RPC][TOPK_CAND];
    __shared__ unsigned long long pair_tops[SEL_RPC][64];
    __shared__ int pair_cnt[SEL_RPC][2];
    const int n_pad = (n_score + 7) & ~7;
    float* sc = reinterpret_cast<float*>(sel_smem);  // [SEL_RPC][n_pad]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int h = blockIdx.y, r0 = blockIdx.x * SEL_RPC;
    const int nr = min(SEL_RPC, R - r0);
    for (int i = tid; i < SEL_RPC * D; i += SEL_THREADS) (&qsum[0][0])[i] = 0.0;
    pdl_launch_dependents();
    pdl_wait();  // Q and pooled_k come from earlier work on the stream
    __syncthreads();

    // ---- phase 1: group means
    {
        const int piece = lane % PIECES, rl = lane / PIECES;
        const uint4* base = q + (int64_t)h * stride_head16 + piece;
        // items: (group g, chunk c of 32 queries)
        const int cpg = (G + 31) / 32;
        for (int item = warp; item < nr * cpg; item += SEL_WARPS) {
            const int g = item / cpg, c = item % cpg;
            const int lo = (r0 + g) * G + c * 32, hi = min(min((r0 + g + 1) * G, n_q), lo + 32);
            double acc[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) acc[i] = 0.0;
            constexpr int NLD = 32 / RL;  // a 32-query item in ONE trip: every load of the lane is in flight before the first add
            for (int s0 = lo + rl; s0 < hi; s0 += NLD * RL) {
                uint4 u[NLD];
#pragma unroll
                for (int j = 0; j < NLD; ++j) {
                    const int s = s0 + j * RL;
                    u[j] = s < hi ? __ldg(base + (int64_t)s * stride_tok16) : make_uint4(0, 0, 0, 0);  // +0.0 terms change nothing
                }
#pragma unroll
                for (int j = 0; j < NLD; ++j) {
                    const uint32_t w[4] = {u[j].x, u[j].y, u[j].z, u[j].w};
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        acc[2 * i] += (double)__uint_as_float(w[i] << 16);
                        acc[2 * i + 1] += (double)__uint_as_float(w[i] & 0xffff0000u);
                    }
                }
            }
#pragma unroll
            for (int o = PIECES; o < 32; o <<= 1)
#pragma unroll
                for (int i = 0; i < 8; ++i) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], o);
            if (lo < hi && rl == 0)
#pragma unroll
                for (int i = 0; i < 8; ++i) atomicAdd(&qsum[g][piece * 8 + i], acc[i]);
        }
    }
    __syncthreads();
    for (int i = tid; i < SEL_RPC * D; i += SEL_THREADS) {
        const int g = i / D, d = i % D;
        float f = 0.f;
        if (g < nr) {
            const int lo = (r0 + g) * G, hi = min(lo + G, n_q);
            f = __fdiv_rn((float)qsum[g][d], (float)(hi - lo));
        }
        qbar_s[g][d] = __float2bfloat16_rn(f);
    }
    __syncthreads();

    // ---- phase 2: scores of the CTA's groups against blocks [0, n_score)
    {
        const int gq = lane >> 2, qd = lane & 3;  // A/C row (group), quad lane
        // This lane's share of a row (group mean or block key) is the 16-byte pieces  [32 i + 8 qd, + 8)  (i < NL); the 8 dims
        // of piece i feed k-steps 2 i and 2 i + 1: words 0, 1 are the two B (A) registers of the first, words 2, 3 of the second.
        uint32_t af[NL][4];
#pragma unroll
        for (int i = 0; i < NL; ++i) {
            const uint4 v = *reinterpret_cast<const uint4*>(&qbar_s[gq][32 * i + 8 * qd]);
            af[i][0] = v.x; af[i][1] = v.y; af[i][2] = v.z; af[i][3] = v.w;
        }
        const __nv_bfloat16* kh = pooled_k + (int64_t)h * max_blocks * D;
        const int n_tiles = n_pad / 8;
        for (int t0 = warp; t0 < n_tiles; t0 += SEL_WARPS * 4) {  // 4 tiles per trip: 4 * NL loads in flight per lane
            uint4 bv[4][NL];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int b = (t0 + SEL_WARPS * u) * 8 + gq;  // B column n = gq: this lane's block
#pragma unroll
                for (int i = 0; i < NL; ++i)
                    bv[u][i] = (t0 + SEL_WARPS * u < n_tiles && b < n_b) ? __ldg(reinterpret_cast<const uint4*>(kh + (int64_t)b * D + 32 * i + 8 * qd))
                                                               : make_uint4(0, 0, 0, 0);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (t0 + SEL_WARPS * u >= n_tiles) break;
                float c4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int i = 0; i < NL; ++i) {
                    const uint32_t bw[4] = {bv[u][i].x, bv[u][i].y, bv[u][i].z, bv[u][i].w};
                    // k-step 2 i: registers (words 0, 1); k-step 2 i + 1: (words 2, 3).  A rows 8-15 are zero.
                    const uint32_t a_lo[4] = {af[i][0], 0u, af[i][1], 0u};
                    const uint32_t a_hi[4] = {af[i][2], 0u, af[i][3], 0u};
                    sel_mma(c4, a_lo, bw[0], bw[1]);
                    sel_mma(c4, a_hi, bw[2], bw[3]);
                }
                const int b = (t0 + SEL_WARPS * u) * 8 + 2 * qd;  // C columns 2 qd, 2 qd + 1 of row gq
                const float s0v = scale * c4[0] + 0.0f, s1v = scale * c4[1] + 0.0f;
                *reinterpret_cast<float2*>(&sc[gq * n_pad + b]) = make_float2(s0v, s1v);
                if (scores_out && gq < nr) {
                    float* dst = scores_out + ((int64_t)h * R + r0 + gq) * n_b;
                    if (b < n_b) dst[b] = s0v;
                    if (b + 1 < n_b) dst[b + 1] = s1v;
                }
            }
        }
    }
    __syncthreads();

    // ---- phase 3: top-k + pointer table.  Warps w and w + 8 share group w's row: each scans half of it (a lane of the pair sees
    // every 64th candidate), the 64 lane tops bound the K-th greatest key from below, each warp compacts the candidates of its
    // half at or above the bound, and warp w finishes (sort, or the exact descent when more than 64 passed) and writes.
    {
        const int rowi = warp & 7, half = warp >> 3;
        if (rowi < nr) {
            const float* row = sc + rowi * n_pad;
            const int64_t row_id = (int64_t)h * R + r0 + rowi;
            int32_t* bi_row = block_idx ? block_idx + row_id * K : nullptr;
            int32_t* ptr_row = ptr_table + row_id * K;
            pair_topk_row<1>(row, n_cand, K, sel[rowi], pair_tops[rowi], pair_cnt[rowi], 1 + rowi, half, lane, page_map, h, max_blocks, bpc,
                             bi_row, ptr_row);
        }
    }
}

// the fused kernel when its rows fit shared memory; false = the caller takes the three-kernel path
bool select_fused_fits(int64_t n_b) { return n_b > 0 && n_b <= SEL_FUSED_MAX_NB; }

int64_t select_launch_ctas(int32_t H, int32_t n_q, int32_t G, int64_t n_b)
{
    if (n_b <= 0) return 0;
    if (!select_fused_fits(n_b)) return INT64_MAX;
    return ceil_div64(ceil_div64(n_q, G), SEL_RPC) * H;
}

int32_t launch_select_fused(const Cache* c, const void* q, int32_t n_q, int64_t stride_tok, int64_t stride_head, int32_t G, int64_t n_b,
                            int64_t n_cand, int32_t K, float scale, float* scores_out, int32_t* block_idx, int32_t* ptr_table, cudaStream_t s)
{
    const int32_t R = (int32_t)ceil_div64(n_q, G);
    const int32_t n_score = scores_out ? (int32_t)n_b : (int32_t)n_cand;
    const size_t smem = (size_t)SEL_RPC * ((n_score + 7) & ~7) * 4;
    dim3 grid((unsigned)ceil_div64(R, SEL_RPC), (unsigned)c->H);
    static std::atomic<uint64_t> attr_devices[2];  // the shared-memory opt-in is per device (and per instantiation)
    int dev = 0;
    cudaGetDevice(&dev);
    const uint64_t bit = 1ull << (dev & 63);
    const int which = c->D == 128 ? 0 : 1;
    if (!(attr_devices[which].load(std::memory_order_acquire) & bit)) {
        const int max_smem = SEL_RPC * SEL_FUSED_MAX_NB * 4;
        cudaError_t e = c->D == 128 ? cudaFuncSetAttribute(select_fused_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem)
                                    : cudaFuncSetAttribute(select_fused_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaFuncSetAttribute(select): %s", cudaGetErrorString(e));
        attr_devices[which].fetch_or(bit, std::memory_order_release);
    }
    cudaError_t e;
    if (c->D == 128)
        e = launch_pdl(select_fused_kernel<128>, grid, dim3(SEL_THREADS), smem, s, (const uint4*)q, n_q, stride_tok / 8, stride_head / 8, G, R,
                       (const __nv_bfloat16*)c->pooled_k, (const int32_t*)c->page_map, c->max_blocks, c->bpc, (int32_t)n_b, n_score, (int32_t)n_cand, K,
                       scale, scores_out, block_idx, ptr_table);
    else
        e = launch_pdl(select_fused_kernel<64>, grid, dim3(SEL_THREADS), smem, s, (const uint4*)q, n_q, stride_tok / 8, stride_head / 8, G, R,
                       (const __nv_bfloat16*)c->pooled_k, (const int32_t*)c->page_map, c->max_blocks, c->bpc, (int32_t)n_b, n_score, (int32_t)n_cand, K,
                       scale, scores_out, block_idx, ptr_table);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "select launch: %s", cudaGetErrorString(e));
    count_launch();
    return check_launch("select");
}

// ---------------------------------------------------------------------------------------------
// a2 under the probability reading (OMNIMEM_SCORE_PROB, reading A1b):
//   sbar[h][r][b] = (1 / |G_r|) * sum_{q in G_r} softmax_b(score_scale * <q, kbar[h][b]>),  b over the head's N_b compressed tokens.
// Unlike the logit mode this does not collapse to one dot product per group: every query needs its own row of logits
// (S x N_b x D per head).  One CTA = one slab of up to 64 queries of one group (4 warps x 16 rows, m16n8k16 with the
// operands loaded straight from global memory under the same k permutation as the fused kernel above):
//   pass A  the row's log-sum-exp over all N_b logits (online max / sum per lane, merged over the quad),
//   pass B  the logits again, p = exp2(x - LSE), summed over the slab's rows per column: a butterfly over the 8 row lanes,
//           then the 4 warps' partial columns are added in a fixed order (no float atomics: results are reproducible).
// A group of more than 64 queries is spread over ceil(G / 64) CTAs whose partial columns land in the workspace and are
// added in slab order by prob_reduce_kernel.
constexpr int PROB_THREADS = 128;
constexpr int PROB_MAX_NB = 11264;  // 4 warps x N_b floats of shared memory

template <int D>
__global__ void __launch_bounds__(PROB_THREADS)
scores_prob_kernel(const uint4* __restrict__ q, int32_t n_q, int64_t stride_tok16, int64_t stride_head16, int32_t G, int32_t R, int32_t spg,
                   const __nv_bfloat16* __restrict__ pooled_k, int32_t max_blocks, int32_t n_b, float scale_log2,
                   float* __restrict__ out /* [H][R * spg][n_b] */)
{
    constexpr int NL = D / 32;
    extern __shared__ __align__(16) unsigned char sel_smem[];
    const int n_pad = (n_b + 7) & ~7;
    float* part = reinterpret_cast<float*>(sel_smem);  // [4][n_pad]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int gq = lane >> 2, qd = lane & 3;
    const int h = blockIdx.y, r = blockIdx.x / spg, j = blockIdx.x % spg;
    const int g_lo = r * G, g_hi = min(g_lo + G, n_q);
    const int row0 = g_lo + j * 64 + warp * 16 + gq, row1 = row0 + 8;  // this lane's two query rows
    const bool on0 = row0 < g_hi, on1 = row1 < g_hi;
    pdl_launch_dependents();
    pdl_wait();
    // A fragments (both rows, every k-step) stay in registers for the whole kernel
    uint32_t a0[NL][4], a1[NL][4];
#pragma unroll
    for (int i = 0; i < NL; ++i) {
        const uint4 z = make_uint4(0, 0, 0, 0);
        const uint4 v0 = on0 ? __ldg(q + (int64_t)h * stride_head16 + (int64_t)row0 * stride_tok16 + 4 * i + qd) : z;
        const uint4 v1 = on1 ? __ldg(q + (int64_t)h * stride_head16 + (int64_t)row1 * stride_tok16 + 4 * i + qd) : z;
        a0[i][0] = v0.x; a0[i][1] = v0.y; a0[i][2] = v0.z; a0[i][3] = v0.w;
        a1[i][0] = v1.x; a1[i][1] = v1.y; a1[i][2] = v1.z; a1[i][3] = v1.w;
    }
    const __nv_bfloat16* kh = pooled_k + (int64_t)h * max_blocks * D;
    const int n_tiles = n_pad / 8;
    // logits (log2 units) of tiles t0 .. t0 + 3: x[u][0..1] row0, x[u][2..3] row1, columns 8 t + 2 qd, + 1
    auto tiles4 = [&](int t0, float (&x)[4][4]) {
        uint4 bv[4][NL];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int b = (t0 + u) * 8 + gq;
#pragma unroll
            for (int i = 0; i < NL; ++i)
                bv[u][i] = (t0 + u < n_tiles && b < n_b) ? __ldg(reinterpret_cast<const uint4*>(kh + (int64_t)b * D + 32 * i + 8 * qd))
                                                         : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float c4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int i = 0; i < NL; ++i) {
                const uint32_t lo4[4] = {a0[i][0], a1[i][0], a0[i][1], a1[i][1]};
                const uint32_t hi4[4] = {a0[i][2], a1[i][2], a0[i][3], a1[i][3]};
                sel_mma(c4, lo4, bv[u][i].x, bv[u][i].y);
                sel_mma(c4, hi4, bv[u][i].z, bv[u][i].w);
            }
            const int b = (t0 + u) * 8 + 2 * qd;
#pragma unroll
            for (int e = 0; e < 4; ++e) x[u][e] = (b + (e & 1) < n_b && t0 + u < n_tiles) ? c4[e] * scale_log2 : -INFINITY;
        }
    };
    // ---- pass A: log-sum-exp per row
    float m[2] = {-INFINITY, -INFINITY}, l[2] = {0.f, 0.f};
    for (int t0 = 0; t0 < n_tiles; t0 += 4) {
        float x[4][4];
        tiles4(t0, x);
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            float mx = m[rr];
#pragma unroll
            for (int u = 0; u < 4; ++u) mx = fmaxf(mx, fmaxf(x[u][2 * rr], x[u][2 * rr + 1]));
            if (mx > m[rr]) { l[rr] *= exp2f(m[rr] - mx); m[rr] = mx; }  // m = -inf: l = 0 stays 0 (exp2f(-inf) = 0)
            if (mx > -INFINITY) {
#pragma unroll
                for (int u = 0; u < 4; ++u) l[rr] += exp2f(x[u][2 * rr] - mx) + exp2f(x[u][2 * rr + 1] - mx);
            }
        }
    }
    float lse[2];
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
        float mm = m[rr], ll = l[rr];
#pragma unroll
        for (int o = 1; o < 4; o <<= 1) {
            const float mo = __shfl_xor_sync(0xffffffffu, mm, o), lo = __shfl_xor_sync(0xffffffffu, ll, o);
            const float mn = fmaxf(mm, mo);
            ll = (mn > -INFINITY) ? ll * exp2f(mm - mn) + lo * exp2f(mo - mn) : 0.f;
            mm = mn;
        }
        lse[rr] = mm + log2f(ll);  // n_b >= 1: ll > 0
    }
    // ---- pass B: probabilities, summed over the slab's rows
    for (int t0 = 0; t0 < n_tiles; t0 += 4) {
        float x[4][4];
        tiles4(t0, x);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (t0 + u >= n_tiles) break;
            float v0 = (on0 ? exp2f(x[u][0] - lse[0]) : 0.f) + (on1 ? exp2f(x[u][2] - lse[1]) : 0.f);
            float v1 = (on0 ? exp2f(x[u][1] - lse[0]) : 0.f) + (on1 ? exp2f(x[u][3] - lse[1]) : 0.f);
#pragma unroll
            for (int o = 4; o < 32; o <<= 1) {
                v0 += __shfl_xor_sync(0xffffffffu, v0, o);
                v1 += __shfl_xor_sync(0xffffffffu, v1, o);
            }
            if (gq == 0) *reinterpret_cast<float2*>(&part[warp * n_pad + (t0 + u) * 8 + 2 * qd]) = make_float2(v0, v1);
        }
    }
    __syncthreads();
    const float inv = 1.0f / (float)(g_hi - g_lo);
    float* dst = out + ((int64_t)h * R * spg + blockIdx.x) * n_b;
    for (int b = tid; b < n_b; b += PROB_THREADS)
        dst[b] = (((part[b] + part[n_pad + b]) + part[2 * n_pad + b]) + part[3 * n_pad + b]) * inv + 0.0f;
}

// scores[h][r][b] = sum over the group's slabs, in slab order
__global__ void __launch_bounds__(256)
prob_reduce_kernel(const float* __restrict__ partial, int32_t spg, int64_t n_b, int64_t n_rows, float* __restrict__ scores)
{
    pdl_launch_dependents();
    pdl_wait();
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n_rows * n_b) return;
    const int64_t row = i / n_b, b = i % n_b;
    float s = 0.f;
    for (int j = 0; j < spg; ++j) s += partial[(row * spg + j) * n_b + b];
    scores[i] = s + 0.0f;
}

bool scores_prob_fits(int64_t n_b) { return n_b <= PROB_MAX_NB; }

// workspace floats the probability path needs beyond the scores themselves (slab partials of groups longer than 64 queries)
size_t scores_prob_partial_floats(int32_t H, int32_t n_q, int32_t G, int64_t n_b)
{
    const int64_t spg = ceil_div64(G, 64), R = ceil_div64(n_q, G);
    return spg > 1 ? (size_t)H * R * spg * n_b : 0;
}

int32_t launch_scores_prob(const Cache* c, const void* q, int32_t n_q, int64_t stride_tok, int64_t stride_head, int32_t G, int64_t n_b,
                           float scale, float* scores, float* partial, cudaStream_t s)
{
    if (n_b <= 0) return OMNIMEM_OK;
    const int32_t R = (int32_t)ceil_div64(n_q, G), spg = (int32_t)ceil_div64(G, 64);
    const size_t smem = (size_t)4 * ((n_b + 7) & ~7) * 4;
    static std::atomic<uint64_t> attr_devices[2];
    int dev = 0;
    cudaGetDevice(&dev);
    const uint64_t bit = 1ull << (dev & 63);
    const int which = c->D == 128 ? 0 : 1;
    if (!(attr_devices[which].load(std::memory_order_acquire) & bit)) {
        const int max_smem = 4 * PROB_MAX_NB * 4;
        cudaError_t e = c->D == 128 ? cudaFuncSetAttribute(scores_prob_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem)
                                    : cudaFuncSetAttribute(scores_prob_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaFuncSetAttribute(scores_prob): %s", cudaGetErrorString(e));
        attr_devices[which].fetch_or(bit, std::memory_order_release);
    }
    float* dst = spg > 1 ? partial : scores;
    dim3 grid((unsigned)(R * spg), (unsigned)c->H);
    const float sl2 = scale * 1.4426950408889634f;
    cudaError_t e;
    if (c->D == 128)
        e = launch_pdl(scores_prob_kernel<128>, grid, dim3(PROB_THREADS), smem, s, (const uint4*)q, n_q, stride_tok / 8, stride_head / 8, G, R, spg,
                       (const __nv_bfloat16*)c->pooled_k, c->max_blocks, (int32_t)n_b, sl2, dst);
    else
        e = launch_pdl(scores_prob_kernel<64>, grid, dim3(PROB_THREADS), smem, s, (const uint4*)q, n_q, stride_tok / 8, stride_head / 8, G, R, spg,
                       (const __nv_bfloat16*)c->pooled_k, c->max_blocks, (int32_t)n_b, sl2, dst);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "scores_prob launch: %s", cudaGetErrorString(e));
    count_launch();
    if (spg > 1) {
        const int64_t n = (int64_t)c->H * R * n_b;
        e = launch_pdl(prob_reduce_kernel, dim3((unsigned)ceil_div64(n, 256)), dim3(256), 0, s, (const float*)partial, spg, n_b, (int64_t)c->H * R, scores);
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "prob_reduce launch: %s", cudaGetErrorString(e));
        count_launch();
    }
    return check_launch("scores_prob");
}

}  // namespace omnimem
