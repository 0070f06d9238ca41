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
// Top-k with a fixed tie-break (a4) + pointer table (a5).
// A candidate's order is the 64-bit key  (order-preserving bits of the fp32 score) << 32 | ~block,
// so "greater key" == (score descending, block index ascending) and no two candidates compare equal.
// A row (one (head, group)) is owned by a TEAM of WARPS warps -- one warp (8 rows per CTA) while the row fits
// 32 * KPL candidates, the whole 8-warp CTA above that -- and its score keys live in REGISTERS, KPL per
// thread, candidate e at thread e % TEAM, register e / TEAM (coalesced loads; -0 canonicalised to +0).
//  1. bitwise descent on the K-th greatest 32-bit score key T: for bit = 31 .. 0 the team counts its keys
//     >= T | bit (a compare + add per register, one redux.sync per warp; 8-warp teams add one shared-memory
//     exchange) and keeps the bit if at least K remain.  No histogram, no shared-memory atomics.
//  2. only if more than K candidates have key >= T (ties at T): the same descent on the low word ~block among
//     the candidates equal to T finds the last block index that still belongs to the K best.
//  3. the K survivors are compacted into shared memory, sorted by their 64-bit key with a warp-level bitonic
//     network and written in (score desc, index asc) order with their page_map entries; slots beyond
//     |Omega| are -1.
// Rows longer than TEAM * KPL candidates (more than 16384 blocks, i.e. a history beyond a million tokens) take
// the STREAM variant: the same algorithm with the keys re-read from global memory in every pass.
__device__ __forceinline__ uint32_t score_key(float s)
{
    s += 0.0f;  // -0 -> +0
    const uint32_t u = __float_as_uint(s);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);  // never 0 for a non-NaN score: 0 marks "no candidate"
}

constexpr int TOPK_THREADS = 256;

template <int WARPS>
__device__ __forceinline__ uint32_t team_sum(uint32_t v, uint32_t* xch, int warp_in_team, int lane, int& flip)
{
    v = __reduce_add_sync(0xffffffffu, v);
    if (WARPS == 1) return v;
    // 8-warp team == the whole CTA; double-buffered exchange slots, one barrier per call
    uint32_t* slot = xch + (flip & 1) * 8;
    flip ^= 1;
    if (lane == 0) slot[warp_in_team] = v;
    __syncthreads();
    uint32_t t = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) t += slot[i];
    return t;
}

template <int KPL, int WARPS, bool STREAM>
__global__ void __launch_bounds__(TOPK_THREADS)
topk_kernel(const float* __restrict__ scores, const int32_t* __restrict__ page_map, int32_t n_rows, int32_t R, int64_t n_b,
            int32_t n_cand, int32_t K, int32_t max_blocks, int32_t* __restrict__ block_idx, int32_t* __restrict__ ptr_table)
{
    constexpr int TEAM = 32 * WARPS;
    constexpr int ROWS = (TOPK_THREADS / 32) / WARPS;  // rows per CTA
    __shared__ unsigned long long sel[ROWS][64];
    __shared__ uint32_t n_sel[ROWS];
    __shared__ uint32_t xch[16];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int team = warp / WARPS, wit = warp % WARPS, t = wit * 32 + lane;  // row team, warp in team, thread in team
    const int row_id = blockIdx.x * ROWS + team;
    const bool live = row_id < n_rows;  // warp-uniform; with WARPS == 8 the whole CTA is one row and always live
    const float* row = scores + (int64_t)(live ? row_id : 0) * n_b;
    int flip = 0;

    if (WARPS == 1) { sel[team][lane] = 0ull; sel[team][lane + 32] = 0ull; }
    else if (tid < 64) sel[0][tid] = 0ull;
    if (t == 0) n_sel[team] = 0;
    pdl_launch_dependents();
    pdl_wait();  // the scores come from scores_kernel (or from the caller's previous kernel)
    if (WARPS == 1 && !live) return;

    uint32_t key[KPL];
    const int n_j = STREAM ? (n_cand + TEAM - 1) / TEAM : KPL;
    if (!STREAM) {
#pragma unroll
        for (int j = 0; j < KPL; ++j) {
            const int e = j * TEAM + t;
            key[j] = e < n_cand ? score_key(__ldg(row + e)) : 0u;
        }
    }
    auto key_at = [&](int j) -> uint32_t {
        if (!STREAM) return key[j];
        const int e = j * TEAM + t;
        return e < n_cand ? score_key(__ldg(row + e)) : 0u;
    };
    if (WARPS > 1) __syncthreads(); else __syncwarp();

    uint32_t T = 0, L = 0;  // take a candidate iff key > T, or key == T and ~block >= L
    if (n_cand > K) {
        for (int bit = 31; bit >= 0; --bit) {
            const uint32_t cand = T | (1u << bit);
            uint32_t c = 0;
            if (STREAM) { for (int j = 0; j < n_j; ++j) c += key_at(j) >= cand; }
            else {
#pragma unroll
                for (int j = 0; j < KPL; ++j) c += key[j] >= cand;
            }
            if (team_sum<WARPS>(c, xch, wit, lane, flip) >= (uint32_t)K) T = cand;
        }
        // T is the K-th greatest score key.  Ties at T: descend on ~block among the candidates equal to T
        uint32_t c_gt = 0, c_eq = 0;
        if (STREAM) { for (int j = 0; j < n_j; ++j) { const uint32_t k = key_at(j); c_gt += k > T; c_eq += k == T; } }
        else {
#pragma unroll
            for (int j = 0; j < KPL; ++j) { c_gt += key[j] > T; c_eq += key[j] == T; }
        }
        c_gt = team_sum<WARPS>(c_gt, xch, wit, lane, flip);
        c_eq = team_sum<WARPS>(c_eq, xch, wit, lane, flip);
        const uint32_t want_eq = (uint32_t)K - c_gt;  // >= 1
        if (c_eq > want_eq) {
            for (int bit = 31; bit >= 0; --bit) {
                const uint32_t cand = L | (1u << bit);
                uint32_t c = 0;
                if (STREAM) { for (int j = 0; j < n_j; ++j) c += (key_at(j) == T) && (~(uint32_t)(j * TEAM + t) >= cand); }
                else {
#pragma unroll
                    for (int j = 0; j < KPL; ++j) c += (key[j] == T) && (~(uint32_t)(j * TEAM + t) >= cand);
                }
                if (team_sum<WARPS>(c, xch, wit, lane, flip) >= want_eq) L = cand;
            }
        }
    } else {
        T = 0;  // at most K candidates: every one of them is taken (the compaction below tests key != 0)
    }
    // compaction of the survivors (at most K <= 64) into sel[team][]
    auto consider = [&](int j) {
        const uint32_t k = key_at(j);
        const uint32_t e = (uint32_t)(j * TEAM + t);
        const bool take = (n_cand > K) ? (k > T || (k == T && ~e >= L)) : (k != 0u);
        const uint32_t m = __ballot_sync(0xffffffffu, take);
        if (m) {
            uint32_t base = 0;
            if (lane == 0) base = atomicAdd(&n_sel[team], (uint32_t)__popc(m));
            base = __shfl_sync(0xffffffffu, base, 0);
            const uint32_t slot = base + __popc(m & ((1u << lane) - 1u));
            if (take && slot < 64) sel[team][slot] = ((unsigned long long)k << 32) | (unsigned long long)(~e);
        }
    };
    if (STREAM) { for (int j = 0; j < n_j; ++j) consider(j); }
    else {
#pragma unroll
        for (int j = 0; j < KPL; ++j) consider(j);
    }
    if (WARPS > 1) __syncthreads(); else __syncwarp();
    if (wit != 0) return;
    // bitonic sort of 64 keys, descending, two per lane (element i = lane + 32*j)
    unsigned long long v0 = sel[team][lane], v1 = sel[team][lane + 32];
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
    const int h = row_id / R;
    const int64_t out0 = (int64_t)row_id * K;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const int s = lane + 32 * j;
        if (s >= K) continue;
        const unsigned long long kv = j ? v1 : v0;
        const int32_t b = kv ? (int32_t)(~(uint32_t)kv) : -1;
        if (block_idx) block_idx[out0 + s] = b;
        ptr_table[out0 + s] = (b < 0) ? -1 : __ldg(page_map + (int64_t)h * max_blocks + b);
    }
}

int32_t launch_topk(const Cache* c, const float* scores, int32_t R, int64_t n_b, int64_t n_cand, int32_t K,
                    int32_t* block_idx, int32_t* ptr_table, cudaStream_t s)
{
    const int32_t n_rows = c->H * R;
    const int32_t nc = (int32_t)n_cand;
    const int32_t* pm = (const int32_t*)c->page_map;
#define OMNIMEM_TOPK(KPL, WARPS, STREAM)                                                                                   \
    launch_pdl(topk_kernel<KPL, WARPS, STREAM>, dim3((unsigned)ceil_div64(n_rows, 8 / WARPS)), dim3(TOPK_THREADS), 0, s, \
               scores, pm, n_rows, R, n_b, nc, K, c->max_blocks, block_idx, ptr_table)
    if (nc <= 32 * 16) OMNIMEM_TOPK(16, 1, false);
    else if (nc <= 32 * 32) OMNIMEM_TOPK(32, 1, false);
    else if (nc <= 32 * 48) OMNIMEM_TOPK(48, 1, false);
    else if (nc <= 32 * 64) OMNIMEM_TOPK(64, 1, false);
    else if (nc <= 256 * 16) OMNIMEM_TOPK(16, 8, false);
    else if (nc <= 256 * 40) OMNIMEM_TOPK(40, 8, false);
    else if (nc <= 256 * 64) OMNIMEM_TOPK(64, 8, false);
    else OMNIMEM_TOPK(1, 8, true);
#undef OMNIMEM_TOPK
    count_launch();
    return check_launch("topk");
}

}  // namespace omnimem
