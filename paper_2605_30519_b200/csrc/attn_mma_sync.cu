// a6-a8, portable kernel: Per-Head Scattered KV Access attention with warp-level mma.sync tiles.
// This is the bring-up kernel (any supported shape: D in {64,128}, B in {64,128}, any G_q, K);
// the tcgen05/TMEM kernel in attn_tcgen05.cu is the fast path.  DESIGN.md section 6.4.
//
// One CTA = 64 query rows of one head (4 warps x 16 rows).  KV arrives one 64-token slot at a time
// (attn_schedule.cuh), double-buffered with cp.async into XOR-swizzled shared memory; pages are read
// in place through the pointer table, no union buffer exists.  Online softmax as in Algorithm 1
// (PAPER.md:382-419), one state per row; GATED mode finalises the SLC branch before the SWA branch.
#include "attn_schedule.cuh"
#include "common.cuh"

namespace omnimem {

struct MmaSyncArgs {
    AttnGeom g;
    const __nv_bfloat16 *q, *k_cur, *v_cur, *k_pages, *v_pages;
    int64_t stride_tok, stride_head;
    const int32_t *ptr_table, *page_map;
    const float *gate_slc, *gate_swa;
    __nv_bfloat16* out;
    float* lse_out;
    float scale_log2;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid)
{
    const int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_trans(uint32_t (&r)[4], uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}

// byte offset of 16-byte chunk `ch` of row `row` in a [64][D] bf16 tile, XOR-swizzled
template <int D>
__device__ __forceinline__ uint32_t tile_off(int row, int ch) { return (uint32_t)(row * (D * 2) + ((ch ^ (row & 7)) << 4)); }

template <int D>
__device__ __forceinline__ void load_rows(uint32_t dst, const __nv_bfloat16* src_row0, int64_t row_stride,
                                          int n_valid_rows, int tid)
{
    constexpr int CH = D / 8;
#pragma unroll
    for (int i = 0; i < 64 * CH / 128; ++i) {
        const int idx = tid + i * 128;
        const int row = idx / CH, ch = idx % CH;
        const bool ok = row < n_valid_rows;
        cp_async16(dst + tile_off<D>(row, ch), ok ? (const void*)(src_row0 + (int64_t)row * row_stride + ch * 8) : (const void*)src_row0, ok);
    }
}

template <int D, bool GATED>
__global__ void __launch_bounds__(128)
attn_mma_sync_kernel(const MmaSyncArgs a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int TILE_BYTES = 64 * D * 2;
    const uint32_t sQ = smem_u32(smem);
    const uint32_t sK = sQ + TILE_BYTES;      // 2 stages
    const uint32_t sV = sK + 2 * TILE_BYTES;  // 2 stages
    const AttnGeom& g = a.g;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int h = blockIdx.y, q0 = blockIdx.x * 64;
    const int gq = lane >> 2, tq = lane & 3;

    TileSched ts;
    ts.init(g, h, q0, 64, 1);

    auto issue_tile = [&](int it, int stage) {
        const Slot s = ts.slot(g, a.ptr_table, a.page_map, it);
        const uint32_t dk = sK + stage * TILE_BYTES, dv = sV + stage * TILE_BYTES;
        if (s.kind == SLOT_HIST) {
            load_rows<D>(dk, a.k_pages + (int64_t)s.row * D, D, 64, tid);
            load_rows<D>(dv, a.v_pages + (int64_t)s.row * D, D, 64, tid);
        } else if (s.kind == SLOT_CUR) {
            const int64_t off = (int64_t)h * a.stride_head + (int64_t)s.row * a.stride_tok;
            load_rows<D>(dk, a.k_cur + off, a.stride_tok, s.hi, tid);
            load_rows<D>(dv, a.v_cur + off, a.stride_tok, s.hi, tid);
        } else {
            load_rows<D>(dk, a.k_pages, D, 0, tid);
            load_rows<D>(dv, a.v_pages, D, 0, tid);
        }
    };

    // prologue: Q tile (rows beyond S zero-filled) + first KV slot
    load_rows<D>(sQ, a.q + (int64_t)h * a.stride_head + (int64_t)q0 * a.stride_tok, a.stride_tok, min(64, g.S - q0), tid);
    if (ts.n_slots > 0) issue_tile(0, 0);
    cp_async_commit();

    float o[D / 8][4];
#pragma unroll
    for (int i = 0; i < D / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
    float o_slc[GATED ? D / 8 : 1][4];
    float m_run[2] = {-INFINITY, -INFINITY};
    float l_slc[2] = {0.f, 0.f}, l_swa[2] = {0.f, 0.f};
    float lse_slc_gated[2] = {-INFINITY, -INFINITY};
    bool slc_closed = false;
    const int row_in_tile[2] = {warp * 16 + gq, warp * 16 + gq + 8};

    auto quad_sum = [](float v) {
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        return v;
    };

    for (int it = 0; it < ts.n_slots; ++it) {
        const int stage = it & 1;
        if (it + 1 < ts.n_slots) issue_tile(it + 1, stage ^ 1);
        cp_async_commit();
        cp_async_wait<1>();
        __syncthreads();

        const Slot s = ts.slot(g, a.ptr_table, a.page_map, it);
        const TileRows tr = ts.rows(g, it);
        if (GATED && !tr.is_slc && !slc_closed) {
            // close the SLC branch: o_slc = g_slc * O_slc (0 if the branch is empty, reading A8)
            slc_closed = true;
            const float gs = __ldg(a.gate_slc + h);
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const float l = quad_sum(l_slc[e]);
                const float inv = l > 0.f ? gs / l : 0.f;
                lse_slc_gated[e] = l > 0.f ? (m_run[e] + log2f(l)) * 0.6931471805599453f : -INFINITY;
#pragma unroll
                for (int i = 0; i < D / 8; ++i) {
                    o_slc[GATED ? i : 0][2 * e] = o[i][2 * e] * inv;
                    o_slc[GATED ? i : 0][2 * e + 1] = o[i][2 * e + 1] * inv;
                    o[i][2 * e] = 0.f;
                    o[i][2 * e + 1] = 0.f;
                }
                m_run[e] = -INFINITY;
                l_slc[e] = 0.f;
            }
        }
        const bool warp_active = s.kind != SLOT_NONE && tr.lo < warp * 16 + 16 && tr.hi > warp * 16;
        if (warp_active) {
            const uint32_t kb = sK + stage * TILE_BYTES, vb = sV + stage * TILE_BYTES;
            float sc[8][4];
#pragma unroll
            for (int i = 0; i < 8; ++i) sc[i][0] = sc[i][1] = sc[i][2] = sc[i][3] = 0.f;
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                uint32_t af[4];
                ldsm_x4(af, sQ + tile_off<D>(warp * 16 + (lane & 7) + ((lane >> 3) & 1) * 8, ks * 2 + (lane >> 4)));
#pragma unroll
                for (int nb2 = 0; nb2 < 4; ++nb2) {
                    uint32_t bf[4];
                    ldsm_x4(bf, kb + tile_off<D>((nb2 * 2 + (lane >> 4)) * 8 + (lane & 7), ks * 2 + ((lane >> 3) & 1)));
                    mma_bf16(sc[nb2 * 2], af, bf[0], bf[1]);
                    mma_bf16(sc[nb2 * 2 + 1], af, bf[2], bf[3]);
                }
            }
            // mask + online softmax (scores in log2 units: t = s * sigma * log2(e))
            float mx[2] = {-INFINITY, -INFINITY};
#pragma unroll
            for (int nb = 0; nb < 8; ++nb)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int col = nb * 8 + 2 * tq + (e & 1);
                    const int row = row_in_tile[e >> 1];
                    const bool ok = col >= s.lo && col < s.hi && row >= tr.lo && row < tr.hi;
                    const float t = ok ? sc[nb][e] * a.scale_log2 : -INFINITY;
                    sc[nb][e] = t;
                    mx[e >> 1] = fmaxf(mx[e >> 1], t);
                }
            float alpha[2], rs[2] = {0.f, 0.f};
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                mx[e] = fmaxf(mx[e], __shfl_xor_sync(0xffffffffu, mx[e], 1));
                mx[e] = fmaxf(mx[e], __shfl_xor_sync(0xffffffffu, mx[e], 2));
                const float m_new = fmaxf(m_run[e], mx[e]);
                const float m_sub = (m_new == -INFINITY) ? 0.f : m_new;
                alpha[e] = exp2f(m_run[e] - m_sub);
                m_run[e] = m_new;
#pragma unroll
                for (int nb = 0; nb < 8; ++nb) {
                    const float p0 = exp2f(sc[nb][2 * e] - m_sub), p1 = exp2f(sc[nb][2 * e + 1] - m_sub);
                    sc[nb][2 * e] = p0;
                    sc[nb][2 * e + 1] = p1;
                    rs[e] += p0 + p1;
                }
                l_slc[e] *= alpha[e];
                l_swa[e] *= alpha[e];
                if (tr.is_slc) l_slc[e] += rs[e]; else l_swa[e] += rs[e];
            }
#pragma unroll
            for (int i = 0; i < D / 8; ++i) {
                o[i][0] *= alpha[0];
                o[i][1] *= alpha[0];
                o[i][2] *= alpha[1];
                o[i][3] *= alpha[1];
            }
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
                uint32_t pf[4];
                pf[0] = pack_bf16(sc[2 * kk][0], sc[2 * kk][1]);
                pf[1] = pack_bf16(sc[2 * kk][2], sc[2 * kk][3]);
                pf[2] = pack_bf16(sc[2 * kk + 1][0], sc[2 * kk + 1][1]);
                pf[3] = pack_bf16(sc[2 * kk + 1][2], sc[2 * kk + 1][3]);
#pragma unroll
                for (int nd2 = 0; nd2 < D / 16; ++nd2) {
                    uint32_t bf[4];
                    ldsm_x4_trans(bf, vb + tile_off<D>(kk * 16 + ((lane >> 3) & 1) * 8 + (lane & 7), nd2 * 2 + (lane >> 4)));
                    mma_bf16(o[nd2 * 2], pf, bf[0], bf[1]);
                    mma_bf16(o[nd2 * 2 + 1], pf, bf[2], bf[3]);
                }
            }
        }
        __syncthreads();
    }
    cp_async_wait<0>();

    // epilogue (a8): normalise, fuse, store bf16; optional natural-log LSE per branch
    const float g_swa = GATED ? __ldg(a.gate_swa + h) : 1.f;
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const int srow = q0 + row_in_tile[e];
        const float ls = quad_sum(l_slc[e]), lw = quad_sum(l_swa[e]);
        float inv, lse0, lse1;
        if (GATED) {
            if (!slc_closed) {  // no SWA tile at all cannot happen (the current chunk is never empty)
                lse_slc_gated[e] = -INFINITY;
            }
            inv = lw > 0.f ? g_swa / lw : 0.f;
            lse0 = lse_slc_gated[e];
            lse1 = lw > 0.f ? (m_run[e] + log2f(lw)) * 0.6931471805599453f : -INFINITY;
        } else {
            const float l = ls + lw;
            inv = l > 0.f ? 1.f / l : 0.f;
            lse0 = ls > 0.f ? (m_run[e] + log2f(ls)) * 0.6931471805599453f : -INFINITY;
            lse1 = lw > 0.f ? (m_run[e] + log2f(lw)) * 0.6931471805599453f : -INFINITY;
        }
        if (srow < g.S) {
            __nv_bfloat16* dst = a.out + ((int64_t)h * g.S + srow) * D;
#pragma unroll
            for (int i = 0; i < D / 8; ++i) {
                float x0 = o[i][2 * e] * inv, x1 = o[i][2 * e + 1] * inv;
                if (GATED) {
                    x0 += o_slc[GATED ? i : 0][2 * e];
                    x1 += o_slc[GATED ? i : 0][2 * e + 1];
                }
                *reinterpret_cast<uint32_t*>(dst + i * 8 + 2 * tq) = pack_bf16(x0, x1);
            }
            if (a.lse_out && tq == 0) {
                a.lse_out[(int64_t)h * g.S + srow] = lse0;
                a.lse_out[(int64_t)g.H * g.S + (int64_t)h * g.S + srow] = lse1;
            }
        }
    }
}

AttnGeom make_attn_geom(const Cache* c, int32_t n_q, const omnimem_attn_params_t& p)
{
    AttnGeom g;
    g.H = c->H;
    g.S = n_q;
    g.B = c->B;
    g.K = p.top_k;
    g.G = p.group_tokens;
    g.R = (int32_t)ceil_div64(n_q, p.group_tokens);
    g.max_blocks = c->max_blocks;
    g.spb = c->B / 64;
    g.n_hist = c->n_hist;
    g.n_b = (int32_t)ceil_div64(c->n_hist, c->B);
    g.last_len = g.n_b > 0 ? (int32_t)(c->n_hist - (int64_t)(g.n_b - 1) * c->B) : c->B;
    int64_t win_start = c->n_hist - p.window_tokens;
    if (win_start < 0) win_start = 0;
    if (p.window_tokens == 0) win_start = c->n_hist;
    g.win_start = win_start;
    g.first_win_blk = (int32_t)(win_start / c->B);
    g.n_win_slots = (win_start < c->n_hist) ? g.spb * (g.n_b - g.first_win_blk) : 0;
    g.n_cur_slots = (int32_t)ceil_div64(n_q, 64);
    g.slc_slots = p.top_k * g.spb;
    return g;
}

int32_t launch_attn_mma_sync(const AttnArgs& x)
{
    const Cache* c = x.cache;
    MmaSyncArgs a;
    a.g = make_attn_geom(c, x.n_q, x.p);
    a.q = (const __nv_bfloat16*)x.q;
    a.k_cur = (const __nv_bfloat16*)x.k_cur;
    a.v_cur = (const __nv_bfloat16*)x.v_cur;
    a.k_pages = c->k_pages;
    a.v_pages = c->v_pages;
    a.stride_tok = x.stride_tok;
    a.stride_head = x.stride_head;
    a.ptr_table = x.ptr_table;
    a.page_map = c->page_map;
    a.gate_slc = x.gate_slc;
    a.gate_swa = x.gate_swa;
    a.out = (__nv_bfloat16*)x.out;
    a.lse_out = x.lse_out;
    a.scale_log2 = x.p.softmax_scale * 1.4426950408889634f;
    dim3 grid((unsigned)ceil_div64(x.n_q, 64), (unsigned)c->H);
    const bool gated = x.p.fuse_mode == OMNIMEM_FUSE_GATED;
    const int smem = 5 * 64 * c->D * 2;
#define OMNIMEM_LAUNCH(DD, GG)                                                                                   \
    do {                                                                                                         \
        cudaError_t e = cudaFuncSetAttribute(attn_mma_sync_kernel<DD, GG>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));    \
        attn_mma_sync_kernel<DD, GG><<<grid, 128, smem, x.stream>>>(a);                                          \
    } while (0)
    if (c->D == 128) {
        if (gated) OMNIMEM_LAUNCH(128, true); else OMNIMEM_LAUNCH(128, false);
    } else {
        if (gated) OMNIMEM_LAUNCH(64, true); else OMNIMEM_LAUNCH(64, false);
    }
#undef OMNIMEM_LAUNCH
    count_launch();
    return check_launch("sparse_attn(mma_sync)");
}

}  // namespace omnimem
