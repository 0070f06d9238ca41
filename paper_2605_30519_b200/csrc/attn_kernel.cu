// a6-a8: Per-Head Scattered KV Access attention (Alg. 1 step 2) fused with the sliding-window
// branch, the current chunk, the compression branch and the gate fusion of Eq. 1 -- ONE persistent kernel
// for sm_100a: TMA-gathered K/V pages, tcgen05.mma tiles, TMEM accumulators.  DESIGN.md section 6.5.
//
// Work decomposition: attn_plan.cuh (units of two 128-row query tiles, 64-token steps, a work tape cut evenly over the
// CTAs, pieces merged through the workspace).  What one CTA does with a piece:
//
//   warp 8      TMA producer: walks the piece's steps, resolves every step's K/V source (page_map for the window,
//               ptr_table for the selected blocks, the current chunk, the compressed cache) 32 steps at a time (one step
//               per lane, so the table reads of a batch are in flight together) and issues ONE 16 KB box per K or V
//               stage into a ring of NST stages.  No union buffer exists: pages are read in place.  The wait on
//               omnimem_select (griddepcontrol.wait) sits right before the first ptr_table read.
//   warp 9, 10  MMA issuers (one elected thread per query tile).  Per step and tile i:  S_i = Q_i K^T  (SS, M128 N64 K16 x D/16)
//               into one of the tile's two S buffers, and  O_i += P_i V  (P from TMEM, V MN-major from smem, M128 N=D
//               K16 x 4).  The K stage and the V stage of a shared step feed BOTH tiles: the SM ingests each window /
//               current-chunk byte once per 256 query rows.  QK of step s+1 is issued before PV of step s.
//   warps 0-3   softmax warpgroup of tile 0, warps 4-7 of tile 1 (thread = query row = TMEM lane): Algorithm 1's online
//               softmax on the tile's own running max / sums / accumulator -- no state is shared between warpgroups.
//               P_i overwrites the first 32 columns of the S buffer it was computed from; the tensor pipe executes in
//               issue order, so QK of step s+2 (same buffer) cannot overtake PV of step s.
//
// TMEM (512 columns): O_0 [0,D) O_1 [D,2D) S_00 S_01 S_10 S_11 (64 columns each) from column 2D.
#include <cuda.h>
#include <stdio.h>
#include <stdlib.h>

#include <atomic>

#include "attn_plan.cuh"
#include "common.cuh"

namespace omnimem {

namespace dq {

constexpr int M_TILE = 128;
constexpr int STEP = 64;
constexpr int NST = 9;           // K/V stages in the ring
constexpr int META_RING = 128;  // a resolved batch (32 steps) + the ring's lead over the softmax warps stays far below it
constexpr int SLOT_RING = 64;
constexpr int THREADS = 384;
constexpr float RESCALE_LOG2 = 8.0f;

enum Src : int32_t { SRC_NONE = 0, SRC_POOL = 1, SRC_CUR = 2, SRC_CMP = 3 };

struct StepSlot {
    int32_t src, row;      // POOL / CMP: first row in the pool viewed as [rows][D]; CUR: first token
    int32_t lo, hi;        // valid tokens [lo, hi) of the 64
    int32_t rlo, rhi;      // query rows of the tile (relative) that attend to this step
    int32_t branch, pad;   // 0 CMP, 1 SLC, 2 SWA: which row sum the step feeds
};
struct StepMeta {          // what a softmax warpgroup needs to know about a step: 16 bytes
    int16_t lo, hi, rlo, rhi;
    int32_t branch, pad;
};

template <int D>
struct Smem {
    static constexpr int Q_BYTES = M_TILE * D * 2;
    static constexpr int ST_BYTES = STEP * D * 2;
    alignas(1024) unsigned char q[2][Q_BYTES];
    alignas(1024) unsigned char st[NST][ST_BYTES];
    alignas(8) unsigned long long q_full[2], q_free;
    unsigned long long kv_full[NST], kv_empty[NST];
    unsigned long long s_full[2][2], p_full[2][2], pv_done[2][2], o_free[2];
    uint32_t tmem_base;
    int32_t is_last[2];
    StepMeta meta[META_RING][2];
    int2 slots[SLOT_RING][2];  // (src, row) of a step's K/V stage, per tile
};

struct Args {
    AttnPlan p;
    const int32_t *ptr_table, *page_map;
    const float *gate_cmp, *gate_slc, *gate_swa;  // [H] fp32 each (GATED); NULL in JOINT mode
    __nv_bfloat16* out;
    float* lse;          // nullable: [n_lse][H][S] natural-log LSE per branch, rows (slc, swa) or (cmp, slc, swa)
    int32_t n_lse;
    int32_t* counters;   // [n_units][2], zero between launches (the merging piece resets its counter)
    float* partial;      // [n_units][max_pieces][2][128][D + 4] fp32
    float scale_log2;
    int32_t pool_rows;   // rows of the page pools: a row coordinate at / after this is out of bounds -> zero fill
    float rescale_thr;
};

// ------------------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ uint64_t global_ns()
{
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// Bounded wait: a protocol bug traps (the launch then reports an error) instead of hanging the GPU.  The bound is elapsed
// time (10 s of %globaltimer, looked at every 4096 failed probes), so a legitimate wait under a profiler's replay, a
// sanitizer or time-slicing never comes near it.
__device__ __forceinline__ void mbar_wait_addr(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) return;
    uint64_t t0 = 0;
    for (uint32_t spins = 1;; ++spins) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if ((spins & 4095u) == 0) {
            const uint64_t t = global_ns();
            if (t0 == 0) t0 = t;
            else if (t - t0 > 10000000000ull) __trap();
        }
    }
}
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity) { mbar_wait_addr(smem_u32(bar), parity); }
// Blocking wait on TWO barriers whose first probes are in flight together (one probe latency, not two).
__device__ __forceinline__ void mbar_wait2(uint32_t bar0, uint32_t par0, uint32_t bar1, uint32_t par1)
{
    uint32_t ok0, ok1;
    asm volatile(
        "{\n\t.reg .pred p, q;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%2], %3;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 q, [%4], %5;\n\t"
        "selp.u32 %0, 1, 0, p;\n\tselp.u32 %1, 1, 0, q;\n\t}"
        : "=r"(ok0), "=r"(ok1) : "r"(bar0), "r"(par0), "r"(bar1), "r"(par1) : "memory");
    if (!ok0) mbar_wait_addr(bar0, par0);
    if (!ok1) mbar_wait_addr(bar1, par1);
}

__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred P;\n\t"
        "elect.sync _|P, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, P;\n\t}"
        : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, void* bar, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, void* bar, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// UMMA shared-memory descriptor, SWIZZLE_128B (layout type 2), version 1.  Operand tiles are [D/64 halves][rows][128 B]:
//   K-major (Q, K):  rows of 128 B (64 bf16 of D), 8-row groups 1024 B apart (SBO); LBO unused (1).
//   MN-major (V):    same bytes; LBO = distance between the two 64-wide halves of D, SBO = 8-token groups (1024 B).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// instruction descriptor, kind::f16: bf16 x bf16 -> fp32, M = 128
__host__ __device__ constexpr uint32_t idesc(uint32_t n, bool b_mn_major)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | (b_mn_major ? (1u << 16) : 0u) | ((n >> 3) << 17) | ((128u >> 4) << 24);
}

// S_i = Q_i K^T for one 64-token stage: D/16 MMAs (M128 N64 K16) + the commits, as ONE asm block (nothing but descriptor
// adds between the MMAs).  kv_empty takes two arrivals per use: `twice` = the stage is private to this tile, so both come from here.
template <int D>
__device__ __forceinline__ void qk_batch(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t bar_s_full, uint32_t bar_empty, bool twice)
{
    constexpr uint32_t ID = idesc(64, false);
    if constexpr (D == 128) {
        asm volatile(
            "{\n\t.reg .pred pa, pr;\n\t.reg .b64 a, b;\n\t"
            "setp.ne.b32 pr, %6, 0;\n\t"
            "setp.ne.b32 pa, 0, 0;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, pa;\n\t"
            "setp.eq.b32 pa, 0, 0;\n\t"
            "add.s64 a, %1, 2;\n\tadd.s64 b, %2, 2;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "add.s64 a, %1, 4;\n\tadd.s64 b, %2, 4;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "add.s64 a, %1, 6;\n\tadd.s64 b, %2, 6;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "add.s64 a, %1, 1024;\n\tadd.s64 b, %2, 512;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "add.s64 a, %1, 1026;\n\tadd.s64 b, %2, 514;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "add.s64 a, %1, 1028;\n\tadd.s64 b, %2, 516;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "add.s64 a, %1, 1030;\n\tadd.s64 b, %2, 518;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%4];\n\t"
            "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t"
            "@pr tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t}"
            :: "r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(ID), "r"(bar_s_full), "r"(bar_empty), "r"((uint32_t)twice)
            : "memory");
    } else {
        asm volatile(
            "{\n\t.reg .pred pa, pr;\n\t.reg .b64 a, b;\n\t"
            "setp.ne.b32 pr, %6, 0;\n\t"
            "setp.ne.b32 pa, 0, 0;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, pa;\n\t"
            "setp.eq.b32 pa, 0, 0;\n\t"
            "add.s64 a, %1, 2;\n\tadd.s64 b, %2, 2;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "add.s64 a, %1, 4;\n\tadd.s64 b, %2, 4;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "add.s64 a, %1, 6;\n\tadd.s64 b, %2, 6;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
            "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%4];\n\t"
            "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t"
            "@pr tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t}"
            :: "r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(ID), "r"(bar_s_full), "r"(bar_empty), "r"((uint32_t)twice)
            : "memory");
    }
}
// O_i (+)= P_i V for one 64-token stage: 4 MMAs (M128 N=D K16), P from TMEM (8 columns per K step), V MN-major from smem
// (16 tokens = 2048 B per step: 128 descriptor units).
template <int D>
__device__ __forceinline__ void pv_batch(uint32_t d_tmem, uint32_t p_tmem, uint64_t vdesc, uint32_t accumulate, uint32_t bar_pv_done,
                                         uint32_t bar_empty, bool twice)
{
    constexpr uint32_t ID = idesc(D, true);
    asm volatile(
        "{\n\t.reg .pred pa, pr;\n\t.reg .b64 b;\n\t.reg .b32 a;\n\t"
        "setp.ne.b32 pr, %7, 0;\n\t"
        "setp.ne.b32 pa, %3, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %4, pa;\n\t"
        "setp.eq.b32 pa, 0, 0;\n\t"
        "add.s32 a, %1, 8;\n\tadd.s64 b, %2, 128;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %4, pa;\n\t"
        "add.s32 a, %1, 16;\n\tadd.s64 b, %2, 256;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %4, pa;\n\t"
        "add.s32 a, %1, 24;\n\tadd.s64 b, %2, 384;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %4, pa;\n\t"
        "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t"
        "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%6];\n\t"
        "@pr tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%6];\n\t}"
        :: "r"(d_tmem), "r"(p_tmem), "l"(vdesc), "r"(accumulate), "r"(ID), "r"(bar_pv_done), "r"(bar_empty), "r"((uint32_t)twice)
        : "memory");
}
__device__ __forceinline__ void commit_to(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32])
{
    uint32_t* r = reinterpret_cast<uint32_t*>(v);
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
          "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]),
          "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]),
          "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
        : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16])
{
    uint32_t* r = reinterpret_cast<uint32_t*>(v);
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
          "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ uint64_t f2(float lo, float hi)
{
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unf2(uint64_t v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c)
{
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b)
{
    uint64_t r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ float max3(float a, float b, float c)
{
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
__device__ __forceinline__ uint32_t pack2(float lo, float hi)
{
    uint32_t r;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}
__device__ __forceinline__ void wg_sync(int tile) { asm volatile("bar.sync %0, 128;" ::"r"(tile + 1) : "memory"); }

// ------------------------------------------------------------------------------------- step sources
// Where tile i's 64 KV tokens of unit-local step s come from.  Returns false when the tile sits the step out.
__device__ __forceinline__ bool resolve_step(const Args& a, const AttnPiece& pc, int s, int i, StepSlot& sl)
{
    const AttnPlan& p = a.p;
    const AttnGeom& g = p.g;
    sl.src = SRC_NONE;
    sl.row = 0;
    sl.lo = 0;
    sl.hi = 0;
    sl.rlo = 0;
    sl.rhi = M_TILE;
    sl.branch = 2;
    sl.pad = 0;
    if (i >= pc.n_tiles) return false;
    if (s < p.n_cmp) {  // compressed tokens [64 s, 64 s + 64) of head h: rows of the pooled_k / pooled_v pools
        sl.branch = 0;
        sl.src = SRC_CMP;
        sl.row = pc.h * g.max_blocks + s * 64;
        sl.hi = min(64, g.n_b - s * 64);
        return true;
    }
    int w = s - p.n_cmp;
    if (w < p.n_swa) {
        if (w < g.n_win_slots) {  // window: history blocks through page_map, token-masked at both ends
            const int b = g.first_win_blk + w / g.spb, sub = w % g.spb;
            const int64_t base = (int64_t)b * g.B + sub * 64;
            const int lo = (int)max((int64_t)0, g.win_start - base);
            const int hi = (int)min((int64_t)64, g.n_hist - base);
            if (lo < hi) {
                const int32_t page = __ldg(a.page_map + (int64_t)pc.h * g.max_blocks + b);
                sl.src = SRC_POOL;
                sl.row = (int32_t)(((int64_t)pc.h * g.max_blocks + page) * g.B + sub * 64);
                sl.lo = lo;
                sl.hi = hi;
            }
            return true;
        }
        w -= g.n_win_slots;  // current chunk, 64 tokens at a time (no mask inside the chunk)
        sl.src = SRC_CUR;
        sl.row = w * 64;
        sl.hi = min(g.S - w * 64, 64);
        return true;
    }
    const int v = w - p.n_swa;  // SLC: group r's K selected blocks through ptr_table (Alg. 1: entry < 0 => skip)
    if (v >= pc.n_slc[i]) return false;
    sl.branch = 1;
    const int r = pc.g_first[i] + v / g.slc_slots, j = v % g.slc_slots;
    const int q0 = (pc.qt0 + i) * M_TILE;
    sl.rlo = max(r * g.G - q0, 0);
    sl.rhi = min(min((r + 1) * g.G, g.S) - q0, M_TILE);
    const int t = j / g.spb, sub = j % g.spb;
    const int32_t page = __ldg(a.ptr_table + ((int64_t)pc.h * g.R + r) * g.K + t);
    if (page < 0) return true;
    int len = g.B;
    if (g.last_len < g.B && page == __ldg(a.page_map + (int64_t)pc.h * g.max_blocks + g.n_b - 1)) len = g.last_len;
    const int hi = min(len - sub * 64, 64);
    if (hi <= 0) return true;
    sl.src = SRC_POOL;
    sl.row = (int32_t)(((int64_t)pc.h * g.max_blocks + page) * g.B + sub * 64);
    sl.hi = hi;
    return true;
}

// ------------------------------------------------------------------------------------- kernel
template <int D>
__global__ void __launch_bounds__(THREADS, 1)
attn_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_kcur,
            const __grid_constant__ CUtensorMap tm_vcur, const __grid_constant__ CUtensorMap tm_kpool,
            const __grid_constant__ CUtensorMap tm_vpool, const __grid_constant__ CUtensorMap tm_kcmp,
            const __grid_constant__ CUtensorMap tm_vcmp, const Args a)
{
    using SM = Smem<D>;
    constexpr uint32_t TM_O = 0, TM_S = 2 * D;  // TMEM columns: O_i at i * D, S buffer (i, b) at TM_S + (2 i + b) * 64
    constexpr int ROW_F = D + 4;                // floats per row of a partial: O[D], m, l_cmp, l_slc, l_swa
    extern __shared__ unsigned char smem_raw[];
    SM& sm = *reinterpret_cast<SM*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    const AttnPlan& p = a.p;
    const AttnGeom& g = p.g;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        mbar_init(&sm.q_full[0], 1);
        mbar_init(&sm.q_full[1], 1);
        mbar_init(&sm.q_free, 2);
        for (int i = 0; i < NST; ++i) { mbar_init(&sm.kv_full[i], 1); mbar_init(&sm.kv_empty[i], 2); }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&sm.o_free[i], 128);
            for (int b = 0; b < 2; ++b) { mbar_init(&sm.s_full[i][b], 1); mbar_init(&sm.p_full[i][b], 128); mbar_init(&sm.pv_done[i][b], 1); }
        }
        fence_barrier_init();
    }
    if (warp == 9) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sm.tmem_base)), "r"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    pdl_launch_dependents();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = sm.tmem_base;
    PieceIter it;  // every role walks the CTA's pieces with its own iterator
    it.init(p, blockIdx.x);
    AttnPiece pc;
    // No griddepcontrol.wait here: Q, the current chunk and the cached pages were complete before the selection kernels were
    // launched, so the window / current-chunk steps run while omnimem_select is still in flight.  The producer waits right
    // before its first ptr_table read, the softmax warps before they touch global memory (output, partials, counters).

    const int off_slc = p.n_cmp + p.n_swa;  // first SLC step of a unit
    if (warp >= 8) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 80;");
        if (warp == 8) {
            // ===================================================================== TMA producer
            // All 32 lanes resolve step sources in batches (one step per lane); lane 0 alone turns resolved steps into TMA
            // boxes, in the MMA issuer's consumption order: K(s0), then for every step s: K(s + 1), V(s).
            if (lane == 0) {
                prefetch_tmap(&tm_q); prefetch_tmap(&tm_kcur); prefetch_tmap(&tm_vcur); prefetch_tmap(&tm_kpool); prefetch_tmap(&tm_vpool);
                if (p.n_cmp > 0) { prefetch_tmap(&tm_kcmp); prefetch_tmap(&tm_vcmp); }
            }
            uint32_t stg = 0, eph = 1;   // ring stage of the next box and the kv_empty parity to wait for (first pass: free)
            uint32_t gbase = 0;          // meta-ring index of the piece's first step
            uint32_t n_units_loaded = 0;
            bool waited = false;
            const uint32_t b_full = smem_u32(&sm.kv_full[0]), b_empty = smem_u32(&sm.kv_empty[0]);
            auto issue = [&](int2 sl, bool is_v, int h) {  // lane 0
                mbar_wait_addr(b_empty + stg * 8, eph);
                const uint32_t bar = b_full + stg * 8;
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((uint32_t)SM::ST_BYTES) : "memory");
                void* dst = sm.st[stg];
                void* barp = &sm.kv_full[stg];
                if (sl.x == SRC_CUR) tma_load_4d(dst, is_v ? &tm_vcur : &tm_kcur, barp, 0, sl.y, 0, h);
                else if (sl.x == SRC_CMP) tma_load_3d(dst, is_v ? &tm_vcmp : &tm_kcmp, barp, 0, sl.y, 0);
                else tma_load_3d(dst, is_v ? &tm_vpool : &tm_kpool, barp, 0, sl.x == SRC_POOL ? sl.y : a.pool_rows, 0);
                if (++stg == NST) { stg = 0; eph ^= 1; }
            };
            while (it.next(p, pc)) {
                if (pc.new_unit && lane == 0) {
                    if (n_units_loaded > 0) mbar_wait(&sm.q_free, (n_units_loaded - 1) & 1);  // every QK^T of the previous unit has completed
                    mbar_expect_tx(&sm.q_full[0], SM::Q_BYTES);
                    tma_load_4d(sm.q[0], &tm_q, &sm.q_full[0], 0, pc.qt0 * M_TILE, 0, pc.h);
                    if (pc.n_tiles == 2) {
                        mbar_expect_tx(&sm.q_full[1], SM::Q_BYTES);
                        tma_load_4d(sm.q[1], &tm_q, &sm.q_full[1], 0, (pc.qt0 + 1) * M_TILE, 0, pc.h);
                    }
                }
                if (pc.new_unit) ++n_units_loaded;
                const bool dual = pc.n_tiles == 2;
                // the steps in which at least one tile takes part form a prefix of [s0, s1): [s0, s_act)
                const int n_slc_any = max(pc.n_slc[0], pc.n_slc[1]);
                const int s_act = min(pc.s1, off_slc + n_slc_any);
                int resolved = pc.s0;  // steps [s0, resolved) sit in the slot / meta rings
                int s = pc.s0;
                bool k_first = true;
                while (s < s_act) {
                    // resolve the next batch when iteration s needs it (it reads the slots of steps s and s + 1)
                    if (resolved < s_act && resolved <= s + 1) {
                        const int n = min(32, s_act - resolved);
                        if (!waited && resolved + n > off_slc) {
                            pdl_wait();  // the batch reaches the SLC steps: ptr_table must be final (omnimem_select has completed)
                            waited = true;
                        }
                        if (lane < n) {
                            const int sr = resolved + lane;
                            StepSlot s0, s1;
                            resolve_step(a, pc, sr, 0, s0);
                            resolve_step(a, pc, sr, 1, s1);
                            sm.slots[sr % SLOT_RING][0] = make_int2(s0.src, s0.row);
                            sm.slots[sr % SLOT_RING][1] = make_int2(s1.src, s1.row);
                            const uint32_t mi = (gbase + (uint32_t)(sr - pc.s0)) % META_RING;
                            StepMeta m0, m1;
                            m0.lo = (int16_t)s0.lo; m0.hi = (int16_t)s0.hi; m0.rlo = (int16_t)s0.rlo; m0.rhi = (int16_t)s0.rhi; m0.branch = s0.branch; m0.pad = 0;
                            m1.lo = (int16_t)s1.lo; m1.hi = (int16_t)s1.hi; m1.rlo = (int16_t)s1.rlo; m1.rhi = (int16_t)s1.rhi; m1.branch = s1.branch; m1.pad = 0;
                            sm.meta[mi][0] = m0;
                            sm.meta[mi][1] = m1;
                        }
                        resolved += n;
                        __syncwarp();
                    }
                    // lane 0 emits every iteration whose slots are resolved: iteration t needs step t + 1 (or the end of the piece)
                    const int s_end = (resolved >= s_act) ? s_act : resolved - 1;
                    if (lane == 0) {
                        for (int t = s; t < s_end; ++t) {
                            // activity of steps t and t + 1 (tile 0 / tile 1 / shared stage)
                            if (k_first) {  // K of the piece's first step
                                const bool sh = dual && (t < off_slc || pc.slc_shared);
                                const int v = t - off_slc;
                                const bool a0 = v < pc.n_slc[0], a1 = dual && v < pc.n_slc[1];
                                const int2 x0 = sm.slots[t % SLOT_RING][0], x1 = sm.slots[t % SLOT_RING][1];
                                if (sh) issue(x0, false, pc.h);
                                else { if (a0) issue(x0, false, pc.h); if (a1) issue(x1, false, pc.h); }
                                k_first = false;
                            }
                            if (t + 1 < s_act) {
                                const int u = t + 1, v = u - off_slc;
                                const bool sh = dual && (u < off_slc || pc.slc_shared);
                                const bool a0 = v < pc.n_slc[0], a1 = dual && v < pc.n_slc[1];
                                const int2 x0 = sm.slots[u % SLOT_RING][0], x1 = sm.slots[u % SLOT_RING][1];
                                if (sh) issue(x0, false, pc.h);
                                else { if (a0) issue(x0, false, pc.h); if (a1) issue(x1, false, pc.h); }
                            }
                            {
                                const int v = t - off_slc;
                                const bool sh = dual && (t < off_slc || pc.slc_shared);
                                const bool a0 = v < pc.n_slc[0], a1 = dual && v < pc.n_slc[1];
                                const int2 x0 = sm.slots[t % SLOT_RING][0], x1 = sm.slots[t % SLOT_RING][1];
                                if (sh) issue(x0, true, pc.h);
                                else { if (a0) issue(x0, true, pc.h); if (a1) issue(x1, true, pc.h); }
                            }
                        }
                    }
                    s = s_end;
                    __syncwarp();
                }
                gbase += (uint32_t)(s_act > pc.s0 ? s_act - pc.s0 : 0);
            }
            if (!waited) pdl_wait();  // grid completion stays ordered behind the previous grid even without SLC steps
        } else if (warp == 9 || warp == 10) {
            // ===================================================================== MMA issuers
            // Warp 9 issues the batches of query tile 0, warp 10 those of tile 1 (one elected thread each).  The tensor pipe
            // accepts only a few MMAs ahead, so an issuing thread runs in lockstep with the pipe and every barrier probe it makes
            // between two batches would idle it -- with one issuer per tile, the probes of one thread overlap the other
            // thread's MMAs.  A tile's QK^T and PV batches stay in ONE thread: P_i aliases S_i, and it is program order in
            // the issuing thread that keeps QK of step s + 2 behind PV of step s.  Both threads walk the same stage ring; a
            // stage is released by two commits (one per reader of a shared stage, both from the owner of a private one).
            if (elect_one()) {
                const int I = warp == 9 ? 0 : 1;
                const uint32_t b_full = smem_u32(&sm.kv_full[0]), b_empty = smem_u32(&sm.kv_empty[0]);
                const uint32_t b_s_full = smem_u32(&sm.s_full[I][0]), b_p_full = smem_u32(&sm.p_full[I][0]);
                const uint32_t b_pv_done = smem_u32(&sm.pv_done[I][0]), b_o_free = smem_u32(&sm.o_free[I]);
                const uint32_t b_q_free = smem_u32(&sm.q_free);
                const uint64_t qd = make_desc(smem_u32(sm.q[I]), 16, 1024);
                const uint64_t kd0 = make_desc(smem_u32(sm.st[0]), 16, 1024);
                const uint64_t vd0 = make_desc(smem_u32(sm.st[0]), STEP * 128, 1024);
                constexpr uint32_t ST_DESC = SM::ST_BYTES >> 4;
                const uint32_t s_tm = tmem + TM_S + (2 * I) * 64, o_tm = tmem + TM_O + I * D;
                uint32_t stg = 0, fph = 0;   // ring stage of the next operand and its kv_full parity
                uint32_t kq = 0, kp = 0;     // QK / PV batches issued (S / P buffer = count & 1, p_full parity = (count >> 1) & 1)
                uint32_t ns = 0, nq = 0;     // softmax states (with at least one PV) closed; Q tiles loaded
#define DQ_RING_NEXT() do { if (++stg == NST) { stg = 0; fph ^= 1; } } while (0)
                while (it.next(p, pc)) {
                    const bool mine = I < pc.n_tiles;
                    if (pc.new_unit && mine) {
                        mbar_wait(&sm.q_full[I], nq & 1);
                        ++nq;
                    }
                    const bool dual = pc.n_tiles == 2;
                    const int n0 = pc.n_slc[0], n1 = pc.n_slc[1];
                    const int s_act = min(pc.s1, off_slc + max(n0, n1));
                    bool first = true;
                    // one stage walk for K (is_v = false) or V: my stage is used, the other tile's private stage is skipped
                    auto qk = [&](int t) {
                        const int v = t - off_slc;
                        const bool a0 = v < n0, a1 = dual && v < n1;
                        const bool sh = dual && (t < off_slc || pc.slc_shared);
                        if (!sh && I == 1 && a0) DQ_RING_NEXT();  // tile 0's private stage comes first
                        if (sh || (I == 0 ? a0 : a1)) {
                            mbar_wait_addr(b_full + stg * 8, fph);
                            tc_fence_after();
                            const uint32_t b = kq & 1;
                            qk_batch<D>(s_tm + b * 64, qd, kd0 + (uint64_t)(stg * ST_DESC), b_s_full + b * 8, b_empty + stg * 8, !sh);
                            ++kq;
                            DQ_RING_NEXT();
                        }
                        if (!sh && I == 0 && a1) DQ_RING_NEXT();  // tile 1's private stage follows
                    };
                    auto pv = [&](int t) {
                        const int v = t - off_slc;
                        const bool a0 = v < n0, a1 = dual && v < n1;
                        const bool sh = dual && (t < off_slc || pc.slc_shared);
                        if (!sh && I == 1 && a0) DQ_RING_NEXT();
                        if (sh || (I == 0 ? a0 : a1)) {
                            const uint32_t b = kp & 1;
                            mbar_wait2(b_full + stg * 8, fph, b_p_full + b * 8, (kp >> 1) & 1);
                            if (first && ns > 0) mbar_wait_addr(b_o_free, (ns - 1) & 1);  // the previous state's O has been read
                            tc_fence_after();
                            pv_batch<D>(o_tm, s_tm + b * 64, vd0 + (uint64_t)(stg * ST_DESC), first ? 0u : 1u, b_pv_done + b * 8, b_empty + stg * 8, !sh);
                            first = false;
                            ++kp;
                            DQ_RING_NEXT();
                        }
                        if (!sh && I == 0 && a1) DQ_RING_NEXT();
                    };
                    // q_free (two arrivals, one per issuer) is committed right behind the unit's last QK^T: it completes when every
                    // MMA this thread issued so far has -- the producer reloads the Q tiles while the last PVs still run
                    if (pc.s0 < s_act) {
                        qk(pc.s0);
                        if (pc.s0 + 1 == s_act && pc.last_of_unit) commit_to(b_q_free);
                        for (int t = pc.s0; t < s_act; ++t) {
                            if (t + 1 < s_act) {
                                qk(t + 1);
                                if (t + 2 == s_act && pc.last_of_unit) commit_to(b_q_free);
                            }
                            pv(t);
                        }
                    } else if (pc.last_of_unit) {
                        commit_to(b_q_free);
                    }
                    if (!first) ++ns;
                }
#undef DQ_RING_NEXT
            }
        }
        __syncwarp();
    } else {
        // ========================================================================= softmax warpgroups
        asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
        const int tile = warp >> 2;                       // the query tile this warpgroup owns
        const int row = (warp & 3) * 32 + lane;           // query row in the tile == TMEM lane
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t o_tmem = tmem + lane_base + TM_O + tile * D;
        const float sl = a.scale_log2;
        uint32_t k = 0;        // active steps of this tile so far (buffer / phase of s_full, p_full, pv_done)
        uint32_t gbase = 0;    // meta-ring index of the piece's first step, as in the producer

        while (it.next(p, pc)) {
            float m = -INFINITY, l3[3] = {0.f, 0.f, 0.f};  // the state's running max (log2 units) and per-branch row sums
            bool any = false;                              // some PV of this state has been issued for this tile
            // this tile takes part in a prefix of the piece's steps: the shared steps and its own SLC steps
            const int s_act = min(pc.s1, off_slc + max(pc.n_slc[0], pc.n_slc[1]));
            const int s_mine = (tile < pc.n_tiles) ? min(pc.s1, off_slc + (tile == 0 ? pc.n_slc[0] : pc.n_slc[1])) : pc.s0;
            for (int s = pc.s0; s < s_mine; ++s) {
                const uint32_t mi = (gbase + (uint32_t)(s - pc.s0)) % META_RING;
                const uint32_t b = k & 1;
                const uint32_t s_tmem = tmem + lane_base + TM_S + (2 * tile + b) * 64;
                mbar_wait(&sm.s_full[tile][b], (k >> 1) & 1);
                tc_fence_after();
                const StepMeta mt = sm.meta[mi][tile];
                const bool row_on = row >= mt.rlo && row < mt.rhi;
                const bool warp_on = __any_sync(0xffffffffu, row_on);
                const bool plain = mt.lo == 0 && mt.hi == 64 && __all_sync(0xffffffffu, row_on);
                float sc[64];
                float (*s2)[32] = reinterpret_cast<float (*)[32]>(sc);
                float mx = -INFINITY;
                if (warp_on) {
                    tmem_ld32(s_tmem, s2[0]);
                    tmem_ld32(s_tmem + 32, s2[1]);
                    tmem_ld_wait();
                    if (!plain) {
#pragma unroll
                        for (int c = 0; c < 64; ++c)
                            if (!(row_on && c >= mt.lo && c < mt.hi)) sc[c] = -INFINITY;
                    }
                    float mx4[4] = {sc[0], sc[1], sc[2], sc[3]};
#pragma unroll
                    for (int c = 4; c < 60; c += 8) {
                        mx4[0] = max3(mx4[0], sc[c], sc[c + 1]);
                        mx4[1] = max3(mx4[1], sc[c + 2], sc[c + 3]);
                        mx4[2] = max3(mx4[2], sc[c + 4], sc[c + 5]);
                        mx4[3] = max3(mx4[3], sc[c + 6], sc[c + 7]);
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) mx4[i] = fmaxf(mx4[i], sc[60 + i]);
                    mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * sl;  // log2 units (sl > 0)
                }
                // lazy rescale (Alg. 1's alpha): keep the stale reference max unless the new max exceeds it by > 2^8
                const bool grow = mx > m + a.rescale_thr;
                if (__any_sync(0xffffffffu, grow)) {
                    const float alpha = grow ? ex2(m - mx) : 1.f;  // m = -inf -> 0
                    if (any) {
                        // every PV of this tile up to the previous step has landed in O (the pipe completes in order); PV of this
                        // step cannot start before this thread's P, so the accumulator is quiescent meanwhile.  (Two barriers per
                        // tile, alternating with the step: QK of step k is issued BEFORE PV of step k - 1, so S_k being ready only
                        // proves PV_{k-2} complete -- a single barrier could be two completions behind, which a parity cannot tell.)
                        mbar_wait(&sm.pv_done[tile][(k - 1) & 1], ((k - 1) >> 1) & 1);
                        tc_fence_after();
#pragma unroll
                        for (int c0 = 0; c0 < D; c0 += 16) {
                            float o[16];
                            tmem_ld16(o_tmem + c0, o);
                            tmem_ld_wait();
                            uint32_t ob[16];
#pragma unroll
                            for (int i = 0; i < 16; ++i) ob[i] = __float_as_uint(o[i] * alpha);
                            tmem_st16(o_tmem + c0, ob);
                        }
                        tmem_st_wait();
                        tc_fence_before();
                    }
                    l3[0] *= alpha;
                    l3[1] *= alpha;
                    l3[2] *= alpha;
                    if (grow) m = mx;
                }
                uint32_t pk[32];
                if (warp_on) {
                    const float m_use = (m == -INFINITY) ? 0.f : m;
                    const uint64_t sl2 = f2(sl, sl), nm2 = f2(-m_use, -m_use);
                    uint64_t rs2[4] = {0ull, 0ull, 0ull, 0ull};
                    // x = s * scale - ref for the whole row first, then one MUFU stream; the sum / bf16 pack of a pair follows its
                    // exponentials LAG pairs later, so the consumers never sit right behind a MUFU result (volatile: keeps this order)
                    constexpr int LAG = 8;
#pragma unroll
                    for (int c = 0; c < 32; ++c) unf2(fma2(f2(sc[2 * c], sc[2 * c + 1]), sl2, nm2), sc[2 * c], sc[2 * c + 1]);
#pragma unroll
                    for (int c = 0; c < 32 + LAG; ++c) {
                        if (c < 32) {
                            asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(sc[2 * c]));
                            asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(sc[2 * c + 1]));
                        }
                        if (c >= LAG) {
                            const int d = c - LAG;
                            uint64_t v;
                            asm volatile("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(sc[2 * d]), "f"(sc[2 * d + 1]));
                            asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(rs2[d & 3]) : "l"(v));
                            asm volatile("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pk[d]) : "f"(sc[2 * d + 1]), "f"(sc[2 * d]));
                        }
                    }
                    float ra, rb;
                    unf2(add2(add2(rs2[0], rs2[1]), add2(rs2[2], rs2[3])), ra, rb);
                    const float rs = ra + rb;
                    if (mt.branch == 0) l3[0] += rs; else if (mt.branch == 1) l3[1] += rs; else l3[2] += rs;
                } else {
#pragma unroll
                    for (int c = 0; c < 32; ++c) pk[c] = 0u;
                }
                // P overwrites the first 32 columns of the S buffer it came from (this thread's S values sit in registers)
                tmem_st32(s_tmem, pk);
                tmem_st_wait();
                tc_fence_before();
                mbar_arrive(&sm.p_full[tile][b]);
                any = true;
                ++k;
            }
            gbase += (uint32_t)(s_act > pc.s0 ? s_act - pc.s0 : 0);
            if (pc.n_tiles <= tile) continue;  // the unit has no second tile: nothing to finish
            // ------------------------------------------------------------------ end of the state: finish or hand over (a8)
            if (any) {
                mbar_wait(&sm.pv_done[tile][(k - 1) & 1], ((k - 1) >> 1) & 1);  // in-order pipe: every PV of this tile has landed
                tc_fence_after();
            }
            pdl_wait();  // everything below touches global memory that the previous grids may still use
            const int srow = (pc.qt0 + tile) * M_TILE + row;
            const int64_t HS = (int64_t)g.H * g.S;
            const float ln2 = 0.6931471805599453f;
            if (pc.npc == 1) {
                // the whole unit was this piece: normalise (GATED: the one branch the piece holds, times its gate) and store
                const float l_all = l3[0] + l3[1] + l3[2];
                float scale = l_all > 0.f ? 1.f / l_all : 0.f;
                if (p.gated) {
                    const float* gp = l3[0] > 0.f ? a.gate_cmp : (l3[1] > 0.f ? a.gate_slc : a.gate_swa);
                    if (gp) scale *= __ldg(gp + pc.h);
                }
#pragma unroll
                for (int c0 = 0; c0 < D; c0 += 32) {
                    float r[32];
                    if (any) {
                        tmem_ld32(o_tmem + c0, r);
                        tmem_ld_wait();
                    }
                    if (srow < g.S) {
                        uint4* dst = reinterpret_cast<uint4*>(a.out + ((int64_t)pc.h * g.S + srow) * D + c0);
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            float x[8];
#pragma unroll
                            for (int e = 0; e < 8; ++e) x[e] = any ? r[8 * i + e] * scale : 0.f;
                            dst[i] = make_uint4(pack2(x[0], x[1]), pack2(x[2], x[3]), pack2(x[4], x[5]), pack2(x[6], x[7]));
                        }
                    }
                }
                if (a.lse && srow < g.S) {
                    const float m_sub = (m == -INFINITY) ? 0.f : m;
                    const int64_t at = (int64_t)pc.h * g.S + srow;
                    for (int br = 3 - a.n_lse; br < 3; ++br)
                        a.lse[(int64_t)(br - (3 - a.n_lse)) * HS + at] = l3[br] > 0.f ? (m_sub + log2f(l3[br])) * ln2 : -INFINITY;
                }
                tc_fence_before();
                if (any) mbar_arrive(&sm.o_free[tile]);  // the MMA issuer counts a state only if it issued a PV for this tile
            } else {
                // leave the unnormalised state in the workspace; the piece that arrives last merges all of them
                float* prow = a.partial + ((((int64_t)pc.unit * p.max_pieces + pc.ord) * 2 + tile) * M_TILE + row) * ROW_F;
#pragma unroll
                for (int c0 = 0; c0 < D; c0 += 32) {
                    float r[32];
                    if (any) {
                        tmem_ld32(o_tmem + c0, r);
                        tmem_ld_wait();
                    }
                    float4* dst = reinterpret_cast<float4*>(prow + c0);
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        dst[i] = any ? make_float4(r[4 * i], r[4 * i + 1], r[4 * i + 2], r[4 * i + 3]) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
                *reinterpret_cast<float4*>(prow + D) = make_float4(m, l3[0], l3[1], l3[2]);
                tc_fence_before();
                if (any) mbar_arrive(&sm.o_free[tile]);  // O is in the workspace: the next state may overwrite the accumulator
                __threadfence();
                wg_sync(tile);
                if ((threadIdx.x & 127) == 0) {
                    const int old = atomicAdd(a.counters + pc.unit * 2 + tile, 1);
                    sm.is_last[tile] = (old == pc.npc - 1);
                }
                wg_sync(tile);
                if (sm.is_last[tile]) {
                    __threadfence();
                    if ((threadIdx.x & 127) == 0) a.counters[pc.unit * 2 + tile] = 0;  // clean for the next launch
                    // pass 1: the row's (m, l_cmp, l_slc, l_swa) of every piece -> per-piece weights
                    const float* base = a.partial + (((int64_t)pc.unit * p.max_pieces * 2 + tile) * M_TILE + row) * ROW_F;
                    const int64_t piece_stride = (int64_t)2 * M_TILE * ROW_F;
                    float wgt[PLAN_MAX_PIECES_PER_UNIT];
                    float M3[3] = {-INFINITY, -INFINITY, -INFINITY}, L3[3] = {0.f, 0.f, 0.f};
                    // a piece holds one branch in GATED mode (which one: its non-zero row sum), SWA and SLC in JOINT mode
                    for (int q = 0; q < pc.npc; ++q) {
                        const float4 ml = __ldcg(reinterpret_cast<const float4*>(base + q * piece_stride + D));
                        const float lq[3] = {ml.y, ml.z, ml.w};
#pragma unroll
                        for (int br = 0; br < 3; ++br) {
                            const int grp = p.gated ? br : 0;  // JOINT: one softmax, one reference
                            if (lq[br] > 0.f) M3[grp] = fmaxf(M3[grp], ml.x);
                        }
                    }
                    for (int q = 0; q < pc.npc; ++q) {
                        const float4 ml = __ldcg(reinterpret_cast<const float4*>(base + q * piece_stride + D));
                        const float lq[3] = {ml.y, ml.z, ml.w};
#pragma unroll
                        for (int br = 0; br < 3; ++br) {
                            const int grp = p.gated ? br : 0;
                            if (lq[br] > 0.f) L3[br] += lq[br] * ex2(ml.x - M3[grp]);
                        }
                    }
                    const float gate[3] = {a.gate_cmp ? __ldg(a.gate_cmp + pc.h) : 1.f, a.gate_slc ? __ldg(a.gate_slc + pc.h) : 1.f,
                                           a.gate_swa ? __ldg(a.gate_swa + pc.h) : 1.f};
                    const float l_joint = L3[0] + L3[1] + L3[2];
#pragma unroll
                    for (int q = 0; q < PLAN_MAX_PIECES_PER_UNIT; ++q) {
                        wgt[q] = 0.f;
                        if (q < pc.npc) {
                            const float4 ml = __ldcg(reinterpret_cast<const float4*>(base + q * piece_stride + D));
                            if (p.gated) {
                                const int br = ml.y > 0.f ? 0 : (ml.z > 0.f ? 1 : 2);
                                const float lb = L3[br];
                                if (lb > 0.f && (ml.y > 0.f || ml.z > 0.f || ml.w > 0.f)) wgt[q] = gate[br] * ex2(ml.x - M3[br]) / lb;
                            } else if (l_joint > 0.f && ml.x > -INFINITY) {
                                wgt[q] = ex2(ml.x - M3[0]) / l_joint;
                            }
                        }
                    }
                    // pass 2: out = sum_q w_q O_q, 32 columns at a time, pieces in order
                    if (srow < g.S) {
#pragma unroll
                        for (int c0 = 0; c0 < D; c0 += 32) {
                            float acc[32];
#pragma unroll
                            for (int i = 0; i < 32; ++i) acc[i] = 0.f;
#pragma unroll
                            for (int q = 0; q < PLAN_MAX_PIECES_PER_UNIT; ++q) {
                                if (q < pc.npc) {
                                    const float4* src = reinterpret_cast<const float4*>(base + q * piece_stride + c0);
#pragma unroll
                                    for (int i = 0; i < 8; ++i) {
                                        const float4 v = __ldcg(src + i);
                                        acc[4 * i] = fmaf(wgt[q], v.x, acc[4 * i]);
                                        acc[4 * i + 1] = fmaf(wgt[q], v.y, acc[4 * i + 1]);
                                        acc[4 * i + 2] = fmaf(wgt[q], v.z, acc[4 * i + 2]);
                                        acc[4 * i + 3] = fmaf(wgt[q], v.w, acc[4 * i + 3]);
                                    }
                                }
                            }
                            uint4* dst = reinterpret_cast<uint4*>(a.out + ((int64_t)pc.h * g.S + srow) * D + c0);
#pragma unroll
                            for (int i = 0; i < 4; ++i)
                                dst[i] = make_uint4(pack2(acc[8 * i], acc[8 * i + 1]), pack2(acc[8 * i + 2], acc[8 * i + 3]),
                                                    pack2(acc[8 * i + 4], acc[8 * i + 5]), pack2(acc[8 * i + 6], acc[8 * i + 7]));
                        }
                        if (a.lse) {
                            const int64_t at = (int64_t)pc.h * g.S + srow;
                            for (int br = 3 - a.n_lse; br < 3; ++br) {
                                const float Mb = M3[p.gated ? br : 0];
                                a.lse[(int64_t)(br - (3 - a.n_lse)) * HS + at] = L3[br] > 0.f ? (Mb + log2f(L3[br])) * ln2 : -INFINITY;
                            }
                        }
                    }
                }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 9) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
    }
}

}  // namespace dq

// ------------------------------------------------------------------------------------- host side
AttnGeom make_attn_geom(const Cache* c, int32_t n_q, const omnimem_attn_params_t& p);

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn()
{
    static std::atomic<EncodeTiledFn> fn{nullptr};
    EncodeTiledFn f = fn.load(std::memory_order_acquire);
    if (!f) {
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) {
            f = (EncodeTiledFn)ptr;
            fn.store(f, std::memory_order_release);
        }
    }
    return f;
}

// bf16 tensor [n2][n1][D] (element strides stride1, stride2) seen as {64 (one half of d), n1 rows, D/64 halves, n2}: one box
// {64, box_rows, D/64, 1} lands in shared memory as [half][box_rows][128 B], the layout the UMMA descriptors read (SWIZZLE_128B).
static int32_t encode_split(CUtensorMap* m, const void* base, int D, uint64_t n1, uint64_t n2, uint64_t stride1_el, uint64_t stride2_el,
                            uint32_t box_rows, bool with_n2)
{
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return fail(OMNIMEM_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    const uint32_t halves = (uint32_t)(D / 64);
    cuuint64_t dims[4] = {64, n1, halves, n2};
    cuuint64_t strides[3] = {stride1_el * 2, 128, stride2_el * 2};
    cuuint32_t box[4] = {64, box_rows, halves, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, with_n2 ? 4u : 3u, const_cast<void*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(OMNIMEM_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return OMNIMEM_OK;
}

static int sm_count()
{
    static std::atomic<int> n{0};
    int v = n.load(std::memory_order_acquire);
    if (v == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
        if (v <= 0) v = 148;
        n.store(v, std::memory_order_release);
    }
    return v;
}

// The work decomposition of one call (attn_plan.cuh): host-only arithmetic, also used to size the workspace.
AttnPlan make_attn_plan(const Cache* c, int32_t n_q, const omnimem_attn_params_t& prm, bool three, int n_sm)
{
    AttnPlan p;
    p.g = make_attn_geom(c, n_q, prm);
    const AttnGeom& g = p.g;
    p.n_qt = (int32_t)ceil_div64(n_q, 128);
    p.units_per_head = (p.n_qt + 1) / 2;
    p.n_units = g.H * p.units_per_head;
    p.gated = prm.fuse_mode == OMNIMEM_FUSE_GATED ? 1 : 0;
    p.n_cmp = three ? (int32_t)ceil_div64(g.n_b, 64) : 0;
    p.n_swa = g.n_win_slots + g.n_cur_slots;
    int max_groups = 0;
    for (int qt = 0; qt < p.n_qt; ++qt) {
        int gf, ng;
        plan_tile_groups(g, qt, &gf, &ng);
        if (ng > max_groups) max_groups = ng;
    }
    p.n_slc = max_groups * g.slc_slots;
    p.T = p.n_cmp + p.n_swa + p.n_slc;
    p.cmp_rows = g.H * g.max_blocks;
    const int64_t total = (int64_t)p.n_units * p.T;
    int64_t min_len = PLAN_MIN_STEPS_PER_CTA;
    if ((p.T + 2) / 3 > min_len) min_len = (p.T + 2) / 3;  // a unit is never split into more than 3 + 1 ranges
    int64_t n_cta = total / min_len;
    if (getenv("OMNIMEM_DQ_NOCUT")) n_cta = p.n_units < n_sm ? p.n_units : n_sm;
    if (n_cta > n_sm) n_cta = n_sm;
    if (n_cta < 1) n_cta = 1;
    p.L = (int32_t)ceil_div64(total, n_cta);
    p.n_cta = (int32_t)ceil_div64(total, p.L);
    int maxp = 1;
    for (int u = 0; u < p.n_units; ++u) {
        int tot, bef;
        plan_unit_pieces(p, u, 0, &tot, &bef);
        if (tot > maxp) maxp = tot;
    }
    p.max_pieces = maxp;
    return p;
}

static size_t plan_workspace_bytes(const AttnPlan& p, int D)
{
    const size_t counters = ((size_t)p.n_units * 2 * 4 + 255) / 256 * 256;
    const size_t partial = p.max_pieces > 1 ? (size_t)p.n_units * p.max_pieces * 2 * 128 * (D + 4) * 4 : 0;
    return counters + partial;
}

// Upper bound for any history length: a unit of T steps meets at most ceil(T / L) + 1 CTA ranges, L >= n_units * T / n_cta,
// and every branch boundary inside the unit (GATED) adds one piece.
size_t attn_workspace_bytes_bound(int32_t H, int32_t D, int32_t n_q, int32_t fuse_mode, bool three)
{
    const int64_t n_qt = ceil_div64(n_q, 128);
    const int64_t n_units = (int64_t)H * ((n_qt + 1) / 2);
    int64_t bound = ceil_div64(sm_count(), n_units) + 1 + (fuse_mode == OMNIMEM_FUSE_GATED ? (three ? 2 : 1) : 0);
    if (bound > PLAN_MAX_PIECES_PER_UNIT) bound = PLAN_MAX_PIECES_PER_UNIT;
    const size_t counters = ((size_t)n_units * 2 * 4 + 255) / 256 * 256;
    return counters + (size_t)n_units * bound * 2 * 128 * (D + 4) * 4;
}

template <int D>
static int32_t launch_dq(const AttnArgs& x, const AttnPlan& p, const CUtensorMap* maps, const dq::Args& a)
{
    const int smem = (int)sizeof(dq::Smem<D>) + 1024;
    static std::atomic<uint64_t> attr_devices{0};  // the shared-memory opt-in is per device
    int dev = 0;
    cudaGetDevice(&dev);
    const uint64_t bit = 1ull << (dev & 63);
    if (!(attr_devices.load(std::memory_order_acquire) & bit)) {
        cudaError_t e = cudaFuncSetAttribute(dq::attn_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
        attr_devices.fetch_or(bit, std::memory_order_release);
    }
    cudaError_t e = launch_pdl(dq::attn_kernel<D>, dim3((unsigned)p.n_cta), dim3(dq::THREADS), (size_t)smem, x.stream, maps[0], maps[1], maps[2],
                               maps[3], maps[4], maps[5], maps[6], a);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "sparse_attn launch: %s", cudaGetErrorString(e));
    count_launch();
    return check_launch("sparse_attn");
}

int32_t launch_attn(const AttnArgs& x)
{
    Cache* c = const_cast<Cache*>(x.cache);
    const bool three = x.gate_cmp != nullptr;
    const AttnPlan p = make_attn_plan(c, x.n_q, x.p, three, sm_count());
    const size_t need = plan_workspace_bytes(p, c->D);
    if (!x.workspace || x.workspace_bytes < need) return fail(OMNIMEM_ECAPACITY, "attn workspace: need %zu bytes, got %zu", need, x.workspace_bytes);
    if (p.max_pieces > PLAN_MAX_PIECES_PER_UNIT) return fail(OMNIMEM_EUNSUPPORTED, "work plan splits a unit into %d pieces (limit %d)", p.max_pieces, PLAN_MAX_PIECES_PER_UNIT);
    // the counters of the merge protocol must be zero before a launch; the kernel leaves them zero, so only a workspace the
    // library has not seen yet (or one whose counter area grew) is cleared here
    const size_t counter_bytes = ((size_t)p.n_units * 2 * 4 + 255) / 256 * 256;
    if (c->ws_seen != x.workspace || c->ws_counter_bytes < counter_bytes) {
        cudaError_t e = cudaMemsetAsync(x.workspace, 0, counter_bytes, x.stream);
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
        c->ws_seen = x.workspace;
        c->ws_counter_bytes = counter_bytes;
    }
    const uint64_t pool_rows = (uint64_t)c->H * c->max_blocks * c->B;
    if (!c->tmaps_ready) {
        if (int32_t rc = encode_split((CUtensorMap*)c->tmap_k, c->k_pages, c->D, pool_rows, 1, c->D, 0, 64, false)) return rc;
        if (int32_t rc = encode_split((CUtensorMap*)c->tmap_v, c->v_pages, c->D, pool_rows, 1, c->D, 0, 64, false)) return rc;
        c->tmaps_ready = true;
    }
    if (three && !c->tmaps_cmp_ready) {
        if (int32_t rc = encode_split((CUtensorMap*)c->tmap_kc, c->pooled_k, c->D, (uint64_t)p.cmp_rows, 1, c->D, 0, 64, false)) return rc;
        if (int32_t rc = encode_split((CUtensorMap*)c->tmap_vc, c->pooled_v, c->D, (uint64_t)p.cmp_rows, 1, c->D, 0, 64, false)) return rc;
        c->tmaps_cmp_ready = true;
    }
    // per-call tensors: re-encoded only when a pointer, a stride or the length changed since the previous call
    if (c->call_q != x.q || c->call_k != x.k_cur || c->call_v != x.v_cur || c->call_n != x.n_q || c->call_st != x.stride_tok || c->call_sh != x.stride_head) {
        if (int32_t rc = encode_split((CUtensorMap*)c->tmap_q, x.q, c->D, x.n_q, c->H, x.stride_tok, x.stride_head, 128, true)) return rc;
        if (int32_t rc = encode_split((CUtensorMap*)c->tmap_kcur, x.k_cur, c->D, x.n_q, c->H, x.stride_tok, x.stride_head, 64, true)) return rc;
        if (int32_t rc = encode_split((CUtensorMap*)c->tmap_vcur, x.v_cur, c->D, x.n_q, c->H, x.stride_tok, x.stride_head, 64, true)) return rc;
        c->call_q = x.q; c->call_k = x.k_cur; c->call_v = x.v_cur; c->call_n = x.n_q; c->call_st = x.stride_tok; c->call_sh = x.stride_head;
    }
    CUtensorMap maps[7];
    maps[0] = *(const CUtensorMap*)c->tmap_q;
    maps[1] = *(const CUtensorMap*)c->tmap_kcur;
    maps[2] = *(const CUtensorMap*)c->tmap_vcur;
    maps[3] = *(const CUtensorMap*)c->tmap_k;
    maps[4] = *(const CUtensorMap*)c->tmap_v;
    maps[5] = three ? *(const CUtensorMap*)c->tmap_kc : maps[3];
    maps[6] = three ? *(const CUtensorMap*)c->tmap_vc : maps[4];

    dq::Args a;
    a.p = p;
    a.ptr_table = x.ptr_table;
    a.page_map = c->page_map;
    a.gate_cmp = three ? x.gate_cmp : nullptr;
    a.gate_slc = p.gated ? x.gate_slc : nullptr;
    a.gate_swa = p.gated ? x.gate_swa : nullptr;
    a.out = (__nv_bfloat16*)x.out;
    a.lse = x.lse_out;
    a.n_lse = three ? 3 : 2;
    a.counters = (int32_t*)x.workspace;
    a.partial = (float*)((char*)x.workspace + counter_bytes);
    a.scale_log2 = x.p.softmax_scale * 1.4426950408889634f;
    a.pool_rows = (int32_t)pool_rows;
    a.rescale_thr = getenv("OMNIMEM_DQ_THR") ? (float)atof(getenv("OMNIMEM_DQ_THR")) : dq::RESCALE_LOG2;
    return c->D == 128 ? launch_dq<128>(x, p, maps, a) : launch_dq<64>(x, p, maps, a);
}

}  // namespace omnimem
