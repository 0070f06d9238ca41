// a6-a8, Blackwell kernel: Per-Head Scattered KV Access attention with TMA-gathered K/V pages,
// tcgen05.mma tiles and TMEM accumulators (sm_100a).  DESIGN.md section 6.5.
//
// One CTA = 128 query rows of one head.  KV arrives as 128-token tiles = two 64-token slots
// (attn_schedule.cuh) fetched straight from the page the pointer table names (or from the current
// chunk) with as few TMA boxes as the operand layouts allow; no union buffer exists.
//
//   warp 8, 10  TMA producers (K tiles, V tiles): walk the slot schedule, one 32 KB tile per ring stage
//   warp 9      MMA issuer (one elected thread runs the whole batch loop): S_t = Q K_t^T (SS),
//               O += P_t V_t (P from TMEM, V MN-major from smem)
//   warps 0-3   softmax warpgroup 0: KV tiles t = 0, 2, 4, ...   (thread = query row, TMEM lane = row)
//   warps 4-7   softmax warpgroup 1: KV tiles t = 1, 3, 5, ...
// Warpgroup p owns score buffer S_p and probability buffer P_p.  It frees S_p as soon as the tile sits
// in registers (s_free), so QK^T of tile t+2 never waits for the exponentials of tile t, and P_p is free
// again once PV of tile t-2 has completed, so no store ever waits for the tensor pipe in steady state.
// Both warpgroups feed ONE accumulator O; its single reference max per row lives in shared memory, and a
// tile's "max step" (read the reference, raise it if the tile max exceeds it by more than 2^8, rescaling
// O) runs in tile order (mbarrier hand-off between the warpgroups) while the exponentials of consecutive
// tiles overlap.
// The tensor pipe accepts only a few MMAs ahead of the one executing (measured: issue of a back-to-back
// stream blocks at 64 clk per 128x128x16 MMA), so whatever the issuing thread does between two MMAs idles
// the pipe.  A batch (8 MMAs + 2 commits) is therefore ONE asm block and the issuer's loop is unrolled
// over rounds of 10 tiles, in which ring slot, barrier phase and S/P buffer of every batch are constants.
// What bounds the kernel is the SM's TMA ingest: hence the 16 / 32 KB boxes below.
//
// TMEM (512 columns): S_0 [0,128) S_1 [128,256) O [256,384) P_0 [384,448) P_1 [448,512).
//
// Branches and fusion (a8, Eq. 1): the KV tile sequence of a CTA is [CMP tiles][SWA tiles][SLC tiles] (the
// compressed cache only in the three-branch call; the SLC tiles, the only ones that need omnimem_select's table, last).
// JOINT runs it as ONE softmax segment.  GATED runs one SEGMENT per branch in the same launch: at a segment's end the
// warpgroups normalise O, scale it by the branch's gate and add it to a per-row fp32 scratch (L2-resident: the CTA that
// writes a row is the one that reads it back), the running max / sums start afresh, and the first PV of the next segment
// overwrites the accumulator.  The tensor pipe, the TMA ring and the S / P buffers run through the boundaries unchanged.
//
// Head dimension: the tiles are 128 wide.  head_dim 64 runs through the SAME kernel: its tensor maps declare one 64-wide
// half of D, so every box's second half lies out of bounds and TMA fills it with zeros -- Q, K and V arrive padded to 128
// (QK^T unchanged, O's upper 64 columns zero) and only the first head_dim output columns are stored.
#include <cuda.h>
#include <stdio.h>

#include <atomic>
#include <type_traits>

#include "attn_schedule.cuh"
#include "common.cuh"

namespace omnimem {

namespace tc {

constexpr int M_TILE = 128;
constexpr int KV_TILE = 128;
constexpr int D = 128;  // tile width; a.d_head (64 or 128) is the tensor's head dimension
constexpr int NSTAGE = 5;
constexpr uint32_t TM_S = 0, TM_O = 256, TM_P = 384;  // TMEM column offsets
constexpr int TILE_BYTES = KV_TILE * D * 2;   // 32 KB
constexpr int HALF_BYTES = TILE_BYTES / 2;    // one 64-wide half of D: [128 rows][128 B]
constexpr int SLOT_BYTES = 64 * 128;          // 64 rows x 128 B
// V tiles are laid out [slot][half of D][64 tokens][128 B]: one 16 KB TMA box per slot (per-copy overhead, not
// bytes, is what separates 8 KB boxes from the SM's L2 ingest limit); K tiles stay [half of D][128 tokens][128 B]
// because the K-major B operand of QK^T needs one uniform stride over its 128 rows.
constexpr int V_SLOT_BYTES = 2 * SLOT_BYTES;  // 16 KB
constexpr int V_HALF_BYTES = SLOT_BYTES;      // distance between the two halves of D inside a V slot
constexpr int META_RING = 16;
constexpr int SLOT_RING = 64;
constexpr int THREADS = 384;
constexpr float RESCALE_LOG2 = 8.0f;
// Tile order.  GATED: [CMP][SWA][SLC], fixed (the segment order) -- the slots that need omnimem_select's table come last, so the
// window tiles run while the selection is still in flight and the producers wait for the table right before the first SLC slot.
// JOINT (one segment): the host picks (Args::swa_first): the same order with 64 / 128-row pages (with the paired tiles of
// attn_schedule.cuh the deferred wait wins there too: config 2 step 298 -> 289 us), [SLC][SWA] with 32-row pages.
constexpr int GATED_SWA_FIRST = 1;

struct TileMeta {
    int32_t lo0, hi0, lo1, hi1;  // pages of 64 / 128 rows: valid tokens [lo, hi) of the tile's two 64-token slots
    int32_t rlo, rhi;            // query rows (relative) that attend
    int32_t branch;              // BR_CMP / BR_SLC / BR_SWA: which row sum the tile feeds; bits 8..: rmid (the one field the softmax
                                 // warps keep across the exponentials)
    int32_t rmid;                // paired SLC tile (attn_schedule.cuh): rows [rlo, rmid) attend slot 0 only, rows [rmid, rhi) slot 1 only; else 0
};
struct TileQuarters {            // 32-row pages: valid tokens [qlo, qhi) of each 32-column quarter of the tile (one page each)
    int8_t qlo[4], qhi[4];
};
enum : int32_t { BR_CMP = 0, BR_SLC = 1, BR_SWA = 2 };
enum : int32_t { SEG_CMP = 0, SEG_SLC = 1, SEG_SWA = 2, SEG_JOINT = 3 };  // SEG_JOINT: SWA tiles then SLC tiles, one softmax

struct Smem {
    alignas(1024) unsigned char q[TILE_BYTES];
    alignas(1024) unsigned char kv[NSTAGE][TILE_BYTES];
    alignas(8) unsigned long long q_full;
    unsigned long long kv_full[NSTAGE], kv_empty[NSTAGE];
    unsigned long long s_full[2], s_free[2], p_full[2], pv_done[2], max_done[2];
    int32_t seg_b[4];           // segment s covers KV tiles [seg_b[s], seg_b[s + 1])
    unsigned long long o_free;  // 256 arrivals per segment boundary: the warpgroups have read O, the next segment may overwrite it
    uint32_t tmem_base;
    float m_ref[M_TILE];  // per query row: reference max (log2 units) that P and O are relative to
    float exch[2 * M_TILE * 4];  // segment end: (m, l_cmp, l_slc, l_swa) of each warpgroup
    TileMeta meta[META_RING];
    TileQuarters metaq[META_RING];
    SlotBase slots[2][SLOT_RING];  // one ring per producer warp
    int32_t slots2[2][SLOT_RING][3];  // 32-row pages: (row2, lo2, hi2) of the slot's second page
};

struct Args {
    AttnGeom g;
    const int32_t *ptr_table, *page_map;
    const float* gate[3];  // [H] fp32 per segment (GATED); NULL = 1
    __nv_bfloat16* out;
    float *lse_cmp, *lse_slc, *lse_swa;  // [H][S] fp32 each, nullable: natural-log LSE of a branch
    float* partial;      // GATED: [H][S][d_head] fp32, the gated sum of the segments finished so far
    float scale_log2;
    int32_t n_seg;       // 1 (JOINT) .. 3
    int32_t seg_kind[3];
    int32_t cmp_blocks;  // three-branch call: the head's N_b compressed tokens lead the sequence, 64 per slot (0 otherwise)
    int32_t cmp_rows;    // H * max_blocks: rows of the compressed-cache pools (out-of-bounds coordinate for their maps)
    int32_t pool_rows;   // H * max_blocks * B: a row coordinate at/after this is out of bounds -> zero fill
    int32_t d_head;      // head dimension of out / partial (64: the tiles' upper half is zero padding)
    int32_t swa_first;   // JOINT: 1 = [SWA][SLC] (the table is needed last: the window tiles overlap omnimem_select), 0 = [SLC][SWA]
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
__device__ __forceinline__ bool mbar_try_wait(void* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug traps (the launch then reports an error) instead of hanging the GPU.  The bound is 2^31
// failed probes -- a probe that fails costs at least ~20 ns (the hardware suspends it for longer), so more than 40 s of
// polling: no legitimate wait comes near it, under a profiler's replay, a sanitizer or time-slicing either.  The retry
// loop is three instructions and keeps ONE register live: these waits sit inside the softmax warps (at the register
// limit) and inside the MMA issuer (whose instruction stream paces the tensor pipe); a %globaltimer-based bound with its
// 64-bit start time cost the headline kernel 10 us of 273 (measured, profiles/r2_microbench.md).
constexpr uint32_t WAIT_PROBES = 1u << 31;
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity)
{
    if (mbar_try_wait(bar, parity)) return;
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > WAIT_PROBES) __trap();
    }
}
__device__ __forceinline__ void mbar_wait_addr(uint32_t bar, uint32_t parity)
{
    uint32_t spins = 0;
    while (true) {
        uint32_t ok;
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if (++spins > WAIT_PROBES) __trap();
    }
}
// One lane of a converged warp (elect.sync): the compiler then knows the region is single-threaded and
// feeds tcgen05.mma / TMA their uniform operands without a per-thread waterfall loop.
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

__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, void* bar, int c0, int c1)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1) : "memory");
}
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

// UMMA shared-memory descriptor, SWIZZLE_128B (layout type 2), version 1.
//   K-major operand  (Q, K):  rows of 128 B (64 bf16 of D), 8-row groups 1024 B apart (SBO); LBO unused (1).
//   MN-major operand (V):     same bytes; LBO = distance between the two 64-wide halves of D,
//                             SBO = distance between 8-token groups (1024 B).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(sbo_bytes >> 4) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}

// instruction descriptor, kind::f16: bf16 x bf16 -> fp32, M = 128, N = 128
constexpr uint32_t IDESC_BASE = (1u << 4) | (1u << 7) | (1u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);
constexpr uint32_t IDESC_QK = IDESC_BASE;              // A, B K-major
constexpr uint32_t IDESC_PV = IDESC_BASE | (1u << 16); // B (V) MN-major


// A tensor-pipe batch = 8 x (M128 N128 K16) MMAs + 2 commits as ONE asm block: nothing but descriptor adds sits
// between the MMAs (measured on B200: a clean stream runs at 64.8 clk per MMA with QK^T and PV batches
// alternating, TMA streaming and eight softmax warps busy; a single data-dependent branch inside the stream
// costs 40 % of that).
// QK^T: SS, descriptors of the Q tile and the K tile ([2 halves of D][128 rows][128 B], SWIZZLE_128B).
__device__ __forceinline__ void qk_batch(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t bar_empty, uint32_t bar_done)
{
    asm volatile(
        "{\n\t.reg .pred pa;\n\t.reg .b64 a, b;\n\t"
        "setp.ne.b32 pa, 0, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, pa;\n\t"
        "setp.eq.b32 pa, 0, 0;\n\t"
        "add.s64 a, %1, 2;\n\tadd.s64 b, %2, 2;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
        "add.s64 a, %1, 4;\n\tadd.s64 b, %2, 4;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
        "add.s64 a, %1, 6;\n\tadd.s64 b, %2, 6;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
        "add.s64 a, %1, 1024;\n\tadd.s64 b, %2, 1024;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
        "add.s64 a, %1, 1026;\n\tadd.s64 b, %2, 1026;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
        "add.s64 a, %1, 1028;\n\tadd.s64 b, %2, 1028;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
        "add.s64 a, %1, 1030;\n\tadd.s64 b, %2, 1030;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], a, b, %3, pa;\n\t"
        "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%4];\n\t"
        "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t}"
        :: "r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(IDESC_QK), "r"(bar_empty), "r"(bar_done)
        : "memory");
}
// PV: O (+)= P V with P from TMEM (8 columns per K = 16 step) and V MN-major from smem: 16 tokens = 2048 B per
// step inside a slot, slots V_SLOT_BYTES apart (descriptor units of 16 B: 128 per step, 1024 per slot).
__device__ __forceinline__ void pv_batch(uint32_t d_tmem, uint32_t p_tmem, uint64_t vdesc, uint32_t acc_first, uint32_t bar_empty, uint32_t bar_done)
{
    asm volatile(
        "{\n\t.reg .pred pa;\n\t.reg .b64 b;\n\t.reg .b32 a;\n\t"
        "setp.ne.b32 pa, %3, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %6, pa;\n\t"
        "setp.eq.b32 pa, 0, 0;\n\t"
        "add.s32 a, %1, 8;\n\tadd.s64 b, %2, 128;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %6, pa;\n\t"
        "add.s32 a, %1, 16;\n\tadd.s64 b, %2, 256;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %6, pa;\n\t"
        "add.s32 a, %1, 24;\n\tadd.s64 b, %2, 384;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %6, pa;\n\t"
        "add.s32 a, %1, 32;\n\tadd.s64 b, %2, 1024;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %6, pa;\n\t"
        "add.s32 a, %1, 40;\n\tadd.s64 b, %2, 1152;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %6, pa;\n\t"
        "add.s32 a, %1, 48;\n\tadd.s64 b, %2, 1280;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %6, pa;\n\t"
        "add.s32 a, %1, 56;\n\tadd.s64 b, %2, 1408;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [a], b, %6, pa;\n\t"
        "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%4];\n\t"
        "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%5];\n\t}"
        :: "r"(d_tmem), "r"(p_tmem), "l"(vdesc), "r"(acc_first), "r"(bar_empty), "r"(bar_done), "r"(IDESC_PV)
        : "memory");
}
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
// packed fp32x2 arithmetic (FFMA2 / FADD2): two lanes per issue slot on the FMA pipe
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

// Column masks without predicates (the softmax warps have none to spare: a compare + select per element became one serial
// chain through a single predicate register): bit c of `mask` = column c is valid; an invalid column gets -inf ADDED.
__device__ __forceinline__ uint32_t range_mask32(int lo, int hi)  // bits [lo, hi) of a 32-column chunk
{
    lo = max(lo, 0);
    hi = min(hi, 32);
    if (hi <= lo) return 0u;
    return (hi == 32 ? 0xffffffffu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u);
}
template <int C>
__device__ __forceinline__ float mask_col(float v, uint32_t mask)
{
    const int m = ((int)(mask << (31 - C))) >> 31;  // 0 or -1
    return v + __int_as_float(~m & (int)0xff800000);  // + 0 or + (-inf)
}
template <int N>
__device__ __forceinline__ void mask_chunk(float* v, uint32_t mask)  // N <= 32 columns, compile-time unrolled
{
    if constexpr (N > 0) {
        mask_chunk<N - 1>(v, mask);
        v[N - 1] = mask_col<N - 1>(v[N - 1], mask);
    }
}

// ------------------------------------------------------------------------------------- kernel
// The tensor-pipe batches of one CTA in issue order: QK_0, QK_1, then for t = 0, 1, ...: QK_{t+2}, PV_t.
// Ring slot i % NSTAGE holds the operand tile of batch position i (K tile for a QK batch, V tile for a PV batch).
// Positions are REGULAR -- QK_t at 2t - 2 (t >= 2), PV_t at 2t + 3 -- also at the end of the sequence, where the
// QK batches have run out and their positions stay unused: ring slot and barrier phase of every batch are then
// compile-time constants of the MMA issuer's 10-tile unrolled loop.
__device__ __forceinline__ constexpr int batch_pos_qk(int t) { return t < 2 ? t : 2 * t - 2; }
__device__ __forceinline__ constexpr int batch_pos_pv(int t) { return 2 * t + 3; }

// ---- MMA issuer: the batch sequence unrolled over rounds of 10 tiles.  Inside a round a tile's index I fixes
// the ring slot and the kv_full phase of both of its batches (20 positions per round = 4 turns of the 5-slot
// ring) and the S / P buffer; only the phase of the S / P barriers alternates between rounds (5 uses per round).
struct MmaCtx {
    uint32_t tmem, b_kv_full, b_kv_empty, b_s_full, b_s_free, b_p_full, b_pv_done, b_o_free;
    uint64_t qd, kd0, vd0;
    int T;
    int first[3];   // first tile of segment s, -1 if the segment has no tile
    int o_waited;   // o_free completions consumed so far
};
// QK_{t0 + J}: J is the tile's index relative to the round start (0 .. 11)
template <int J>
__device__ __forceinline__ void mma_qk(const MmaCtx& c, int t0, uint32_t rp)
{
    static_assert(NSTAGE == 5, "the unrolled issuer assumes a 5-slot ring");
    if (t0 + J >= c.T) return;
    constexpr int pos = batch_pos_qk(J >= 2 ? J : J);          // position inside the round (round offset 20 = 4 ring turns)
    constexpr int posr = J < 2 ? J : 2 * J - 2;
    constexpr int st = posr % NSTAGE, ph = (posr / NSTAGE) & 1;
    constexpr int par = J & 1;
    (void)pos;
    if (J < 2 && t0 == 0) {
        mbar_wait_addr(c.b_kv_full + st * 8, ph);               // S_p has no previous tenant
    } else {
        // S_par was last used by tile t - 2: completion number (t >> 1) - 1 of s_free[par]
        const uint32_t sph = ((uint32_t)(((J >> 1) - 1) & 1)) ^ rp;
        mbar_wait2(c.b_kv_full + st * 8, ph, c.b_s_free + par * 8, sph);
    }
    tc_fence_after();
    qk_batch(c.tmem + TM_S + par * 128, c.qd, c.kd0 + (uint64_t)(st * (TILE_BYTES >> 4)), c.b_kv_empty + st * 8, c.b_s_full + par * 8);
}
// SEG: the sequence has more than one segment (GATED); otherwise tile 0 alone starts an accumulation and the issuing thread's
// instruction stream between two batches stays as short as it can be (it paces the tensor pipe).
template <int I, bool SEG>
__device__ __forceinline__ void mma_pv(MmaCtx& c, int t0, uint32_t rp)
{
    if (t0 + I >= c.T) return;
    const int t = t0 + I;
    int seg = t == 0 ? 0 : -1;
    if constexpr (SEG) {
        // the first PV of a segment overwrites the accumulator: the warpgroups must have read the previous segment's O
        seg = t == c.first[2] ? 2 : (t == c.first[1] ? 1 : (t == c.first[0] ? 0 : -1));
        while (seg > c.o_waited) {  // completions are consumed in order (a parity cannot tell two of them apart)
            mbar_wait_addr(c.b_o_free, (uint32_t)c.o_waited & 1u);
            ++c.o_waited;
        }
    }
    constexpr int posr = 2 * I + 3;
    constexpr int st = posr % NSTAGE, ph = (posr / NSTAGE) & 1;
    constexpr int par = I & 1;
    const uint32_t pph = ((uint32_t)((I >> 1) & 1)) ^ rp;        // completion number t >> 1 of p_full[par]
    mbar_wait2(c.b_kv_full + st * 8, ph, c.b_p_full + par * 8, pph);
    tc_fence_after();
    pv_batch(c.tmem + TM_O, c.tmem + TM_P + par * 64, c.vd0 + (uint64_t)(st * (TILE_BYTES >> 4)), seg < 0, c.b_kv_empty + st * 8,
             c.b_pv_done + par * 8);
}
template <int I, bool SEG>
__device__ __forceinline__ void mma_tile(MmaCtx& c, int t0, uint32_t rp)
{
    mma_qk<I + 2>(c, t0, rp);
    mma_pv<I, SEG>(c, t0, rp);
}

// SEG: more than one softmax segment (GATED); P32: 32-row pages (two pages per slot).  Both are compile-time so that the
// common configuration carries none of the other's instructions in its producer / issuer / softmax loops.
template <bool SEG, bool P32>
__global__ void __launch_bounds__(THREADS, 1)
attn_tcgen05_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_kcur,
                    const __grid_constant__ CUtensorMap tm_kcur128, const __grid_constant__ CUtensorMap tm_vcur,
                    const __grid_constant__ CUtensorMap tm_kpool, const __grid_constant__ CUtensorMap tm_vpool,
                    const __grid_constant__ CUtensorMap tm_kcmp, const __grid_constant__ CUtensorMap tm_vcmp, const Args a)
{
    extern __shared__ unsigned char smem_raw[];
    Smem& sm = *reinterpret_cast<Smem*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    const AttnGeom& g = a.g;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = blockIdx.y, q0 = blockIdx.x * M_TILE;

    TileSched ts;
    // GATED: the segment order is fixed ([CMP] SWA SLC); JOINT: one segment, the host picks the order (Args::swa_first)
    const int SWA_FIRST = SEG ? GATED_SWA_FIRST : a.swa_first;
    ts.init(g, h, q0, M_TILE, 2, SWA_FIRST);
    // slot sequence: [cmp_pad compressed-cache slots][ts: SWA slots, SLC slots]; tile = two slots
    // (the three-branch call is GATED: without segments there is no compressed-cache part and its code folds away)
    const int cmp_slots = SEG ? (a.cmp_blocks + 63) / 64 : 0, cmp_pad = (cmp_slots + 1) / 2 * 2;
    const int T = (cmp_pad + ts.n_slots) / 2;  // KV tiles
    // segment s covers tiles [seg_b[s], seg_b[s + 1]): kept in shared memory (the softmax loop has no register to spare)
    if (threadIdx.x == 0) {
        int at = 0;
        for (int sg = 0; sg < 4; ++sg) {
            sm.seg_b[sg] = sg < a.n_seg ? at : T;
            if (sg < a.n_seg)
                at += a.n_seg == 1 ? T : (a.seg_kind[sg] == SEG_CMP ? cmp_pad : (a.seg_kind[sg] == SEG_SWA ? ts.n_swa_slots : ts.n_slc_slots)) / 2;
        }
    }

    if (threadIdx.x == 0) {
        mbar_init(&sm.q_full, 1);
        for (int i = 0; i < NSTAGE; ++i) { mbar_init(&sm.kv_full[i], 1); mbar_init(&sm.kv_empty[i], 1); }
        for (int b = 0; b < 2; ++b) {
            mbar_init(&sm.s_full[b], 1);
            mbar_init(&sm.s_free[b], 128);
            mbar_init(&sm.p_full[b], 128);
            mbar_init(&sm.pv_done[b], 1);
            mbar_init(&sm.max_done[b], 128);
        }
        mbar_init(&sm.o_free, 256);
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
    // No griddepcontrol.wait here: Q, the current chunk and the cached pages were complete before the selection kernels were
    // launched, so the window / current-chunk tiles run while omnimem_select is still in flight.  The producers wait right
    // before they read ptr_table for the first SLC slot, the softmax warps before the epilogue touches global memory.

    if (warp >= 8) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
        if (warp == 8 || warp == 10) {
            // ===================================================================== TMA producers
            // warp 8 fetches the K tiles, warp 10 the V tiles (one warp alone cannot issue 8 boxes per KV tile
            // at the pace the tensor pipe consumes them: its instruction stream shares a scheduler with two
            // softmax warps).  Each warp resolves the slot schedule 32 slots at a time (one slot per lane: the
            // ptr_table / page_map reads of a batch are independent loads in flight together) into its own
            // shared ring; one elected lane then turns ring entries into TMA boxes, one 32 KB tile per stage.
            const bool is_v = warp == 10;
            using RingSlot = typename std::conditional<P32, Slot, SlotBase>::type;
            SlotBase* ring = sm.slots[is_v ? 1 : 0];
            int32_t (*ring2)[3] = sm.slots2[is_v ? 1 : 0];
            auto ring_get = [&](int i) {  // a slot of the ring; with 32-row pages its second page comes from the side array
                RingSlot r;
                static_cast<SlotBase&>(r) = ring[i % SLOT_RING];
                if constexpr (P32) { r.row2 = ring2[i % SLOT_RING][0]; r.lo2 = ring2[i % SLOT_RING][1]; r.hi2 = ring2[i % SLOT_RING][2]; }
                return r;
            };
            if (!is_v && T > 0 && elect_one()) {  // T == 0: nobody waits for Q, so no copy may be left in flight at exit
                prefetch_tmap(&tm_q); prefetch_tmap(&tm_kcur); prefetch_tmap(&tm_kcur128); prefetch_tmap(&tm_kpool);
                if (a.cmp_blocks > 0) prefetch_tmap(&tm_kcmp);
                mbar_expect_tx(&sm.q_full, TILE_BYTES);
                tma_load_3d(sm.q, &tm_q, &sm.q_full, 0, q0, h);
                tma_load_3d(sm.q + HALF_BYTES, &tm_q, &sm.q_full, 64, q0, h);
            }
            if (is_v && elect_one()) { prefetch_tmap(&tm_vcur); prefetch_tmap(&tm_vpool); if (a.cmp_blocks > 0) prefetch_tmap(&tm_vcmp); }
            int resolved = 0;  // slots [0, resolved) are in the ring
            bool waited = false;
            for (int t = 0; t < T; ++t) {
                while (resolved < 2 * t + 2) {  // warp-uniform
                    if (!waited && ts.n_slc_slots > 0 && resolved + 32 > cmp_pad + (SWA_FIRST ? ts.n_swa_slots : 0)) {
                        pdl_wait();  // the batch reaches the SLC slots: ptr_table must be final (omnimem_select has completed)
                        waited = true;
                    }
                    const int idx = resolved + lane;
                    Slot sl;
                    sl.row2 = -1; sl.lo2 = 0; sl.hi2 = 0;
                    if (idx < cmp_pad) {  // compressed tokens [64 idx, 64 idx + 64) of head h: contiguous rows of pooled_k / pooled_v
                        sl.kind = idx < cmp_slots ? SLOT_CMP : SLOT_NONE;
                        sl.row = h * g.max_blocks + idx * 64;
                        sl.lo = 0;
                        sl.hi = idx < cmp_slots ? min(64, a.cmp_blocks - idx * 64) : 0;
                    } else {
                        sl = ts.template slot<P32>(g, a.ptr_table, a.page_map, idx - cmp_pad);
                    }
                    ring[idx % SLOT_RING] = static_cast<const SlotBase&>(sl);
                    if constexpr (P32) { ring2[idx % SLOT_RING][0] = sl.row2; ring2[idx % SLOT_RING][1] = sl.lo2; ring2[idx % SLOT_RING][2] = sl.hi2; }
                    resolved += 32;
                    __syncwarp();
                }
                if (elect_one()) {
                    const int item = is_v ? batch_pos_pv(t) : batch_pos_qk(t);
                    const int stage = item % NSTAGE;
                    const RingSlot s0 = ring_get(2 * t);
                    const RingSlot s1 = ring_get(2 * t + 1);
                    if (!is_v) {
                        TileMeta m;
                        TileRows tr;
                        if (2 * t < cmp_pad) { tr.lo = 0; tr.hi = M_TILE; tr.is_slc = 0; tr.mid = 0; }
                        else tr = ts.rows(g, 2 * t - cmp_pad);
                        if constexpr (P32) {
                            TileQuarters mq;
#pragma unroll
                            for (int sl = 0; sl < 2; ++sl) {
                                const RingSlot& s = sl ? s1 : s0;
                                if (s.kind == SLOT_HIST) {  // two pages, each with its own valid range
                                    mq.qlo[2 * sl] = (int8_t)s.lo; mq.qhi[2 * sl] = (int8_t)s.hi;
                                    mq.qlo[2 * sl + 1] = (int8_t)s.lo2; mq.qhi[2 * sl + 1] = (int8_t)s.hi2;
                                } else {  // current chunk / compressed cache: one range over the slot's 64 tokens
                                    mq.qlo[2 * sl] = (int8_t)min(s.lo, 32); mq.qhi[2 * sl] = (int8_t)min(s.hi, 32);
                                    mq.qlo[2 * sl + 1] = (int8_t)(max(s.lo, 32) - 32); mq.qhi[2 * sl + 1] = (int8_t)(max(s.hi, 32) - 32);
                                }
                            }
                            sm.metaq[t % META_RING] = mq;
                        }
                        m.lo0 = s0.lo; m.hi0 = s0.hi; m.lo1 = s1.lo; m.hi1 = s1.hi;
                        m.rlo = tr.lo; m.rhi = tr.hi; m.branch = (2 * t < cmp_pad ? BR_CMP : (tr.is_slc ? BR_SLC : BR_SWA)) | (tr.mid << 8); m.rmid = tr.mid;
                        sm.meta[t % META_RING] = m;
                    }
                    mbar_wait(&sm.kv_empty[stage], ((item / NSTAGE) & 1) ^ 1);
                    unsigned char* dst = sm.kv[stage];
                    mbar_expect_tx(&sm.kv_full[stage], TILE_BYTES);
                    if (is_v) {
                        // one 16 KB box {64 d, 64 tokens, 2 halves} per slot
#pragma unroll
                        for (int sl = 0; sl < 2; ++sl) {
                            const RingSlot& s = sl ? s1 : s0;
                            unsigned char* d = dst + sl * V_SLOT_BYTES;
                            if (s.kind == SLOT_CUR) tma_load_4d(d, &tm_vcur, &sm.kv_full[stage], 0, s.row, 0, h);
                            else if (SEG && s.kind == SLOT_CMP) tma_load_3d(d, &tm_vcmp, &sm.kv_full[stage], 0, s.row, 0);
                            else if constexpr (P32) {
                                // 32-row pages: one 4 KB box per (page, half of D); a missing page reads out of bounds (zeros)
#pragma unroll
                                for (int u = 0; u < 2; ++u) {
                                    const bool ok = s.kind == SLOT_HIST && (u ? s.hi2 > s.lo2 : s.hi > s.lo);
                                    const int row = ok ? (u ? s.row2 : s.row) : a.pool_rows;
#pragma unroll
                                    for (int c = 0; c < 2; ++c)
                                        tma_load_2d(d + c * V_HALF_BYTES + u * 32 * 128, &tm_vpool, &sm.kv_full[stage], c * 64, row);  // P32: a 2-D map, 32-row boxes
                                }
                            }
                            else tma_load_3d(d, &tm_vpool, &sm.kv_full[stage], 0, s.kind == SLOT_HIST ? s.row : a.pool_rows, 0);
                        }
                    } else if (s0.kind == SLOT_CUR && s1.kind != SLOT_HIST) {
                        // 128 consecutive tokens of the current chunk: one 32 KB box {64 d, 128 tokens, 2 halves}
                        tma_load_4d(dst, &tm_kcur128, &sm.kv_full[stage], 0, s0.row, 0, h);
                    } else {
#pragma unroll
                        for (int sl = 0; sl < 2; ++sl) {
                            const RingSlot& s = sl ? s1 : s0;
#pragma unroll
                            for (int c = 0; c < 2; ++c) {
                                unsigned char* d = dst + c * HALF_BYTES + sl * SLOT_BYTES;
                                if (s.kind == SLOT_CUR) tma_load_3d(d, &tm_kcur, &sm.kv_full[stage], c * 64, s.row, h);
                                else if (SEG && s.kind == SLOT_CMP) tma_load_2d(d, &tm_kcmp, &sm.kv_full[stage], c * 64, s.row);
                                else if constexpr (P32) {
#pragma unroll
                                    for (int u = 0; u < 2; ++u) {
                                        const bool ok = s.kind == SLOT_HIST && (u ? s.hi2 > s.lo2 : s.hi > s.lo);
                                        tma_load_2d(d + u * 32 * 128, &tm_kpool, &sm.kv_full[stage], c * 64, ok ? (u ? s.row2 : s.row) : a.pool_rows);  // P32: 32-row boxes
                                    }
                                }
                                else tma_load_2d(d, &tm_kpool, &sm.kv_full[stage], c * 64, s.kind == SLOT_HIST ? s.row : a.pool_rows);
                            }
                        }
                    }
                }
                __syncwarp();
            }
            if (!waited) pdl_wait();
        } else if (warp == 9) {
            // ===================================================================== MMA issuer
            // One elected thread runs the whole loop (the other lanes park at the __syncwarp below).  Batch order:
            // QK_0, QK_1, then QK_{t+2}, PV_t for t = 0, 1, ...; every batch waits for its own operands only.
            if (elect_one() && T > 0) {
                MmaCtx cx;
                cx.tmem = tmem;
                cx.T = T;
                cx.b_kv_full = smem_u32(&sm.kv_full[0]); cx.b_kv_empty = smem_u32(&sm.kv_empty[0]);
                cx.b_s_full = smem_u32(&sm.s_full[0]); cx.b_s_free = smem_u32(&sm.s_free[0]);
                cx.b_p_full = smem_u32(&sm.p_full[0]); cx.b_pv_done = smem_u32(&sm.pv_done[0]);
                cx.b_o_free = smem_u32(&sm.o_free);
                cx.o_waited = 0;
                for (int sg = 0; sg < 3; ++sg) cx.first[sg] = (sg < a.n_seg && sm.seg_b[sg] < sm.seg_b[sg + 1]) ? sm.seg_b[sg] : -1;
                cx.qd = make_desc(smem_u32(sm.q), 16, 1024);
                cx.kd0 = make_desc(smem_u32(sm.kv[0]), 16, 1024);
                cx.vd0 = make_desc(smem_u32(sm.kv[0]), V_HALF_BYTES, 1024);
                mbar_wait(&sm.q_full, 0);
                mma_qk<0>(cx, 0, 0);
                mma_qk<1>(cx, 0, 0);
                for (int t0 = 0; t0 < T; t0 += 10) {
                    const uint32_t rp = (uint32_t)(t0 / 10) & 1;  // tiles of odd rounds see every S / P barrier one phase later
                    mma_tile<0, SEG>(cx, t0, rp); mma_tile<1, SEG>(cx, t0, rp); mma_tile<2, SEG>(cx, t0, rp); mma_tile<3, SEG>(cx, t0, rp);
                    mma_tile<4, SEG>(cx, t0, rp); mma_tile<5, SEG>(cx, t0, rp); mma_tile<6, SEG>(cx, t0, rp); mma_tile<7, SEG>(cx, t0, rp);
                    mma_tile<8, SEG>(cx, t0, rp); mma_tile<9, SEG>(cx, t0, rp);
                }
            }
        }
        __syncwarp();
    } else {
        // ========================================================================= softmax warpgroups
        asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
        const int p = warp >> 2;                          // parity of the tiles this warpgroup owns
        const int row = (warp & 3) * 32 + lane;           // query row in the tile == TMEM lane
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t o_tmem = tmem + lane_base + TM_O;
        const uint32_t s_tmem = tmem + lane_base + TM_S + p * 128;
        const uint32_t p_tmem = tmem + lane_base + TM_P + p * 64;
        const int srow = q0 + row;
        // m_mine: the shared reference max as this thread last saw it; l3: this warpgroup's partial row sums (CMP, SLC, SWA),
        // relative to m_mine.  Both start afresh with every segment.
        const float sl = a.scale_log2;
        const float ln2 = 0.6931471805599453f;
        int t = p;  // next KV tile of this warpgroup (tiles alternate between the warpgroups across segment boundaries)
        if (p == 0) sm.m_ref[row] = -INFINITY;  // read by the other warpgroup only after max_done (tile 0)
        const int n_seg = SEG ? a.n_seg : 1;
        const int t_slc0 = SWA_FIRST ? (cmp_pad + ts.n_swa_slots) / 2 : 0;  // first tile that may be a paired SLC tile
        for (int sg = 0; sg < n_seg; ++sg) {
          float m_mine = -INFINITY, l3[3] = {0.f, 0.f, 0.f};
          const int t_end = SEG ? sm.seg_b[sg + 1] : T;
          // The tile loop exists twice: the window / current-chunk / compressed-cache tiles (the bulk; their loop carries no
          // instruction of the paired-tile path) and the SLC tiles behind them.
#pragma unroll
          for (int pass = P32 ? 1 : 0; pass < 2; ++pass) {  // 32-row pages never pair: one copy of the loop
          const bool PAIRED = !P32 && pass == 1;  // a constant in each unrolled copy
          const int t_stop = pass == 0 ? min(t_end, t_slc0) : t_end;
          for (; t < t_stop; t += 2) {
            const uint32_t ph = (t >> 1) & 1;
            mbar_wait(&sm.s_full[p], ph);
            tc_fence_after();
            const TileMeta mt = sm.meta[t % META_RING];
            const bool row_on = row >= mt.rlo && row < mt.rhi;
            const bool warp_on = __any_sync(0xffffffffu, row_on);
            float s[128];
            float mx = -INFINITY;
            TileQuarters mq = {};
            if constexpr (P32) mq = sm.metaq[t % META_RING];
            const bool full = P32 ? (*reinterpret_cast<const uint32_t*>(mq.qlo) == 0u && *reinterpret_cast<const uint32_t*>(mq.qhi) == 0x20202020u)
                                  : (mt.lo0 == 0 && mt.hi0 == 64 && mt.lo1 == 0 && mt.hi1 == 64 && (!PAIRED || mt.rmid == 0));
            // 32-row pages: a page holds B < 32 tokens, so no tile is ever `full`; but the regular case -- every page valid from its
            // first row up to at least its 24th -- only masks the last columns of each quarter: it takes the pipelined path below too
            const bool tail_only = P32 && *reinterpret_cast<const uint32_t*>(mq.qlo) == 0u && mq.qhi[0] >= 24 && mq.qhi[1] >= 24 &&
                                   mq.qhi[2] >= 24 && mq.qhi[3] >= 24;
            const bool rows_all = __all_sync(0xffffffffu, row_on);  // no row masked in this warp's 32 rows
            // colmask: only COLUMN ranges are masked (the window's first / last block, the ragged end of the chunk): the pipelined
            // path below, with the chunks of 32 columns that a range cuts masked as they arrive
            const bool plain = (full || tail_only) && rows_all;
            float (*s4)[32] = reinterpret_cast<float (*)[32]>(s);
            if (plain) {
                // the row maximum of 32 columns is taken while the next 32 are on their way out of TMEM
                float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
                tmem_ld32(s_tmem, s4[0]);
                tmem_ld_wait();
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    if (k < 3) tmem_ld32(s_tmem + 32 * (k + 1), s4[k + 1]);
                    if constexpr (P32) {  // the pad columns of this quarter's page ("mask the two extra positions")
#pragma unroll
                        for (int c = 24; c < 32; ++c)
                            if (c >= mq.qhi[k]) s[32 * k + c] = -INFINITY;
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {  // FMNMX3: two new values per instruction
                        const int b = 32 * k + 8 * i;
                        mx4[i] = max3(mx4[i], s[b], s[b + 1]);
                        mx4[i] = max3(mx4[i], s[b + 2], s[b + 3]);
                        mx4[i] = max3(mx4[i], s[b + 4], s[b + 5]);
                        mx4[i] = max3(mx4[i], s[b + 6], s[b + 7]);
                    }
                    if (k < 3) tmem_ld_wait();
                }
                tc_fence_before();
                mbar_arrive(&sm.s_free[p]);  // the tile sits in registers: QK_{t+2} may overwrite S_p
                mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * sl;  // log2 units (sl > 0)
            } else if (PAIRED && !P32 && mt.rmid > 0) {
                // paired SLC tile: this warp's rows attend ONE 64-token slot -- half the columns, half the exponentials
                const int hsel = (warp & 3) * 32 >= mt.rmid ? 1 : 0;  // warp-uniform: G_q is a multiple of 32
                if (warp_on) {
                    tmem_ld32(s_tmem + 64 * hsel, s4[0]);
                    tmem_ld32(s_tmem + 64 * hsel + 32, s4[1]);
                    tmem_ld_wait();
                }
                tc_fence_before();
                mbar_arrive(&sm.s_free[p]);
                if (warp_on) {
                    const int lo = hsel ? mt.lo1 : mt.lo0, hi = row_on ? (hsel ? mt.hi1 : mt.hi0) : 0;
                    if (!(rows_all && (hsel ? (mt.lo1 == 0 && mt.hi1 == 64) : (mt.lo0 == 0 && mt.hi0 == 64)))) {
                        mask_chunk<32>(s, range_mask32(lo, hi));
                        mask_chunk<32>(s + 32, range_mask32(lo - 32, hi - 32));
                    }
                    float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
#pragma unroll
                        for (int c = 0; c < 16; c += 2) mx4[i] = max3(mx4[i], s[16 * i + c], s[16 * i + c + 1]);
                    }
                    mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * sl;
                }
            } else if (!P32 && rows_all) {
                // only COLUMN ranges are masked (the window's first / last block, the ragged end of the chunk)
                tmem_ld32(s_tmem, s4[0]);
                tmem_ld32(s_tmem + 32, s4[1]);
                tmem_ld32(s_tmem + 64, s4[2]);
                tmem_ld32(s_tmem + 96, s4[3]);
                tmem_ld_wait();
                tc_fence_before();
                mbar_arrive(&sm.s_free[p]);
                float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                for (int k = 0; k < 4; ++k) {  // CTA-uniform tests: only the chunks of 32 columns that a range cuts pay for the mask
                    const int lo = (k < 2 ? mt.lo0 : mt.lo1) - 32 * (k & 1), hi = (k < 2 ? mt.hi0 : mt.hi1) - 32 * (k & 1);
                    if (lo > 0 || hi < 32) mask_chunk<32>(s + 32 * k, range_mask32(lo, hi));
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int b = 32 * k + 8 * i;
                        mx4[i] = max3(mx4[i], s[b], s[b + 1]);
                        mx4[i] = max3(mx4[i], s[b + 2], s[b + 3]);
                        mx4[i] = max3(mx4[i], s[b + 4], s[b + 5]);
                        mx4[i] = max3(mx4[i], s[b + 6], s[b + 7]);
                    }
                }
                mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * sl;
            } else {
                if (warp_on) {
                    tmem_ld32(s_tmem, s4[0]);
                    tmem_ld32(s_tmem + 32, s4[1]);
                    tmem_ld32(s_tmem + 64, s4[2]);
                    tmem_ld32(s_tmem + 96, s4[3]);
                    tmem_ld_wait();
                }
                tc_fence_before();
                mbar_arrive(&sm.s_free[p]);
                if (warp_on) {
                    const uint32_t on = row_on ? 0xffffffffu : 0u;
                    if constexpr (P32) {
#pragma unroll
                        for (int c = 0; c < 32; ++c) {
#pragma unroll
                            for (int qt = 0; qt < 4; ++qt)
                                if (!(row_on && c >= mq.qlo[qt] && c < mq.qhi[qt])) s[32 * qt + c] = -INFINITY;
                        }
                    } else {
                        mask_chunk<32>(s, range_mask32(mt.lo0, mt.hi0) & on);
                        mask_chunk<32>(s + 32, range_mask32(mt.lo0 - 32, mt.hi0 - 32) & on);
                        mask_chunk<32>(s + 64, range_mask32(mt.lo1, mt.hi1) & on);
                        mask_chunk<32>(s + 96, range_mask32(mt.lo1 - 32, mt.hi1 - 32) & on);
                    }
                    float mx4[4] = {s[0], s[1], s[2], s[3]};
#pragma unroll
                    for (int c = 4; c < 124; c += 8) {
                        mx4[0] = max3(mx4[0], s[c], s[c + 1]);
                        mx4[1] = max3(mx4[1], s[c + 2], s[c + 3]);
                        mx4[2] = max3(mx4[2], s[c + 4], s[c + 5]);
                        mx4[3] = max3(mx4[3], s[c + 6], s[c + 7]);
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) mx4[i] = fmaxf(mx4[i], s[124 + i]);
                    mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3])) * sl;
                }
            }
            // ---- max step, in tile order: tile t-1's step (other warpgroup) has published its reference
            if (t > 0) mbar_wait(&sm.max_done[(t - 1) & 1], ((t - 1) >> 1) & 1);
            {
                const float m_cur = sm.m_ref[row];
                if (m_cur != m_mine) {  // raised by the other warpgroup: bring this warpgroup's sums along
                    const float f = ex2(m_mine - m_cur);  // m_mine = -inf -> 0 (sums are 0 then anyway)
                    l3[0] *= f;
                    l3[1] *= f;
                    l3[2] *= f;
                    m_mine = m_cur;
                }
            }
            // lazy rescale: keep the stale reference max unless the new max exceeds it by > 2^8
            const bool grow = mx > m_mine + RESCALE_LOG2;
            if (__any_sync(0xffffffffu, grow)) {
                const float alpha = grow ? ex2(m_mine - mx) : 1.f;  // m_mine = -inf -> 0
                if (t > (SEG ? sm.seg_b[sg] : 0)) {
                    // every PV of this segment up to tile t-1 must have landed in O (the pipe completes in order); PV_t
                    // cannot start before this thread's P_t, so the accumulator is quiescent meanwhile
                    mbar_wait(&sm.pv_done[(t - 1) & 1], ((t - 1) >> 1) & 1);
                    tc_fence_after();
#pragma unroll
                    for (int c0 = 0; c0 < 128; c0 += 16) {
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
                if (grow) { m_mine = mx; sm.m_ref[row] = mx; }
            }
            mbar_arrive(&sm.max_done[t & 1]);  // release: m_ref and the rescaled O are visible to tile t+1's step
            // ---- exponentials of this tile against the reference (overlaps tile t+1's max step)
            uint32_t pk[64];
            if (PAIRED && warp_on && (mt.branch >> 8) != 0) {
                // paired tile, 64 columns: the other slot's half of P is zero for these rows
                const float m_use = (m_mine == -INFINITY) ? 0.f : m_mine;
                const uint64_t sl2 = f2(sl, sl), nm2 = f2(-m_use, -m_use);
                uint64_t rs2[4] = {0ull, 0ull, 0ull, 0ull};
                constexpr int LAG = 8;
#pragma unroll
                for (int c = 0; c < 32; ++c) unf2(fma2(f2(s[2 * c], s[2 * c + 1]), sl2, nm2), s[2 * c], s[2 * c + 1]);
#pragma unroll
                for (int c = 0; c < 32 + LAG; ++c) {
                    if (c < 32) {
                        asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(s[2 * c]));
                        asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(s[2 * c + 1]));
                    }
                    if (c >= LAG) {
                        const int d = c - LAG;
                        uint64_t v;
                        asm volatile("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(s[2 * d]), "f"(s[2 * d + 1]));
                        asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(rs2[d & 3]) : "l"(v));
                        asm volatile("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pk[d]) : "f"(s[2 * d + 1]), "f"(s[2 * d]));
                    }
                }
                float ra, rb;
                unf2(add2(add2(rs2[0], rs2[1]), add2(rs2[2], rs2[3])), ra, rb);
                l3[1] += ra + rb;  // a paired tile is an SLC tile
#pragma unroll
                for (int c = 32; c < 64; ++c) pk[c] = 0u;
            } else if (warp_on) {
                const float m_use = (m_mine == -INFINITY) ? 0.f : m_mine;
                const uint64_t sl2 = f2(sl, sl), nm2 = f2(-m_use, -m_use);
                uint64_t rs2[4] = {0ull, 0ull, 0ull, 0ull};
                // x = s * scale - ref for the whole row first, then one MUFU stream; the sum / bf16 pack of a pair follows its
                // exponentials 16 pairs later, so the consumers never sit right behind a MUFU result (volatile: keeps this order)
                constexpr int LAG = 16;
#pragma unroll
                for (int c = 0; c < 64; ++c) unf2(fma2(f2(s[2 * c], s[2 * c + 1]), sl2, nm2), s[2 * c], s[2 * c + 1]);
#pragma unroll
                for (int c = 0; c < 64 + LAG; ++c) {
                    if (c < 64) {
                        asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(s[2 * c]));
                        asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(s[2 * c + 1]));
                    }
                    if (c >= LAG) {
                        const int d = c - LAG;
                        uint64_t v;
                        asm volatile("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(s[2 * d]), "f"(s[2 * d + 1]));
                        asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(rs2[d & 3]) : "l"(v));
                        asm volatile("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(pk[d]) : "f"(s[2 * d + 1]), "f"(s[2 * d]));
                    }
                }
                float ra, rb;
                unf2(add2(add2(rs2[0], rs2[1]), add2(rs2[2], rs2[3])), ra, rb);
                const float rs = ra + rb;
                if ((mt.branch & 3) == BR_CMP) l3[0] += rs; else if ((mt.branch & 3) == BR_SLC) l3[1] += rs; else l3[2] += rs;
            } else {
#pragma unroll
                for (int c = 0; c < 64; ++c) pk[c] = 0u;
            }
            // ---- P_t -> TMEM: P_p is free once PV_{t-2} has completed (it is issued right behind QK_t, so it
            // has long finished when the exponentials of tile t are done; waiting earlier would stall)
            if (t >= 2) {
                mbar_wait(&sm.pv_done[p], ((t - 2) >> 1) & 1);
                tc_fence_after();
            }
            // (paired tile: the warp's 64 probabilities go to its slot's half of P, zeros to the other half)
            const int hsel = (PAIRED && (mt.branch >> 8) != 0 && (warp & 3) * 32 >= (mt.branch >> 8)) ? 1 : 0;
            tmem_st32(p_tmem + 32 * hsel, reinterpret_cast<uint32_t (*)[32]>(pk)[0]);
            tmem_st32(p_tmem + 32 * (hsel ^ 1), reinterpret_cast<uint32_t (*)[32]>(pk)[1]);
            tmem_st_wait();
            tc_fence_before();
            mbar_arrive(&sm.p_full[p]);
          }
          }

          // ---------------------------------------------------------------- end of the segment: gate, fuse, store (a8)
          const int tb = SEG ? sm.seg_b[sg] : 0, te = t_end;
          if (te > tb) mbar_wait(&sm.pv_done[(te - 1) & 1], ((te - 1) >> 1) & 1);  // in-order pipe: every PV of the segment has landed
          tc_fence_after();
          pdl_wait();  // the stores below (and the scratch they may read) are ordered behind the previous grid
          // exchange (m, l_cmp, l_slc, l_swa) between the two warpgroups
          float* exch = sm.exch;
          exch[(p * 128 + row) * 4 + 0] = m_mine;
          exch[(p * 128 + row) * 4 + 1] = l3[0];
          exch[(p * 128 + row) * 4 + 2] = l3[1];
          exch[(p * 128 + row) * 4 + 3] = l3[2];
          asm volatile("bar.sync 1, 256;" ::: "memory");
          const float m_o = exch[((p ^ 1) * 128 + row) * 4 + 0];
          // O is relative to the final shared reference (every raise rescaled it); a warpgroup that did not see
          // the last raise brings its sums along here
          const float m_all = sm.m_ref[row];
          const float m_sub = (m_all == -INFINITY) ? 0.f : m_all;
          const float a_me = ex2(m_mine - m_sub), a_ot = ex2(m_o - m_sub);
          float lb[3];
#pragma unroll
          for (int i = 0; i < 3; ++i) lb[i] = a_me * l3[i] + a_ot * exch[((p ^ 1) * 128 + row) * 4 + 1 + i];
          asm volatile("bar.sync 1, 256;" ::: "memory");  // exch and m_ref may be rewritten from here on
          tc_fence_after();
          // the next segment starts from an empty reference: reset by the warpgroup that owns its first tile (the other one
          // reads m_ref only behind that tile's max_done)
          if (sg + 1 < n_seg && p == (te & 1)) sm.m_ref[row] = -INFINITY;
          const float l_all = lb[0] + lb[1] + lb[2];
          float scale = l_all > 0.f ? 1.f / l_all : 0.f;
          if (a.gate[sg]) scale *= __ldg(a.gate[sg] + h);
          const bool first_seg = sg == 0, last_seg = sg == n_seg - 1;
          // warpgroup p handles output columns [64 p, 64 p + 64) of every row
#pragma unroll
          for (int cc = 0; cc < 2; ++cc) {
              const int c0 = p * 64 + cc * 32;
              if (c0 >= a.d_head) continue;  // head_dim 64: columns 64 .. 127 are padding
              float r[32];
              if (te > tb) {
                  tmem_ld32(o_tmem + c0, r);
                  tmem_ld_wait();
              }
#pragma unroll
              for (int i = 0; i < 32; ++i) r[i] = te > tb ? r[i] * scale : 0.f;
              if (srow < g.S) {
                  float4* acc = reinterpret_cast<float4*>(a.partial + ((int64_t)h * g.S + srow) * a.d_head + c0);
                  if (!first_seg) {  // add what the earlier segments left (written by this very thread)
#pragma unroll
                      for (int i = 0; i < 8; ++i) {
                          const float4 v = acc[i];
                          r[4 * i] += v.x; r[4 * i + 1] += v.y; r[4 * i + 2] += v.z; r[4 * i + 3] += v.w;
                      }
                  }
                  if (!last_seg) {
#pragma unroll
                      for (int i = 0; i < 8; ++i) acc[i] = make_float4(r[4 * i], r[4 * i + 1], r[4 * i + 2], r[4 * i + 3]);
                  } else {
                      uint4* dst = reinterpret_cast<uint4*>(a.out + ((int64_t)h * g.S + srow) * a.d_head + c0);
#pragma unroll
                      for (int i = 0; i < 4; ++i)
                          dst[i] = make_uint4(pack2(r[8 * i], r[8 * i + 1]), pack2(r[8 * i + 2], r[8 * i + 3]),
                                              pack2(r[8 * i + 4], r[8 * i + 5]), pack2(r[8 * i + 6], r[8 * i + 7]));
                  }
              }
          }
          if (p == 0 && srow < g.S) {
              const int kind = a.seg_kind[sg];
              const int64_t at = (int64_t)h * g.S + srow;
              if (a.lse_cmp && kind == SEG_CMP) a.lse_cmp[at] = lb[0] > 0.f ? (m_sub + log2f(lb[0])) * ln2 : -INFINITY;
              if (a.lse_slc && (kind == SEG_SLC || kind == SEG_JOINT)) a.lse_slc[at] = lb[1] > 0.f ? (m_sub + log2f(lb[1])) * ln2 : -INFINITY;
              if (a.lse_swa && (kind == SEG_SWA || kind == SEG_JOINT)) a.lse_swa[at] = lb[2] > 0.f ? (m_sub + log2f(lb[2])) * ln2 : -INFINITY;
          }
          if (!last_seg) {
              tc_fence_before();
              mbar_arrive(&sm.o_free);  // O has been read: the first PV of the next segment may overwrite it
          }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 9) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512));
    }
}

}  // namespace tc

// ------------------------------------------------------------------------------------- host side
static AttnGeom make_attn_geom(const Cache* c, int32_t n_q, const omnimem_attn_params_t& p)
{
    AttnGeom g;
    g.H = c->H;
    g.S = n_q;
    g.B = c->B;
    g.K = p.top_k;
    g.G = p.group_tokens;
    g.R = (int32_t)ceil_div64(n_q, p.group_tokens);
    g.max_blocks = c->max_blocks;
    g.pool_blocks = c->pool_blocks;
    g.P = c->P;
    g.bpc = c->bpc;
    g.spb = c->P / 64;  // 0 with 32-row pages: a slot then holds two blocks
    g.n_hist = c->n_hist;
    g.n_b = (int32_t)ceil_div64(c->n_hist, c->B);
    g.last_len = g.n_b > 0 ? (int32_t)(c->n_hist - (int64_t)(g.n_b - 1) * c->B) : c->B;
    int64_t win_start = c->n_hist - p.window_tokens;
    if (win_start < 0) win_start = 0;
    if (p.window_tokens == 0) win_start = c->n_hist;
    g.win_start = win_start;
    g.first_win_blk = (int32_t)(win_start / c->B);
    const int32_t n_win_blk = (win_start < c->n_hist) ? g.n_b - g.first_win_blk : 0;
    g.n_win_slots = c->P == 32 ? (n_win_blk + 1) / 2 : g.spb * n_win_blk;
    g.n_cur_slots = (int32_t)ceil_div64(n_q, 64);
    g.slc_slots = c->P == 32 ? (p.top_k + 1) / 2 : p.top_k * g.spb;
    return g;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// bf16 tensor [n2][n1][d] (d = 64 or 128) with element strides (stride1, stride2); box = 64 x box_rows (x 1), SWIZZLE_128B.
// With d = 64 a box at d-coordinate 64 lies out of bounds: TMA writes zeros (the padding half of a 128-wide tile).
static int32_t encode_map(CUtensorMap* m, const void* base, int d, int rank, uint64_t n1, uint64_t n2, uint64_t stride1_el,
                          uint64_t stride2_el, uint32_t box_rows)
{
    EncodeTiledFn enc = get_encode();
    if (!enc) return fail(OMNIMEM_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint64_t dims[3] = {(cuuint64_t)d, n1, n2};
    cuuint64_t strides[2] = {stride1_el * 2, stride2_el * 2};
    cuuint32_t box[3] = {64, box_rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(OMNIMEM_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return OMNIMEM_OK;
}

// bf16 tensor [n2][n1][d] seen as {64 (one half of d), n1 rows, d / 64 halves, n2}: one box {64, box_rows, 2, 1}
// lands in shared memory as [half][box_rows][128 B], the layout the UMMA descriptors read (SWIZZLE_128B); with d = 64 the
// second half of every box is out of bounds and arrives as zeros.
static int32_t encode_map_split(CUtensorMap* m, const void* base, int d, int rank, uint64_t n1, uint64_t n2, uint64_t stride1_el,
                                uint64_t stride2_el, uint32_t box_rows)
{
    EncodeTiledFn enc = get_encode();
    if (!enc) return fail(OMNIMEM_ECUDA, "cuTensorMapEncodeTiled entry point not found");
    cuuint64_t dims[4] = {64, n1, (cuuint64_t)(d / 64), n2};
    cuuint64_t strides[3] = {stride1_el * 2, 128, stride2_el * 2};
    cuuint32_t box[4] = {64, box_rows, 2, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, (cuuint32_t)rank, const_cast<void*>(base), dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(OMNIMEM_ECUDA, "cuTensorMapEncodeTiled (split-d map) failed (%d)", (int)r);
    return OMNIMEM_OK;
}

size_t attn_tcgen05_workspace_bytes(int32_t H, int32_t n_q, int32_t D, int32_t fuse_mode)
{
    if (fuse_mode != OMNIMEM_FUSE_GATED) return 0;
    return (size_t)H * n_q * D * 4;
}

int32_t launch_attn_tcgen05(const AttnArgs& x)
{
    Cache* c = const_cast<Cache*>(x.cache);
    const bool gated = x.p.fuse_mode == OMNIMEM_FUSE_GATED;
    const bool three = x.gate_cmp != nullptr;  // full Eq. 1: CMP + SLC + SWA (GATED only, checked by the caller)
    if (gated) {
        const size_t need = attn_tcgen05_workspace_bytes(c->H, x.n_q, c->D, x.p.fuse_mode);
        if (!x.workspace || x.workspace_bytes < need) return fail(OMNIMEM_ECAPACITY, "attn workspace: need %zu bytes, got %zu", need, x.workspace_bytes);
    }
    const uint64_t pool_rows = (uint64_t)c->H * c->pool_blocks * c->P;
    if (!c->tmaps_ready) {
        if (int32_t rc = encode_map((CUtensorMap*)c->tmap_k, c->k_pages, c->D, 2, pool_rows, 1, c->D, 0, 64)) return rc;
        if (int32_t rc = encode_map_split((CUtensorMap*)c->tmap_v, c->v_pages, c->D, 3, pool_rows, 1, c->D, 0, 64)) return rc;
        // 32-row pages: boxes of one page x one half of D, for K and V alike
        if (int32_t rc = encode_map((CUtensorMap*)c->tmap_k32, c->k_pages, c->D, 2, pool_rows, 1, c->D, 0, 32)) return rc;
        if (int32_t rc = encode_map((CUtensorMap*)c->tmap_v32, c->v_pages, c->D, 2, pool_rows, 1, c->D, 0, 32)) return rc;
        c->tmaps_ready = true;
    }
    const uint64_t cmp_rows = (uint64_t)c->H * c->max_blocks;
    if (three && !c->tmaps_cmp_ready) {
        // the compressed cache [H][max_blocks][D] seen as one pool of rows, like the page pools
        if (int32_t rc = encode_map((CUtensorMap*)c->tmap_kc, c->pooled_k, c->D, 2, cmp_rows, 1, c->D, 0, 64)) return rc;
        if (int32_t rc = encode_map_split((CUtensorMap*)c->tmap_vc, c->pooled_v, c->D, 3, cmp_rows, 1, c->D, 0, 64)) return rc;
        c->tmaps_cmp_ready = true;
    }
    // per-call tensors: re-encoded only when a pointer, a stride or the length changed since the previous call on this cache
    if (c->call_q != x.q || c->call_k != x.k_cur || c->call_v != x.v_cur || c->call_n != x.n_q || c->call_st != x.stride_tok || c->call_sh != x.stride_head) {
        c->call_q = nullptr;
        if (int32_t rc = encode_map((CUtensorMap*)c->tmap_q, x.q, c->D, 3, x.n_q, c->H, x.stride_tok, x.stride_head, 128)) return rc;
        if (int32_t rc = encode_map((CUtensorMap*)c->tmap_kcur, x.k_cur, c->D, 3, x.n_q, c->H, x.stride_tok, x.stride_head, 64)) return rc;
        if (int32_t rc = encode_map_split((CUtensorMap*)c->tmap_kcur128, x.k_cur, c->D, 4, x.n_q, c->H, x.stride_tok, x.stride_head, 128)) return rc;
        if (int32_t rc = encode_map_split((CUtensorMap*)c->tmap_vcur, x.v_cur, c->D, 4, x.n_q, c->H, x.stride_tok, x.stride_head, 64)) return rc;
        c->call_q = x.q; c->call_k = x.k_cur; c->call_v = x.v_cur; c->call_n = x.n_q; c->call_st = x.stride_tok; c->call_sh = x.stride_head;
    }
    const CUtensorMap &tq = *(const CUtensorMap*)c->tmap_q, &tk = *(const CUtensorMap*)c->tmap_kcur, &tk128 = *(const CUtensorMap*)c->tmap_kcur128,
                      &tv = *(const CUtensorMap*)c->tmap_vcur;

    tc::Args a;
    a.g = make_attn_geom(c, x.n_q, x.p);
    a.ptr_table = x.ptr_table;
    a.page_map = c->page_map;
    a.out = (__nv_bfloat16*)x.out;
    a.partial = (float*)x.workspace;
    a.scale_log2 = x.p.softmax_scale * 1.4426950408889634f;
    a.pool_rows = (int32_t)pool_rows;
    a.cmp_rows = (int32_t)cmp_rows;
    a.d_head = c->D;
    // JOINT tile order.  64 / 128-row pages: SLC last (paired tiles are cheap anywhere in the sequence and the selection overlaps the
    // window tiles).  32-row pages (the paper's geometry): SLC first -- its selection fills every SM for its whole duration (R = 312
    // groups per head), so nothing overlaps, and the mostly masked G_q = 15 tiles cost less at the head of a CTA than at its tail
    // (attend 538 against 555 us).
    a.swa_first = c->P == 32 ? 0 : 1;
    const int64_t HS = (int64_t)c->H * x.n_q;
    float* lse = x.lse_out;  // [2][H][S] (slc, swa) or, with the CMP branch, [3][H][S] (cmp, slc, swa)
    a.lse_cmp = three ? lse : nullptr;
    a.lse_slc = lse ? lse + (three ? HS : 0) : nullptr;
    a.lse_swa = lse ? lse + (three ? 2 * HS : HS) : nullptr;
    a.cmp_blocks = three ? (int32_t)ceil_div64(c->n_hist, c->B) : 0;
    // segments in sequence order: [CMP] SWA SLC, each with its own softmax and gate (Eq. 1); JOINT: one segment, no gate
    a.gate[0] = a.gate[1] = a.gate[2] = nullptr;
    a.seg_kind[0] = a.seg_kind[1] = a.seg_kind[2] = tc::SEG_JOINT;
    if (!gated) {
        a.n_seg = 1;
    } else {
        int n = 0;
        if (three) { a.seg_kind[n] = tc::SEG_CMP; a.gate[n] = x.gate_cmp; ++n; }
        if (tc::GATED_SWA_FIRST) {
            a.seg_kind[n] = tc::SEG_SWA; a.gate[n] = x.gate_swa; ++n;
            a.seg_kind[n] = tc::SEG_SLC; a.gate[n] = x.gate_slc; ++n;
        } else {
            a.seg_kind[n] = tc::SEG_SLC; a.gate[n] = x.gate_slc; ++n;
            a.seg_kind[n] = tc::SEG_SWA; a.gate[n] = x.gate_swa; ++n;
        }
        a.n_seg = n;
    }
    const int smem = (int)sizeof(tc::Smem) + 1024;
    {   // the opt-in is per device: remember which devices already have it
        static std::atomic<uint64_t> attr_devices{0};
        int dev = 0;
        cudaGetDevice(&dev);
        const uint64_t bit = 1ull << (dev & 63);
        if (!(attr_devices.load(std::memory_order_acquire) & bit)) {
            cudaError_t e = cudaFuncSetAttribute(tc::attn_tcgen05_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(tc::attn_tcgen05_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(tc::attn_tcgen05_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(tc::attn_tcgen05_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
            attr_devices.fetch_or(bit, std::memory_order_release);
        }
    }
    dim3 grid((unsigned)ceil_div64(x.n_q, tc::M_TILE), (unsigned)c->H);
    const CUtensorMap* pk = (const CUtensorMap*)c->tmap_k;
    const CUtensorMap* pv = (const CUtensorMap*)c->tmap_v;
    const CUtensorMap* ck = three ? (const CUtensorMap*)c->tmap_kc : pk;
    const CUtensorMap* cv = three ? (const CUtensorMap*)c->tmap_vc : pv;
    const bool seg = a.n_seg > 1, p32 = c->P == 32;
    if (p32) {  // 32-row pages: the pool maps are the 2-D maps with boxes of one page x one half of D
        pk = (const CUtensorMap*)c->tmap_k32;
        pv = (const CUtensorMap*)c->tmap_v32;
        if (!three) { ck = pk; cv = pv; }
    }
    // Launch policy.  Behind a selection that fits one wave of CTAs (config 2: 120 CTAs of select_fused_kernel) the kernel is
    // launched programmatically: its CTAs start on the SMs the selection leaves free and run the window tiles while the selection
    // finishes (step 305 -> 295 us).  Behind a selection of several waves or several kernels (long histories, 40 heads, G_q = 15) an
    // attention CTA that slips in holds its SM for its whole lifetime and the selection behind it loses that SM: plain stream
    // order is faster there (config 3: step 416 -> 379 us, wan14b 1008 -> 989 us).
    bool early = true;
    {
        static std::atomic<int> sm_count[64];
        int dev = 0;
        cudaGetDevice(&dev);
        int n_sm = sm_count[dev & 63].load(std::memory_order_relaxed);
        if (n_sm == 0) {
            cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
            sm_count[dev & 63].store(n_sm, std::memory_order_relaxed);
        }
        early = select_launch_ctas(c->H, x.n_q, x.p.group_tokens, a.g.n_b) <= (int64_t)n_sm;
    }
    auto launch = [&](auto kernel) {
        if (!early) return launch_plain(kernel, grid, dim3(tc::THREADS), (size_t)smem, x.stream, tq, tk, tk128, tv, *pk, *pv, *ck, *cv, a);
        return launch_pdl(kernel, grid, dim3(tc::THREADS), (size_t)smem, x.stream, tq, tk, tk128, tv, *pk, *pv, *ck, *cv, a);
    };
    cudaError_t le = seg ? (p32 ? launch(tc::attn_tcgen05_kernel<true, true>) : launch(tc::attn_tcgen05_kernel<true, false>))
                         : (p32 ? launch(tc::attn_tcgen05_kernel<false, true>) : launch(tc::attn_tcgen05_kernel<false, false>));
    if (le != cudaSuccess) return fail(OMNIMEM_ECUDA, "sparse_attn launch: %s", cudaGetErrorString(le));
    count_launch();
    return check_launch("sparse_attn(tcgen05)");
}

}  // namespace omnimem
