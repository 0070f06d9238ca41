// Work decomposition of the attention kernel (a6-a8): units, steps, the work tape and its pieces.
// Shared by the host (workspace sizing, launch geometry) and every warp role of the kernel, which all
// derive the same piece list from (plan, blockIdx) -- nothing but data moves through memory.
//
//   unit   = two adjacent 128-row query tiles of one head (the last unit of a head may hold one tile).
//            Both tiles consume every window / current-chunk / compressed K,V stage that the CTA loads,
//            so a stage's bytes enter the SM once per TWO tiles of tensor work.
//   step   = 64 KV tokens.  A unit's step sequence is  [CMP: ceil(N_b/64) steps over the compressed cache,
//            three-branch call only] [SWA: window blocks through page_map, then the current chunk]
//            [SLC: per tile, the K selected blocks of every query group that overlaps the tile, through
//            ptr_table].  CMP and SWA steps are shared by the two tiles; an SLC step serves each tile from
//            its own block (shared only when both tiles lie in one query group).  The SLC steps -- the only
//            ones that depend on omnimem_select -- come last.
//   tape   = the units' step sequences laid end to end, T steps each.  CTA c of n_cta owns tape positions
//            [cut(c), cut(c+1)); cuts fall anywhere inside a unit (a unit's KV range is split between CTAs
//            when that balances the SMs), but snap to a unit boundary that is only a few steps away.
//   piece  = the steps of one unit inside one CTA that belong to one softmax state: the whole range in
//            JOINT mode, one piece per branch in GATED mode (Eq. 1 keeps a separate softmax per branch,
//            PAPER.md:66).  A unit with a single piece is finished by its CTA; otherwise every piece leaves an
//            unnormalised partial (O, m, l per branch) in the workspace and the piece that arrives last
//            merges them in piece order (deterministic) and writes the output.
#pragma once
#include <stdint.h>

#include "attn_schedule.cuh"

namespace omnimem {

constexpr int PLAN_MAX_PIECES_PER_UNIT = 8;
constexpr int PLAN_MIN_STEPS_PER_CTA = 16;
constexpr int PLAN_SNAP = 6;

struct AttnPlan {
    AttnGeom g;
    int32_t n_qt;             // 128-row query tiles per head
    int32_t units_per_head;   // ceil(n_qt / 2)
    int32_t n_units;          // H * units_per_head
    int32_t n_cmp, n_swa;     // shared steps per unit
    int32_t n_slc;            // SLC steps per unit = max over tiles of (groups overlapping the tile) * K * B/64
    int32_t T;                // steps per unit
    int32_t L;                // tape positions per CTA
    int32_t n_cta;
    int32_t gated;            // 1: one softmax state per branch; 0: one state for SWA + SLC (JOINT)
    int32_t max_pieces;       // most pieces any unit is split into (workspace stride)
    int32_t cmp_rows;         // rows of the compressed-cache pools (H * max_blocks)
};

struct AttnPiece {
    int32_t unit, h, qt0, n_tiles;  // head, first query tile, 1 or 2 tiles
    int32_t s0, s1;                 // steps [s0, s1) in the unit's sequence
    int32_t ord, npc;               // position among the unit's pieces, number of them
    int32_t new_unit;               // first piece of this unit in the CTA: Q tiles must be loaded
    int32_t last_of_unit;           // last piece of this unit in the CTA: Q tiles are free afterwards
    int32_t n_slc[2];               // SLC steps of each tile
    int32_t g_first[2];             // first query group of each tile
    int32_t slc_shared;             // both tiles lie in ONE query group: SLC steps are shared too
};

__host__ __device__ inline int64_t plan_cut(const AttnPlan& p, int c)
{
    const int64_t total = (int64_t)p.n_units * p.T;
    int64_t x = (int64_t)c * p.L;
    if (x >= total) return total;
    const int64_t r = x % p.T;
    if (r < PLAN_SNAP) x -= r;
    else if (p.T - r < PLAN_SNAP) x += p.T - r;
    return x;
}

// number of softmax states the unit-local step range [lo, hi) touches
__host__ __device__ inline int plan_states(const AttnPlan& p, int lo, int hi)
{
    if (hi <= lo) return 0;
    if (!p.gated) return 1;
    const int b1 = p.n_cmp, b2 = p.n_cmp + p.n_swa;
    return (lo < b1 && hi > 0 ? 1 : 0) + (lo < b2 && hi > b1 ? 1 : 0) + (hi > b2 && lo < p.T ? 1 : 0);
}

// the CTA that owns tape position x
__host__ __device__ inline int plan_owner(const AttnPlan& p, int64_t x)
{
    int c = (int)(x / p.L);
    if (c >= p.n_cta) c = p.n_cta - 1;
    while (c > 0 && plan_cut(p, c) > x) --c;
    while (c + 1 < p.n_cta && plan_cut(p, c + 1) <= x) ++c;
    return c;
}

// pieces of unit u: total count, and how many precede tape position `before` (the ordinal of a piece starting there)
__host__ __device__ inline void plan_unit_pieces(const AttnPlan& p, int u, int64_t before, int* n_total, int* n_before)
{
    const int64_t u0 = (int64_t)u * p.T, u1 = u0 + p.T;
    int tot = 0, bef = 0;
    for (int c = plan_owner(p, u0); c < p.n_cta; ++c) {
        const int64_t a = plan_cut(p, c), b = plan_cut(p, c + 1);
        if (a >= u1) break;
        const int lo = (int)((a > u0 ? a : u0) - u0), hi = (int)((b < u1 ? b : u1) - u0);
        const int n = plan_states(p, lo, hi);
        tot += n;
        if (u0 + lo < before) bef += n;  // ranges are disjoint and ascending: a range starting before `before` lies wholly before it
    }
    *n_total = tot;
    *n_before = bef;
}

__host__ __device__ inline void plan_tile_groups(const AttnGeom& g, int qt, int* g_first, int* n_groups)
{
    const int q0 = qt * 128;
    const int q_last = (q0 + 128 < g.S ? q0 + 128 : g.S) - 1;
    *g_first = q0 / g.G;
    *n_groups = (g.n_hist > 0 && q0 < g.S) ? (q_last / g.G - q0 / g.G + 1) : 0;
}

// Pieces of CTA c in PROCESSING order: units in descending tape order (the head of the next unit, which holds no SLC
// step, comes first; whatever reaches a unit's SLC tail comes as late as possible), a unit's pieces in branch order.
// Every warp role walks its own iterator: a CTA may own any number of pieces, none is stored.
struct PieceIter {
    int64_t a, b;     // the CTA's tape range
    int u, u_lo;      // current unit (descending), last unit
    int k;            // next branch slot of the current unit (0 .. 2)
    int lo, hi;       // the CTA's step range inside the current unit
    int tot, bef;     // pieces of the current unit; pieces before this CTA's range
    int emitted;      // pieces of the current unit emitted by this CTA so far
    bool have_next;   // `next` was produced ahead of time (to know whether a piece is the unit's last in this CTA)
    AttnPiece nxt;

    __host__ __device__ void load_unit(const AttnPlan& p)
    {
        const int64_t u0 = (int64_t)u * p.T;
        lo = (int)((a > u0 ? a : u0) - u0);
        hi = (int)((b < u0 + p.T ? b : u0 + p.T) - u0);
        plan_unit_pieces(p, u, u0 + lo, &tot, &bef);
        k = 0;
        emitted = 0;
    }
    __host__ __device__ bool produce(const AttnPlan& p, AttnPiece& pc)
    {
        while (u >= u_lo) {
            while (k < 3) {
                const int kk = k++;
                int s0, s1;
                if (p.gated) {
                    const int b0 = kk == 0 ? 0 : (kk == 1 ? p.n_cmp : p.n_cmp + p.n_swa);
                    const int b1 = kk == 0 ? p.n_cmp : (kk == 1 ? p.n_cmp + p.n_swa : p.T);
                    s0 = lo > b0 ? lo : b0;
                    s1 = hi < b1 ? hi : b1;
                    if (s1 <= s0) continue;
                } else {
                    if (kk != 0) continue;  // JOINT: the single state covers the whole range
                    s0 = lo;
                    s1 = hi;
                }
                pc.unit = u;
                pc.h = u / p.units_per_head;
                pc.qt0 = (u % p.units_per_head) * 2;
                pc.n_tiles = (pc.qt0 + 1 < p.n_qt) ? 2 : 1;
                pc.s0 = s0;
                pc.s1 = s1;
                pc.ord = bef + emitted;
                pc.npc = tot;
                pc.new_unit = emitted == 0;
                pc.last_of_unit = 0;
                {
                    int gf = 0, ng = 0;
                    plan_tile_groups(p.g, pc.qt0, &gf, &ng);
                    pc.g_first[0] = gf;
                    pc.n_slc[0] = ng * p.g.slc_slots;
                    gf = 0;
                    ng = 0;
                    if (pc.n_tiles == 2) plan_tile_groups(p.g, pc.qt0 + 1, &gf, &ng);
                    pc.g_first[1] = gf;
                    pc.n_slc[1] = ng * p.g.slc_slots;
                }
                pc.slc_shared = pc.n_tiles == 2 && pc.n_slc[0] == p.g.slc_slots && pc.n_slc[1] == p.g.slc_slots && pc.g_first[0] == pc.g_first[1];
                ++emitted;
                return true;
            }
            --u;
            if (u >= u_lo) load_unit(p);
        }
        return false;
    }
    __host__ __device__ void init(const AttnPlan& p, int c)
    {
        a = plan_cut(p, c);
        b = plan_cut(p, c + 1);
        have_next = false;
        if (b <= a) { u = -1; u_lo = 0; return; }
        u_lo = (int)(a / p.T);
        u = (int)((b - 1) / p.T);
        load_unit(p);
        have_next = produce(p, nxt);
    }
    // next piece of the CTA; false when none is left
    __host__ __device__ bool next(const AttnPlan& p, AttnPiece& pc)
    {
        if (!have_next) return false;
        pc = nxt;
        have_next = produce(p, nxt);
        pc.last_of_unit = (!have_next || nxt.unit != pc.unit) ? 1 : 0;
        return true;
    }
};

// activity of a step: which tiles take part, and whether they share the K / V stage
struct StepAct {
    bool act0, act1, shared;
};
__host__ __device__ inline StepAct plan_step(const AttnPlan& p, const AttnPiece& pc, int s)
{
    StepAct r;
    const int off = p.n_cmp + p.n_swa;
    if (s < off) {
        r.act0 = true;
        r.act1 = pc.n_tiles == 2;
        r.shared = r.act1;
    } else {
        const int v = s - off;
        r.act0 = v < pc.n_slc[0];
        r.act1 = pc.n_tiles == 2 && v < pc.n_slc[1];
        r.shared = pc.slc_shared && r.act0 && r.act1;
    }
    return r;
}

}  // namespace omnimem
