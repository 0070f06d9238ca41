// KV "slot" schedule shared by the attention kernels (a6-a8).
//
// A slot is 64 consecutive KV tokens from one source.  For a query tile (head h, rows
// [q0, q0 + M)) the slot sequence is
//     [ SLC: for every query group r that overlaps the tile, its K selected blocks, read through
//            ptr_table (B/64 slots per block), padded to a multiple of SPT slots per group ]
//     [ SWA: the history blocks that intersect the window, through page_map ]
//     [ SWA: the current chunk, 64 tokens at a time ]                    padded to a multiple of SPT
// where SPT = slots per KV tile of the kernel.  PAIRED SLC tiles (pair != 0; SPT = 2, G a multiple of 32, pages of 64 / 128
// rows, at least two groups in the tile): the groups are taken two at a time and a tile holds slot j of the even group AND
// slot j of the odd group -- rows of the even group attend the tile's first 64 columns only, rows of the odd group its last
// 64 -- so that every softmax warp has work in every SLC tile, and only 64 columns of it (with two slots of ONE group per tile
// the other group's warps sit the tile out while its own warps pay for all 128 columns).  With swa_first the two SWA segments lead and the SLC segment -- the only
// one that depends on omnimem_select's output -- comes last, so a kernel launched behind the selection by programmatic
// dependent launch needs ptr_table only for its final slots.  Every role of a kernel (loader, MMA issuer,
// softmax) recomputes the same slot from (h, q0, index), so nothing but data moves through smem.
#pragma once
#include <stdint.h>

#include "common.cuh"

namespace omnimem {

struct AttnGeom {
    int32_t H, S, B, K, G, R;
    int32_t max_blocks;
    int32_t pool_blocks;    // pages per head of the K / V pools (= max_blocks unless chunks are offloaded)
    int32_t P;              // rows per page (32, 64, 128); a block's B <= P tokens are its first rows
    int32_t bpc;            // blocks per chunk of the two-level page map (0: one entry per block)
    int32_t spb;            // slots per block = P / 64 (P >= 64); with P = 32 a slot holds TWO blocks (spb = 0)
    int32_t n_b;            // ceil(n_hist / B)
    int32_t last_len;       // valid tokens of logical block n_b - 1 (B if not ragged)
    int32_t first_win_blk;  // first logical block that intersects the window
    int32_t n_win_slots;    // spb * (n_b - first_win_blk), 0 if the window holds no history
    int32_t n_cur_slots;    // ceil(S / 64)
    int32_t slc_slots;      // K * spb (per group, before padding)
    int64_t n_hist, win_start;
};

enum SlotKind : int32_t { SLOT_NONE = 0, SLOT_HIST = 1, SLOT_CUR = 2, SLOT_CMP = 3 };  // CMP: rows of the compressed cache

struct SlotBase {
    int32_t kind;
    int32_t row;     // HIST: first row in the page pool viewed as [H*max_blocks*P][D]; CUR: first token
    int32_t lo, hi;  // valid tokens of the slot: [lo, hi) within 0..64  (P = 32: of its FIRST page, within 0..32)
};
struct Slot : SlotBase {  // 32-row pages only: the slot's second page
    int32_t row2;      // its first pool row, -1 = none (zero fill, masked)
    int32_t lo2, hi2;  // its valid tokens, within 0..32
};

struct TileRows {
    int32_t lo, hi;  // query rows of the tile (relative to q0) that attend to this KV tile
    int32_t is_slc;
    int32_t mid;     // paired SLC tile: rows [lo, mid) attend slot 0 only, rows [mid, hi) slot 1 only; 0 otherwise
};

// Per query tile: counts derived from the geometry.
struct TileSched {
    int32_t h, q0, m_rows;    // m_rows: tile height M
    int32_t g_first, n_groups;
    int32_t slc_slots_padded;  // per group, multiple of SPT
    int32_t n_slc_slots;       // n_groups * slc_slots_padded
    int32_t n_swa_slots;       // (n_win_slots + n_cur_slots) padded to SPT
    int32_t n_slots;
    int32_t swa_first;         // 1: [SWA][SLC] -- the slots that depend on omnimem_select come last; 0: [SLC][SWA]
    int32_t pair;              // 1: paired SLC tiles (two groups per tile, one slot each)

    // index of a slot inside its segment
    __device__ __forceinline__ bool in_slc(int slot_idx) const { return swa_first ? slot_idx >= n_swa_slots : slot_idx < n_slc_slots; }
    __device__ __forceinline__ int slc_index(int slot_idx) const { return swa_first ? slot_idx - n_swa_slots : slot_idx; }
    __device__ __forceinline__ int swa_index(int slot_idx) const { return swa_first ? slot_idx : slot_idx - n_slc_slots; }

    __device__ __forceinline__ void init(const AttnGeom& g, int h_, int q0_, int M, int spt, int swa_first_ = 0)
    {
        swa_first = swa_first_;
        h = h_;
        q0 = q0_;
        m_rows = M;
        const int q_last = min(q0 + M, g.S) - 1;
        g_first = q0 / g.G;
        n_groups = (g.n_hist > 0) ? (q_last / g.G - g_first + 1) : 0;
        pair = (spt == 2 && g.P >= 64 && g.G % 32 == 0 && n_groups >= 2) ? 1 : 0;
        slc_slots_padded = pair ? g.slc_slots : (g.slc_slots + spt - 1) / spt * spt;
        n_slc_slots = pair ? (n_groups + 1) / 2 * 2 * slc_slots_padded : n_groups * slc_slots_padded;
        n_swa_slots = (g.n_win_slots + g.n_cur_slots + spt - 1) / spt * spt;
        n_slots = n_slc_slots + n_swa_slots;
    }

    __device__ __forceinline__ TileRows rows(const AttnGeom& g, int slot_idx) const
    {
        TileRows t;
        t.mid = 0;
        if (in_slc(slot_idx) && pair) {  // called with the tile's first slot: groups ra (slot 0) and ra + 1 (slot 1)
            const int ra = g_first + 2 * ((slc_index(slot_idx) >> 1) / slc_slots_padded);
            t.lo = max(ra * g.G - q0, 0);
            t.mid = min(min((ra + 1) * g.G, g.S) - q0, m_rows);
            t.hi = max(min(min((ra + 2) * g.G, g.S) - q0, m_rows), t.mid);
            t.is_slc = 1;
        } else if (in_slc(slot_idx)) {
            const int r = g_first + slc_index(slot_idx) / slc_slots_padded;
            t.lo = max(r * g.G - q0, 0);
            t.hi = min(min((r + 1) * g.G, g.S) - q0, m_rows);
            t.is_slc = 1;
        } else {
            t.lo = 0;
            t.hi = m_rows;
            t.is_slc = 0;
        }
        return t;
    }

    template <bool P32>
    __device__ __forceinline__ Slot slot(const AttnGeom& g, const int32_t* __restrict__ ptr_table,
                                         const int32_t* __restrict__ page_map, int slot_idx) const
    {
        Slot s;
        s.kind = SLOT_NONE;
        s.row = 0;
        s.lo = 0;
        s.hi = 0;
        s.row2 = -1;
        s.lo2 = 0;
        s.hi2 = 0;
        if (in_slc(slot_idx)) {
            const int si = slc_index(slot_idx);
            // paired tiles: slot si = (tile si / 2, half si % 2): group 2 * (tile / slots per group) + half, slot tile % slots per group
            const int r = g_first + (pair ? 2 * ((si >> 1) / slc_slots_padded) + (si & 1) : si / slc_slots_padded);
            const int j = pair ? (si >> 1) % slc_slots_padded : si % slc_slots_padded;
            if (j >= g.slc_slots || r >= g_first + n_groups) return s;
            const int32_t last_page = g.last_len < g.B ? page_of(page_map, h, g.n_b - 1, g.max_blocks, g.bpc) : -1;
            if constexpr (P32) {  // two selected blocks per slot, each in the first B rows of its 32-row page
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const int t = 2 * j + u;
                    const int32_t page = t < g.K ? __ldg(ptr_table + ((int64_t)h * g.R + r) * g.K + t) : -1;
                    if (page < 0) continue;
                    const int len = page == last_page ? g.last_len : g.B;
                    const int32_t row = (int32_t)(((int64_t)h * g.pool_blocks + page) * 32);
                    s.kind = SLOT_HIST;
                    if (u == 0) { s.row = row; s.hi = len; } else { s.row2 = row; s.hi2 = len; }
                }
                if (s.kind == SLOT_HIST && s.hi == 0) s.row = -1;  // only the second page exists
                return s;
            }
            const int t = j / g.spb, sub = j % g.spb;
            const int32_t page = __ldg(ptr_table + ((int64_t)h * g.R + r) * g.K + t);
            if (page < 0) return s;  // Alg. 1 lines 20-22: skip
            const int len = page == last_page ? g.last_len : g.B;
            const int hi = min(len - sub * 64, 64);
            if (hi <= 0) return s;
            s.kind = SLOT_HIST;
            s.row = (int32_t)(((int64_t)h * g.pool_blocks + page) * g.P + sub * 64);
            s.hi = hi;
            return s;
        }
        int w = swa_index(slot_idx);
        if (w < g.n_win_slots) {
            if constexpr (P32) {  // two window blocks per slot
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const int b = g.first_win_blk + 2 * w + u;
                    if (b >= g.n_b) continue;
                    const int64_t base = (int64_t)b * g.B;
                    const int lo = (int)max((int64_t)0, g.win_start - base);
                    const int hi = (int)min((int64_t)g.B, g.n_hist - base);
                    if (lo >= hi) continue;
                    const int32_t wp = page_of(page_map, h, b, g.max_blocks, g.bpc);
                    if (wp < 0) continue;  // a window chunk is always resident; a missing one is skipped, never dereferenced
                    const int32_t row = (int32_t)(((int64_t)h * g.pool_blocks + wp) * 32);
                    s.kind = SLOT_HIST;
                    if (u == 0) { s.row = row; s.lo = lo; s.hi = hi; } else { s.row2 = row; s.lo2 = lo; s.hi2 = hi; }
                }
                if (s.kind == SLOT_HIST && s.hi == 0) s.row = -1;
                return s;
            }
            const int b = g.first_win_blk + w / g.spb, sub = w % g.spb;
            const int64_t base = (int64_t)b * g.B + sub * 64;
            const int lo = (int)max((int64_t)0, g.win_start - base);
            const int hi = (int)min((int64_t)min(64, g.B - sub * 64), g.n_hist - base);
            if (lo >= hi) return s;
            const int32_t page = page_of(page_map, h, b, g.max_blocks, g.bpc);
            if (page < 0) return s;
            s.kind = SLOT_HIST;
            s.row = (int32_t)(((int64_t)h * g.pool_blocks + page) * g.P + sub * 64);
            s.lo = lo;
            s.hi = hi;
            return s;
        }
        w -= g.n_win_slots;
        if (w < g.n_cur_slots) {
            s.kind = SLOT_CUR;
            s.row = w * 64;
            s.hi = min(g.S - w * 64, 64);
        }
        return s;
    }
};

}  // namespace omnimem
