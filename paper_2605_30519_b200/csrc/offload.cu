// NEXT-4: offload / reload of full-resolution KV chunks.
// HBM holds G chunk slots per head; every appended chunk is written through to a pinned host store; the per-head LRU
// order, the slot tables and the page_map mirror live on the host (this file), the copies are cudaMemcpyAsync on the
// caller's stream, and two small kernels do the device-side bookkeeping (which chunks a selection touches; the pointer
// table of Alg. 1 step 1 through the current map).  Residency is per (head, chunk): page_map[h][c] = base page or -1.
#include <string.h>

#include <vector>

#include "common.cuh"

namespace omnimem {

struct Offload {
    char *host_k, *host_v;     // pinned host store, [H][n_chunks][chunk_bytes]
    size_t chunk_bytes;        // B_pc * P * D * 2
    int32_t n_chunks;          // ceil(max_blocks / B_pc): entries per head of page_map
    int32_t n_slots;           // G
    int32_t pinned_recent;     // W most recent chunks are never evicted
    int64_t n_appended;        // chunks appended so far (chunk ids 0 .. n_appended - 1 exist)
    std::vector<int32_t> slot_chunk;  // [H][G]: chunk in the slot, -1 = free
    std::vector<int32_t> chunk_slot;  // [H][n_chunks]: slot of the chunk, -1 = not resident
    std::vector<uint64_t> last_use;   // [H][G]: LRU clock of the slot's chunk
    uint64_t clock;
    // caller-owned scratch: pinned host = [MAP_RING page_map snapshots][need bitmap]; device = need bitmap
    int32_t* map_ring;
    int32_t ring_pos;
    cudaEvent_t ring_ev[4];
    int32_t *need_host, *need_dev;
    omnimem_offload_stats_t st;
};
constexpr int MAP_RING = 4;

void offload_destroy(Offload* o)
{
    if (!o) return;
    for (int i = 0; i < MAP_RING; ++i) cudaEventDestroy(o->ring_ev[i]);
    delete o;
}

// need[h][c] = 1 for every chunk c that head h's selection touches (c = block / B_pc)
__global__ void __launch_bounds__(256)
chunk_need_kernel(const int32_t* __restrict__ block_idx, int64_t per_head, int64_t n, int32_t bpc, int32_t n_chunks, int32_t* __restrict__ need)
{
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const int32_t b = block_idx[i];
    if (b < 0) return;
    const int32_t c = b / bpc;
    if (c < n_chunks) need[(i / per_head) * n_chunks + c] = 1;
}

// Alg. 1 step 1 as a standalone kernel: P = Pi[h][I / B_pc] + I % B_pc, -1 for masked slots and for
// chunks that are not resident
__global__ void __launch_bounds__(256)
build_ptr_kernel(const int32_t* __restrict__ block_idx, const int32_t* __restrict__ page_map, int64_t per_head, int64_t n, int32_t max_blocks,
                 int32_t bpc, int32_t* __restrict__ ptr_table)
{
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const int32_t b = block_idx[i];
    ptr_table[i] = b < 0 ? -1 : page_of(page_map, i / per_head, b, max_blocks, bpc);
}

// entries of ptr_table that are -1 although their block was selected (skipped because the chunk is not resident)
__global__ void __launch_bounds__(256)
count_skipped_kernel(const int32_t* __restrict__ block_idx, const int32_t* __restrict__ ptr_table, int64_t n, int32_t* __restrict__ out)
{
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    const bool sk = i < n && block_idx[i] >= 0 && ptr_table[i] < 0;
    const unsigned m = __ballot_sync(0xffffffffu, sk);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(out, __popc(m));
}

static char* slot_ptr(const Cache* c, const __nv_bfloat16* pages, int h, int slot)
{
    return (char*)pages + ((size_t)h * c->pool_blocks + (size_t)slot * c->bpc) * c->P * c->D * 2;
}

// publish the host mirror of page_map: snapshot into the next ring buffer (pinned), async copy, event guards the reuse
static int32_t publish_map(Cache* c, cudaStream_t s)
{
    Offload* o = c->off;
    const size_t n = (size_t)c->H * o->n_chunks;
    int32_t* snap = o->map_ring + (size_t)o->ring_pos * n;
    cudaEventSynchronize(o->ring_ev[o->ring_pos]);  // the copy that last used this snapshot has run
    for (int h = 0; h < c->H; ++h)
        for (int ch = 0; ch < o->n_chunks; ++ch) {
            const int32_t sl = o->chunk_slot[(size_t)h * o->n_chunks + ch];
            snap[(size_t)h * o->n_chunks + ch] = sl < 0 ? -1 : sl * c->bpc;
        }
    cudaError_t e = cudaMemcpyAsync(c->page_map, snap, n * 4, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "page_map upload: %s", cudaGetErrorString(e));
    cudaEventRecord(o->ring_ev[o->ring_pos], s);
    o->ring_pos = (o->ring_pos + 1) % MAP_RING;
    return OMNIMEM_OK;
}

// the slot the next chunk of head h goes to: a free one, else the least recently used whose chunk is neither pinned
// (one of the W most recent) nor needed by the call in progress; -1 if there is none
static int pick_slot(const Cache* c, Offload* o, int h, int64_t newest, const int32_t* need_row)
{
    int best = -1;
    uint64_t best_t = ~0ull;
    for (int sl = 0; sl < o->n_slots; ++sl) {
        const int32_t ch = o->slot_chunk[(size_t)h * o->n_slots + sl];
        if (ch < 0) return sl;
        if (ch > newest - o->pinned_recent) continue;       // pinned: the window reads it
        if (need_row && need_row[ch]) continue;               // this step's attention reads it
        const uint64_t t = o->last_use[(size_t)h * o->n_slots + sl];
        if (t < best_t) { best_t = t; best = sl; }
    }
    (void)c;
    return best;
}

// Before the append kernel runs: give the new chunk (id n_appended) a slot in every head, evicting if needed.
int32_t offload_on_append(Cache* c, int32_t n_tokens, cudaStream_t s)
{
    Offload* o = c->off;
    if (!o) return fail(OMNIMEM_ESTATE, "resident_chunks > 0: call omnimem_offload_attach before appending");
    const int64_t chunk_tokens = (int64_t)c->bpc * c->B;
    if (n_tokens != chunk_tokens || c->n_hist % chunk_tokens != 0)
        return fail(OMNIMEM_EINVAL, "with offloading a chunk of exactly %lld tokens is appended at a time", (long long)chunk_tokens);
    const int64_t ch = o->n_appended;
    if (ch >= o->n_chunks) return fail(OMNIMEM_ECAPACITY, "chunk %lld exceeds the cache's %d chunks", (long long)ch, o->n_chunks);
    for (int h = 0; h < c->H; ++h) {
        const int sl = pick_slot(c, o, h, ch, nullptr);
        if (sl < 0) return fail(OMNIMEM_ECAPACITY, "no evictable slot: resident_chunks must exceed pinned_recent");
        const int32_t old = o->slot_chunk[(size_t)h * o->n_slots + sl];
        if (old >= 0) { o->chunk_slot[(size_t)h * o->n_chunks + old] = -1; ++o->st.evictions; }
        o->slot_chunk[(size_t)h * o->n_slots + sl] = (int32_t)ch;
        o->chunk_slot[(size_t)h * o->n_chunks + ch] = sl;
        o->last_use[(size_t)h * o->n_slots + sl] = ++o->clock;
    }
    return publish_map(c, s);
}

// After the append kernel: write the chunk through to the pinned host store (stream-ordered behind the kernel).
int32_t offload_after_append(Cache* c, int64_t ch, cudaStream_t s)
{
    Offload* o = c->off;
    for (int h = 0; h < c->H; ++h) {
        const int sl = o->chunk_slot[(size_t)h * o->n_chunks + ch];
        const size_t off = ((size_t)h * o->n_chunks + (size_t)ch) * o->chunk_bytes;
        cudaError_t e = cudaMemcpyAsync(o->host_k + off, slot_ptr(c, c->k_pages, h, sl), o->chunk_bytes, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(o->host_v + off, slot_ptr(c, c->v_pages, h, sl), o->chunk_bytes, cudaMemcpyDeviceToHost, s);
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "write-through copy: %s", cudaGetErrorString(e));
    }
    o->n_appended = ch + 1;
    return OMNIMEM_OK;
}

}  // namespace omnimem

using namespace omnimem;

extern "C" {

size_t omnimem_offload_scratch_bytes(const omnimem_cache_desc_t* d)
{
    if (!d || d->blocks_per_chunk <= 0 || d->block_tokens <= 0) return 0;
    const size_t max_blocks = (size_t)ceil_div64(d->max_tokens, d->block_tokens);
    const size_t n = (size_t)d->n_heads * (size_t)ceil_div64((int64_t)max_blocks, d->blocks_per_chunk);
    return (MAP_RING + 1) * n * 4 + 256;
}

int32_t omnimem_offload_attach(omnimem_cache_t* cache, void* host_k, void* host_v, int32_t pinned_recent, void* scratch_host,
                               void* scratch_dev, size_t scratch_bytes)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    Cache* c = reinterpret_cast<Cache*>(cache);
    if (c->resident_chunks <= 0) return fail(OMNIMEM_ESTATE, "the cache was created with resident_chunks = 0");
    if (c->off) return fail(OMNIMEM_ESTATE, "offloading is already attached");
    if (c->n_hist != 0) return fail(OMNIMEM_ESTATE, "attach before the first append");
    if (!host_k || !host_v || !scratch_host || !scratch_dev) return fail(OMNIMEM_EINVAL, "NULL buffer");
    if (pinned_recent < 1 || pinned_recent >= c->resident_chunks)
        return fail(OMNIMEM_EINVAL, "pinned_recent %d not in [1, resident_chunks)", pinned_recent);
    const int32_t n_chunks = (int32_t)ceil_div64(c->max_blocks, c->bpc);
    const size_t n = (size_t)c->H * n_chunks;
    if (scratch_bytes < (MAP_RING + 1) * n * 4) return fail(OMNIMEM_ECAPACITY, "offload scratch: need %zu bytes", (MAP_RING + 1) * n * 4);
    Offload* o = new (std::nothrow) Offload();
    if (!o) return fail(OMNIMEM_ECAPACITY, "out of host memory");
    o->host_k = (char*)host_k;
    o->host_v = (char*)host_v;
    o->chunk_bytes = (size_t)c->bpc * c->P * c->D * 2;
    o->n_chunks = n_chunks;
    o->n_slots = c->resident_chunks;
    o->pinned_recent = pinned_recent;
    o->n_appended = 0;
    o->slot_chunk.assign((size_t)c->H * o->n_slots, -1);
    o->chunk_slot.assign(n, -1);
    o->last_use.assign((size_t)c->H * o->n_slots, 0);
    o->clock = 0;
    o->map_ring = (int32_t*)scratch_host;
    o->need_host = o->map_ring + MAP_RING * n;
    o->need_dev = (int32_t*)scratch_dev;
    o->ring_pos = 0;
    for (int i = 0; i < MAP_RING; ++i) cudaEventCreateWithFlags(&o->ring_ev[i], cudaEventDisableTiming);
    memset(&o->st, 0, sizeof(o->st));
    c->off = o;
    return OMNIMEM_OK;
}

int32_t omnimem_offload_step(omnimem_cache_t* cache, const int32_t* block_idx, int32_t n_groups, int32_t top_k, int32_t mode,
                             int32_t* ptr_table, omnimem_offload_stats_t* stats_out, void* stream)
{
    if (!cache) return fail(OMNIMEM_EINVAL, "cache is NULL");
    Cache* c = reinterpret_cast<Cache*>(cache);
    Offload* o = c->off;
    if (!o) return fail(OMNIMEM_ESTATE, "offloading is not attached");
    if (!block_idx || !ptr_table || n_groups < 1 || top_k < 1) return fail(OMNIMEM_EINVAL, "bad argument");
    if (mode != OMNIMEM_OFFLOAD_SKIP && mode != OMNIMEM_OFFLOAD_WAIT) return fail(OMNIMEM_EINVAL, "mode %d", mode);
    cudaStream_t s = (cudaStream_t)stream;
    const size_t n_map = (size_t)c->H * o->n_chunks;
    const int64_t per_head = (int64_t)n_groups * top_k, n = per_head * c->H;
    // which chunks does the selection touch?  (device bitmap -> pinned host; the one synchronisation of the host step)
    cudaError_t e = cudaMemsetAsync(o->need_dev, 0, (n_map + 1) * 4, s);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
    chunk_need_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, s>>>(block_idx, per_head, n, c->bpc, o->n_chunks, o->need_dev);
    count_launch();
    e = cudaMemcpyAsync(o->need_host, o->need_dev, n_map * 4, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "need bitmap: %s", cudaGetErrorString(e));
    // LRU bookkeeping and reloads, head by head, chunks in ascending order
    const int64_t newest = o->n_appended - 1;
    bool changed = false;
    for (int h = 0; h < c->H; ++h) {
        const int32_t* need = o->need_host + (size_t)h * o->n_chunks;
        for (int ch = 0; ch < o->n_chunks; ++ch) {  // hits first: their clocks must be fresh before victims are chosen
            if (!need[ch]) continue;
            const int32_t sl = o->chunk_slot[(size_t)h * o->n_chunks + ch];
            ++o->st.requests;
            if (sl >= 0) { ++o->st.hits; o->last_use[(size_t)h * o->n_slots + sl] = ++o->clock; }
        }
        for (int ch = 0; ch < o->n_chunks; ++ch) {
            if (!need[ch] || ch > newest || o->chunk_slot[(size_t)h * o->n_chunks + ch] >= 0) continue;
            const int sl = pick_slot(c, o, h, newest, need);
            if (sl < 0) continue;  // more chunks needed than slots: the rest stays on the host (skipped)
            const int32_t old = o->slot_chunk[(size_t)h * o->n_slots + sl];
            if (old >= 0) { o->chunk_slot[(size_t)h * o->n_chunks + old] = -1; ++o->st.evictions; }
            const size_t off = ((size_t)h * o->n_chunks + (size_t)ch) * o->chunk_bytes;
            e = cudaMemcpyAsync(slot_ptr(c, c->k_pages, h, sl), o->host_k + off, o->chunk_bytes, cudaMemcpyHostToDevice, s);
            if (e == cudaSuccess) e = cudaMemcpyAsync(slot_ptr(c, c->v_pages, h, sl), o->host_v + off, o->chunk_bytes, cudaMemcpyHostToDevice, s);
            if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "reload copy: %s", cudaGetErrorString(e));
            o->slot_chunk[(size_t)h * o->n_slots + sl] = ch;
            o->chunk_slot[(size_t)h * o->n_chunks + ch] = sl;
            o->last_use[(size_t)h * o->n_slots + sl] = ++o->clock;
            ++o->st.reloads;
            changed = true;
        }
    }
    if (mode == OMNIMEM_OFFLOAD_WAIT) {
        if (changed)
            if (int32_t rc = publish_map(c, s)) return rc;
        build_ptr_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, s>>>(block_idx, c->page_map, per_head, n, c->max_blocks, c->bpc, ptr_table);
        count_launch();
    }
    // how many selected entries the attention will skip (counted against the table it is going to read)
    int32_t* cnt = o->need_dev + n_map;
    count_skipped_kernel<<<(unsigned)ceil_div64(n, 256), 256, 0, s>>>(block_idx, ptr_table, n, cnt);
    count_launch();
    if (mode == OMNIMEM_OFFLOAD_SKIP && changed)
        if (int32_t rc = publish_map(c, s)) return rc;  // the reloaded chunks serve the NEXT selection
    if (stats_out) {
        int32_t sk = 0;
        e = cudaMemcpyAsync(&sk, cnt, 4, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) return fail(OMNIMEM_ECUDA, "stats: %s", cudaGetErrorString(e));
        o->st.skipped = sk;
        *stats_out = o->st;
    }
    return check_launch("offload_step");
}

}  // extern "C"
