/*
 * omnimem_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU restatement of the OmniMem hot path, written from the
 * paper (/root/reference/PAPER.md, cited as PAPER.md:<line>) and the readings listed in
 * DESIGN.md section 3.  It shares no code, header, table or helper with the CUDA path
 * under paper_2605_30519_b200/csrc/, and nothing under the package may import, link or
 * execute it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs call it.
 *
 * Conventions: every tensor is a dense C array of float32 whose values are exactly
 * representable in bf16 (the generators round once); all sums are accumulated in double;
 * softmax is the plain two-pass definition, NOT Algorithm 1's online form, so that it can
 * be checked against the paper by eye.
 *
 *   paged cache     k_pages, v_pages : [H][n_pages][B][D]      (PAPER.md:337 full-resolution
 *                                                               cache; page = one KV block)
 *   page map        page_map         : [H][n_pages] int32       logical block -> physical page
 *                                                               (PAPER.md:356 per-head ptr table)
 *   pooled keys     pooled_k         : [H][n_pages][D]          (PAPER.md:335 compressed cache)
 *   pooled values   pooled_v         : [H][n_pages][D]          (same cache, CMP branch of Eq. 1;
 *                                                               SURVEY.md 8f NEXT-1)
 *   queries         q                : [H][S][D]
 *   current chunk   k_cur, v_cur     : [H][S][D]
 *   block ids       block_idx        : [H][R][K] int32, -1 = masked
 *   pointer table   ptr_table        : [H][R][K] int32 physical page id, -1 = skip
 *
 *
 * Parity pins (tests/test_oracle_pins.py): every function below is pinned against
 * something other than itself -- closed forms, the paper's counting examples, brute force
 * in independent numpy code, invariants.  No function is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* round an fp32 value to the nearest bf16 (ties to even), returned as fp32 */
static float bf16_rne(float x)
{
    uint32_t u;
    memcpy(&u, &x, 4);
    if ((u & 0x7fffffffu) > 0x7f800000u) return x; /* NaN: contract violation, pass through */
    uint32_t lsb = (u >> 16) & 1u;
    u += 0x7fffu + lsb;
    u &= 0xffff0000u;
    memcpy(&x, &u, 4);
    return x;
}

float oracle_bf16_round(float x) { return bf16_rne(x); }

static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

/* ------------------------------------------------------------------------------------ */
/* a0  append one finished chunk to the paged cache ("list of chunk
 *     tensors", flat token stream paged in blocks of B: DESIGN.md reading R-paging).
 *     A page that receives its first token in this call is zero-filled first
 *     (reading A10).  Returns the new N_hist.                                   */
int64_t oracle_append_chunk(float* k_pages, float* v_pages, const int32_t* page_map,
                            int32_t H, int32_t D, int32_t B, int32_t n_pages, int64_t n_hist,
                            const float* k_chunk, const float* v_chunk, int32_t n_tokens)
{
    for (int32_t h = 0; h < H; ++h) {
        for (int32_t t = 0; t < n_tokens; ++t) {
            int64_t pos = n_hist + t;
            int64_t b = pos / B, o = pos % B;
            int64_t page = page_map[(int64_t)h * n_pages + b];
            float* kp = k_pages + (((int64_t)h * n_pages + page) * B) * D;
            float* vp = v_pages + (((int64_t)h * n_pages + page) * B) * D;
            if (o == 0) { /* fresh page */
                memset(kp, 0, sizeof(float) * (size_t)B * D);
                memset(vp, 0, sizeof(float) * (size_t)B * D);
            }
            memcpy(kp + o * D, k_chunk + ((int64_t)h * n_tokens + t) * D, sizeof(float) * D);
            memcpy(vp + o * D, v_chunk + ((int64_t)h * n_tokens + t) * D, sizeof(float) * D);
        }
    }
    return n_hist + n_tokens;
}

/* ------------------------------------------------------------------------------------ */
/* a1  block keys: "plain mean pool" of post-RoPE K over each KV block (PAPER.md:319,
 *     :335, :581).  Mean over the VALID tokens of the block (reading A10); the mean is
 *     stored in bf16 (reading A13): sum in double -> float -> divide by (float)len -> RNE. */
static void pool_pages(const float* pages, const int32_t* page_map, int32_t H, int32_t D,
                       int32_t B, int32_t n_pages, int64_t n_hist, int64_t first_block,
                       int64_t n_blocks, float* pooled)
{
    for (int32_t h = 0; h < H; ++h) {
        for (int64_t b = first_block; b < first_block + n_blocks; ++b) {
            int64_t len = n_hist - b * B;
            if (len > B) len = B;
            if (len <= 0) continue;
            int64_t page = page_map[(int64_t)h * n_pages + b];
            const float* kp = pages + (((int64_t)h * n_pages + page) * B) * D;
            for (int32_t d = 0; d < D; ++d) {
                double sum = 0.0;
                for (int64_t t = 0; t < len; ++t) sum += (double)kp[t * D + d];
                float f = (float)sum;
                f = f / (float)len;
                pooled[((int64_t)h * n_pages + b) * D + d] = bf16_rne(f);
            }
        }
    }
}

void oracle_pool_keys(const float* k_pages, const int32_t* page_map, int32_t H, int32_t D,
                      int32_t B, int32_t n_pages, int64_t n_hist, int64_t first_block,
                      int64_t n_blocks, float* pooled_k)
{
    pool_pages(k_pages, page_map, H, D, B, n_pages, n_hist, first_block, n_blocks, pooled_k);
}

/* NEXT-1: the compressed cache also holds block VALUES, pooled exactly like the
 * keys ("we pool its KV states into compressed KV blocks"; plain mean pool, :319). */
void oracle_pool_values(const float* v_pages, const int32_t* page_map, int32_t H, int32_t D,
                        int32_t B, int32_t n_pages, int64_t n_hist, int64_t first_block,
                        int64_t n_blocks, float* pooled_v)
{
    pool_pages(v_pages, page_map, H, D, B, n_pages, n_hist, first_block, n_blocks, pooled_v);
}

/* ------------------------------------------------------------------------------------ */
/* a2  Query-Shared KV Selection, query side (Eq. 3):
 *     R = ceil(S / G_q) adjacent groups; qbar[h][r] = mean of the group's valid queries,
 *     same rounding recipe as the block keys.                                            */
void oracle_group_mean_q(const float* q, int32_t H, int32_t S, int32_t D, int32_t G, float* qbar)
{
    int32_t R = (int32_t)ceil_div(S, G);
    for (int32_t h = 0; h < H; ++h)
        for (int32_t r = 0; r < R; ++r) {
            int32_t lo = r * G, hi = lo + G;
            if (hi > S) hi = S;
            for (int32_t d = 0; d < D; ++d) {
                double sum = 0.0;
                for (int32_t s = lo; s < hi; ++s) sum += (double)q[((int64_t)h * S + s) * D + d];
                float f = (float)sum;
                f = f / (float)(hi - lo);
                qbar[((int64_t)h * R + r) * D + d] = bf16_rne(f);
            }
        }
}

/* a2  scores sbar[h][r][b] = sigma_s * <qbar[h][r], kbar[h][b]>  (Eq. 3 with logit scores,
 *     reading A1: AvgPool_q of the per-query logits equals this by linearity).
 *     Sum in double, one rounding to fp32, -0 canonicalised to +0.                         */
void oracle_scores(const float* qbar, const float* pooled_k, int32_t H, int32_t R, int32_t D,
                   int32_t n_pages, int64_t n_b, float score_scale, float* scores)
{
    for (int32_t h = 0; h < H; ++h)
        for (int32_t r = 0; r < R; ++r)
            for (int64_t b = 0; b < n_b; ++b) {
                double sum = 0.0;
                const float* qv = qbar + ((int64_t)h * R + r) * D;
                const float* kv = pooled_k + ((int64_t)h * n_pages + b) * D;
                for (int32_t d = 0; d < D; ++d) sum += (double)qv[d] * (double)kv[d];
                float s = (float)((double)score_scale * sum);
                s += 0.0f;
                scores[((int64_t)h * R + r) * n_b + b] = s;
            }
}

/* a2, probability reading of "compression-attention scores" ("Selection attention uses
 *     compression-attention scores", :87; the NSA-style variant of reading A1, reading A1b):
 *     p[h][q][b] = softmax over the head's N_b compressed tokens b of  sigma_s * <q[h][q], kbar[h][b]>
 *     (the distribution the CMP branch of Eq. 1 attends with), and Eq. 3's AvgPool over the group:
 *     sbar[h][r][b] = (1 / |G_r|) * sum_{q in G_r} p[h][q][b].
 *     Plain two-pass softmax per query, everything in double, one rounding to fp32.              */
void oracle_scores_prob(const float* q, const float* pooled_k, int32_t H, int32_t S, int32_t D, int32_t G,
                        int32_t n_pages, int64_t n_b, float score_scale, float* scores)
{
    int32_t R = (int32_t)ceil_div(S, G);
    if (n_b <= 0) return;
    double* logit = (double*)malloc(sizeof(double) * (size_t)n_b);
    double* acc = (double*)malloc(sizeof(double) * (size_t)n_b);
    for (int32_t h = 0; h < H; ++h)
        for (int32_t r = 0; r < R; ++r) {
            int32_t lo = r * G, hi = lo + G;
            if (hi > S) hi = S;
            for (int64_t b = 0; b < n_b; ++b) acc[b] = 0.0;
            for (int32_t s = lo; s < hi; ++s) {
                const float* qv = q + ((int64_t)h * S + s) * D;
                double mx = -INFINITY;
                for (int64_t b = 0; b < n_b; ++b) {
                    const float* kv = pooled_k + ((int64_t)h * n_pages + b) * D;
                    double sum = 0.0;
                    for (int32_t d = 0; d < D; ++d) sum += (double)qv[d] * (double)kv[d];
                    logit[b] = (double)score_scale * sum;
                    if (logit[b] > mx) mx = logit[b];
                }
                double den = 0.0;
                for (int64_t b = 0; b < n_b; ++b) den += exp(logit[b] - mx);
                for (int64_t b = 0; b < n_b; ++b) acc[b] += exp(logit[b] - mx) / den;
            }
            for (int64_t b = 0; b < n_b; ++b) {
                float v = (float)(acc[b] / (double)(hi - lo));
                v += 0.0f;
                scores[((int64_t)h * R + r) * n_b + b] = v;
            }
        }
    free(logit);
    free(acc);
}

/* ------------------------------------------------------------------------------------ */
/* a3  Adaptive Window Exclusion (Eq. 2, threshold :319; readings A2-A4).
 *     out[0] = b_w (first block that intersects the window), out[1] = active,
 *     out[2] = omega_end (candidates are blocks [0, omega_end)), out[3] = N_b.            */
void oracle_awe(int64_t n_hist, int32_t B, int64_t n_wt, int32_t K, int64_t t_awe, int64_t* out)
{
    int64_t n_b = ceil_div(n_hist, B);
    int64_t win_start = n_hist - n_wt;
    if (win_start < 0) win_start = 0;
    int64_t b_w = (n_wt == 0) ? n_b : win_start / B;
    int64_t need = t_awe > K ? t_awe : K;
    int64_t active = (b_w >= need) ? 1 : 0;
    out[0] = b_w;
    out[1] = active;
    out[2] = active ? b_w : n_b;
    out[3] = n_b;
}

/* ------------------------------------------------------------------------------------ */
/* a4  per-(head, group) top-k: sort the candidates by
 *     (score descending, block index ascending) -- reading A6 -- keep the first
 *     K_eff = min(K, |Omega|); remaining slots are -1 (reading A7, the paper's mask M).    */
typedef struct { float s; int32_t b; } cand_t;

static int cand_cmp(const void* pa, const void* pb)
{
    const cand_t* a = (const cand_t*)pa;
    const cand_t* b = (const cand_t*)pb;
    if (a->s > b->s) return -1;
    if (a->s < b->s) return 1;
    if (a->b < b->b) return -1;
    if (a->b > b->b) return 1;
    return 0;
}

void oracle_topk(const float* scores, int32_t H, int32_t R, int64_t n_b, int64_t omega_end,
                 int32_t K, int32_t* block_idx)
{
    cand_t* c = (cand_t*)malloc(sizeof(cand_t) * (size_t)(omega_end > 0 ? omega_end : 1));
    for (int32_t h = 0; h < H; ++h)
        for (int32_t r = 0; r < R; ++r) {
            const float* row = scores + ((int64_t)h * R + r) * n_b;
            for (int64_t b = 0; b < omega_end; ++b) { c[b].s = row[b] + 0.0f; c[b].b = (int32_t)b; }
            qsort(c, (size_t)omega_end, sizeof(cand_t), cand_cmp);
            int32_t* out = block_idx + ((int64_t)h * R + r) * K;
            for (int32_t t = 0; t < K; ++t) out[t] = (t < omega_end) ? c[t].b : -1;
        }
    free(c);
}

/* a5  pointer table (Alg. 1 step 1 with B_pc = 1: DESIGN.md reading
 *     R-paging): P = page_map[h][I], masked slots stay -1 (the paper's 0 = skip).          */
void oracle_ptr_table(const int32_t* block_idx, const int32_t* page_map, int32_t H, int32_t R,
                      int32_t K, int32_t n_pages, int32_t* ptr_table)
{
    for (int32_t h = 0; h < H; ++h)
        for (int64_t i = 0; i < (int64_t)R * K; ++i) {
            int32_t b = block_idx[(int64_t)h * R * K + i];
            ptr_table[(int64_t)h * R * K + i] = (b < 0) ? -1 : page_map[(int64_t)h * n_pages + b];
        }
}

/* a5, the paper's own two-level map (Alg. 1 step 1 lines 7-12; App. C "each selected block index is
 *     mapped to a chunk index and an intra-chunk block offset"): c = I div B_pc, o = I mod B_pc, P = Pi[h][c] + offset(o).
 *     chunk_map[h][c] is the physical page of chunk c's first block for head h and a chunk's B_pc blocks are contiguous
 *     pages, so offset(o) = o pages (reading R-paging2).  Masked slots (-1) stay -1 (the paper's M = 0 => P = 0).  */
void oracle_ptr_table_chunked(const int32_t* block_idx, const int32_t* chunk_map, int32_t H, int32_t R, int32_t K,
                              int32_t n_chunks, int32_t B_pc, int32_t* ptr_table)
{
    for (int32_t h = 0; h < H; ++h)
        for (int64_t i = 0; i < (int64_t)R * K; ++i) {
            int32_t I = block_idx[(int64_t)h * R * K + i];
            if (I < 0) { ptr_table[(int64_t)h * R * K + i] = -1; continue; }
            int32_t c = I / B_pc;
            int32_t o = I % B_pc;
            ptr_table[(int64_t)h * R * K + i] = chunk_map[(int64_t)h * n_chunks + c] + o;
        }
}

/* Tile padding of a pooling block ("pad each tile to 32 tokens inside the kernel and mask the two extra
 *     positions"; Tab. H1 :506-526 "the padded block size is rounded to the next power of two"): returns the padded size. */
int32_t oracle_padded_block(int32_t block_tokens)
{
    int32_t p = 1;
    while (p < block_tokens) p *= 2;
    return p;
}

/* Union accounting (Eqs. 4-5): per_head[h] = |U_h|, returns |U_{h} U_h|. */
int64_t oracle_union_counts(const int32_t* block_idx, int32_t H, int32_t R, int32_t K,
                            int64_t n_b, int64_t* per_head)
{
    uint8_t* any = (uint8_t*)calloc((size_t)(n_b > 0 ? n_b : 1), 1);
    uint8_t* mine = (uint8_t*)malloc((size_t)(n_b > 0 ? n_b : 1));
    for (int32_t h = 0; h < H; ++h) {
        memset(mine, 0, (size_t)(n_b > 0 ? n_b : 1));
        for (int64_t i = 0; i < (int64_t)R * K; ++i) {
            int32_t b = block_idx[(int64_t)h * R * K + i];
            if (b >= 0) { mine[b] = 1; any[b] = 1; }
        }
        int64_t c = 0;
        for (int64_t b = 0; b < n_b; ++b) c += mine[b];
        per_head[h] = c;
    }
    int64_t u = 0;
    for (int64_t b = 0; b < n_b; ++b) u += any[b];
    free(any);
    free(mine);
    return u;
}

/* ------------------------------------------------------------------------------------ */
/* a6-a8  attention for a list of (head, query) rows.
 *   T_slc = valid tokens of the group's selected blocks, read THROUGH the pointer table
 *           from the paged storage (Alg. 1 line 23);
 *   T_swa = history tokens [win_start, N_hist) (through page_map) + all S tokens of the
 *           current chunk, no mask inside the chunk (readings A4, A5).
 *   Each branch is plain two-pass softmax attention in double (Alg. 1 computes the same
 *   thing online).  Empty branch: O = 0, LSE = -inf (reading A8).
 *   fuse_mode 0 JOINT: one softmax over T_slc (+) T_swa, i.e. the LSE-weighted merge;
 *   fuse_mode 1 GATED: O = g_slc[h] O_slc + g_swa[h] O_swa   (Eq. 1 without CMP, A11).
 *   out: [n_rows][D] float, lse: [2][n_rows] float (slc, swa).                            */
typedef struct { double m, l; int any; } branch_t;

static void branch_begin(branch_t* s) { s->m = -INFINITY; s->l = 0.0; s->any = 0; }

void oracle_sparse_attn_rows(const int32_t* row_h, const int32_t* row_q, int64_t n_rows,
                             const float* q, const float* k_cur, const float* v_cur,
                             const float* k_pages, const float* v_pages, const int32_t* page_map,
                             const int32_t* block_idx, const int32_t* ptr_table,
                             int32_t H, int32_t S, int32_t D, int32_t B, int32_t n_pages,
                             int64_t n_hist, int64_t n_wt, int32_t G, int32_t K,
                             float softmax_scale, int32_t fuse_mode,
                             const float* g_slc, const float* g_swa, float* out, float* lse)
{
    (void)H;
    int32_t R = (int32_t)ceil_div(S, G);
    int64_t win_start = n_hist - n_wt;
    if (win_start < 0) win_start = 0;
    if (n_wt == 0) win_start = n_hist;
    int64_t max_tok = (int64_t)K * B + (n_hist - win_start) + S;
    double* u = (double*)malloc(sizeof(double) * (size_t)max_tok);
    const float** vrow = (const float**)malloc(sizeof(float*) * (size_t)max_tok);
    double* o_slc = (double*)malloc(sizeof(double) * D);
    double* o_swa = (double*)malloc(sizeof(double) * D);

    for (int64_t i = 0; i < n_rows; ++i) {
        int32_t h = row_h[i], s = row_q[i];
        int32_t r = s / G;
        const float* qv = q + ((int64_t)h * S + s) * D;
        double lse2[2];
        for (int br = 0; br < 2; ++br) {
            /* gather the branch's token set: logits u[], value rows vrow[] */
            int64_t n = 0;
            if (br == 0) {
                for (int32_t t = 0; t < K; ++t) {
                    int32_t blk = block_idx[((int64_t)h * R + r) * K + t];
                    int32_t page = ptr_table[((int64_t)h * R + r) * K + t];
                    if (blk < 0 || page < 0) continue; /* Alg. 1 lines 20-22: skip */
                    int64_t len = n_hist - (int64_t)blk * B;
                    if (len > B) len = B;
                    const float* kp = k_pages + (((int64_t)h * n_pages + page) * B) * D;
                    const float* vp = v_pages + (((int64_t)h * n_pages + page) * B) * D;
                    for (int64_t tt = 0; tt < len; ++tt) {
                        double dot = 0.0;
                        for (int32_t d = 0; d < D; ++d) dot += (double)qv[d] * (double)kp[tt * D + d];
                        u[n] = (double)softmax_scale * dot;
                        vrow[n] = vp + tt * D;
                        ++n;
                    }
                }
            } else {
                for (int64_t pos = win_start; pos < n_hist; ++pos) {
                    int64_t page = page_map[(int64_t)h * n_pages + pos / B];
                    const float* kp = k_pages + ((((int64_t)h * n_pages + page) * B) + pos % B) * D;
                    const float* vp = v_pages + ((((int64_t)h * n_pages + page) * B) + pos % B) * D;
                    double dot = 0.0;
                    for (int32_t d = 0; d < D; ++d) dot += (double)qv[d] * (double)kp[d];
                    u[n] = (double)softmax_scale * dot;
                    vrow[n] = vp;
                    ++n;
                }
                for (int32_t t = 0; t < S; ++t) {
                    const float* kp = k_cur + ((int64_t)h * S + t) * D;
                    double dot = 0.0;
                    for (int32_t d = 0; d < D; ++d) dot += (double)qv[d] * (double)kp[d];
                    u[n] = (double)softmax_scale * dot;
                    vrow[n] = v_cur + ((int64_t)h * S + t) * D;
                    ++n;
                }
            }
            /* two-pass softmax */
            double* o = br == 0 ? o_slc : o_swa;
            for (int32_t d = 0; d < D; ++d) o[d] = 0.0;
            branch_t st;
            branch_begin(&st);
            for (int64_t t = 0; t < n; ++t) if (u[t] > st.m) st.m = u[t];
            for (int64_t t = 0; t < n; ++t) {
                double w = exp(u[t] - st.m);
                st.l += w;
                for (int32_t d = 0; d < D; ++d) o[d] += w * (double)vrow[t][d];
            }
            if (n > 0) {
                for (int32_t d = 0; d < D; ++d) o[d] /= st.l;
                lse2[br] = st.m + log(st.l);
            } else {
                lse2[br] = -INFINITY;
            }
        }
        float* orow = out + i * D;
        if (fuse_mode == 0) {
            double M = lse2[0] > lse2[1] ? lse2[0] : lse2[1];
            double a = (lse2[0] == -INFINITY) ? 0.0 : exp(lse2[0] - M);
            double b = (lse2[1] == -INFINITY) ? 0.0 : exp(lse2[1] - M);
            for (int32_t d = 0; d < D; ++d)
                orow[d] = (a + b > 0.0) ? (float)((a * o_slc[d] + b * o_swa[d]) / (a + b)) : 0.0f;
        } else {
            for (int32_t d = 0; d < D; ++d)
                orow[d] = (float)((double)g_slc[h] * o_slc[d] + (double)g_swa[h] * o_swa[d]);
        }
        lse[i] = (float)lse2[0];
        lse[n_rows + i] = (float)lse2[1];
    }
    free(u);
    free(vrow);
    free(o_slc);
    free(o_swa);
}

/* ------------------------------------------------------------------------------------ */
/* NEXT-1  compression attention (CMP): Attn(Q, K^cmp, V^cmp) over the pooled historical KV
 *   cache (Eq. 1): every query attends to the N_b compressed tokens
 *   (kbar[h][b], vbar[h][b]) of its head; plain two-pass softmax in double.  N_b = 0: O = 0,
 *   LSE = -inf.  out: [n_rows][D] float (O_cmp, not gated), lse: [n_rows] float.            */
void oracle_cmp_attn_rows(const int32_t* row_h, const int32_t* row_q, int64_t n_rows, const float* q,
                          const float* pooled_k, const float* pooled_v, int32_t S, int32_t D,
                          int32_t n_pages, int64_t n_b, float softmax_scale, float* out, float* lse)
{
    double* u = (double*)malloc(sizeof(double) * (size_t)(n_b > 0 ? n_b : 1));
    double* o = (double*)malloc(sizeof(double) * D);
    for (int64_t i = 0; i < n_rows; ++i) {
        int32_t h = row_h[i], s = row_q[i];
        const float* qv = q + ((int64_t)h * S + s) * D;
        double m = -INFINITY, l = 0.0;
        for (int64_t b = 0; b < n_b; ++b) {
            const float* kp = pooled_k + ((int64_t)h * n_pages + b) * D;
            double dot = 0.0;
            for (int32_t d = 0; d < D; ++d) dot += (double)qv[d] * (double)kp[d];
            u[b] = (double)softmax_scale * dot;
            if (u[b] > m) m = u[b];
        }
        for (int32_t d = 0; d < D; ++d) o[d] = 0.0;
        for (int64_t b = 0; b < n_b; ++b) {
            const float* vp = pooled_v + ((int64_t)h * n_pages + b) * D;
            double w = exp(u[b] - m);
            l += w;
            for (int32_t d = 0; d < D; ++d) o[d] += w * (double)vp[d];
        }
        for (int32_t d = 0; d < D; ++d) out[i * D + d] = n_b > 0 ? (float)(o[d] / l) : 0.0f;
        lse[i] = n_b > 0 ? (float)(m + log(l)) : -INFINITY;
    }
    free(u);
    free(o);
}
