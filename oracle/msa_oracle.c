/*
 * msa_oracle.c -- fp64 CPU oracle for Multi-Segment Attention (MSA).
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (paper_2606_02964_b200/,
 * include/) may include, link or call this file; only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs do.  It shares no code, header,
 * table or helper with the CUDA path and takes the raw descriptors, not the CUDA
 * path's plan.
 *
 * What it computes (MSA is exact attention, "lossless ... bitwise-equivalent outputs",
 * PAPER.md:24; it is "a combination of multiple individual self-attention",
 * PAPER.md:102), written as the plain definition:
 *
 *   Eq. (1), PAPER.md:55-58      A = Q K^T / sqrt(d_k),  O = softmax(A) V
 *   Eq. (2), PAPER.md:104-112    every query run attends to all K/V that precede it
 *                                (O1 = Attn(Q1,K1,V1), O2 = Attn(Q2,K,V); reading c1)
 *   PAPER.md:116, :124           only attention needs the token dependency; each token
 *                                block has an "equivalent seq_len" = its causal horizon
 *
 * For a query row at absolute position p and q head h (KV head kvh = q_to_kv[h]):
 *   gather:  the context is the concatenation of all segments of the run's segment list;
 *            token idx of a segment sits at absolute position a = abs_start + idx and at
 *              pool[block_table[block_off + idx/16]][idx%16][kvh][:]   (kind 0, paged)
 *              arena[row_off + idx][kvh][:]                            (kind 1/2, contiguous)
 *   visible: a <= p                        (causal by absolute position, reading c2)
 *   s_j  = (double)scale_f32 * sum_d q[d] * K_j[d]        (bf16 -> double is exact)
 *   m    = max_j s_j ;  l = sum_j exp(s_j - m)
 *   LSE  = m + log(l)   (natural log; reading c9) ;  O[d] = sum_j exp(s_j - m) V_j[d] / l
 *   no visible key  =>  O = 0, LSE = -inf
 *
 * No blocking, no online softmax, no reordering: two plain passes per (row, head).
 * OpenMP only spreads independent (row, head) pairs over cores.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): torch SDPA fp64 with an explicit mask
 * and the Eq. (2) two-call decomposition; brute force over the generator's un-segmented
 * copy; segment-cut / block-table-permutation invariance; LSE-merge identity; closed
 * forms (uniform scores -> mean of V and ln n; V==1; V[0]=position -> p/2; position 0);
 * future-independence; key-shift invariance; Eq. (4) pair counts.
 *
 * fp8 KV pool (motive: the KV footprint; reading c20):
 * msa_oracle_forward_kv8 is the same definition with the PAGED pool stored as OCP FP8 E4M3 bytes
 * (1 sign, 4 exponent bits with bias 7, 3 mantissa bits; no infinities; S.1111.111 = NaN) and one
 * fp32 scale per KV head for K and for V:  K_j[kvh][d] = e4m3(byte) * k_scale[kvh], likewise V.  The
 * arena (CONTIG / SELF) stays bf16.  Dequantisation happens here, in fp64, from the same bytes the
 * CUDA path reads.  Pins: all 256 codes against torch's float8_e4m3fn -> float conversion and the
 * format's closed forms (448, 2^-9, 1.0); the whole function against msa_oracle_forward on a pool
 * that holds the dequantised values as bf16 (exact for power-of-two scales).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_BLOCK 16

static double bf16_to_double(uint16_t h)
{
    uint32_t u = ((uint32_t)h) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* OCP FP8 E4M3 ("e4m3fn"): value = (-1)^s * 2^(e-7) * (1 + m/8) for e in 1..15, (-1)^s * 2^-6 * (m/8) for e = 0;
 * the code with e = 15, m = 7 is NaN; there is no infinity (the largest finite value is 448). */
double msa_oracle_e4m3_to_double(uint8_t b)
{
    const int s = b >> 7, e = (b >> 3) & 15, m = b & 7;
    double v;
    if (e == 15 && m == 7) return NAN;
    if (e == 0) v = ldexp((double)m / 8.0, -6);
    else v = ldexp(1.0 + (double)m / 8.0, e - 7);
    return s ? -v : v;
}

int msa_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * rows to compute are given as (row_req[i], row_idx[i]) = (request index, row within the
 * run), grouped by request in any order.  O is [n_rows][Hq][D] doubles, LSE [n_rows][Hq].
 * Returns 0, or -1 on allocation failure, -2 on a malformed descriptor.
 */
static int forward_impl(
    int Hq, int Hkv, int D, const int32_t *q_to_kv,
    const uint16_t *q,                                   /* bf16 [total_q][Hq][D]          */
    const void *pool_k_any, const void *pool_v_any,      /* [num_blocks][16][Hkv][D]: bf16, or e4m3 bytes when kv8 */
    int kv8, const float *k_scale, const float *v_scale, /* kv8: fp32 scale per KV head    */
    const int32_t *block_table,
    const uint16_t *contig_k, const uint16_t *contig_v,  /* bf16 [rows][Hkv][D]            */
    int n_req, const int32_t *req_q_row_start, const int32_t *req_q_len,
    const int32_t *req_q_abs_start, const int32_t *req_seg_begin, const int32_t *req_seg_count,
    const int32_t *seg_kind, const int32_t *seg_abs_start, const int32_t *seg_len,
    const int32_t *seg_block_off, const int64_t *seg_row_off,
    float scale,
    int64_t n_rows, const int32_t *row_req, const int32_t *row_idx,
    double *O, double *LSE)
{
    const double scale_d = (double)scale;
    const uint16_t *pool_k = (const uint16_t *)pool_k_any, *pool_v = (const uint16_t *)pool_v_any;
    const uint8_t *pool_k8 = (const uint8_t *)pool_k_any, *pool_v8 = (const uint8_t *)pool_v_any;
    for (int r = 0; r < n_req; ++r) {
        /* any row of this request asked for? */
        int64_t wanted = 0;
        for (int64_t i = 0; i < n_rows; ++i) wanted += (row_req[i] == r);
        if (!wanted) continue;

        /* ---- gather: the concatenated context of request r, in fp64 ---------------- */
        int64_t n_ctx = 0;
        for (int s = req_seg_begin[r]; s < req_seg_begin[r] + req_seg_count[r]; ++s) {
            if (seg_len[s] < 0) return -2;
            n_ctx += seg_len[s];
        }
        const size_t per_tok = (size_t)Hkv * (size_t)D;
        double *Kc = (double *)malloc(sizeof(double) * per_tok * (size_t)(n_ctx > 0 ? n_ctx : 1));
        double *Vc = (double *)malloc(sizeof(double) * per_tok * (size_t)(n_ctx > 0 ? n_ctx : 1));
        int64_t *pos = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n_ctx > 0 ? n_ctx : 1));
        if (!Kc || !Vc || !pos) { free(Kc); free(Vc); free(pos); return -1; }
        int64_t base = 0;   /* index of the segment's first token in the concatenation */
        for (int s = req_seg_begin[r]; s < req_seg_begin[r] + req_seg_count[r]; ++s) {
            if (seg_kind[s] < 0 || seg_kind[s] > 2) {
                free(Kc); free(Vc); free(pos);
                return -2;
            }
#pragma omp parallel for schedule(static)
            for (int idx = 0; idx < seg_len[s]; ++idx) {
                const int64_t j = base + idx;
                const uint16_t *ksrc, *vsrc;
                pos[j] = (int64_t)seg_abs_start[s] + idx;
                if (seg_kind[s] == 0 && kv8) {   /* paged, fp8 pool: e4m3 byte times the KV head's scale */
                    int64_t blk = block_table[seg_block_off[s] + idx / ORACLE_BLOCK];
                    size_t off = ((size_t)blk * ORACLE_BLOCK + (size_t)(idx % ORACLE_BLOCK)) * per_tok;
                    for (size_t e = 0; e < per_tok; ++e) {
                        const size_t kvh = e / (size_t)D;
                        Kc[(size_t)j * per_tok + e] = msa_oracle_e4m3_to_double(pool_k8[off + e]) * (double)k_scale[kvh];
                        Vc[(size_t)j * per_tok + e] = msa_oracle_e4m3_to_double(pool_v8[off + e]) * (double)v_scale[kvh];
                    }
                    continue;
                }
                if (seg_kind[s] == 0) {          /* paged: through the block table */
                    int64_t blk = block_table[seg_block_off[s] + idx / ORACLE_BLOCK];
                    size_t off = ((size_t)blk * ORACLE_BLOCK + (size_t)(idx % ORACLE_BLOCK)) * per_tok;
                    ksrc = pool_k + off;
                    vsrc = pool_v + off;
                } else {                         /* contiguous arena (recomputed run / own chunk) */
                    size_t off = (size_t)(seg_row_off[s] + idx) * per_tok;
                    ksrc = contig_k + off;
                    vsrc = contig_v + off;
                }
                for (size_t e = 0; e < per_tok; ++e) {
                    Kc[(size_t)j * per_tok + e] = bf16_to_double(ksrc[e]);
                    Vc[(size_t)j * per_tok + e] = bf16_to_double(vsrc[e]);
                }
            }
            base += seg_len[s];
        }

        /* ---- plain attention for every requested (row, head) of request r ---------- */
        int fail = 0;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
        for (int64_t i = 0; i < n_rows; ++i) {
            for (int h = 0; h < Hq; ++h) {
                if (row_req[i] != r) continue;
                const int kvh = q_to_kv ? q_to_kv[h] : h / (Hq / Hkv);
                const int64_t p = (int64_t)req_q_abs_start[r] + row_idx[i];
                const uint16_t *qrow = q + ((size_t)(req_q_row_start[r] + row_idx[i]) * Hq + h) * D;
                double *o = O + ((size_t)i * Hq + h) * D;
                double *sc = (double *)malloc(sizeof(double) * (size_t)(n_ctx > 0 ? n_ctx : 1));
                double *qd = (double *)malloc(sizeof(double) * (size_t)D);
                if (!sc || !qd) { fail = 1; free(sc); free(qd); continue; }
                for (int d = 0; d < D; ++d) qd[d] = bf16_to_double(qrow[d]);
                /* pass 1: scores of visible keys and their maximum */
                double m = -INFINITY;
                int64_t n_vis = 0;
                for (int64_t t = 0; t < n_ctx; ++t) {
                    if (pos[t] > p) { sc[t] = -INFINITY; continue; }
                    const double *kk = Kc + (size_t)t * per_tok + (size_t)kvh * D;
                    double dot = 0.0;
                    for (int d = 0; d < D; ++d) dot += qd[d] * kk[d];
                    sc[t] = scale_d * dot;
                    if (sc[t] > m) m = sc[t];
                    ++n_vis;
                }
                for (int d = 0; d < D; ++d) o[d] = 0.0;
                if (n_vis == 0) {
                    LSE[(size_t)i * Hq + h] = -INFINITY;
                } else {
                    /* pass 2: l = sum exp(s-m), O = sum exp(s-m) V / l */
                    double l = 0.0;
                    for (int64_t t = 0; t < n_ctx; ++t) {
                        if (pos[t] > p) continue;
                        const double w = exp(sc[t] - m);
                        const double *vv = Vc + (size_t)t * per_tok + (size_t)kvh * D;
                        l += w;
                        for (int d = 0; d < D; ++d) o[d] += w * vv[d];
                    }
                    for (int d = 0; d < D; ++d) o[d] /= l;
                    LSE[(size_t)i * Hq + h] = m + log(l);
                }
                free(sc);
                free(qd);
            }
        }
        free(Kc); free(Vc); free(pos);
        if (fail) return -1;
    }
    return 0;
}

int msa_oracle_forward(
    int Hq, int Hkv, int D, const int32_t *q_to_kv,
    const uint16_t *q,                                   /* bf16 [total_q][Hq][D]          */
    const uint16_t *pool_k, const uint16_t *pool_v,      /* bf16 [num_blocks][16][Hkv][D]  */
    const int32_t *block_table,
    const uint16_t *contig_k, const uint16_t *contig_v,  /* bf16 [rows][Hkv][D]            */
    int n_req, const int32_t *req_q_row_start, const int32_t *req_q_len,
    const int32_t *req_q_abs_start, const int32_t *req_seg_begin, const int32_t *req_seg_count,
    const int32_t *seg_kind, const int32_t *seg_abs_start, const int32_t *seg_len,
    const int32_t *seg_block_off, const int64_t *seg_row_off,
    float scale,
    int64_t n_rows, const int32_t *row_req, const int32_t *row_idx,
    double *O, double *LSE)
{
    return forward_impl(Hq, Hkv, D, q_to_kv, q, pool_k, pool_v, 0, NULL, NULL, block_table, contig_k, contig_v, n_req,
                        req_q_row_start, req_q_len, req_q_abs_start, req_seg_begin, req_seg_count, seg_kind, seg_abs_start,
                        seg_len, seg_block_off, seg_row_off, scale, n_rows, row_req, row_idx, O, LSE);
}

/* The same with an fp8 (E4M3) paged pool: pool_k / pool_v are bytes [num_blocks][16][Hkv][D], k_scale / v_scale
 * fp32 [Hkv]; everything else as above. */
int msa_oracle_forward_kv8(
    int Hq, int Hkv, int D, const int32_t *q_to_kv,
    const uint16_t *q,
    const uint8_t *pool_k, const uint8_t *pool_v, const float *k_scale, const float *v_scale,
    const int32_t *block_table,
    const uint16_t *contig_k, const uint16_t *contig_v,
    int n_req, const int32_t *req_q_row_start, const int32_t *req_q_len,
    const int32_t *req_q_abs_start, const int32_t *req_seg_begin, const int32_t *req_seg_count,
    const int32_t *seg_kind, const int32_t *seg_abs_start, const int32_t *seg_len,
    const int32_t *seg_block_off, const int64_t *seg_row_off,
    float scale,
    int64_t n_rows, const int32_t *row_req, const int32_t *row_idx,
    double *O, double *LSE)
{
    if (!k_scale || !v_scale) return -2;
    return forward_impl(Hq, Hkv, D, q_to_kv, q, pool_k, pool_v, 1, k_scale, v_scale, block_table, contig_k, contig_v, n_req,
                        req_q_row_start, req_q_len, req_q_abs_start, req_seg_begin, req_seg_count, seg_kind, seg_abs_start,
                        seg_len, seg_block_off, seg_row_off, scale, n_rows, row_req, row_idx, O, LSE);
}
