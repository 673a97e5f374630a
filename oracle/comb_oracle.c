/*
 * comb_oracle.c — ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, obviously-correct fp64 CPU statement of what the COMB link-stage cross-attention
 * computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this.  It shares no code, header, table or helper with the CUDA path under
 * paper_2602_01519_b200/ and neither imports the other.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md at authoring time):
 *   - PAPER.md:112-115, §4.2 Eq. 7-8:  A = softmax(Q K^T / sqrt(d)) row-wise over l_doc, NO mask;
 *     H = A V.                                        (reading I1-I3 in DESIGN.md §4)
 *   - PAPER.md:119, §4.2: the PICaches of several chunks are "concatenated along the l_doc during
 *     inference (link stage)"; l_doc = sum_i l_doc,i  => ONE joint softmax over
 *     the explicit concatenation, in link order.     (reading I4-I5)
 *   - PAPER.md:66, §4: generated tokens are "treated identically to the initial query tokens"
 *     => decode is the same function with one query row. (reading I17)
 *   - PAPER.md:62, §3: "possibly none ... contexts" => kv_len = 0 gives O = 0, LSE = -inf. (I13)
 *   - multi-head "extension is standard": per head, q-head h reads kv-head h / G. (I8)
 *
 * The oracle reads the ORIGINAL chunk tensors (never pages or block tables), widens bf16 to fp64
 * exactly, and rounds nothing.  No blocking, no online softmax, no fusion: concatenate, score,
 * max, exp, sum, weighted sum, divide.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): brute force without max-subtraction,
 * library fp64 SDPA special case, single key, equal scores (mean of V, LSE = ln n), two-level
 * closed form sigma(1), permutation invariance, split == whole, merge identity, shift
 * invariance, V-affinity, empty link.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static inline double bf16_to_f64(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f; /* exact: every bf16 is a float, every float is a double */
}

/* One query row against the concatenated K/V of its request, one q-head. Eq. 7-8. */
static void attend_row(const uint16_t *q_row,  /* [Dqk] bf16 bits of Q[i][h][:] */
                       const double *Kcat,     /* [kv][Hkv][Dqk] */
                       const double *Vcat,     /* [kv][Hkv][Dv]  */
                       int64_t kv, int Hkv, int g, int Dqk, int Dv, double scale,
                       double *s_buf,          /* scratch [kv] */
                       double *o_out,          /* [Dv] */
                       double *lse_out) {
    if (kv == 0) { /* reading I13: no contexts => zero contribution */
        for (int c = 0; c < Dv; ++c) o_out[c] = 0.0;
        *lse_out = -INFINITY;
        return;
    }
    double m = -INFINITY;
    for (int64_t j = 0; j < kv; ++j) { /* s_j = scale * sum_c Q[i][h][c] * K[j][g][c] */
        const double *krow = Kcat + ((size_t)j * Hkv + g) * Dqk;
        double acc = 0.0;
        for (int c = 0; c < Dqk; ++c) acc += bf16_to_f64(q_row[c]) * krow[c];
        s_buf[j] = scale * acc;
        if (s_buf[j] > m) m = s_buf[j];
    }
    double l = 0.0;
    for (int64_t j = 0; j < kv; ++j) { /* p_j = exp(s_j - m); l = sum p_j */
        s_buf[j] = exp(s_buf[j] - m);
        l += s_buf[j];
    }
    for (int c = 0; c < Dv; ++c) o_out[c] = 0.0;
    for (int64_t j = 0; j < kv; ++j) { /* O = sum_j p_j V[j][g][:] */
        const double *vrow = Vcat + ((size_t)j * Hkv + g) * Dv;
        const double p = s_buf[j];
        for (int c = 0; c < Dv; ++c) o_out[c] += p * vrow[c];
    }
    for (int c = 0; c < Dv; ++c) o_out[c] /= l;
    *lse_out = m + log(l);
}

/* Explicit concatenation of one request's chunks in link order. Valid tokens only. */
static int64_t concat_request(const int32_t *chunk_indptr, const int32_t *chunk_sel, int r,
                              const uint16_t *const *k_chunks, const uint16_t *const *v_chunks,
                              const int32_t *chunk_len, int Hkv, int Dqk, int Dv,
                              double **Kcat_out, double **Vcat_out) {
    int64_t kv = 0;
    for (int32_t e = chunk_indptr[r]; e < chunk_indptr[r + 1]; ++e) kv += chunk_len[chunk_sel[e]];
    double *Kcat = (double *)malloc(sizeof(double) * (size_t)(kv > 0 ? kv : 1) * Hkv * Dqk);
    double *Vcat = (double *)malloc(sizeof(double) * (size_t)(kv > 0 ? kv : 1) * Hkv * Dv);
    if (!Kcat || !Vcat) { free(Kcat); free(Vcat); return -1; }
    int64_t at = 0;
    for (int32_t e = chunk_indptr[r]; e < chunk_indptr[r + 1]; ++e) {
        const int32_t c = chunk_sel[e];
        const int64_t T = chunk_len[c];
        const size_t nk = (size_t)T * Hkv * Dqk, nv = (size_t)T * Hkv * Dv;
        for (size_t x = 0; x < nk; ++x) Kcat[(size_t)at * Hkv * Dqk + x] = bf16_to_f64(k_chunks[c][x]);
        for (size_t x = 0; x < nv; ++x) Vcat[(size_t)at * Hkv * Dv + x] = bf16_to_f64(v_chunks[c][x]);
        at += T;
    }
    *Kcat_out = Kcat;
    *Vcat_out = Vcat;
    return kv;
}

/*
 * O1 — full attention output.
 *   q          bf16 bits [sum lq][Hq][Dqk], rows of request r are q_indptr[r]..q_indptr[r+1]
 *   chunk_sel  for request r, entries chunk_indptr[r]..chunk_indptr[r+1]: index into the chunk
 *              arrays below, IN LINK ORDER
 *   k_chunks[c] / v_chunks[c]  bf16 bits [chunk_len[c]][Hkv][Dqk] / [..][Hkv][Dv]
 *   out  fp64 [sum lq][Hq][Dv];  lse fp64 [sum lq][Hq]
 * returns 0, or -1 on allocation failure.
 */
int comb_oracle_attention(int R, const int32_t *q_indptr, const uint16_t *q, int Hq, int Hkv, int Dqk,
                          int Dv, const int32_t *chunk_indptr, const int32_t *chunk_sel,
                          const uint16_t *const *k_chunks, const uint16_t *const *v_chunks,
                          const int32_t *chunk_len, double scale, double *out, double *lse,
                          int num_threads) {
    const int G = Hq / Hkv;
#ifdef _OPENMP
    if (num_threads > 0) omp_set_num_threads(num_threads);
#else
    (void)num_threads;
#endif
    for (int r = 0; r < R; ++r) {
        double *Kcat = NULL, *Vcat = NULL;
        const int64_t kv = concat_request(chunk_indptr, chunk_sel, r, k_chunks, v_chunks, chunk_len, Hkv,
                                          Dqk, Dv, &Kcat, &Vcat);
        if (kv < 0) return -1;
        const int32_t row0 = q_indptr[r], rows = q_indptr[r + 1] - q_indptr[r];
        int failed = 0;
#pragma omp parallel
        {
            double *s_buf = (double *)malloc(sizeof(double) * (size_t)(kv > 0 ? kv : 1));
            if (!s_buf) {
#pragma omp atomic write
                failed = 1;
            }
#pragma omp barrier
            if (!failed) {
#pragma omp for collapse(2) schedule(dynamic, 1)
                for (int32_t i = 0; i < rows; ++i) {
                    for (int h = 0; h < Hq; ++h) { /* no mask: every row sees every key (Eq. 7) */
                        const size_t row = (size_t)(row0 + i);
                        attend_row(q + (row * Hq + h) * Dqk, Kcat, Vcat, kv, Hkv, h / G, Dqk, Dv, scale,
                                   s_buf, out + (row * Hq + h) * Dv, lse + row * Hq + h);
                    }
                }
            }
            free(s_buf);
        }
        free(Kcat);
        free(Vcat);
        if (failed) return -1;
    }
    return 0;
}

/*
 * O1 on sampled outputs: the same definition evaluated only for the listed (row, head) pairs of
 * ONE request (used at full BASELINE sizes where all outputs would take too long).
 *   sample_rows[n] are global row indices inside request r's range; sample_heads[n] q-heads.
 *   out fp64 [n][Dv], lse fp64 [n].
 */
int comb_oracle_attention_samples(int r, const int32_t *q_indptr, const uint16_t *q, int Hq, int Hkv,
                                  int Dqk, int Dv, const int32_t *chunk_indptr, const int32_t *chunk_sel,
                                  const uint16_t *const *k_chunks, const uint16_t *const *v_chunks,
                                  const int32_t *chunk_len, double scale, int n, const int32_t *sample_rows,
                                  const int32_t *sample_heads, double *out, double *lse) {
    const int G = Hq / Hkv;
    double *Kcat = NULL, *Vcat = NULL;
    const int64_t kv =
        concat_request(chunk_indptr, chunk_sel, r, k_chunks, v_chunks, chunk_len, Hkv, Dqk, Dv, &Kcat, &Vcat);
    if (kv < 0) return -1;
    double *s_buf = (double *)malloc(sizeof(double) * (size_t)(kv > 0 ? kv : 1));
    if (!s_buf) { free(Kcat); free(Vcat); return -1; }
    for (int x = 0; x < n; ++x) {
        const size_t row = (size_t)sample_rows[x];
        const int h = sample_heads[x];
        if ((int32_t)row < q_indptr[r] || (int32_t)row >= q_indptr[r + 1]) { free(s_buf); free(Kcat); free(Vcat); return -2; }
        attend_row(q + (row * Hq + h) * Dqk, Kcat, Vcat, kv, Hkv, h / G, Dqk, Dv, scale, s_buf,
                   out + (size_t)x * Dv, lse + x);
    }
    free(s_buf);
    free(Kcat);
    free(Vcat);
    return 0;
}

int comb_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
