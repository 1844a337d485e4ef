/*
 * fp64 CPU oracle for the SparseX Sparse-KV recomputation step -- heavy loops (stages b and c).
 *
 * TEST INFRASTRUCTURE ONLY. Nothing in the product path (paper_2606_01751_b200/) may link, load or
 * call this file. It shares no code, header, table or constant with the CUDA library.
 *
 * Everything is the plain definition, written out:
 *   Eq. (1)  A_sq = softmax(Q_sq K^T / sqrt(d) + M_causal[I_nr, :])
 *   Eq. (2)  s_j  = sum_i A_sq[i, j]
 *            summed over all query heads ("a global score aggregated across
 *            attention heads"; reading A5: plain sum)
 *   Alg. 1 line 21
 *            O[R] = SparseAttn(Q[R], K_cur[1:T], V_cur[1:T], M_causal)
 * Positions are 0-based; the query at absolute position i sees keys j <= i (reading A6).
 * GQA: query head h reads KV head h / (Hq / Hkv).
 * Keys/values are read through the block table from the paged bf16 pool
 *   pool[num_blocks][Hkv][block_size][head_dim]   (bf16 bit patterns, widened exactly to double).
 * Parallelism: OpenMP over independent (query row) work items only; no blocking, no fusion.
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
    return (double)f;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* dense [seq_len][head_dim] double view of one KV head of one request, read through the block table */
static double *gather_head(const uint16_t *pool, int num_kv_heads, int head_dim, int block_size,
                           const int32_t *table, int seq_len, int kvh) {
    double *dst = (double *)malloc((size_t)seq_len * head_dim * sizeof(double));
    if (!dst) return NULL;
    for (int j = 0; j < seq_len; ++j) {
        const int64_t blk = table[j / block_size];
        const uint16_t *src =
            pool + (((blk * num_kv_heads + kvh) * block_size) + (j % block_size)) * (int64_t)head_dim;
        for (int d = 0; d < head_dim; ++d) dst[(size_t)j * head_dim + d] = bf16_to_f64(src[d]);
    }
    return dst;
}

static inline double dot(const double *a, const double *b, int n) {
    double acc = 0.0;
#pragma omp simd reduction(+ : acc)
    for (int d = 0; d < n; ++d) acc += a[d] * b[d];
    return acc;
}

/*
 * Stage (b) scores, one request. scores[seq_len] (overwritten) = Eq. (2) summed over heads;
 * lse[n_new][Hq] (optional) = log sum_j exp(l_j), l_j = <q,k_j>/sqrt(d), natural log.
 */
int orc_scores(const uint16_t *pool_k, int num_kv_heads, int num_q_heads, int head_dim, int block_size,
               const int32_t *k_table, int seq_len, const uint16_t *q_new, const int32_t *new_idx,
               int n_new, double *scores, double *lse) {
    const int g = num_q_heads / num_kv_heads;
    const double inv_sqrt_d = 1.0 / sqrt((double)head_dim);
    const int nt = orc_num_threads();
    double *priv = (double *)calloc((size_t)nt * seq_len, sizeof(double));
    if (!priv) return -1;
    for (int kvh = 0; kvh < num_kv_heads; ++kvh) {
        double *K = gather_head(pool_k, num_kv_heads, head_dim, block_size, k_table, seq_len, kvh);
        if (!K) { free(priv); return -1; }
        for (int h = kvh * g; h < (kvh + 1) * g; ++h) {
#pragma omp parallel
            {
#ifdef _OPENMP
                double *s = priv + (size_t)omp_get_thread_num() * seq_len;
#else
                double *s = priv;
#endif
                double *q = (double *)malloc(head_dim * sizeof(double));
                double *l = (double *)malloc((size_t)seq_len * sizeof(double));
#pragma omp for schedule(static, 1)
                for (int n = 0; n < n_new; ++n) {
                    const int i = new_idx[n]; /* absolute position of this Sparse-Q query */
                    const uint16_t *qb = q_new + ((size_t)n * num_q_heads + h) * head_dim;
                    for (int d = 0; d < head_dim; ++d) q[d] = bf16_to_f64(qb[d]);
                    double m = -INFINITY;
                    for (int j = 0; j <= i; ++j) { /* causal: keys j <= i */
                        l[j] = dot(q, K + (size_t)j * head_dim, head_dim) * inv_sqrt_d;
                        if (l[j] > m) m = l[j];
                    }
                    double z = 0.0;
                    for (int j = 0; j <= i; ++j) { l[j] = exp(l[j] - m); z += l[j]; }
                    for (int j = 0; j <= i; ++j) s[j] += l[j] / z; /* Eq. (2): column sum of A_sq */
                    if (lse) lse[(size_t)n * num_q_heads + h] = m + log(z);
                }
                free(q);
                free(l);
            }
        }
        free(K);
    }
    for (int j = 0; j < seq_len; ++j) scores[j] = 0.0;
    for (int t = 0; t < nt; ++t) /* fixed thread order */
        for (int j = 0; j < seq_len; ++j) scores[j] += priv[(size_t)t * seq_len + j];
    free(priv);
    return 0;
}

/*
 * Stage (c), one request: out[n_rows][Hq][head_dim] (double), row n is the query at absolute position
 * rows[n]; q_rows[n_rows][Hq][head_dim] bf16. lse optional [n_rows][Hq].
 */
int orc_attention(const uint16_t *pool_k, const uint16_t *pool_v, int num_kv_heads, int num_q_heads,
                  int head_dim, int block_size, const int32_t *k_table, const int32_t *v_table,
                  int seq_len, const uint16_t *q_rows, const int32_t *rows, int n_rows, double *out,
                  double *lse) {
    const int g = num_q_heads / num_kv_heads;
    const double inv_sqrt_d = 1.0 / sqrt((double)head_dim);
    for (int kvh = 0; kvh < num_kv_heads; ++kvh) {
        double *K = gather_head(pool_k, num_kv_heads, head_dim, block_size, k_table, seq_len, kvh);
        double *V = gather_head(pool_v, num_kv_heads, head_dim, block_size, v_table, seq_len, kvh);
        if (!K || !V) { free(K); free(V); return -1; }
        for (int h = kvh * g; h < (kvh + 1) * g; ++h) {
#pragma omp parallel
            {
                double *q = (double *)malloc(head_dim * sizeof(double));
                double *l = (double *)malloc((size_t)seq_len * sizeof(double));
#pragma omp for schedule(static, 1)
                for (int n = 0; n < n_rows; ++n) {
                    const int r = rows[n];
                    const uint16_t *qb = q_rows + ((size_t)n * num_q_heads + h) * head_dim;
                    for (int d = 0; d < head_dim; ++d) q[d] = bf16_to_f64(qb[d]);
                    double m = -INFINITY;
                    for (int j = 0; j <= r; ++j) {
                        l[j] = dot(q, K + (size_t)j * head_dim, head_dim) * inv_sqrt_d;
                        if (l[j] > m) m = l[j];
                    }
                    double z = 0.0;
                    for (int j = 0; j <= r; ++j) { l[j] = exp(l[j] - m); z += l[j]; }
                    double *o = out + ((size_t)n * num_q_heads + h) * head_dim;
                    for (int d = 0; d < head_dim; ++d) o[d] = 0.0;
                    for (int j = 0; j <= r; ++j) {
                        const double p = l[j] / z;
                        const double *v = V + (size_t)j * head_dim;
                        for (int d = 0; d < head_dim; ++d) o[d] += p * v[d];
                    }
                    if (lse) lse[(size_t)n * num_q_heads + h] = m + log(z);
                }
                free(q);
                free(l);
            }
        }
        free(K);
        free(V);
    }
    return 0;
}
