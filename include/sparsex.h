/*
 * sparsex.h -- C ABI of the B200 (sm_100a) Sparse-KV recomputation step of SparseX
 * (arxiv/paper_2606_01751). Citations are PAPER.md line numbers (+ section / equation / Algorithm 1).
 *
 * One layer of the method is four stages over a paged bf16 KV pool (BASELINE.json north_star):
 *   (a) sx_rope_realign  k^_{p'+j} <- R_{p'-p} k^_{p+j}, v^ copied      PAPER.md:151-165 (S3.1), Alg. 1 l.502-504
 *   (b) sx_score_select  A_sq = softmax(Q_sq K^T/sqrt(d) + M_causal)      Eq. (1)
 *                        s_j = sum_heads sum_{i in I_nr} A_sq[i,j]         Eq. (2)
 *                        S_key = TopK(s, k) over cached positions          Eq. (3)
 *                        R = I_nr U S_key                                  Alg. 1 l.537-539
 *   (c) sx_sparse_attn   O[R] = SparseAttn(Q[R], K_cur[1:T], V_cur[1:T])   Alg. 1 l.546-548 (full mode: l.507-511)
 *   (d) sx_scatter_kv    write fresh K,V of the computed rows into pages   Alg. 1 l.509-510, 544-545
 *
 * Conventions
 *   - "device" pointers are CUDA device memory owned by the caller; "host" values are plain integers
 *     in the structs below. The library allocates nothing and frees nothing. The only process-wide state it
 *     keeps is (i) a bounded cache of encoded TMA tensor maps keyed by (base pointer, shape) -- a pure function
 *     of its key, so it cannot go stale -- (ii) the kernel-launch counter of sx_launch_count(), (iii) the
 *     thread-local text of sx_last_error() and (iv) the built-in device scratch of sx_sparse_attn_noalloc (9.1 MiB
 *     per GPU, used by that entry point only). All entry points may be called from several threads; calls of
 *     sx_sparse_attn_noalloc must not overlap on the GPU (see there).
 *   - Every stage call is asynchronous on `stream` and never synchronises the device (the two validation calls
 *     sx_check_batch / sx_check_rows do: they are for descriptor construction time). A non-zero status
 *     means nothing was launched (argument errors) or a launch failed (SX_ERR_CUDA);
 *     sx_last_error() then returns a thread-local description.
 *   - The workspace `ws` is scratch that calls write: calls that may run concurrently (different streams)
 *     need their own workspace; consecutive calls on one stream may share it.
 *   - bf16 tensors are raw 16-bit patterns. All device pointers must be 16-byte aligned.
 *   - head_dim must be 128 and block_size 16 (SX_ERR_UNSUPPORTED otherwise);
 *     num_q_heads % num_kv_heads == 0, group size g = Hq/Hkv <= 128.
 *   - Positions are 0-based; the query at absolute position i sees keys j <= i (Eq. 1 M_causal).
 *   - Same inputs => bit-identical outputs (no floating-point atomics anywhere).
 *   - There is no CPU fallback: without a CUDA device every stage call returns SX_ERR_CUDA.
 */
#ifndef SPARSEX_H_
#define SPARSEX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SX_OK = 0,
  SX_ERR_INVALID_ARG = -1, /* null pointer, negative size, inconsistent counts                 */
  SX_ERR_UNSUPPORTED = -2, /* head_dim != 128, block_size != 16, bad head grouping, bad style  */
  SX_ERR_WORKSPACE = -3,   /* ws_bytes smaller than sx_workspace_size()                        */
  SX_ERR_CUDA = -4,        /* a CUDA runtime / driver call or a launch failed                  */
  SX_ERR_MISALIGNED = -5   /* a device pointer is not 16-byte aligned                          */
} sx_status;

typedef struct CUstream_st *sx_stream; /* a cudaStream_t / CUstream; NULL = legacy default stream */

/* Paged KV pool of ONE layer (a block holds the K/V of block_size tokens).
 * Layout chosen here (the paper fixes none): separate K and V arrays, each
 *   bf16 [num_blocks][num_kv_heads][block_size=16][head_dim=128]
 * so that one (page, kv head) tile is 4 KB contiguous = 16 rows of 256 B. */
typedef struct {
  void *k;            /* device */
  void *v;            /* device */
  int32_t num_blocks; /* host */
  int32_t block_size; /* host, must be 16 */
  int32_t num_kv_heads;
  int32_t num_q_heads;
  int32_t head_dim;   /* host, must be 128 */
} sx_pool;

/* One reused segment S_m of one request (Alg. 1 inputs l.497, l.502).
 * len, old_pos (p_m) and new_pos (p'_m) are multiples of block_size (segment
 * boundaries are padded to the block size). delta = new_pos - old_pos may be negative or zero.
 * src_off indexes src_blocks[]; segments must be stored so that src_off is the running sum of
 * len/block_size of the segments before it (segment i's pages follow segment i-1's). */
typedef struct {
  int32_t req;
  int32_t len;
  int32_t old_pos;
  int32_t new_pos;
  int32_t src_off;
} sx_segment;

/* Block-table / segment-map descriptor of one scheduling batch (scheduler output of PAPER.md:333:
 * request layout, block table, slot mapping, sparse mask). Host fields mirror sizes so that grids
 * can be sized without reading device memory. */
typedef struct {
  /* host mirrors */
  int32_t num_reqs;
  int32_t num_segments;
  int32_t max_pages_per_req; /* row pitch of the block tables                                   */
  int32_t total_tokens;      /* sum_r T_r                                                        */
  int32_t total_new;         /* sum_r |I_nr|                                                     */
  int32_t total_seg_pages;   /* sum_m len_m / block_size                                         */
  int32_t max_seq_len;       /* max_r T_r                                                        */
  /* device arrays */
  const int32_t *seq_len;    /* [num_reqs]     T_r (any value >= 1; last page may be partial)   */
  const int32_t *tok_off;    /* [num_reqs+1]   prefix sum of seq_len                             */
  int32_t *k_block_table;    /* [num_reqs][max_pages_per_req] logical page -> physical K page    */
  int32_t *v_block_table;    /* same for V; may alias k_block_table; written only under COW      */
  const int32_t *cow_private;/* [num_reqs][max_pages_per_req] reserved private page or -1; may be NULL */
  const sx_segment *segments;/* [num_segments]                                                   */
  const int32_t *src_blocks; /* [total_seg_pages] physical source pages (shared, never written)  */
  const int32_t *new_off;    /* [num_reqs+1]   CSR offsets into new_idx                          */
  const int32_t *new_idx;    /* [total_new]    sorted positions of I_nr per request (sparse mask m_i = 1) */
  /* RoPE: theta_i = rope_theta^(-2i/head_dim); rotation by angle delta*theta_i */
  double rope_theta;         /* host */
  int32_t rope_style;        /* host: 0 = pairs (i, i+head_dim/2) ("half-split"), 1 = pairs (2i, 2i+1) */
  int32_t zero_copy;         /* host: 0 = reused K is re-aligned into private pages by sx_rope_realign;
                                1 = zero-copy mode, see below                                            */
} sx_batch;

/* Zero-copy mode (batch->zero_copy = 1; the paper's remark that position-independent blocks can be SHARED between
 * requests, taken to its end for K as well as V). Nothing is re-aligned up front: the caller
 * points the k_block_table (and v_block_table) entries of reused pages straight at the cached source pages, whose
 * keys are stored rotated for their OLD positions, and the stage kernels apply R_{delta_m} while they read:
 *   - a logical page lp of request r that a segment m covers and whose k_block_table entry equals m's source page
 *     for lp is read ROTATED by delta_m (same arithmetic, same bits as sx_rope_realign would have stored);
 *     every other page (fresh, prefix hit, or already made private) is read as stored;
 *   - sx_score_select[_ex] and sx_sparse_attn rotate each K tile in shared memory between its TMA load and the MMA
 *     (in attention the softmax warpgroups do it; CTA pairs and the CUDA-core kernels are not available:
 *     SX_ERR_UNSUPPORTED);
 *   - sx_scatter_kv needs batch->cow_private: the first row written to a still-shared page copies it to its private
 *     page -- K rotated on the way, V bit-copied -- and flips the table entries; later calls see a private page;
 *   - sx_rope_realign[_layers] refuses the descriptor (SX_ERR_INVALID_ARG): its destination would be the shared
 *     source pages.
 * Memory: a request holds private pages only for the positions it recomputes (|R| / 16 pages, worst case one page
 * per recomputed token) instead of all of its reused pages. Cost: every sweep over K pays the rotation again
 * (measured in DESIGN.md S9). The tables belong to ONE layer, as under copy-on-write. */

/* Bytes of caller-provided workspace that any stage call on (pool, batch) may need. Host only. */
sx_status sx_workspace_size(const sx_pool *pool, const sx_batch *batch, size_t *bytes);

/* (a) PAPER.md:151-165, Alg. 1 l.502-504. For every segment m and token j < len:
 *   K[k_block_table[req][(new_pos+j)/16]][h][(new_pos+j)%16][:] = RNE_bf16(R_{delta_m} K[src page][h][j%16][:])
 *   V[v_block_table[...]] = V[src page] (bit copy; skipped when the V table entry IS the source
 *   page, i.e. the page is still shared copy-on-write).
 * Rotation in fp32 on angles computed in fp64 on the device; one rounding to bf16.
 * One launch for the whole batch ("fused copy-Delta-RoPE"). Source pages are
 * only read. Uses ws. */
sx_status sx_rope_realign(const sx_pool *pool, const sx_batch *batch, void *ws, size_t ws_bytes,
                          sx_stream stream);
/* (both realign calls return SX_ERR_INVALID_ARG for a batch in zero-copy mode) */

/* (a) for a stack of layers in ONE launch: pools[0..num_layers) are the per-layer pools (host array; same
 * num_blocks / num_kv_heads), all addressed through the same batch descriptor (block tables and segment map
 * are per request, not per layer). The re-alignment reads only cached source pages, never an output of the
 * current step, so it can be completed for every layer of the scheduling batch before the first layer runs
 * ("completes RoPE alignment for all requests in a scheduling batch", 331).
 * Not available with copy-on-write (batch->cow_private != NULL and num_layers > 1 -> SX_ERR_UNSUPPORTED): the
 * COW state is the v_block_table, which then belongs to ONE layer (page contents are per layer, so every layer
 * needs its own table and its own sx_batch; see sx_scatter_kv). */
sx_status sx_rope_realign_layers(const sx_pool *pools, int32_t num_layers, const sx_batch *batch, void *ws,
                                 size_t ws_bytes, sx_stream stream);

/* (d) Alg. 1 l.509-510 / 544-545; slot mapping PAPER.md:333. Rows of request r are
 * rows[rows_off[r] .. rows_off[r+1]) (absolute positions, strictly ascending within a request);
 * k_fresh / v_fresh are bf16 [n][Hkv][128] in the same order. For each row p:
 *   K[k_block_table[r][p/16]][:][p%16][:] = k_fresh[n],  V likewise through v_block_table.
 * Copy-on-write (batch->cow_private != NULL): before any row is written, a touched page whose
 * table entry differs from its reserved private page (>= 0) is copied there and the entry is
 * flipped (K and V tables independently). Rows not listed are untouched. The flipped table describes THIS
 * layer's pool only: under COW every layer of a stack has its own block tables (its own sx_batch).
 * max_rows (host) >= rows_off[num_reqs] sizes the grid. */
sx_status sx_scatter_kv(const sx_pool *pool, const sx_batch *batch, const void *k_fresh,
                        const void *v_fresh, const int32_t *rows, const int32_t *rows_off,
                        int32_t max_rows, sx_stream stream);

/* (b) Eq. (1)-(3); Alg. 1 l.515-531, 537-539.
 *   q_new     device bf16 [total_new][Hq][128]: queries of I_nr in new_idx order, already rotated.
 *   lse_new   device fp32 natural-log softmax normaliser of those rows over the CURRENT pool, or
 *             NULL (then a first QK^T sweep computes it). lse_by_token = 0: [total_new][Hq] in
 *             new_idx order; 1: [total_tokens][Hq] indexed by batch token tok_off[r]+position (the
 *             lse output of a full-mode sx_sparse_attn: boundary layer of Alg. 1 l.507-531).
 *   sel_off   device [num_reqs+1]: request r selects k_r = sel_off[r+1]-sel_off[r] cached tokens
 *             (k_r <= number of cached tokens of r); rows_off device [num_reqs+1] with
 *             rows_off[r+1]-rows_off[r] = |I_nr(r)| + k_r.
 *   scores    device fp32 [total_tokens] or NULL: s_j of every position (token (r,j) at tok_off[r]+j).
 *   sel_idx   device int32 [sel_off[num_reqs]]: S_key per request, ascending positions.
 *   rows_R    device int32 [rows_off[num_reqs]]: R = I_nr U S_key per request, ascending.
 * Candidates are the REUSED positions only (those covered by a segment of the request; see "Token classes" below);
 * order = (score descending, position ascending); k is clamped to their number.
 * Scores are fp32 sums in a fixed order (deterministic). Uses ws. */
sx_status sx_score_select(const sx_pool *pool, const sx_batch *batch, const void *q_new,
                          const float *lse_new, int32_t lse_by_token, const int32_t *sel_off,
                          const int32_t *rows_off,
                          float *scores, int32_t *sel_idx, int32_t *rows_R, void *ws,
                          size_t ws_bytes, sx_stream stream);

/* (b) with the two additions that complete the paper's recompute set (Alg. 1 l.535-539):
 *   R = I_nr U S_key U S_ov U S_tail
 *   S_ov   (overflow): every maximal contiguous interval of I_nr is expanded by
 *          overflow_blocks pages (the paper uses 1) on both sides, clipped to the request;
 *   S_tail (tail fallback): if the last position of the request is a reused token, the last
 *          tail_tokens (the paper uses 64) positions of the reused segment that holds it.
 * S_key is still the top-k of ALL cached positions (it may overlap S_ov / S_tail), so |R| depends on the data:
 *   rows_off      device [num_reqs+1]: CAPACITY offsets; slot r must hold |I_nr(r)| + k_r + |S_ov U S_tail|
 *                 positions (host-computable from the layout; rows beyond the capacity would be dropped);
 *   rows_R        device int32 [rows_off[num_reqs]]: R of all requests, packed back to back;
 *   rows_off_out  device [num_reqs+1]: the actual CSR offsets into rows_R. Pass (rows_R, rows_off_out) to
 *                 sx_scatter_kv / sx_sparse_attn with max_rows / total_rows = rows_off[num_reqs] (upper bound).
 * With overflow_blocks = tail_tokens = 0 this is sx_score_select (rows_off_out may then be NULL). */
sx_status sx_score_select_ex(const sx_pool *pool, const sx_batch *batch, const void *q_new,
                             const float *lse_new, int32_t lse_by_token, const int32_t *sel_off,
                             const int32_t *rows_off, int32_t overflow_blocks, int32_t tail_tokens,
                             float *scores, int32_t *sel_idx, int32_t *rows_R, int32_t *rows_off_out, void *ws,
                             size_t ws_bytes, sx_stream stream);

/* Token classes (Alg. 1 l.500-501). A position of a request is NEW if it is listed in new_idx (I_nr), REUSED if a
 * segment covers it (I_reuse: re-aligned by sx_rope_realign, the candidates of the top-k, the only members of
 * S_ov / S_tail), otherwise a PREFIX-CACHE HIT: its K/V are already in the request's pages at the right position
 * ("excluded from the current prefill computation"): visible as a key everywhere, never a candidate, never a query
 * row. With prefix hits, full-attention layers are run in mode 0 with the non-prefix positions as rows_R. */
#define SX_ATTN_CUDA_CORE 2 /* flag for sx_sparse_attn's mode: CUDA-core kernels for small row sets */
#define SX_ATTN_CTA_PAIR 4  /* flag for sx_sparse_attn's mode: force 2-CTA clusters (tcgen05.mma.cta_group::2) */
#define SX_ATTN_SINGLE_CTA 8 /* flag for sx_sparse_attn's mode: force the single-CTA tensor-core kernel */

/* (c) Alg. 1 l.546-548 (sparse) / l.507-511 (full). mode 0: query rows are rows_R (as produced by
 * sx_score_select); mode 1: rows_R and rows_off are ignored, every position of every request is
 * a query row (R = {0..T-1}, row n of the batch = token tok_off[r]+j).
 *   q    device bf16 [total_rows][Hq][128], compact in rows order; out same shape (bf16);
 *   lse  device fp32 [total_rows][Hq] natural-log normaliser, or NULL.
 *   total_rows (host) >= rows_off[num_reqs] (mode 0; equal unless the row list came from sx_score_select_ex,
 *   then its capacity) or = total_tokens (mode 1); q / out / lse are sized by total_rows.
 * O[n][h] = sum_{j <= pos(n)} softmax_j(<q, k_j>/sqrt(128)) v_j with kv head h / g, K and V read
 * through the block tables. Kernels, chosen from host-visible sizes only:
 *   - general kernel: tcgen05 tensor-core tiles with the query rows on the M dimension, bf16 x bf16 -> fp32
 *     accumulate, fp32 softmax, P rounded to bf16 before PV. When the row set fills fewer than 148 CTAs (few query
 *     tiles against a long context) the key range is cut into splits that merge themselves in a fixed order (the
 *     splits of a row pair wait for one another through an arrival word in ws: one launch); uses ws in that case.
 *   - mode | SX_ATTN_CUDA_CORE: row sets with total_rows * g < 64 * num_reqs (fewer than 64 query rows per
 *     KV head on average; g = Hq/Hkv <= 32) take CUDA-core split-KV kernels, fp32 FMA throughout (the rule of
 *     BASELINE.json north_star; measured slower than the padded tensor-core tile on B200). Uses ws.
 *   - CTA pairs: when the general kernel runs without key splits it exists in two forms with the same arithmetic
 *     per row (hence the same results): one CTA per pair of query tiles, or clusters of two CTAs on adjacent pairs
 *     with M = 256 MMAs (tcgen05.mma.cta_group::2), where every K/V tile is fetched once per cluster, half into
 *     each CTA. Measured (S10): clusters are 1-2 % faster for a batch of ONE request (long uniform
 *     launches) and 5-6 % slower for batches of several requests, so that is the default rule;
 *     mode | SX_ATTN_CTA_PAIR / mode | SX_ATTN_SINGLE_CTA force one or the other.
 * Every kernel is launched with programmatic dependent launch allowed: its prologue may overlap the tail of the
 * previous kernel in the stream; it touches global memory only after that kernel has completed.
 * All are deterministic and meet the same tolerance against fp64. */
sx_status sx_sparse_attn(const sx_pool *pool, const sx_batch *batch, int32_t mode, const void *q,
                         const int32_t *rows_R, const int32_t *rows_off, int32_t total_rows,
                         void *out, float *lse, void *ws, size_t ws_bytes, sx_stream stream);

/* (c) for SMALL row sets without a workspace and without any allocation: for callers that cannot allocate device
 * memory where they call from (code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc).
 * Same operation, same kernel and same results as sx_sparse_attn in mode 0 (the single-CTA tensor-core kernel with
 * self-merging key splits); the scratch of the key splits lives in a file-scope device array of
 * SX_NOALLOC_SCRATCH_BYTES (9.1 MiB) that every GPU which loads the library holds until the process exits.
 *   Limit: total_rows * num_q_heads <= SX_NOALLOC_MAX_PAIRS (row, query head) pairs (e.g. 32 rows x 32 heads);
 *          beyond it SX_ERR_UNSUPPORTED with the sizes in sx_last_error(), nothing launched. The number of key
 *          splits is reduced until its partials fit the array (18 at the limit), so a row set near the limit may be
 *          cut differently from sx_sparse_attn (same tolerance, different rounding); equal cuts give equal bits.
 *   Not available for batches in zero-copy mode (their page classification needs the workspace).
 *   The call makes no cudaMalloc / cudaFree and uses no allocating library routine; the first call on a device looks
 *   the array's device address up once (make that call outside a graph capture).
 *   SHARED STATE: every call on a device uses the same array. Calls ordered on one stream (or by events / graph
 *   edges) are safe, and nothing has to be cleared between them; calls that OVERLAP on the GPU race on the array
 *   (wrong results or a hang): concurrent callers use sx_sparse_attn with a workspace each. */
#define SX_NOALLOC_MAX_PAIRS 1024
#define SX_NOALLOC_SCRATCH_BYTES 9512096
sx_status sx_sparse_attn_noalloc(const sx_pool *pool, const sx_batch *batch, const void *q, const int32_t *rows_R,
                                 const int32_t *rows_off, int32_t total_rows, void *out, float *lse,
                                 sx_stream stream);

/* Validation of the DEVICE-resident descriptor arrays, which the stage calls cannot see from the host mirrors:
 * seq_len / tok_off / new_off consistent with the host counts; new_idx strictly ascending inside its request;
 * every segment's len / old_pos / new_pos a positive multiple of block_size, src_off the running
 * sum of len / block_size, segments sorted by (req, new_pos) and non-overlapping, inside the request's pages;
 * src_blocks, the block-table entries of used pages and cow_private inside the pool; every table entry that still is
 * its segment's shared source page (copy-on-write V, zero-copy K and V) has a reserved private page. One small kernel, one error
 * word copied back: this call SYNCHRONISES `stream`. Returns SX_OK or SX_ERR_INVALID_ARG with the failing check
 * and its index in sx_last_error(). A descriptor that fails here would corrupt pages in the stage calls. Uses ws. */
sx_status sx_check_batch(const sx_pool *pool, const sx_batch *batch, void *ws, size_t ws_bytes, sx_stream stream);

/* Same for a row list handed to sx_scatter_kv / sx_sparse_attn: rows_off ascending from 0 with
 * rows_off[num_reqs] <= max_rows; rows strictly ascending inside [0, seq_len) of their request.
 * SYNCHRONISES `stream`. Uses ws. */
sx_status sx_check_rows(const sx_pool *pool, const sx_batch *batch, const int32_t *rows, const int32_t *rows_off,
                        int32_t max_rows, void *ws, size_t ws_bytes, sx_stream stream);

/* Number of kernels this library has launched in the process so far (diagnostic; monotone, thread safe). */
uint64_t sx_launch_count(void);

/* Diagnostic, not part of the method: instruction-pipe rate probe, the denominator of the roofline of the scoring
 * sweeps (one exponential per 256 flop: bound by the special-function pipe). Launches num_ctas CTAs of 1024 threads,
 * each running 8 * iters dependent-chain operations per thread on ONE pipe, and writes the clock64() cycles of every
 * CTA's loop to cycles[0 .. num_ctas) (device, uint64; one more word behind them is scratch):
 *   pipe 0 = MUFU.EX2, 1 = FFMA, 2 = FFMA2 (two fused multiply-adds per lane), 3 = the sweeps' mix (of every 8
 *   exponentials 6 on MUFU.EX2 and 2 by the FMA-pipe polynomial).
 * Lane-operations per clock and SM = 1024 * 8 * iters / cycles with one CTA per SM. Asynchronous on `stream`. */
sx_status sx_probe_pipe(int32_t pipe, int32_t iters, uint64_t *cycles, int32_t num_ctas, sx_stream stream);

/* Thread-local text of the last error returned on this thread ("" if none). Static storage. */
const char *sx_last_error(void);

/* Library build tag, e.g. "sparsex-b200 sm_100a". Static storage. */
const char *sx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPARSEX_H_ */
