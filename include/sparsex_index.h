/*
 * sparsex_index.h -- host-side segment index of SparseX (arxiv/paper_2606_01751 S4, PAPER.md:285-337;
 * Alg. 1 l.500-501): the step BEFORE the GPU path. It turns a prompt with candidate reuse segments into the
 * pieces of the sx_batch descriptor (segment map, source pages, Sparse-Q mask) that include/sparsex.h consumes.
 * Pure host code, no CUDA calls; lives in the same shared library.
 *
 *   virtual block a position-, prefix- and context-independent view of ONE physical KV
 *                   block: (physical block id, position of its first token when it was cached, virtual hash).
 *   virtual hash    h = H(B, e) over the block's token ids B and the namespace ("extra") key e
 *                   (PAPER.md:301-311). The paper does not fix H: here 64-bit FNV-1a over e then the tokens
 *                   (reading A25); a hit additionally requires the stored token ids and e to be equal.
 *   frozen block an entry that is not dropped when its reference count reaches zero; it
 *                   leaves the pool only through sx_index_erase or the utilisation-triggered eviction, which
 *                   removes the least-referenced unreferenced frozen entries first.
 *
 * All functions are thread-compatible (no internal locking). Sizes are in tokens unless stated; every segment
 * length and position must be a multiple of block_size. Return values < 0 are sx_status codes
 * (SX_ERR_INVALID_ARG = -1).
 */
#ifndef SPARSEX_INDEX_H_
#define SPARSEX_INDEX_H_

#include <stdint.h>

#include "sparsex.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sx_index sx_index; /* opaque; owned by the caller through create / destroy */

sx_index *sx_index_create(int32_t block_size);
void sx_index_destroy(sx_index *ix);

/* Number of virtual blocks currently indexed. */
int32_t sx_index_size(const sx_index *ix);

/* Register a cached segment: tokens[len] were prefilled at positions [old_pos, old_pos + len) and their K/V
 * live in blocks[len / block_size] (host array of physical page ids). One virtual block per page is
 * inserted under namespace extra_key; an entry with the same (tokens, extra_key) is overwritten.
 * frozen != 0 marks the entries as frozen blocks. Returns the number of entries inserted or overwritten. */
int32_t sx_index_insert(sx_index *ix, const int32_t *tokens, int32_t len, uint64_t extra_key, int32_t old_pos,
                        const int32_t *blocks, int32_t frozen);

/* Remove the virtual blocks of tokens[len] under extra_key (insert / delete API of PAPER.md:291).
 * Returns how many were removed. */
int32_t sx_index_erase(sx_index *ix, const int32_t *tokens, int32_t len, uint64_t extra_key);

/* Alg. 1 l.500 for one request. The prompt is tokens[seq_len]; cand[i] = {start, len} (host arrays of
 * num_cand pairs, ascending, non-overlapping, block aligned) are the candidate reuse segments, all looked up
 * under extra_key. A candidate hits only if EVERY one of its blocks is indexed (token ids and key equal).
 * A hit candidate is emitted as one sx_segment per maximal run of blocks whose cached positions are
 * contiguous (constant delta): {req, len, old_pos, new_pos, src_off}, with src_off the running offset into
 * src_blocks_out. Positions not covered by a hit form I_nr (Alg. 1 l.501, sparse mask m_i = 1), written
 * ascending to new_idx_out. Every block handed out gets its reference count and its hit count increased.
 *   segments_out   capacity seq_len / block_size entries
 *   src_blocks_out capacity seq_len / block_size
 *   new_idx_out    capacity seq_len
 *   counts_out[3]  {number of segments, number of source pages, |I_nr|}
 * Returns the number of candidates that hit. */
int32_t sx_index_plan_request(sx_index *ix, int32_t req, const int32_t *tokens, int32_t seq_len,
                              const int32_t *cand, int32_t num_cand, uint64_t extra_key,
                              sx_segment *segments_out, int32_t *src_blocks_out, int32_t *new_idx_out,
                              int32_t *counts_out);

/* The request is done with these source pages (after the copy-Delta-RoPE): drop one reference each.
 * Non-frozen entries whose count reaches zero are removed (ordinary blocks return to the engine's free list,
 * PAPER.md:289). Returns the number of entries removed. */
int32_t sx_index_release(sx_index *ix, const int32_t *src_blocks, int32_t n);

/* Utilisation-triggered eviction ("when KV Cache block utilization exceeds 90 % ... delete the
 * least-referenced blocks from the frozen-block pool"): while used_blocks / total_blocks > threshold, remove
 * physical blocks whose virtual blocks are ALL frozen and unreferenced (several namespaces / token views may sit
 * on one physical block; one referenced or non-frozen view keeps the block), in order (hit count summed over the
 * block's views ascending, then its oldest insertion first). All views of an evicted block leave the index and
 * the block is reported once: evicted_out (capacity max_out) receives the distinct physical ids. Returns how
 * many blocks were freed. */
int32_t sx_index_evict(sx_index *ix, int32_t used_blocks, int32_t total_blocks, double threshold,
                       int32_t *evicted_out, int32_t max_out);

#ifdef __cplusplus
}
#endif
#endif /* SPARSEX_INDEX_H_ */
