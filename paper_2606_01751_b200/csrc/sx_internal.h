// sx_internal.h -- declarations shared by the translation units of libsparsex.so (not installed).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/sparsex.h"

namespace sx {

constexpr int kHeadDim = 128;   // D
constexpr int kPage = 16;       // block_size b
constexpr int kTile = 128;      // keys per K/V tile = 8 pages; rows per Q tile
constexpr double kLog2e = 1.4426950408889634;

// Workspace carve-up (all offsets 256-B aligned). Computed from host mirrors only.
struct WsLayout {
  size_t rope_table;   // float2 [num_segments][64]       (cos, sin)(delta_m * theta_i)
  size_t page_desc;    // int4   [total_seg_pages]        (segment, source, destination K, destination V) per page
  size_t lse_new;      // float  [8][total_new][Hq]       sweep-1 normaliser (natural log) per key split
  size_t partial;      // float  [Hkv][total_tokens]      per-kv-head column sums of A_sq
  size_t scores;       // float  [total_tokens]           head-summed scores when the caller passes none
  size_t col_tab;      // float2 [query tiles][Hkv][128]  (log2-domain lse, position) of every sweep-2 column
  size_t rows_tmp;     // int32  [total_tokens]           capacity-slotted R of the extended selection
  size_t rows_cnt;     // int32  [num_reqs]
  size_t sel_scratch;  // int    [num_reqs][4*256 + 4*64] digit histograms and slice counters of the multi-CTA select
  size_t attn_part;    // float  key-split partials of the tcgen05 attention (few CTAs, long context)
  size_t small_part;   // float  split-KV partials of the CUDA-core attention path (sx_attn_small.cu)
  size_t page_seg;     // int32  [num_reqs][max_pages]    zero-copy mode: segment whose source page the entry still is, or -1
  size_t total;
};
WsLayout ws_layout(const sx_pool *pool, const sx_batch *batch);

sx_status set_error(sx_status st, const char *fmt, ...);
sx_status check_launch(const char *what);

// kernels (one launcher per translation unit)
sx_status launch_realign(const sx_pool *pools, int num_layers, const sx_batch *b, float2 *table, int4 *page_desc,
                         cudaStream_t st);
// zero-copy mode: rotation table + page_seg of the workspace (sx_realign.cu); run before a stage that rotates on the fly
sx_status launch_zc_prepare(const sx_batch *b, float2 *table, int32_t *page_seg, cudaStream_t st);
struct ZcArgs {  // what a rotating kernel needs; style < 0: not in zero-copy mode
  int style = -1;
  const float2 *table = nullptr;
  const int32_t *page_seg = nullptr;
};
sx_status launch_scatter(const sx_pool *pool, const sx_batch *b, const void *k_fresh, const void *v_fresh,
                         const int32_t *rows, const int32_t *rows_off, int32_t max_rows, cudaStream_t st);
sx_status launch_select(const sx_pool *pool, const sx_batch *b, const float *partial, const int32_t *sel_off,
                        const int32_t *rows_off, float *scores, int32_t *sel_idx, int32_t *rows_R, int ov_blocks,
                        int tail_tokens, int32_t *rows_tmp, int32_t *rows_cnt, int32_t *rows_off_out, int *scratch,
                        cudaStream_t st);
size_t select_scratch_bytes(const sx_batch *b);
// tcgen05 kernels. q_rows: bf16 [total_rows][Hq][128]; rows == nullptr => row n is position n - off[req].
sx_status launch_attn(const sx_pool *pool, const sx_batch *b, const void *q, const int32_t *rows,
                      const int32_t *rows_off, int32_t total_rows, void *out, float *lse, int kv_splits,
                      float *part, bool cta_pair, const ZcArgs &zc, cudaStream_t st,
                      unsigned long long *tickets = nullptr);  // tickets == nullptr: the words behind `part` (attn_tickets)
// the same kernel with its key-split scratch in a file-scope device array (sx_attn_noalloc.cu): no workspace argument
sx_status launch_attn_noalloc(const sx_pool *pool, const sx_batch *b, const void *q, const int32_t *rows,
                              const int32_t *rows_off, int32_t total_rows, void *out, float *lse, cudaStream_t st);
int attn_pv_splits(const sx_pool *pool, const sx_batch *b, int32_t total_rows, int tiles_per_cta);
size_t attn_part_bytes();
unsigned long long *attn_tickets(float *part);  // rendezvous words of the key splits, behind the partial buffer
// first sweep of stage (b) (sx_lse.cu): partial log-sum-exps [kv_splits][total_new][Hq] of the Sparse-Q rows
int lse_splits(const sx_pool *pool, const sx_batch *b);
sx_status launch_lse(const sx_pool *pool, const sx_batch *b, const void *q_new, float *lse_ws, int kv_splits,
                     const ZcArgs &zc, cudaStream_t st);
// CUDA-core split-KV attention for fewer than 64 (row, head) pairs per KV head; part = ws.small_part
sx_status launch_attn_small(const sx_pool *pool, const sx_batch *b, const void *q, const int32_t *rows,
                            const int32_t *rows_off, int32_t total_rows, void *out, float *lse, float *part,
                            cudaStream_t st);
size_t small_ws_bytes(int num_reqs, int num_kv_heads, int group);
sx_status launch_colsum(const sx_pool *pool, const sx_batch *b, const void *q_new, const float *lse_new,
                        int lse_by_token, int lse_splits, float *partial, float2 *col_tab, const ZcArgs &zc,
                        cudaStream_t st);
size_t colsum_tab_bytes(const sx_pool *pool, const sx_batch *b);

// descriptor validation (sx_check.cu): one kernel + one error word copied back; synchronises the stream
sx_status run_check_batch(const sx_pool *pool, const sx_batch *b, void *ws, cudaStream_t st);
sx_status run_check_rows(const sx_batch *b, const int32_t *rows, const int32_t *rows_off, int32_t max_rows, void *ws,
                         cudaStream_t st);

// instruction-pipe rate probe (sx_probe.cu)
sx_status launch_probe(int pipe, int iters, unsigned long long *cycles, int num_ctas, cudaStream_t st);

// TMA descriptor construction (driver entry point fetched through the runtime; no libcuda link)
sx_status make_tmap_pool(CUtensorMap *out, const void *base, int num_blocks, int num_kv_heads);
sx_status make_tmap_q(CUtensorMap *out, const void *base, int total_rows, int num_q_heads, int group,
                      int rows_per_tile);

// Launch with programmatic dependent launch allowed (and optionally a cluster dimension): the kernel must call
// griddep_wait() (sx_ptx.cuh) before its first global-memory access.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, int cluster,
                              Args &&...args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  int n = 0;
  attr[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[n].val.programmaticStreamSerializationAllowed = 1;
  ++n;
  if (cluster > 1) {
    attr[n].id = cudaLaunchAttributeClusterDimension;
    attr[n].val.clusterDim.x = cluster;
    attr[n].val.clusterDim.y = 1;
    attr[n].val.clusterDim.z = 1;
    ++n;
  }
  cfg.attrs = attr;
  cfg.numAttrs = n;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

}  // namespace sx
