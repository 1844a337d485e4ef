// sx_check.cu -- validation of the device-resident parts of the block-table / segment-map descriptor
// (sx_check_batch, sx_check_rows in include/sparsex.h). The stage calls validate only what the host mirrors
// show; the arrays themselves live on the device, so a misaligned segment (reuse-segment
// boundaries are block aligned) or an out-of-range page id would silently corrupt pages. These two calls
// run one small kernel over the arrays, copy one error word back and -- unlike every stage call --
// SYNCHRONISE the stream: they are meant for descriptor construction time, not for the hot path.
#include "sx_internal.h"

namespace sx {

// first failing check wins: the error word is min over (check id << 32 | index)
enum CheckId : int {
  kChkSeqLen = 1, kChkTokOff, kChkNewOff, kChkNewIdx, kChkSegReq, kChkSegAlign, kChkSegRange, kChkSegSrcOff,
  kChkSegOrder, kChkSegPages, kChkSrcBlock, kChkKTable, kChkVTable, kChkCow, kChkShared, kChkRowsOff, kChkRows
};

static const char *check_text(int id) {
  switch (id) {
    case kChkSeqLen: return "seq_len[r] outside [1, max_seq_len]";
    case kChkTokOff: return "tok_off is not the prefix sum of seq_len ending at total_tokens";
    case kChkNewOff: return "new_off not ascending, or new_off[num_reqs] != total_new";
    case kChkNewIdx: return "new_idx not strictly ascending inside [0, seq_len) of its request";
    case kChkSegReq: return "segment request index out of range";
    case kChkSegAlign: return "segment len / old_pos / new_pos not a positive multiple of block_size (PAPER.md:327)";
    case kChkSegRange: return "segment exceeds the pages of its request";
    case kChkSegSrcOff: return "segment src_off is not the running sum of len / block_size";
    case kChkSegOrder: return "segments not sorted by (req, new_pos) or overlapping";
    case kChkSegPages: return "total_seg_pages != sum of len / block_size";
    case kChkSrcBlock: return "src_blocks entry outside [0, num_blocks)";
    case kChkKTable: return "k_block_table entry of a used page outside [0, num_blocks)";
    case kChkVTable: return "v_block_table entry of a used page outside [0, num_blocks)";
    case kChkCow: return "cow_private entry outside [-1, num_blocks)";
    case kChkShared:
      return "a table entry that still is its segment's shared source page has no reserved private page (cow_private)";
    case kChkRowsOff: return "rows_off not ascending from 0, or rows_off[num_reqs] > max_rows";
    case kChkRows: return "row list not strictly ascending inside [0, seq_len) of its request";
  }
  return "unknown check";
}

__device__ __forceinline__ void fail(unsigned long long *err, int id, int index) {
  atomicMin(err, ((unsigned long long)id << 32) | (unsigned)index);
}

__global__ void __launch_bounds__(1024)
check_batch_kernel(sx_batch b, int num_blocks, unsigned long long *err) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  for (int r = tid; r < b.num_reqs; r += nth) {
    const int t = b.seq_len[r];
    if (t < 1 || t > b.max_seq_len) fail(err, kChkSeqLen, r);
    if (b.tok_off[r + 1] - b.tok_off[r] != t || (r == 0 && b.tok_off[0] != 0) ||
        (r == b.num_reqs - 1 && b.tok_off[r + 1] != b.total_tokens))
      fail(err, kChkTokOff, r);
    if (b.new_off[r + 1] < b.new_off[r] || (r == 0 && b.new_off[0] != 0) ||
        (r == b.num_reqs - 1 && b.new_off[r + 1] != b.total_new))
      fail(err, kChkNewOff, r);
  }
  // new_idx: every element against its predecessor; its request by binary search in new_off
  for (int i = tid; i < b.total_new; i += nth) {
    int lo = 0, hi = b.num_reqs - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (b.new_off[mid] <= i) lo = mid; else hi = mid - 1;
    }
    const int p = b.new_idx[i], t = b.seq_len[lo];
    if (p < 0 || p >= t || (i > b.new_off[lo] && b.new_idx[i - 1] >= p)) fail(err, kChkNewIdx, i);
  }
  for (int m = tid; m < b.num_segments; m += nth) {
    const sx_segment s = b.segments[m];
    if (s.req < 0 || s.req >= b.num_reqs) {
      fail(err, kChkSegReq, m);
      continue;
    }
    if (s.len <= 0 || s.len % kPage || s.old_pos < 0 || s.old_pos % kPage || s.new_pos < 0 || s.new_pos % kPage) {
      fail(err, kChkSegAlign, m);
      continue;
    }
    const int pages_r = (b.seq_len[s.req] + kPage - 1) / kPage;
    if ((s.new_pos + s.len) / kPage > pages_r || (s.new_pos + s.len) / kPage > b.max_pages_per_req)
      fail(err, kChkSegRange, m);
    if (m == 0) {
      if (s.src_off != 0) fail(err, kChkSegSrcOff, m);
    } else {
      const sx_segment q = b.segments[m - 1];
      if (s.src_off != q.src_off + q.len / kPage) fail(err, kChkSegSrcOff, m);
      if (q.req > s.req || (q.req == s.req && q.new_pos + q.len > s.new_pos)) fail(err, kChkSegOrder, m);
    }
    if (m == b.num_segments - 1 && s.src_off + s.len / kPage != b.total_seg_pages) fail(err, kChkSegPages, m);
  }
  if (b.num_segments == 0 && b.total_seg_pages != 0 && tid == 0) fail(err, kChkSegPages, 0);
  for (int i = tid; i < b.total_seg_pages; i += nth) {
    const int blk = b.src_blocks[i];
    if (blk < 0 || blk >= num_blocks) fail(err, kChkSrcBlock, i);
    // copy-on-write / zero-copy: an entry that still aliases the shared page must have somewhere to go when written
    int lo = 0, hi = b.num_segments - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (b.segments[mid].src_off <= i) lo = mid; else hi = mid - 1;
    }
    const sx_segment s = b.segments[lo];
    const int lp = s.new_pos / kPage + (i - s.src_off);
    if (s.req >= 0 && s.req < b.num_reqs && s.new_pos >= 0 && i >= s.src_off && lp < b.max_pages_per_req) {
      const size_t e = (size_t)s.req * b.max_pages_per_req + lp;
      if (b.k_block_table[e] == blk || b.v_block_table[e] == blk) {
        const int cp = b.cow_private ? b.cow_private[e] : -1;
        if (cp < 0 || cp == blk) fail(err, kChkShared, i);
      }
    }
  }
  const int entries = b.num_reqs * b.max_pages_per_req;
  for (int i = tid; i < entries; i += nth) {
    const int r = i / b.max_pages_per_req, pg = i - r * b.max_pages_per_req;
    const bool used = pg < (b.seq_len[r] + kPage - 1) / kPage;
    if (used) {
      const int kb = b.k_block_table[i], vb = b.v_block_table[i];
      if (kb < 0 || kb >= num_blocks) fail(err, kChkKTable, i);
      if (vb < 0 || vb >= num_blocks) fail(err, kChkVTable, i);
    }
    if (b.cow_private) {
      const int cp = b.cow_private[i];
      if (cp < -1 || cp >= num_blocks) fail(err, kChkCow, i);
    }
  }
}

__global__ void __launch_bounds__(1024)
check_rows_kernel(int num_reqs, const int32_t *seq_len, const int32_t *rows, const int32_t *rows_off, int max_rows,
                  unsigned long long *err) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  for (int r = tid; r < num_reqs; r += nth)
    if (rows_off[r + 1] < rows_off[r] || (r == 0 && rows_off[0] != 0) ||
        (r == num_reqs - 1 && rows_off[r + 1] > max_rows))
      fail(err, kChkRowsOff, r);
  int total = rows_off[num_reqs];
  if (total > max_rows) total = max_rows;
  for (int i = tid; i < total; i += nth) {
    int lo = 0, hi = num_reqs - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (rows_off[mid] <= i) lo = mid; else hi = mid - 1;
    }
    const int p = rows[i];
    if (p < 0 || p >= seq_len[lo] || (i > rows_off[lo] && rows[i - 1] >= p)) fail(err, kChkRows, i);
  }
}

static sx_status finish_check(unsigned long long *err_dev, cudaStream_t st, const char *what) {
  unsigned long long h = ~0ull;
  cudaError_t e = cudaMemcpyAsync(&h, err_dev, sizeof h, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
  if (h == ~0ull) return SX_OK;
  return set_error(SX_ERR_INVALID_ARG, "%s: %s (index %u)", what, check_text((int)(h >> 32)), (unsigned)(h & 0xffffffffu));
}

sx_status run_check_batch(const sx_pool *pool, const sx_batch *b, void *ws, cudaStream_t st) {
  unsigned long long *err = reinterpret_cast<unsigned long long *>(ws);
  cudaError_t e = cudaMemsetAsync(err, 0xff, sizeof(unsigned long long), st);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "check memset: %s", cudaGetErrorString(e));
  check_batch_kernel<<<32, 1024, 0, st>>>(*b, pool->num_blocks, err);
  sx_status s = check_launch("check_batch_kernel");
  if (s != SX_OK) return s;
  return finish_check(err, st, "sx_check_batch");
}

sx_status run_check_rows(const sx_batch *b, const int32_t *rows, const int32_t *rows_off, int32_t max_rows, void *ws,
                         cudaStream_t st) {
  unsigned long long *err = reinterpret_cast<unsigned long long *>(ws);
  cudaError_t e = cudaMemsetAsync(err, 0xff, sizeof(unsigned long long), st);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "check memset: %s", cudaGetErrorString(e));
  check_rows_kernel<<<32, 1024, 0, st>>>(b->num_reqs, b->seq_len, rows, rows_off, max_rows, err);
  sx_status s = check_launch("check_rows_kernel");
  if (s != SX_OK) return s;
  return finish_check(err, st, "sx_check_rows");
}

}  // namespace sx
