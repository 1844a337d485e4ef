// sx_scatter.cu -- stage (d): write the fresh K,V rows of the computed positions into their paged
// slots (Alg. 1 l.509-510 / 544-545 "write fresh K,V into the current request cache"; slot mapping
// PAPER.md:333), with copy-on-write of still-shared pages (reading A14).
//
// HBM-bound bit copy: 8*Hkv*128 bytes per row. One warp per row, 16-byte vector loads/stores; the
// 256 B of one (row, head) are written by 16 consecutive lanes.
#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

__device__ __forceinline__ int find_req(const int32_t *__restrict__ off, int num_reqs, int n) {
  int r = 0;
  while (r + 1 < num_reqs && n >= off[r + 1]) ++r;
  return r;
}

// Copy-on-write resolve: the first listed row of every touched page copies the page it still
// aliases into the reserved private page and flips the table entry (K and V independently).
// Rows are ascending within a request, so "first row of its page" is a local test: no atomics.
__global__ void __launch_bounds__(128)
cow_kernel(uint4 *pool_k, uint4 *pool_v, int num_kv_heads, int num_reqs, int max_pages, int32_t *k_table,
           int32_t *v_table, const int32_t *__restrict__ cow_private, const int32_t *__restrict__ rows,
           const int32_t *__restrict__ rows_off) {
  const int n = blockIdx.x;
  if (n >= rows_off[num_reqs]) return;
  const int req = find_req(rows_off, num_reqs, n);
  const int p = rows[n];
  const int pg = p / kPage;
  if (n > rows_off[req] && rows[n - 1] / kPage == pg) return;  // not the first row of this page
  const size_t e = (size_t)req * max_pages + pg;
  const int priv = cow_private[e];
  if (priv < 0) return;
  const int page_chunks = num_kv_heads * kPage * 16;
  const int ck = k_table[e], cv = v_table[e];
  if (ck != priv) {
    const uint4 *s = pool_k + (size_t)ck * page_chunks;
    uint4 *d = pool_k + (size_t)priv * page_chunks;
    for (int i = threadIdx.x; i < page_chunks; i += blockDim.x) d[i] = s[i];
  }
  if (cv != priv) {
    const uint4 *s = pool_v + (size_t)cv * page_chunks;
    uint4 *d = pool_v + (size_t)priv * page_chunks;
    for (int i = threadIdx.x; i < page_chunks; i += blockDim.x) d[i] = s[i];
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    if (ck != priv) k_table[e] = priv;
    if (cv != priv && v_table + e != k_table + e) v_table[e] = priv;
  }
}

constexpr int kScatterWarps = 8;

__global__ void __launch_bounds__(kScatterWarps * 32)
scatter_kernel(uint4 *pool_k, uint4 *pool_v, int num_kv_heads, int num_reqs, int max_pages,
               const int32_t *__restrict__ k_table, const int32_t *__restrict__ v_table,
               const uint4 *__restrict__ k_fresh, const uint4 *__restrict__ v_fresh, const int32_t *__restrict__ rows,
               const int32_t *__restrict__ rows_off) {
  const int n = blockIdx.x * kScatterWarps + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (n >= rows_off[num_reqs]) return;
  const int req = find_req(rows_off, num_reqs, n);
  const int p = rows[n];
  const int pg = p / kPage, o = p % kPage;
  const size_t e = (size_t)req * max_pages + pg;
  const int kb = k_table[e], vb = v_table[e];
  const int row_chunks = num_kv_heads * 16;  // 16-byte chunks of one fresh row
  const uint4 *ks = k_fresh + (size_t)n * row_chunks;
  const uint4 *vs = v_fresh + (size_t)n * row_chunks;
  for (int c = lane; c < row_chunks; c += 32) {
    const int h = c >> 4, cc = c & 15;
    const size_t dst = (((size_t)kb * num_kv_heads + h) * kPage + o) * 16 + cc;
    const size_t dstv = (((size_t)vb * num_kv_heads + h) * kPage + o) * 16 + cc;
    uint4 a = __ldg(ks + c);
    uint4 b = __ldg(vs + c);
    pool_k[dst] = a;
    pool_v[dstv] = b;
  }
}

sx_status launch_scatter(const sx_pool *pool, const sx_batch *b, const void *k_fresh, const void *v_fresh,
                         const int32_t *rows, const int32_t *rows_off, int32_t max_rows, cudaStream_t st) {
  uint4 *pk = reinterpret_cast<uint4 *>(pool->k);
  uint4 *pv = reinterpret_cast<uint4 *>(pool->v);
  if (b->cow_private) {
    cow_kernel<<<max_rows, 128, 0, st>>>(pk, pv, pool->num_kv_heads, b->num_reqs, b->max_pages_per_req,
                                         b->k_block_table, b->v_block_table, b->cow_private, rows, rows_off);
    sx_status s = check_launch("cow_kernel");
    if (s != SX_OK) return s;
  }
  int grid = (max_rows + kScatterWarps - 1) / kScatterWarps;
  scatter_kernel<<<grid, kScatterWarps * 32, 0, st>>>(pk, pv, pool->num_kv_heads, b->num_reqs, b->max_pages_per_req,
                                                     b->k_block_table, b->v_block_table,
                                                     reinterpret_cast<const uint4 *>(k_fresh),
                                                     reinterpret_cast<const uint4 *>(v_fresh), rows, rows_off);
  return check_launch("scatter_kernel");
}

}  // namespace sx
