// sx_scatter.cu -- stage (d): write the fresh K,V rows of the computed positions into their paged
// slots (Alg. 1 l.509-510 / 544-545 "write fresh K,V into the current request cache"; slot mapping
// PAPER.md:333), with copy-on-write of still-shared pages (reading A14).
//
// HBM-bound bit copy: 8*Hkv*128 bytes per row. ONE launch: a warp per listed row, 16-byte vector loads/stores
// (the 256 B of one (row, head) are written by 16 consecutive lanes), all loads of a row in flight before the
// first store; the request of a row is found by binary search in rows_off. Under copy-on-write the unit of work
// is the touched PAGE (the warp of the page's first listed row copies the aliased page, flips the table entry
// and then writes every listed row of that page itself: the copy and the row writes are ordered inside one
// warp, no atomics, no second launch). The kernel is launched with programmatic dependent launch allowed.
#include "sx_internal.h"
#include "sx_ptx.cuh"
#include "sx_rotate.cuh"

namespace sx {

// request r with off[r] <= n < off[r+1] (off ascending, off[0] = 0; empty requests are skipped)
__device__ __forceinline__ int find_req(const int32_t *__restrict__ off, int num_reqs, int n) {
  int lo = 0, hi = num_reqs - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (ld_dep(off + mid) <= n) lo = mid; else hi = mid - 1;
  }
  return lo;
}

constexpr int kScatterWarps = 8;
constexpr int kScatterMaxChunks = 4;  // 16-byte chunks per lane and tensor held in registers: Hkv <= 8

// one row: K and V, every 16-byte chunk of the row loaded before the first store
__device__ __forceinline__ void scatter_row(uint4 *pool_k, uint4 *pool_v, int num_kv_heads, int kb, int vb, int o,
                                            const uint4 *__restrict__ ks, const uint4 *__restrict__ vs, int lane) {
  const int row_chunks = num_kv_heads * 16;  // 16-byte chunks of one fresh row
  if (row_chunks <= 32 * kScatterMaxChunks) {
    uint4 a[kScatterMaxChunks], b[kScatterMaxChunks];
#pragma unroll
    for (int i = 0; i < kScatterMaxChunks; ++i) {
      const int c = lane + 32 * i;
      if (c < row_chunks) {
        a[i] = __ldg(ks + c);  // (read-only path: the fresh rows are inputs of the call, never written by this library)
        b[i] = __ldg(vs + c);
      }
    }
#pragma unroll
    for (int i = 0; i < kScatterMaxChunks; ++i) {
      const int c = lane + 32 * i;
      if (c < row_chunks) {
        const int h = c >> 4, cc = c & 15;
        pool_k[(((size_t)kb * num_kv_heads + h) * kPage + o) * 16 + cc] = a[i];
        pool_v[(((size_t)vb * num_kv_heads + h) * kPage + o) * 16 + cc] = b[i];
      }
    }
  } else {
    for (int c = lane; c < row_chunks; c += 32) {
      const int h = c >> 4, cc = c & 15;
      const uint4 a = __ldg(ks + c), b = __ldg(vs + c);
      pool_k[(((size_t)kb * num_kv_heads + h) * kPage + o) * 16 + cc] = a;
      pool_v[(((size_t)vb * num_kv_heads + h) * kPage + o) * 16 + cc] = b;
    }
  }
}

// zero-copy mode (include/sparsex.h): what the copy-on-write of a K page needs to rotate a still-shared source page
struct ScatterZc {
  const sx_segment *segs;
  const int32_t *src_blocks;
  int num_segments;
  int style;  // -1: not in zero-copy mode
  double theta;
};

// bit copy of one page by one warp: n (a multiple of 256) 16-byte chunks, eight loads in flight per lane (source and
// destination never overlap: a shared source page / a reserved private page)
__device__ __forceinline__ void copy_page(const uint4 *__restrict__ s, uint4 *__restrict__ d, int n, int lane) {
  for (int i = lane; i < n; i += 256) {
    uint4 t[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) t[k] = s[i + 32 * k];
#pragma unroll
    for (int k = 0; k < 8; ++k) d[i + 32 * k] = t[k];
  }
}

// copy-on-write of one K page in zero-copy mode: K[priv] = R_delta K[src], one warp (same arithmetic as realign_kernel)
__device__ __forceinline__ void cow_rotate_page(const uint4 *__restrict__ s, uint4 *__restrict__ d, int num_kv_heads,
                                                int style, double theta, int delta, int lane) {
  if (style == 0) {
    // items (head, row, c < 8): chunks c and c + 8 of the row; i = lane + 32 k keeps c = lane & 7
    const int c = lane & 7;
    // the 64 (cos, sin) pairs of the segment: two per lane in fp64, handed round by shuffles (lane needs 8c .. 8c+7)
    const float2 t0 = rope_cos_sin(theta, delta, 2 * lane), t1 = rope_cos_sin(theta, delta, 2 * lane + 1);
    float2 cs[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      const int src = (8 * c + e) >> 1;
      const float2 a = make_float2(__shfl_sync(0xffffffffu, t0.x, src), __shfl_sync(0xffffffffu, t0.y, src));
      const float2 b = make_float2(__shfl_sync(0xffffffffu, t1.x, src), __shfl_sync(0xffffffffu, t1.y, src));
      cs[e] = (e & 1) ? b : a;
    }
    const int items = num_kv_heads * kPage * 8;  // a multiple of 128: four items per lane and step, loads first
    for (int i = lane; i < items; i += 128) {
      uint4 a[4], b[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int o = ((i + 32 * k) >> 3) * 16 + c;
        a[k] = s[o];
        b[k] = s[o + 8];
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int o = ((i + 32 * k) >> 3) * 16 + c;
        rotate_split(a[k], b[k], cs);
        d[o] = a[k];
        d[o + 8] = b[k];
      }
    }
  } else {
    const int c16 = lane & 15;
    const float2 t0 = rope_cos_sin(theta, delta, 2 * lane), t1 = rope_cos_sin(theta, delta, 2 * lane + 1);
    float2 cs[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int src = (4 * c16 + e) >> 1;
      const float2 a = make_float2(__shfl_sync(0xffffffffu, t0.x, src), __shfl_sync(0xffffffffu, t0.y, src));
      const float2 b = make_float2(__shfl_sync(0xffffffffu, t1.x, src), __shfl_sync(0xffffffffu, t1.y, src));
      cs[e] = (e & 1) ? b : a;
    }
    const int items = num_kv_heads * kPage * 16;  // a multiple of 256
    for (int i = lane; i < items; i += 256) {
      uint4 a[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) a[k] = s[i + 32 * k];
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        rotate_inter(a[k], cs);
        d[i + 32 * k] = a[k];
      }
    }
  }
}

template <bool kCow, bool kZc = false>
__global__ void __launch_bounds__(kScatterWarps * 32)
scatter_kernel(uint4 *pool_k, uint4 *pool_v, int num_kv_heads, int num_reqs, int max_pages, int32_t *k_table,
               int32_t *v_table, const int32_t *__restrict__ cow_private, const uint4 *__restrict__ k_fresh,
               const uint4 *__restrict__ v_fresh, const int32_t *__restrict__ rows,
               const int32_t *__restrict__ rows_off, const ScatterZc zc) {
  griddep_launch();  // the next kernel's prologue may overlap this one
  griddep_wait();    // the row list / the pool may be outputs of the previous kernel
  const int n = blockIdx.x * kScatterWarps + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (n >= ld_dep(rows_off + num_reqs)) return;
  const int req = find_req(rows_off, num_reqs, n);
  const int p = ld_dep(rows + n);
  const int pg = p / kPage;
  const size_t e = (size_t)req * max_pages + pg;
  const int row_chunks = num_kv_heads * 16;
  if (!kCow) {
    scatter_row(pool_k, pool_v, num_kv_heads, k_table[e], v_table[e], p % kPage, k_fresh + (size_t)n * row_chunks,
                v_fresh + (size_t)n * row_chunks, lane);
    return;
  }
  // copy-on-write: the warp of the FIRST listed row of a page owns the page (rows are ascending inside a request)
  if (n > ld_dep(rows_off + req) && ld_dep(rows + n - 1) / kPage == pg) return;
  const int priv = cow_private[e];
  int kb = k_table[e], vb = v_table[e];
  if (priv >= 0) {
    const int page_chunks = num_kv_heads * kPage * 16;
    if (kb != priv) {
      const uint4 *s = pool_k + (size_t)kb * page_chunks;
      uint4 *d = pool_k + (size_t)priv * page_chunks;
      // zero-copy mode: a page that still is the cached source page of its segment holds keys at their OLD positions
      int m = -1;
      if (kZc) {
        m = find_segment(zc.segs, zc.num_segments, req, pg * kPage);
        if (m >= 0 && kb != zc.src_blocks[zc.segs[m].src_off + pg - zc.segs[m].new_pos / kPage]) m = -1;
      }
      if (kZc && m >= 0)
        cow_rotate_page(s, d, num_kv_heads, zc.style, zc.theta, zc.segs[m].new_pos - zc.segs[m].old_pos, lane);
      else
        copy_page(s, d, page_chunks, lane);
    }
    if (vb != priv) {
      copy_page(pool_v + (size_t)vb * page_chunks, pool_v + (size_t)priv * page_chunks, page_chunks, lane);
    }
    __syncwarp();  // orders the page copy before the row writes of other lanes below
    if (lane == 0) {
      if (kb != priv) k_table[e] = priv;
      if (vb != priv && v_table + e != k_table + e) v_table[e] = priv;
    }
    kb = vb = priv;
  }
  const int n_end = ld_dep(rows_off + req + 1);
  for (int m = n; m < n_end; ++m) {
    const int q = ld_dep(rows + m);
    if (q / kPage != pg) break;
    scatter_row(pool_k, pool_v, num_kv_heads, kb, vb, q % kPage, k_fresh + (size_t)m * row_chunks,
                v_fresh + (size_t)m * row_chunks, lane);
  }
}

sx_status launch_scatter(const sx_pool *pool, const sx_batch *b, const void *k_fresh, const void *v_fresh,
                         const int32_t *rows, const int32_t *rows_off, int32_t max_rows, cudaStream_t st) {
  uint4 *pk = reinterpret_cast<uint4 *>(pool->k);
  uint4 *pv = reinterpret_cast<uint4 *>(pool->v);
  const int grid = (max_rows + kScatterWarps - 1) / kScatterWarps;
  const uint4 *kf = reinterpret_cast<const uint4 *>(k_fresh), *vf = reinterpret_cast<const uint4 *>(v_fresh);
  ScatterZc zc;
  zc.segs = b->segments;
  zc.src_blocks = b->src_blocks;
  zc.num_segments = b->num_segments;
  zc.style = (b->zero_copy && b->num_segments > 0) ? b->rope_style : -1;
  zc.theta = b->rope_theta;
  cudaError_t e;
  if (b->cow_private && zc.style >= 0)
    e = launch_pdl(scatter_kernel<true, true>, dim3(grid), dim3(kScatterWarps * 32), 0, st, 1, pk, pv, pool->num_kv_heads,
                   b->num_reqs, b->max_pages_per_req, b->k_block_table, b->v_block_table, b->cow_private, kf, vf, rows,
                   rows_off, zc);
  else if (b->cow_private)
    e = launch_pdl(scatter_kernel<true>, dim3(grid), dim3(kScatterWarps * 32), 0, st, 1, pk, pv, pool->num_kv_heads,
                   b->num_reqs, b->max_pages_per_req, b->k_block_table, b->v_block_table, b->cow_private, kf, vf, rows,
                   rows_off, zc);
  else
    e = launch_pdl(scatter_kernel<false>, dim3(grid), dim3(kScatterWarps * 32), 0, st, 1, pk, pv, pool->num_kv_heads,
                   b->num_reqs, b->max_pages_per_req, b->k_block_table, b->v_block_table, b->cow_private, kf, vf, rows,
                   rows_off, zc);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "scatter launch: %s", cudaGetErrorString(e));
  return check_launch("scatter_kernel");
}

}  // namespace sx
