// sx_colsum.cu -- stage (b), second sweep: column sums of the Sparse-Q attention matrix,
//   s_j = sum_{i in I_nr} A_sq[i, j],  A_sq = softmax(Q_sq K^T / sqrt(d) + M_causal[I_nr, :])
// (Eq. (1)-(2)), per KV head; the head sum of PAPER.md:225 is finished in
// fixed order by the select kernel.
//
// K-stationary tcgen05 design: a CTA owns one tile of 128 keys of one (request, KV head) and keeps
// it in shared memory as the A operand (M = keys); it streams every GQA-packed tile of Sparse-Q
// queries that can see it as the B operand (N = (query, head) pairs), D = K Q^T lands in TMEM
// with lane = key. Each consumer thread owns one key: p = exp2(s*c - lse_i) summed over its TMEM
// row -> the column sum needs no cross-thread reduction and no atomics (deterministic).
// The row normaliser lse_i comes from the first sweep (attn_kernel<false>) or from the caller.
#include <math.h>

#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

constexpr int kCsThreads = 192;
constexpr int kCsTileBytes = kTile * kHeadDim * 2;
constexpr int kCsHalf = kCsTileBytes / 2;
constexpr int kCsStages = 3;
constexpr int kCsOffK = 0;
constexpr int kCsOffQ = kCsOffK + kCsTileBytes;
constexpr int kCsOffCol = kCsOffQ + kCsStages * kCsTileBytes;  // [2][128] float lse2 + [2][128] int pos
constexpr int kCsOffBar = kCsOffCol + 2 * 128 * 8;
constexpr int kCsSmemBytes = kCsOffBar + 256 + 1024;

struct ColsumParams {
  const int32_t *seq_len, *tok_off, *new_off, *new_idx, *k_table;
  const float *lse;  // natural log; [total_new][Hq], or [total_tokens][Hq] when lse_by_token
  int lse_by_token;
  float *partial;    // [Hkv][total_tokens]
  int num_reqs, max_pages, num_q_heads, num_kv_heads, group, rows_per_tile, total_tokens;
  float scale_log2;
};

struct CsBars {
  uint64_t k_full;
  uint64_t q_full[kCsStages], q_empty[kCsStages];
  uint64_t d_full[2], d_empty[2];
  uint32_t tmem_base;
};

__global__ void __launch_bounds__(kCsThreads, 1)
colsum_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
              const ColsumParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  CsBars *bars = reinterpret_cast<CsBars *>(smem + kCsOffBar);
  float *col_lse = reinterpret_cast<float *>(smem + kCsOffCol);       // [2][128]
  int *col_pos = reinterpret_cast<int *>(smem + kCsOffCol + 2 * 128 * 4);  // [2][128]

  // ---- (request, key tile, KV head); early key tiles (seen by the most queries) first
  const int g = p.group, rpt = p.rows_per_tile;
  int req = 0, base = 0, ktiles = 0;
  for (; req < p.num_reqs; ++req) {
    ktiles = (p.seq_len[req] + kTile - 1) / kTile;
    if ((int)blockIdx.x < base + ktiles * p.num_kv_heads) break;
    base += ktiles * p.num_kv_heads;
  }
  if (req >= p.num_reqs) return;
  const int local = blockIdx.x - base;
  const int kvh = local % p.num_kv_heads;
  const int kt = local / p.num_kv_heads;
  const int T = p.seq_len[req];
  const int j0 = kt * kTile;
  const int n_pages = (T + kPage - 1) / kPage;
  const int nq0 = p.new_off[req], nn = p.new_off[req + 1] - nq0;
  // first Sparse-Q query that can see key j0: lower_bound(new_idx, j0)
  int lo = 0, hi = nn;
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (p.new_idx[nq0 + mid] < j0) lo = mid + 1; else hi = mid;
  }
  const int qt0 = lo / rpt;                          // first query tile with a visible query
  const int n_qt = (nn + rpt - 1) / rpt;
  const int n_it = (lo < nn) ? n_qt - qt0 : 0;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_q);
    tma_prefetch_desc(&tm_k);
    mbar_init(&bars->k_full, 1);
    for (int i = 0; i < kCsStages; ++i) {
      mbar_init(&bars->q_full[i], 1);
      mbar_init(&bars->q_empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bars->d_full[i], 1);
      mbar_init(&bars->d_empty[i], 128);
    }
    fence_mbar_init();
  }
  if (warp == 1) {
    tmem_alloc(&bars->tmem_base, 256);
    tmem_relinquish();
  }
  // rows of the Q stages that the TMA box never writes (128 - rpt*g pad columns) must be finite
  if (rpt * g < kTile) {
    const int pad = kTile - rpt * g;
    for (int i = threadIdx.x; i < kCsStages * 2 * pad * 8; i += kCsThreads) {
      int c16 = i & 7, r = (i >> 3) % pad, hs = (i >> 3) / pad;  // hs = stage*2 + half
      *reinterpret_cast<uint4 *>(smem + kCsOffQ + hs * kCsHalf + (rpt * g + r) * 128 + c16 * 16) =
          make_uint4(0, 0, 0, 0);
    }
    fence_proxy_async_smem();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;

  if (warp == 0) {
    // ================================================================ TMA producer
    if (n_it > 0) {
      const int pg_in_tile = lane >> 1, half = lane & 1;
      if (lane == 0) mbar_expect_tx(&bars->k_full, kCsTileBytes);
      __syncwarp();
      if (lane < 16) {
        int lp = kt * 8 + pg_in_tile;
        if (lp > n_pages - 1) lp = n_pages - 1;
        const int blk = p.k_table[(size_t)req * p.max_pages + lp];
        tma_load_2d(smem + kCsOffK + half * kCsHalf + pg_in_tile * 2048, &tm_k, &bars->k_full, half * 64,
                    (blk * p.num_kv_heads + kvh) * kPage);
      }
      for (int it = 0; it < n_it; ++it) {
        const int s = it % kCsStages, u = it / kCsStages;
        mbar_wait(&bars->q_empty[s], (u & 1) ^ 1);
        if (lane == 0) {
          mbar_expect_tx(&bars->q_full[s], (uint32_t)(2 * rpt * g * 128));
          const int r0 = nq0 + (qt0 + it) * rpt;
          tma_load_3d(smem + kCsOffQ + s * kCsTileBytes, &tm_q, &bars->q_full[s], 0, kvh * g, r0);
          tma_load_3d(smem + kCsOffQ + s * kCsTileBytes + kCsHalf, &tm_q, &bars->q_full[s], 64, kvh * g, r0);
        }
        __syncwarp();
      }
    }
  } else if (warp == 1) {
    // ================================================================ MMA issuer: D[b] = K_tile * Q_tile^T
    if (n_it > 0) {
      constexpr uint32_t idesc = umma_idesc_bf16(128, 128, 0, 0);
      const uint32_t k_addr = smem_u32(smem + kCsOffK);
      mbar_wait(&bars->k_full, 0);
      for (int it = 0; it < n_it; ++it) {
        const int s = it % kCsStages, b = it & 1;
        mbar_wait(&bars->q_full[s], (it / kCsStages) & 1);
        if (it >= 2) mbar_wait(&bars->d_empty[b], ((it >> 1) + 1) & 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t q_addr = smem_u32(smem + kCsOffQ + s * kCsTileBytes);
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const uint32_t o = (kk >> 2) * kCsHalf + (kk & 3) * 32;
            umma_ss(tmem + b * 128, umma_smem_desc(k_addr + o, 16, 1024), umma_smem_desc(q_addr + o, 16, 1024),
                    idesc, kk > 0);
          }
          umma_commit(&bars->d_full[b]);
          umma_commit(&bars->q_empty[s]);
        }
        __syncwarp();
      }
    }
  } else {
    // ================================================================ consumers: thread = one key
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;   // key j0 + row = TMEM lane
    const int ct = threadIdx.x - 64;       // 0..127: column staged by this thread
    const int j = j0 + row;
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    const int cn = ct / g, ch = ct - cn * g;  // column ct = (query cn of the tile, head ch of the group)
    float acc = 0.f;

    auto load_col = [&](int it, float &lse2, int &qpos) {
      const int n = (qt0 + it) * rpt + cn;  // query index within the request
      if (cn < rpt && n < nn) {
        qpos = p.new_idx[nq0 + n];
        const size_t lrow = p.lse_by_token ? (size_t)(p.tok_off[req] + qpos) : (size_t)(nq0 + n);
        lse2 = p.lse[lrow * p.num_q_heads + kvh * g + ch] * (float)kLog2e;
      } else {
        lse2 = INFINITY;  // pad column: exp2(-inf) = 0
        qpos = -1;
      }
    };
    float nx_lse = 0.f;
    int nx_pos = 0;
    if (n_it > 0) load_col(0, nx_lse, nx_pos);
    for (int it = 0; it < n_it; ++it) {
      const int b = it & 1;
      col_lse[b * 128 + ct] = nx_lse;
      col_pos[b * 128 + ct] = nx_pos;
      if (it + 1 < n_it) load_col(it + 1, nx_lse, nx_pos);
      named_bar_sync(1, 128);
      // queries are sorted by position: columns below `first` cannot see key j
      const bool need_mask = col_pos[b * 128] < j0 + kTile - 1;  // some column may be masked for some key
      mbar_wait(&bars->d_full[b], (it >> 1) & 1);
      tc_fence_after();
      const float4 *lse4 = reinterpret_cast<const float4 *>(col_lse + b * 128);
      const int4 *pos4 = reinterpret_cast<const int4 *>(col_pos + b * 128);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t d[32];
        tmem_ld32(tmem + lane_addr + b * 128 + c * 32, d);
        tmem_wait_ld();
        if (!need_mask) {
#pragma unroll
          for (int i = 0; i < 32; i += 4) {
            const float4 ls = lse4[(c * 32 + i) >> 2];
            acc += ex2_approx(fmaf(__uint_as_float(d[i + 0]), p.scale_log2, -ls.x));
            acc += ex2_approx(fmaf(__uint_as_float(d[i + 1]), p.scale_log2, -ls.y));
            acc += ex2_approx(fmaf(__uint_as_float(d[i + 2]), p.scale_log2, -ls.z));
            acc += ex2_approx(fmaf(__uint_as_float(d[i + 3]), p.scale_log2, -ls.w));
          }
        } else {
#pragma unroll
          for (int i = 0; i < 32; i += 4) {
            const float4 ls = lse4[(c * 32 + i) >> 2];
            const int4 qp = pos4[(c * 32 + i) >> 2];
            float e0 = ex2_approx(fmaf(__uint_as_float(d[i + 0]), p.scale_log2, -ls.x));
            float e1 = ex2_approx(fmaf(__uint_as_float(d[i + 1]), p.scale_log2, -ls.y));
            float e2 = ex2_approx(fmaf(__uint_as_float(d[i + 2]), p.scale_log2, -ls.z));
            float e3 = ex2_approx(fmaf(__uint_as_float(d[i + 3]), p.scale_log2, -ls.w));
            acc += (qp.x >= j) ? e0 : 0.f;
            acc += (qp.y >= j) ? e1 : 0.f;
            acc += (qp.z >= j) ? e2 : 0.f;
            acc += (qp.w >= j) ? e3 : 0.f;
          }
        }
      }
      tc_fence_before();
      mbar_arrive(&bars->d_empty[b]);
    }
    if (j < T) p.partial[(size_t)kvh * p.total_tokens + p.tok_off[req] + j] = acc;
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 256);
}

sx_status launch_colsum(const sx_pool *pool, const sx_batch *b, const void *q_new, const float *lse_new,
                        int lse_by_token, float *partial, cudaStream_t st) {
  const int g = pool->num_q_heads / pool->num_kv_heads;
  const int rpt = kTile / g;
  CUtensorMap tm_q, tm_k;
  sx_status s = make_tmap_q(&tm_q, q_new, b->total_new, pool->num_q_heads, g, rpt);
  if (s != SX_OK) return s;
  s = make_tmap_pool(&tm_k, pool->k, pool->num_blocks, pool->num_kv_heads);
  if (s != SX_OK) return s;
  ColsumParams p;
  p.seq_len = b->seq_len;
  p.tok_off = b->tok_off;
  p.new_off = b->new_off;
  p.new_idx = b->new_idx;
  p.k_table = b->k_block_table;
  p.lse = lse_new;
  p.lse_by_token = lse_by_token;
  p.partial = partial;
  p.num_reqs = b->num_reqs;
  p.max_pages = b->max_pages_per_req;
  p.num_q_heads = pool->num_q_heads;
  p.num_kv_heads = pool->num_kv_heads;
  p.group = g;
  p.rows_per_tile = rpt;
  p.total_tokens = b->total_tokens;
  p.scale_log2 = (float)(kLog2e / sqrt((double)kHeadDim));
  const int grid = (b->total_tokens / kTile + b->num_reqs) * pool->num_kv_heads;
  cudaError_t e = cudaFuncSetAttribute(colsum_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kCsSmemBytes);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "colsum smem attr: %s", cudaGetErrorString(e));
  colsum_kernel<<<grid, kCsThreads, kCsSmemBytes, st>>>(tm_q, tm_k, p);
  return check_launch("colsum_kernel");
}

}  // namespace sx
