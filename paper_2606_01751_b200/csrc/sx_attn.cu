// sx_attn.cu -- stage (c): causal attention of the sparse query set R over the full paged K/V
//   O[R] = SparseAttn(Q[R], K_cur[1:T], V_cur[1:T], M_causal)          Alg. 1 l.546-548 (sparse)
//   full causal attention on all positions                                Alg. 1 l.507-511 (layers <= l*)
// and, with kWithPV = false, the first sweep of stage (b): the softmax normaliser (log-sum-exp) of
// the Sparse-Q rows of Eq. (1).
//
// tcgen05 design (one CTA per (request, KV head, tile of R rows)):
//   * GQA packing: the M = 128 rows of a tile are (row of R, query head of the KV group) pairs,
//     rows_per_tile = 128 / g consecutive rows of R times g heads -> one K/V tile feeds g heads.
//     Q arrives by one 3-D TMA box per 64-column half, already in the 128-B-swizzled K-major layout.
//   * K/V tiles of 128 keys = 8 pages: the producer warp reads 8 block-table entries and issues
//     16 TMA boxes (64 columns x 16 rows, 128-B swizzle) per tile; the 8 boxes of a half stack into
//     a 128-row operand. K is the K-major B operand of S = Q K^T, V the MN-major B operand of O += P V.
//   * warp 0 = TMA producer, warp 1 = MMA issuer (one elected lane), warps 2-5 = softmax: thread =
//     one row of S in TMEM (tcgen05.ld), fp32 online softmax in the exp2 domain with lazy rescale
//     (O in TMEM is rescaled only when the row maximum grew by more than 2^8), P rounded to bf16
//     into swizzled shared memory as the A operand of the PV MMA. S is double-buffered in TMEM so
//     QK^T of tile t+1 overlaps the softmax of tile t.
//   * causality with a sparse, sorted row list: key tiles run up to the largest position of the
//     tile; each row masks keys beyond its own position.
#include <math.h>

#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

constexpr int kAttnThreads = 192;
constexpr int kTileBytes = kTile * kHeadDim * 2;  // 32 KB: two 16-KB halves [half][row][64 bf16]
constexpr int kHalfBytes = kTileBytes / 2;

struct AttnParams {
  const int32_t *rows;      // [total_rows] positions, or nullptr (row n of request r = position n - rows_off[r])
  const int32_t *rows_off;  // [num_reqs+1]
  const int32_t *seq_len;
  const int32_t *k_table;
  const int32_t *v_table;
  __nv_bfloat16 *out;  // [total_rows][Hq][128]
  float *lse;          // [total_rows][Hq] or nullptr
  int num_reqs, max_pages, num_q_heads, num_kv_heads, group, rows_per_tile;
  float scale_log2;  // log2(e) / sqrt(128)
  float scale;       // 1 / sqrt(128)
};

template <bool kWithPV>
struct AttnCfg {
  static constexpr int kStagesK = kWithPV ? 2 : 4;
  static constexpr int kStagesV = kWithPV ? 2 : 0;
  static constexpr int kOffQ = 0;
  static constexpr int kOffK = kOffQ + kTileBytes;
  static constexpr int kOffV = kOffK + kStagesK * kTileBytes;
  static constexpr int kOffP = kOffV + kStagesV * kTileBytes;
  static constexpr int kOffBar = kOffP + (kWithPV ? kTileBytes : 0);
  static constexpr int kSmemBytes = kOffBar + 512 + 1024;  // + alignment slack
  static constexpr uint32_t kTmemCols = kWithPV ? 512 : 256;
};

struct AttnBars {
  uint64_t q_full;
  uint64_t k_full[4], k_empty[4];
  uint64_t v_full[2], v_empty[2];
  uint64_t s_full[2], s_empty[2];
  uint64_t p_full, pv_done;
  uint32_t tmem_base;
};

template <bool kWithPV>
__global__ void __launch_bounds__(kAttnThreads, 1)
attn_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
            const __grid_constant__ CUtensorMap tm_v, const AttnParams p) {
  using Cfg = AttnCfg<kWithPV>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  AttnBars *bars = reinterpret_cast<AttnBars *>(smem + Cfg::kOffBar);

  // ---- which (request, KV head, row tile) is this CTA; heavy (late) tiles of a request first
  const int g = p.group, rpt = p.rows_per_tile;
  int req = 0, base = 0, tiles = 0, n_r = 0;
  for (; req < p.num_reqs; ++req) {
    n_r = p.rows_off[req + 1] - p.rows_off[req];
    tiles = (n_r + rpt - 1) / rpt;
    if ((int)blockIdx.x < base + tiles * p.num_kv_heads) break;
    base += tiles * p.num_kv_heads;
  }
  if (req >= p.num_reqs) return;
  const int local = blockIdx.x - base;
  const int kvh = local % p.num_kv_heads;
  const int tile = tiles - 1 - local / p.num_kv_heads;
  const int row_base = p.rows_off[req] + tile * rpt;     // first row (batch-wide index) of this tile
  const int nrows = min(rpt, n_r - tile * rpt);          // valid rows of R in this tile
  const int T = p.seq_len[req];
  const int pos_max = p.rows ? p.rows[row_base + nrows - 1] : tile * rpt + nrows - 1;
  const int n_tiles = pos_max / kTile + 1;
  const int n_pages = (T + kPage - 1) / kPage;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_q);
    tma_prefetch_desc(&tm_k);
    if (kWithPV) tma_prefetch_desc(&tm_v);
    mbar_init(&bars->q_full, 1);
    for (int i = 0; i < 4; ++i) {
      mbar_init(&bars->k_full[i], 1);
      mbar_init(&bars->k_empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bars->v_full[i], 1);
      mbar_init(&bars->v_empty[i], 1);
      mbar_init(&bars->s_full[i], 1);
      mbar_init(&bars->s_empty[i], 128);
    }
    mbar_init(&bars->p_full, 128);
    mbar_init(&bars->pv_done, 1);
    fence_mbar_init();
  }
  if (warp == 1) {
    tmem_alloc(&bars->tmem_base, Cfg::kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;
  const uint32_t tmem_o = tmem + 256;

  if (warp == 0) {
    // ================================================================ TMA producer
    if (lane == 0) {
      mbar_expect_tx(&bars->q_full, (uint32_t)(2 * rpt * g * 128));
      tma_load_3d(smem + Cfg::kOffQ, &tm_q, &bars->q_full, 0, kvh * g, row_base);
      tma_load_3d(smem + Cfg::kOffQ + kHalfBytes, &tm_q, &bars->q_full, 64, kvh * g, row_base);
    }
    const int pg_in_tile = lane >> 1, half = lane & 1;
    for (int t = 0; t < n_tiles; ++t) {
      int lp = t * 8 + pg_in_tile;
      if (lp > n_pages - 1) lp = n_pages - 1;  // pages past the sequence: any valid page (keys are masked)
      {
        const int s = t % Cfg::kStagesK, u = t / Cfg::kStagesK;
        mbar_wait(&bars->k_empty[s], (u & 1) ^ 1);
        if (lane == 0) mbar_expect_tx(&bars->k_full[s], kTileBytes);
        __syncwarp();
        if (lane < 16) {
          const int blk = p.k_table[(size_t)req * p.max_pages + lp];
          tma_load_2d(smem + Cfg::kOffK + s * kTileBytes + half * kHalfBytes + pg_in_tile * 2048, &tm_k,
                      &bars->k_full[s], half * 64, (blk * p.num_kv_heads + kvh) * kPage);
        }
      }
      if (kWithPV) {
        const int s = t % 2, u = t / 2;
        mbar_wait(&bars->v_empty[s], (u & 1) ^ 1);
        if (lane == 0) mbar_expect_tx(&bars->v_full[s], kTileBytes);
        __syncwarp();
        if (lane < 16) {
          const int blk = p.v_table[(size_t)req * p.max_pages + lp];
          tma_load_2d(smem + Cfg::kOffV + s * kTileBytes + half * kHalfBytes + pg_in_tile * 2048, &tm_v,
                      &bars->v_full[s], half * 64, (blk * p.num_kv_heads + kvh) * kPage);
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================ MMA issuer
    constexpr uint32_t idesc_qk = umma_idesc_bf16(128, 128, 0, 0);
    constexpr uint32_t idesc_pv = umma_idesc_bf16(128, 128, 0, 1);
    const uint32_t q_addr = smem_u32(smem + Cfg::kOffQ);
    const uint32_t p_addr = smem_u32(smem + Cfg::kOffP);
    mbar_wait(&bars->q_full, 0);
    auto issue_qk = [&](int t) {
      const int s = t % Cfg::kStagesK;
      mbar_wait(&bars->k_full[s], (t / Cfg::kStagesK) & 1);
      if (t >= 2) mbar_wait(&bars->s_empty[t & 1], ((t >> 1) + 1) & 1);
      tc_fence_after();
      if (lane == 0) {
        const uint32_t k_addr = smem_u32(smem + Cfg::kOffK + s * kTileBytes);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t o = (kk >> 2) * kHalfBytes + (kk & 3) * 32;
          umma_ss(tmem + (t & 1) * 128, umma_smem_desc(q_addr + o, 16, 1024), umma_smem_desc(k_addr + o, 16, 1024),
                  idesc_qk, kk > 0);
        }
        umma_commit(&bars->s_full[t & 1]);
        umma_commit(&bars->k_empty[s]);
      }
      __syncwarp();
    };
    issue_qk(0);
    for (int t = 0; t < n_tiles; ++t) {
      if (t + 1 < n_tiles) issue_qk(t + 1);
      if (kWithPV) {
        const int s = t & 1;
        mbar_wait(&bars->v_full[s], (t >> 1) & 1);
        mbar_wait(&bars->p_full, t & 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t v_addr = smem_u32(smem + Cfg::kOffV + s * kTileBytes);
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {  // 16 keys per MMA
            const uint32_t po = (kk >> 2) * kHalfBytes + (kk & 3) * 32;
            umma_ss(tmem_o, umma_smem_desc(p_addr + po, 16, 1024),
                    umma_smem_desc(v_addr + kk * 2048, kHalfBytes, 1024), idesc_pv, (t > 0 || kk > 0));
          }
          umma_commit(&bars->pv_done);
          umma_commit(&bars->v_empty[s]);
        }
        __syncwarp();
      }
    }
  } else {
    // ================================================================ softmax / epilogue (128 threads)
    const int quarter = warp & 3;              // TMEM lane quarter this warp may access
    const int row = quarter * 32 + lane;       // row of the tile = TMEM lane
    const int n_local = row / g, hh = row - n_local * g;
    const bool valid = n_local < nrows;
    const int pos = valid ? (p.rows ? p.rows[row_base + n_local] : tile * rpt + n_local) : 0;
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    float m_used = -INFINITY, l = 0.f;

    for (int t = 0; t < n_tiles; ++t) {
      const int b = t & 1;
      mbar_wait(&bars->s_full[b], (t >> 1) & 1);
      tc_fence_after();
      uint32_t sr[4][32];
#pragma unroll
      for (int c = 0; c < 4; ++c) tmem_ld32(tmem + lane_addr + b * 128 + c * 32, sr[c]);
      tmem_wait_ld();
      tc_fence_before();
      mbar_arrive(&bars->s_empty[b]);

      const int nvalid = pos - t * kTile + 1;  // keys [0, nvalid) of this tile are visible to this row
      if (nvalid < kTile) {
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (c * 32 + i >= nvalid) sr[c][i] = 0xFF800000u;  // -inf
      }
      float tmax = -INFINITY;
#pragma unroll
      for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int i = 0; i < 32; ++i) tmax = fmaxf(tmax, __uint_as_float(sr[c][i]));
      const float m_new = fmaxf(m_used, tmax);
      const bool upd = (m_new - m_used) * p.scale_log2 > 8.0f;  // lazy rescale threshold: 2^8
      float alpha = 1.f;
      if (upd) {
        alpha = ex2_approx((m_used - m_new) * p.scale_log2);
        m_used = m_new;
      }
      const float neg_m = -m_used * p.scale_log2;
      float rsum = 0.f;
#pragma unroll
      for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          float e = ex2_approx(fmaf(__uint_as_float(sr[c][i]), p.scale_log2, neg_m));
          rsum += e;
          sr[c][i] = __float_as_uint(e);
        }
      l = l * alpha + rsum;

      if (kWithPV) {
        if (t > 0) mbar_wait(&bars->pv_done, (t - 1) & 1);  // P buffer free, O accumulator quiescent
        if (t > 0 && __any_sync(0xffffffffu, upd)) {
          tc_fence_after();
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            uint32_t o[32];
            tmem_ld32(tmem_o + lane_addr + c * 32, o);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st32(tmem_o + lane_addr + c * 32, o);
          }
          tmem_wait_st();
        }
        // V rows of keys beyond the sequence may hold anything (even NaN patterns): zero them
        if (t == n_tiles - 1 && (t + 1) * kTile > T) {
          mbar_wait(&bars->v_full[t & 1], (t >> 1) & 1);
          if (t * kTile + row >= T) {
            uint4 z = make_uint4(0, 0, 0, 0);
            uint8_t *v0 = smem + Cfg::kOffV + (t & 1) * kTileBytes + row * 128;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              *reinterpret_cast<uint4 *>(v0 + i * 16) = z;
              *reinterpret_cast<uint4 *>(v0 + kHalfBytes + i * 16) = z;
            }
          }
        }
        // P (bf16) -> swizzled K-major A operand: chunk j = keys [8j, 8j+8) of this row
        uint8_t *prow = smem + Cfg::kOffP + row * 128;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int c = j >> 2, i0 = (j & 3) * 8;
          uint4 v;
          v.x = pack_bf16x2(__uint_as_float(sr[c][i0 + 0]), __uint_as_float(sr[c][i0 + 1]));
          v.y = pack_bf16x2(__uint_as_float(sr[c][i0 + 2]), __uint_as_float(sr[c][i0 + 3]));
          v.z = pack_bf16x2(__uint_as_float(sr[c][i0 + 4]), __uint_as_float(sr[c][i0 + 5]));
          v.w = pack_bf16x2(__uint_as_float(sr[c][i0 + 6]), __uint_as_float(sr[c][i0 + 7]));
          *reinterpret_cast<uint4 *>(prow + (j >> 3) * kHalfBytes + (((j & 7) ^ (row & 7)) << 4)) = v;
        }
        fence_proxy_async_smem();
        tc_fence_before();
        mbar_arrive(&bars->p_full);
      }
    }

    // ---- epilogue
    const size_t out_row = (size_t)(row_base + n_local) * p.num_q_heads + kvh * g + hh;
    if (kWithPV) {
      mbar_wait(&bars->pv_done, (n_tiles - 1) & 1);
      tc_fence_after();
      const float inv = 1.f / l;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        uint32_t o[32];
        tmem_ld32(tmem_o + lane_addr + c * 32, o);
        tmem_wait_ld();
        if (valid) {
          uint4 *dst = reinterpret_cast<uint4 *>(p.out + out_row * kHeadDim + c * 32);
#pragma unroll
          for (int v4 = 0; v4 < 4; ++v4) {
            uint4 v;
            v.x = pack_bf16x2(__uint_as_float(o[v4 * 8 + 0]) * inv, __uint_as_float(o[v4 * 8 + 1]) * inv);
            v.y = pack_bf16x2(__uint_as_float(o[v4 * 8 + 2]) * inv, __uint_as_float(o[v4 * 8 + 3]) * inv);
            v.z = pack_bf16x2(__uint_as_float(o[v4 * 8 + 4]) * inv, __uint_as_float(o[v4 * 8 + 5]) * inv);
            v.w = pack_bf16x2(__uint_as_float(o[v4 * 8 + 6]) * inv, __uint_as_float(o[v4 * 8 + 7]) * inv);
            dst[v4] = v;
          }
        }
      }
    }
    if (p.lse && valid) p.lse[out_row] = m_used * p.scale + logf(l);
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, Cfg::kTmemCols);
}

sx_status launch_attn(const sx_pool *pool, const sx_batch *b, bool with_pv, const void *q, const int32_t *rows,
                      const int32_t *rows_off, int32_t total_rows, void *out, float *lse, cudaStream_t st) {
  const int g = pool->num_q_heads / pool->num_kv_heads;
  const int rpt = kTile / g;
  CUtensorMap tm_q, tm_k, tm_v;
  sx_status s = make_tmap_q(&tm_q, q, total_rows, pool->num_q_heads, g, rpt);
  if (s != SX_OK) return s;
  s = make_tmap_pool(&tm_k, pool->k, pool->num_blocks, pool->num_kv_heads);
  if (s != SX_OK) return s;
  s = make_tmap_pool(&tm_v, pool->v, pool->num_blocks, pool->num_kv_heads);
  if (s != SX_OK) return s;
  AttnParams p;
  p.rows = rows;
  p.rows_off = rows_off;
  p.seq_len = b->seq_len;
  p.k_table = b->k_block_table;
  p.v_table = b->v_block_table;
  p.out = reinterpret_cast<__nv_bfloat16 *>(out);
  p.lse = lse;
  p.num_reqs = b->num_reqs;
  p.max_pages = b->max_pages_per_req;
  p.num_q_heads = pool->num_q_heads;
  p.num_kv_heads = pool->num_kv_heads;
  p.group = g;
  p.rows_per_tile = rpt;
  p.scale = (float)(1.0 / sqrt((double)kHeadDim));
  p.scale_log2 = (float)(kLog2e / sqrt((double)kHeadDim));
  const int grid = (total_rows / rpt + b->num_reqs) * pool->num_kv_heads;
  cudaError_t e;
  if (with_pv) {
    e = cudaFuncSetAttribute(attn_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnCfg<true>::kSmemBytes);
    if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "attn smem attr: %s", cudaGetErrorString(e));
    attn_kernel<true><<<grid, kAttnThreads, AttnCfg<true>::kSmemBytes, st>>>(tm_q, tm_k, tm_v, p);
  } else {
    e = cudaFuncSetAttribute(attn_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttnCfg<false>::kSmemBytes);
    if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "lse smem attr: %s", cudaGetErrorString(e));
    attn_kernel<false><<<grid, kAttnThreads, AttnCfg<false>::kSmemBytes, st>>>(tm_q, tm_k, tm_v, p);
  }
  return check_launch(with_pv ? "attn_kernel<pv>" : "attn_kernel<lse>");
}

}  // namespace sx
