// sx_lse.cu -- stage (b), first sweep: the softmax normaliser (log-sum-exp) of every Sparse-Q row of Eq. (1),
//   lse_i = log sum_{j <= i} exp(<q_i, k_j> / sqrt(d)),  i in I_nr
// per query head, over the keys of the current pool. The second sweep (sx_colsum.cu) turns it into the column
// sums of Eq. (2).
//
// The sweep has no PV product: per 128 x 128 score tile it needs 128^2 exponentials against 512 tensor-pipe
// cycles, so MUFU.EX2 (16 / clk / SM) is the roof, and what matters is keeping that pipe fed. Shape (the one
// of the column-sum kernel, transposed): a CTA owns ONE GQA-packed tile of 128 (query, head) rows as the A
// operand and streams the 128-key tiles it can see through a 2-slot TMA ring as B; S = Q K^T lands in a
// double-buffered TMEM accumulator (256 columns, so TWO CTAs share an SM); TWO consumer threads share a row,
// each running its own online (max, sum) over 64 of the 128 key columns of every tile -- a log-sum-exp over keys
// splits freely, so the two halves never exchange anything until the end. A fixed fraction of the exponentials
// is evaluated on the FMA pipe (Cody-Waite + cubic). Long single requests are cut into key splits; the partial
// normalisers are merged by coltab_kernel.
#include <math.h>

#include "sx_internal.h"
#include "sx_ptx.cuh"
#include "sx_rotate.cuh"

namespace sx {

constexpr int kLseThreads = 320;  // warps 0-7 consumers, warp 8 TMA producer, warp 9 MMA issuer
constexpr int kLseTileBytes = kTile * kHeadDim * 2;
constexpr int kLseHalf = kLseTileBytes / 2;
constexpr int kLseStages = 2;
constexpr int kLseOffQ = 0;
constexpr int kLseOffK = kLseOffQ + kLseTileBytes;
constexpr int kLseOffBar = kLseOffK + kLseStages * kLseTileBytes;
constexpr int kLseOffX = kLseOffBar + 128;                 // float2 [128] exchange of the second half's (m, l)
constexpr int kLseSmemBytes = kLseOffX + 1024 + 1024;      // + alignment slack; 2 CTAs per SM
#ifndef SX_LSE_POLY
#define SX_LSE_POLY 2  // of every 8 pairs of exponentials, this many pairs go to the FMA pipe (0..8)
#endif

struct LseParams {
  const int32_t *new_idx;  // [total_new] positions of the Sparse-Q rows
  const int32_t *new_off;  // [num_reqs+1]
  const int32_t *seq_len;
  const int32_t *k_table;
  float *lse;              // [split][total_new][Hq] natural-log partial normalisers
  int num_reqs, max_pages, num_q_heads, num_kv_heads, group, rows_per_tile, total_new, kv_splits;
  float scale_log2, scale;
  const float2 *zc_table;  // zero-copy mode: (cos, sin) per segment and the page classification (sx_rotate.cuh)
  const int32_t *zc_page_seg;
};

struct LseBars {
  uint64_t q_full;
  uint64_t k_rot[kLseStages];  // zero-copy mode: the consumers have rotated the K tile of the slot (256 arrivals)
  uint64_t k_full[kLseStages], k_empty[kLseStages];
  uint64_t s_full[2], s_free[2];
  uint32_t tmem_base;
};

// kZc: 0 = K is read as stored; 1 / 2 = zero-copy mode with half-split / interleaved RoPE pairs: before they turn to
// S(t), the consumers rotate the rows of K tile t + 1 that still are cached source pages; the MMA of a tile waits for
// its rotation instead of its TMA completion.
template <int kZc>
__global__ void __launch_bounds__(kLseThreads, 2)
lse_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k, const LseParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  LseBars *bars = reinterpret_cast<LseBars *>(smem + kLseOffBar);
  float2 *xch = reinterpret_cast<float2 *>(smem + kLseOffX);
  const int g = p.group, rpt = p.rows_per_tile;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  constexpr int kWarpProd = 8, kWarpMma = 9;

  // ---- prologue without global memory (may overlap the previous kernel: programmatic dependent launch)
  griddep_launch();
  if (warp == kWarpProd && lane == 0) {
    tma_prefetch_desc(&tm_q);
    tma_prefetch_desc(&tm_k);
    mbar_init(&bars->q_full, 1);
    for (int i = 0; i < kLseStages; ++i) {
      mbar_init(&bars->k_full[i], 1);
      mbar_init(&bars->k_empty[i], 1);
      mbar_init(&bars->k_rot[i], 256);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bars->s_full[i], 1);
      mbar_init(&bars->s_free[i], 256);
    }
    fence_mbar_init();
  }
  if (warp == kWarpMma) {
    tmem_alloc(&bars->tmem_base, 256);
    tmem_relinquish();
  }
  // rows of the query tile that the TMA box never writes (128 - rpt*g pad rows) must be finite
  if (rpt * g < kTile) {
    const int pad = kTile - rpt * g;
    for (int i = threadIdx.x; i < 2 * pad * 8; i += kLseThreads) {
      const int c16 = i & 7, r = (i >> 3) % pad, h = (i >> 3) / pad;
      *reinterpret_cast<uint4 *>(smem + kLseOffQ + h * kLseHalf + (rpt * g + r) * 128 + c16 * 16) = make_uint4(0, 0, 0, 0);
    }
    fence_proxy_async_smem();
  }
  griddep_wait();

  // ---- (request, query tile, KV head, key split); late (heavy) query tiles of a request first
  const int split = (int)blockIdx.x % p.kv_splits;
  const int bid = (int)blockIdx.x / p.kv_splits;
  int req = 0, base = 0, tiles = 0, nn = 0;
  for (; req < p.num_reqs; ++req) {
    nn = p.new_off[req + 1] - p.new_off[req];
    tiles = (nn + rpt - 1) / rpt;
    if (bid < base + tiles * p.num_kv_heads) break;
    base += tiles * p.num_kv_heads;
  }
  const bool active = req < p.num_reqs;
  if (!active) req = 0;
  const int local = active ? bid - base : 0;
  const int kvh = local % p.num_kv_heads;
  const int qt = active ? tiles - 1 - local / p.num_kv_heads : 0;
  const int row_base = active ? p.new_off[req] + qt * rpt : p.total_new;  // first Sparse-Q row of this tile
  const int n_rows = active ? min(rpt, nn - qt * rpt) : 0;
  const int T = p.seq_len[req];
  const int n_pages = (T + kPage - 1) / kPage;
  const int pos_max = n_rows > 0 ? p.new_idx[row_base + n_rows - 1] : -1;
  const int all_tiles = pos_max / kTile + 1;  // (pos_max = -1 -> 0 tiles... see below)
  int t0 = 0, n_tiles = n_rows > 0 ? all_tiles : 0;
  if (p.kv_splits > 1) {
    const int per = (n_tiles + p.kv_splits - 1) / p.kv_splits;
    t0 = split * per;
    n_tiles = max(0, min(n_tiles, t0 + per) - t0);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;

  if (!active) {
    // grid overshoot
  } else if (warp == kWarpProd) {
    // ================================================================ TMA producer: Q once, then the K tiles
    if (n_tiles > 0) {
      if (lane == 0) {
        mbar_expect_tx(&bars->q_full, (uint32_t)(2 * rpt * g * 128));
        tma_load_3d(smem + kLseOffQ, &tm_q, &bars->q_full, 0, kvh * g, row_base);
        tma_load_3d(smem + kLseOffQ + kLseHalf, &tm_q, &bars->q_full, 64, kvh * g, row_base);
      }
      const int pg = lane >> 1, half = lane & 1;
      auto table_entry = [&](int t) -> int {
        int lp = (t0 + t) * 8 + pg;
        if (lp > n_pages - 1) lp = n_pages - 1;  // pages past the sequence: any valid page (keys are masked)
        return p.k_table[(size_t)req * p.max_pages + lp];
      };
      int blk = lane < 16 ? table_entry(0) : 0;
      for (int t = 0; t < n_tiles; ++t) {
        const int blk_next = (t + 1 < n_tiles && lane < 16) ? table_entry(t + 1) : 0;
        const int s = t % kLseStages, u = t / kLseStages;
        mbar_wait(&bars->k_empty[s], (u & 1) ^ 1);
        if (lane == 0) mbar_expect_tx(&bars->k_full[s], kLseTileBytes);
        __syncwarp();
        if (lane < 16)
          tma_load_2d(smem + kLseOffK + s * kLseTileBytes + half * kLseHalf + pg * 2048, &tm_k, &bars->k_full[s],
                      half * 64, (blk * p.num_kv_heads + kvh) * kPage);
        blk = blk_next;
      }
    }
  } else if (warp == kWarpMma) {
    // ================================================================ MMA issuer: S[b] = Q K(t)^T
    if (n_tiles > 0 && elect_one()) {
      constexpr uint32_t idesc = umma_idesc_bf16(128, 128, 0, 0);
      const uint64_t q_desc = umma_smem_desc(smem_u32(smem + kLseOffQ), 16, 1024);
      const uint64_t k_desc = umma_smem_desc(smem_u32(smem + kLseOffK), 16, 1024);
      const uint32_t q_lo = (uint32_t)q_desc, k_lo = (uint32_t)k_desc, hi32 = (uint32_t)(k_desc >> 32);
      mbar_wait(&bars->q_full, 0);
      for (int t = 0; t < n_tiles; ++t) {
        const int b = t & 1, s = t % kLseStages;
        mbar_wait(kZc ? &bars->k_rot[s] : &bars->k_full[s], (t / kLseStages) & 1);
        if (t >= 2) mbar_wait(&bars->s_free[b], ((t >> 1) + 1) & 1);
        tc_fence_after();
        const uint32_t kd = k_lo + (uint32_t)s * (kLseTileBytes >> 4);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t o = ((kk >> 2) * kLseHalf + (kk & 3) * 32) >> 4;
          umma_ss2(tmem + b * 128, q_lo + o, hi32, kd + o, hi32, idesc, kk > 0);
        }
        umma_commit(&bars->s_full[b]);
        umma_commit(&bars->k_empty[s]);
      }
    }
  } else {
    // ================================================================ consumers: two threads per row
    const int hf = warp >> 2;             // key columns [64 hf, 64 hf + 64) of every tile
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;  // (query, head) row = TMEM lane
    const int n_local = row / g, hh = row - n_local * g;
    const bool valid = n_local < n_rows;
    // rows without a query (pad rows when g does not divide 128, the tail of a request's last tile) are treated as
    // seeing every key: their S is finite (zero or another request's Q rows) and their result is never stored, but
    // with position -1 they would drag their whole warp through the masking path on every tile
    const int pos = valid ? p.new_idx[row_base + n_local] : 0x3fffffff;
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    float m = -INFINITY, l = 0.f;  // running maximum (log2 domain) and sum of this thread's key columns
    auto rotate_tile = [&](int t) {
      const int s = t % kLseStages;
      mbar_wait(&bars->k_full[s], (t / kLseStages) & 1);
      rotate_k_tile<(kZc > 0 ? kZc - 1 : 0), 256>(smem + kLseOffK + s * kLseTileBytes, kLseHalf,
                                                   p.zc_page_seg + (size_t)req * p.max_pages + (t0 + t) * 8,
                                                   n_pages - (t0 + t) * 8, p.zc_table, (int)threadIdx.x);
      fence_proxy_async_smem();
      mbar_arrive(&bars->k_rot[s]);
    };
    if (kZc != 0 && n_tiles > 0) rotate_tile(0);
    for (int t = 0; t < n_tiles; ++t) {
      const int b = t & 1;
      if (kZc != 0 && t + 1 < n_tiles) rotate_tile(t + 1);
      mbar_wait(&bars->s_full[b], (t >> 1) & 1);
      tc_fence_after();
      uint32_t sr[2][32];
      tmem_ld32(tmem + lane_addr + b * 128 + hf * 64, sr[0]);
      tmem_ld32(tmem + lane_addr + b * 128 + hf * 64 + 32, sr[1]);
      tmem_wait_ld();
      tc_fence_before();
      mbar_arrive(&bars->s_free[b]);
      // keys [j0, j0 + 64) of this thread; the first nvalid of them are visible to the row
      const int nvalid = pos - ((t0 + t) * kTile + hf * 64) + 1;
      if (nvalid < 64) {
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (c * 32 + i >= nvalid) sr[c][i] = 0xFF800000u;  // -inf
      }
      float tm0 = -INFINITY, tm1 = -INFINITY;
#pragma unroll
      for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int i = 0; i < 32; i += 4) {
          tm0 = fmaxf(tm0, fmaxf(__uint_as_float(sr[c][i]), __uint_as_float(sr[c][i + 1])));
          tm1 = fmaxf(tm1, fmaxf(__uint_as_float(sr[c][i + 2]), __uint_as_float(sr[c][i + 3])));
        }
      const float m_new = fmaxf(m, fmaxf(tm0, tm1) * p.scale_log2);
      if (m_new > -INFINITY) {  // (a tile this row cannot see at all leaves the state untouched)
        l *= ex2_approx(m - m_new);  // exp2(-inf) = 0 on the first visible tile
        m = m_new;
        const float2 sc2 = make_float2(p.scale_log2, p.scale_log2), nm2 = make_float2(-m, -m);
        float2 acc2 = make_float2(0.f, 0.f);
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
          for (int i = 0; i < 32; i += 2) {
            const float2 x = __ffma2_rn(make_float2(__uint_as_float(sr[c][i]), __uint_as_float(sr[c][i + 1])), sc2, nm2);
            float2 e;
            if ((i & 15) < 2 * SX_LSE_POLY) {
              e = ex2_poly2(x);
            } else {
              e.x = ex2_approx(x.x);
              e.y = ex2_approx(x.y);
            }
            acc2 = __fadd2_rn(acc2, e);
          }
        l += acc2.x + acc2.y;
      }
    }
    // the two halves of a row combine in a fixed order: lse = log(sum over both halves)
    named_bar_sync(1, 256);
    if (hf == 1) xch[row] = make_float2(m, l);
    named_bar_sync(1, 256);
    if (hf == 0 && valid) {
      const float2 o = xch[row];
      const float mm = fmaxf(m, o.x);
      float out = -INFINITY;  // a key split that holds no visible key of the row reports -inf
      if (mm > -INFINITY) {
        const float ls = (m == -INFINITY ? 0.f : l * ex2_approx(m - mm)) + (o.x == -INFINITY ? 0.f : o.y * ex2_approx(o.x - mm));
        out = (mm + log2f(ls)) * 0.6931471805599453f;
      }
      p.lse[((size_t)split * p.total_new + row_base + n_local) * p.num_q_heads + kvh * g + hh] = out;
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == kWarpMma) tmem_dealloc(tmem, 256);
}

// Key splits of the sweep: enough CTAs for about four waves at two CTAs per SM (a long single request gives few
// query tiles: C5 has 64 x 4 KV heads), at most 8 (the workspace holds 8 partial normalisers per row).
int lse_splits(const sx_pool *pool, const sx_batch *b) {
  const int g = pool->num_q_heads / pool->num_kv_heads;
  const int grid = (b->total_new / (kTile / g) + b->num_reqs) * pool->num_kv_heads;
  int s = (4 * 296 + grid - 1) / grid;
  const int tiles = (b->max_seq_len + kTile - 1) / kTile;
  if (s > tiles / 4) s = tiles / 4;  // at least four key tiles per split
  return s < 1 ? 1 : (s > 8 ? 8 : s);
}

sx_status launch_lse(const sx_pool *pool, const sx_batch *b, const void *q_new, float *lse_ws, int kv_splits,
                     const ZcArgs &zc, cudaStream_t st) {
  const int g = pool->num_q_heads / pool->num_kv_heads;
  const int rpt = kTile / g;
  CUtensorMap tm_q, tm_k;
  sx_status s = make_tmap_q(&tm_q, q_new, b->total_new, pool->num_q_heads, g, rpt);
  if (s != SX_OK) return s;
  s = make_tmap_pool(&tm_k, pool->k, pool->num_blocks, pool->num_kv_heads);
  if (s != SX_OK) return s;
  LseParams p;
  p.new_idx = b->new_idx;
  p.new_off = b->new_off;
  p.seq_len = b->seq_len;
  p.k_table = b->k_block_table;
  p.lse = lse_ws;
  p.num_reqs = b->num_reqs;
  p.max_pages = b->max_pages_per_req;
  p.num_q_heads = pool->num_q_heads;
  p.num_kv_heads = pool->num_kv_heads;
  p.group = g;
  p.rows_per_tile = rpt;
  p.total_new = b->total_new;
  p.kv_splits = kv_splits < 1 ? 1 : kv_splits;
  p.scale = (float)(1.0 / sqrt((double)kHeadDim));
  p.scale_log2 = (float)(kLog2e / sqrt((double)kHeadDim));
  const int grid = (b->total_new / rpt + b->num_reqs) * pool->num_kv_heads;  // >= sum_r ceil(|I_nr(r)| / rpt) * Hkv
  p.zc_table = zc.table;
  p.zc_page_seg = zc.page_seg;
  auto kern = zc.style < 0 ? lse_kernel<0> : (zc.style == 0 ? lse_kernel<1> : lse_kernel<2>);
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kLseSmemBytes);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "lse smem attr: %s", cudaGetErrorString(e));
  e = launch_pdl(kern, dim3(grid * p.kv_splits), dim3(kLseThreads), kLseSmemBytes, st, 1, tm_q, tm_k, p);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "lse launch: %s", cudaGetErrorString(e));
  return check_launch("lse_kernel");
}

}  // namespace sx
