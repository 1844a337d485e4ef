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
// The sweep is bound by the exponentials (128 x 128 per tile against 512 tensor-pipe cycles), so two
// CTAs share an SM, two consumer threads share a key (64 columns each), and a fixed fraction of the
// exponentials runs on the FMA pipe (Cody-Waite + cubic) beside MUFU.EX2.
#include <math.h>

#include "sx_internal.h"
#include "sx_ptx.cuh"
#include "sx_rotate.cuh"

namespace sx {

constexpr int kCsThreads = 320;  // warps 0-7 consumers, warp 8 TMA producer, warp 9 MMA issuer
constexpr int kCsTileBytes = kTile * kHeadDim * 2;
constexpr int kCsHalf = kCsTileBytes / 2;
constexpr int kCsStages = 2;
#ifndef SX_COLSUM_KSLOT
#define SX_COLSUM_KSLOT 1  // 1: the normaliser rides through the MMA as a ninth K step (see colsum_kernel); 0: added per element
#endif
constexpr bool kCsKslot = SX_COLSUM_KSLOT != 0;
// extra operand blocks of the ninth K step: 128 rows x 16 bf16 (32 B), K-major, NO swizzle: core matrices of
// 8 rows x 16 B; (row group, K chunk) at group * 256 + chunk * 128, i.e. LBO = 128 B, SBO = 256 B
constexpr int kCsExtBytes = kCsKslot ? kTile * 32 : 0;
constexpr int kCsOffK = 0;
constexpr int kCsOffAext = kCsOffK + kCsTileBytes;              // A side: [1, 1, 1, 0 ...] for every key row
constexpr int kCsOffQ = kCsOffAext + kCsExtBytes;
constexpr int kCsQStage = kCsTileBytes + kCsExtBytes;           // a Q stage = the tile, then its extra block
constexpr int kCsColStages = kCsKslot ? 6 : 8;                  // ring of column rows (see producer)
constexpr int kCsColRow = kCsKslot ? 512 : 1024;                // K-slot form: positions only (mask tiles only)
constexpr int kCsOffCol = kCsOffQ + kCsStages * kCsQStage;
constexpr int kCsOffBar = kCsOffCol + kCsColStages * kCsColRow;
constexpr int kCsSmemBytes = kCsOffBar + 256 + 1024;  // 2 CTAs per SM: 2 x (this + 1 KB) <= 228 KB
static_assert(2 * (kCsSmemBytes + 1024) <= 233472, "two CTAs per SM");
static_assert(kCsQStage % 1024 == 0, "128-B swizzle atoms need 1024-B aligned tiles");
constexpr int kCsTabEntry = 1024 + (kCsKslot ? 4096 : 0);       // bytes per (query tile, KV head) in the workspace
#ifndef SX_COLSUM_POLY
#define SX_COLSUM_POLY 2  // of every 8 pairs of exponentials, this many pairs go to the FMA pipe (0..8);
                          // measured on C2 / C4 / C5 (MUFU pipe 77 % busy at 1): 2 and 3 are 1-2 % faster than 1, 4 slower
#endif

struct ColsumParams {
  const int32_t *seq_len, *tok_off, *new_off, *new_idx, *k_table;
  const float *lse;  // natural log; [total_new][Hq], or [total_tokens][Hq] when lse_by_token
  int lse_by_token;
  int lse_splits;     // > 1: lse holds that many partial normalisers [split][total_new][Hq] (key splits)
  size_t lse_stride;  // total_new * Hq
  float2 *col_tab;   // [query tiles of the batch][Hkv] entries of kCsTabEntry bytes: float lse * log2 e [128], int position
                     // [128], then (K-slot form) the 4-KB extra B block of the tile in its shared-memory layout
  float *partial;    // [Hkv][total_tokens]
  int num_reqs, max_pages, num_q_heads, num_kv_heads, group, rows_per_tile, total_tokens;
  float scale_log2;
  const float2 *zc_table;     // zero-copy mode: (cos, sin) per segment and the page classification (sx_rotate.cuh)
  const int32_t *zc_page_seg;
  int4 *plan;                 // [colsum grid][2] work record of every colsum CTA, written by coltab_kernel (see there)
  int n_qt_blocks, cs_grid;   // coltab grid: blockIdx.x < n_qt_blocks build column rows, the rest build the plan
};

struct CsBars {
  uint64_t k_full;
  uint64_t k_rot;  // zero-copy mode: the consumers have rotated the K tile (256 arrivals)
  uint64_t q_full[kCsStages], q_empty[kCsStages];
  uint64_t d_full[2], d_empty[2];
  uint64_t c_full[kCsColStages];
  uint32_t tmem_base;
};

// Column table of sweep 2: for every GQA-packed query tile (rows_per_tile queries x g heads = up to 128
// columns) the log2-domain normaliser and the position of each column; pad columns get (+inf, -1) so that
// their exp2 is 0. One 1-KB row per (query tile, KV head): the colsum producer fetches it with one bulk copy.
// Normalisers and positions are stored one after the other (128 floats, then 128 ints): tiles that need no
// causal mask (the majority) read the normalisers only, four columns per 16-byte shared-memory load.
__global__ void __launch_bounds__(128)
coltab_kernel(const ColsumParams p) {
  griddep_launch();  // programmatic dependent launch: the next kernel may become resident now ...
  griddep_wait();    // ... and this one touches global memory only after its predecessor has completed
  const int g = p.group, rpt = p.rows_per_tile;
  if ((int)blockIdx.x >= p.n_qt_blocks) {
    // ---- work records of the colsum CTAs: which (request, key tile, KV head) a CTA owns and which query tiles can
    // see its keys is a serial walk over the requests plus two binary searches over new_idx -- a dozen DEPENDENT
    // global loads (clock64 trace: 6 300 clk per CTA, a quarter of a C4 CTA's life). One thread per CTA does them
    // here, once; the CTA then starts from a single 32-byte load.
    const int cta = (((int)blockIdx.x - p.n_qt_blocks) * (int)gridDim.y + (int)blockIdx.y) * 128 + (int)threadIdx.x;
    if (cta >= p.cs_grid) return;
    int req = 0, base = 0, ktiles = 0, qt_base = 0;  // qt_base: query tiles of the requests before this one
    for (; req < p.num_reqs; ++req) {
      ktiles = (p.seq_len[req] + kTile - 1) / kTile;
      if (cta < base + ktiles * p.num_kv_heads) break;
      base += ktiles * p.num_kv_heads;
      qt_base += (p.new_off[req + 1] - p.new_off[req] + rpt - 1) / rpt;
    }
    int4 r0 = make_int4(-1, 0, 0, 0), r1 = make_int4(0, 0, 0, 0);
    if (req < p.num_reqs) {
      const int local = cta - base;
      const int kvh = local % p.num_kv_heads, kt = local / p.num_kv_heads;  // early key tiles (seen by the most queries) first
      const int j0 = kt * kTile;
      const int nq0 = p.new_off[req], nn = p.new_off[req + 1] - nq0;
      int lo = 0, hi = nn;  // first Sparse-Q query that can see key j0: lower_bound(new_idx, j0)
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (p.new_idx[nq0 + mid] < j0) lo = mid + 1; else hi = mid;
      }
      const int qt0 = lo / rpt;  // first query tile with a visible query
      const int n_it = (lo < nn) ? (nn + rpt - 1) / rpt - qt0 : 0;
      // queries are sorted by position: only the leading tiles, whose first query sits below the tile's last key,
      // need a causal mask: tiles it < n_mask (first query index (qt0 + it) * rpt below lower_bound(new_idx, j0 + 127))
      int lo2 = lo, hi2 = nn;
      while (lo2 < hi2) {
        const int mid = (lo2 + hi2) >> 1;
        if (p.new_idx[nq0 + mid] < j0 + kTile - 1) lo2 = mid + 1; else hi2 = mid;
      }
      r0 = make_int4(req, kt | (kvh << 24), p.seq_len[req], nq0 + qt0 * rpt);
      r1 = make_int4(n_it, max(0, (lo2 + rpt - 1) / rpt - qt0), qt_base + qt0, p.tok_off[req]);
    }
    p.plan[2 * cta] = r0;
    p.plan[2 * cta + 1] = r1;
    return;
  }
  int req = 0, base = 0;
  for (; req < p.num_reqs; ++req) {
    const int nq = (p.new_off[req + 1] - p.new_off[req] + rpt - 1) / rpt;
    if ((int)blockIdx.x < base + nq) break;
    base += nq;
  }
  if (req >= p.num_reqs) return;
  const int qt = blockIdx.x - base, kvh = blockIdx.y, ct = threadIdx.x;
  const int nq0 = p.new_off[req], nn = p.new_off[req + 1] - nq0;
  const int cn = ct / g, ch = ct - cn * g, n = qt * rpt + cn;
  float lse2 = INFINITY;
  int qpos = -1;
  if (cn < rpt && n < nn) {
    qpos = p.new_idx[nq0 + n];
    const size_t lrow = p.lse_by_token ? (size_t)(p.tok_off[req] + qpos) : (size_t)(nq0 + n);
    const size_t idx = lrow * p.num_q_heads + kvh * g + ch;
    float l = p.lse[idx];
    if (p.lse_splits > 1) {  // log-sum-exp of the key splits, fixed order
      float mx = l;
      for (int s = 1; s < p.lse_splits; ++s) mx = fmaxf(mx, p.lse[s * p.lse_stride + idx]);
      float sum = 0.f;
      for (int s = 0; s < p.lse_splits; ++s) sum += expf(p.lse[s * p.lse_stride + idx] - mx);
      l = mx + logf(sum);
    }
    lse2 = l * (float)kLog2e;
  }
  uint8_t *entry = reinterpret_cast<uint8_t *>(p.col_tab) + ((size_t)blockIdx.x * p.num_kv_heads + kvh) * kCsTabEntry;
  float *row = reinterpret_cast<float *>(entry);
  row[ct] = lse2;
  row[128 + ct] = __int_as_float(qpos);
  if (kCsKslot) {
    // -lse2 / scale_log2 = -lse * sqrt(d), split into three bf16 (hi + mid + lo carries 24 bits): the MMA adds it to
    // the raw score of every key of the column. Pad columns: -inf (their exponential is 0), mid = lo = 0.
    const float v = (lse2 == INFINITY) ? -INFINITY : -lse2 / p.scale_log2;
    const __nv_bfloat16 h = __float2bfloat16_rn(v);
    float rem = (lse2 == INFINITY) ? 0.f : v - __bfloat162float(h);
    const __nv_bfloat16 m = __float2bfloat16_rn(rem);
    rem -= __bfloat162float(m);
    const __nv_bfloat16 l = __float2bfloat16_rn(rem);
    const uint32_t w0 = (uint32_t)__bfloat16_as_ushort(h) | ((uint32_t)__bfloat16_as_ushort(m) << 16);
    const uint32_t w1 = (uint32_t)__bfloat16_as_ushort(l);
    uint4 *ext = reinterpret_cast<uint4 *>(entry + 1024);
    ext[(ct >> 3) * 16 + (ct & 7)] = make_uint4(w0, w1, 0, 0);   // K chunk 0 of column ct
    ext[(ct >> 3) * 16 + 8 + (ct & 7)] = make_uint4(0, 0, 0, 0);  // K chunk 1
  }
}

// One consumer thread, one D tile: sum of exp2(s * c - lse_col) over its 64 columns (d[2][32] = raw scores of its key
// against the 64 (query, head) columns; `col` = shared-memory address of their normalisers, positions 512 B further).
template <bool kMask>
__device__ __forceinline__ float2 cs_consume(const uint32_t (&d)[2][32], uint32_t col, float2 sc2, int j, float2 acc2) {
#pragma unroll
  for (int c = 0; c < 2; ++c)
#pragma unroll
    for (int i = 0; i < 32; i += 4) {
      float4 l4 = make_float4(0.f, 0.f, 0.f, 0.f);
      if (!kCsKslot) l4 = lds_f4(col + (c * 32 + i) * 4);  // lse of four columns (K-slot form: already inside d)
      float4 p4 = make_float4(0.f, 0.f, 0.f, 0.f);
      if (kMask) p4 = lds_f4(col + (kCsKslot ? 0 : 512) + (c * 32 + i) * 4);  // their positions (int bits)
#pragma unroll
      for (int h2 = 0; h2 < 2; ++h2) {
        const int ii = i + 2 * h2;
        const float la = h2 ? l4.z : l4.x, lb = h2 ? l4.w : l4.y;
        const float2 dv = make_float2(__uint_as_float(d[c][ii]), __uint_as_float(d[c][ii + 1]));
        const float2 x = kCsKslot ? __fmul2_rn(dv, sc2) : __ffma2_rn(dv, sc2, make_float2(-la, -lb));
        float2 e;
        if ((ii & 15) < 2 * SX_COLSUM_POLY) {
          e = ex2_poly2(x);
        } else {
          e.x = ex2_approx(x.x);
          e.y = ex2_approx(x.y);
        }
        if (kMask) {  // a query sees key j iff its position is >= j
          e.x = (__float_as_int(h2 ? p4.z : p4.x) >= j) ? e.x : 0.f;
          e.y = (__float_as_int(h2 ? p4.w : p4.y) >= j) ? e.y : 0.f;
        }
        acc2 = __fadd2_rn(acc2, e);
      }
    }
  return acc2;
}

// kZc: 0 = K is read as stored; 1 / 2 = zero-copy mode with half-split / interleaved RoPE pairs: the consumers rotate
// the rows of the K tile that still are cached source pages before the first MMA reads the tile.
template <int kZc>
__global__ void __launch_bounds__(kCsThreads, 2)
colsum_kernel(const __grid_constant__ CUtensorMap tm_q, const __grid_constant__ CUtensorMap tm_k,
              const ColsumParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = reinterpret_cast<uint8_t *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  CsBars *bars = reinterpret_cast<CsBars *>(smem + kCsOffBar);
  uint8_t *col_sm = smem + kCsOffCol;  // [kCsColStages] rows of kCsColRow bytes: (lse2[128],) position[128]
  const int g = p.group, rpt = p.rows_per_tile;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  constexpr int kWarpProd = 8, kWarpMma = 9;

  // ---- prologue without global memory (may overlap the previous kernel: programmatic dependent launch)
  griddep_launch();
  if (warp == kWarpProd && lane == 0) {
    tma_prefetch_desc(&tm_q);
    tma_prefetch_desc(&tm_k);
    mbar_init(&bars->k_full, 1);
    mbar_init(&bars->k_rot, 256);
    for (int i = 0; i < kCsStages; ++i) {
      mbar_init(&bars->q_full[i], 1);
      mbar_init(&bars->q_empty[i], 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bars->d_full[i], 1);
      mbar_init(&bars->d_empty[i], 256);
    }
    for (int i = 0; i < kCsColStages; ++i) mbar_init(&bars->c_full[i], 1);
    fence_mbar_init();
  }
  if (warp == kWarpMma) {
    tmem_alloc(&bars->tmem_base, 256);
    tmem_relinquish();
  }
  // rows of the Q stages that the TMA box never writes (128 - rpt*g pad columns) must be finite
  if (rpt * g < kTile) {
    const int pad = kTile - rpt * g;
    for (int i = threadIdx.x; i < kCsStages * 2 * pad * 8; i += kCsThreads) {
      int c16 = i & 7, r = (i >> 3) % pad, hs = (i >> 3) / pad;  // hs = stage*2 + half
      *reinterpret_cast<uint4 *>(smem + kCsOffQ + (hs >> 1) * kCsQStage + (hs & 1) * kCsHalf + (rpt * g + r) * 128 +
                                 c16 * 16) = make_uint4(0, 0, 0, 0);
    }
    fence_proxy_async_smem();
  }
  if (kCsKslot) {
    // A side of the ninth K step: every key row is [1, 1, 1, 0 ...] (bf16 1.0 = 0x3F80); 256 chunks of 16 B
    if (threadIdx.x < 256) {
      const int ch = threadIdx.x;  // chunk (row group, K chunk, row): K chunk = bit 3
      reinterpret_cast<uint4 *>(smem + kCsOffAext)[ch] =
          ((ch >> 3) & 1) ? make_uint4(0, 0, 0, 0) : make_uint4(0x3F803F80u, 0x00003F80u, 0, 0);
    }
    fence_proxy_async_smem();
  }
  griddep_wait();

  // ---- this CTA's work record (coltab_kernel): (request, key tile, KV head), the query tiles that see its keys
  // (plain loads: the record is an OUTPUT of the preceding kernel, and under programmatic dependent launch this CTA
  // may have become resident before that kernel wrote it -- the read-only (.nc) path must not be used for it)
  const int4 w0 = p.plan[2 * blockIdx.x], w1 = p.plan[2 * blockIdx.x + 1];
  const int req = w0.x, kt = w0.y & 0xFFFFFF, kvh = w0.y >> 24, T = w0.z, r_first = w0.w;
  const int n_it = req >= 0 ? w1.x : 0, n_mask = w1.y, qt_first = w1.z, tok0 = w1.w;
  const int j0 = kt * kTile;
  const int n_pages = (T + kPage - 1) / kPage;

  // The producer warp does not wait for the others: it initialised the barriers itself and needs neither TMEM nor
  // the operand rows the others zero, so it ARRIVES at the block-wide meeting and starts loading at once.
  if (warp == kWarpProd) named_bar_arrive(2, kCsThreads);
  else {
    tc_fence_before();
    named_bar_sync(2, kCsThreads);
    tc_fence_after();
  }
  const uint32_t tmem = bars->tmem_base;  // (not used by the producer warp)

  if (warp == kWarpProd) {
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
      __syncwarp();
      if (elect_one()) {
        int s = 0, ph = 1;
        for (int it = 0; it < n_it; ++it) {
          mbar_wait(&bars->q_empty[s], ph);
          mbar_expect_tx(&bars->q_full[s], (uint32_t)(2 * rpt * g * 128 + kCsExtBytes));
          const int r0 = r_first + it * rpt;
          uint8_t *qs = smem + kCsOffQ + s * kCsQStage;
          tma_load_3d(qs, &tm_q, &bars->q_full[s], 0, kvh * g, r0);
          tma_load_3d(qs + kCsHalf, &tm_q, &bars->q_full[s], 64, kvh * g, r0);
          const uint8_t *entry = reinterpret_cast<const uint8_t *>(p.col_tab) +
                                 ((size_t)(qt_first + it) * p.num_kv_heads + kvh) * kCsTabEntry;
          // Column row of this query tile, own ring: this thread is at most 2 tiles ahead of the MMA issuer, which is
          // at most 2 tiles ahead of the consumers' D loads, so 5 slots suffice.
          const int cs = it % kCsColStages;
          if (kCsKslot) {
            // the tile's extra B block (normalisers) lands behind the tile on the same barrier; positions are needed by
            // the leading mask tiles only
            bulk_load_1d(qs + kCsTileBytes, entry + 1024, kCsExtBytes, &bars->q_full[s]);
            if (it < n_mask) {
              mbar_expect_tx(&bars->c_full[cs], 512);
              bulk_load_1d(col_sm + cs * kCsColRow, entry + 512, 512, &bars->c_full[cs]);
            }
          } else {
            mbar_expect_tx(&bars->c_full[cs], 1024);
            bulk_load_1d(col_sm + cs * kCsColRow, entry, 1024, &bars->c_full[cs]);
          }
          if (++s == kCsStages) { s = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == kWarpMma) {
    // ================================================================ MMA issuer: D[b] = K_tile * Q_tile^T
    if (n_it > 0 && elect_one()) {
      constexpr uint32_t idesc = umma_idesc_bf16(128, 128, 0, 0);
      const uint64_t k_desc = umma_smem_desc(smem_u32(smem + kCsOffK), 16, 1024);
      const uint64_t q_desc = umma_smem_desc(smem_u32(smem + kCsOffQ), 16, 1024);
      const uint32_t k_lo = (uint32_t)k_desc, q_lo = (uint32_t)q_desc, hi32 = (uint32_t)(k_desc >> 32);
      mbar_wait(kZc ? &bars->k_rot : &bars->k_full, 0);
      int s = 0, ph = 0;
      for (int it = 0; it < n_it; ++it) {
        const int b = it & 1;
        mbar_wait(&bars->q_full[s], ph);
        if (it >= 2) mbar_wait(&bars->d_empty[b], ((it >> 1) + 1) & 1);
        tc_fence_after();
        const uint32_t qd = q_lo + (uint32_t)s * (kCsQStage >> 4);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t o = ((kk >> 2) * kCsHalf + (kk & 3) * 32) >> 4;
          umma_ss2(tmem + b * 128, k_lo + o, hi32, qd + o, hi32, idesc, kk > 0);
        }
        if (kCsKslot) {
          // ninth K step: D += [1 1 1 0 ...] x [hi mid lo 0 ...]^T = -lse * sqrt(d) of every column, added to every
          // key row. Unswizzled K-major blocks: LBO = 128 B (K chunks), SBO = 256 B (8-row groups), layout type 0.
          constexpr uint32_t ext_hi = (256u >> 4) | (1u << 14);
          const uint32_t a_ext = ((smem_u32(smem + kCsOffAext) & 0x3FFFF) >> 4) | ((128u >> 4) << 16);
          const uint32_t b_ext = ((smem_u32(smem + kCsOffQ + s * kCsQStage + kCsTileBytes) & 0x3FFFF) >> 4) | ((128u >> 4) << 16);
          umma_ss2(tmem + b * 128, a_ext, ext_hi, b_ext, ext_hi, idesc, 1);
        }
        umma_commit(&bars->d_full[b]);
        umma_commit(&bars->q_empty[s]);
        if (++s == kCsStages) { s = 0; ph ^= 1; }
      }
    }
  } else {
    // ================================================================ consumers: two threads per key
    const int hf = warp >> 2;              // column half [64 hf, 64 hf + 64) of every D tile
    const int quarter = warp & 3;
    const int row = quarter * 32 + lane;   // key j0 + row = TMEM lane
    const int j = j0 + row;
    const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
    float2 acc2 = make_float2(0.f, 0.f);
    const float2 sc2 = make_float2(p.scale_log2, p.scale_log2);
    if (kZc != 0 && n_it > 0) {
      mbar_wait(&bars->k_full, 0);
      rotate_k_tile<kZc - 1, 256>(smem + kCsOffK, kCsHalf, p.zc_page_seg + (size_t)req * p.max_pages + kt * 8,
                                  n_pages - kt * 8, p.zc_table, (int)threadIdx.x);
      fence_proxy_async_smem();
      mbar_arrive(&bars->k_rot);
    }
    for (int it = 0; it < n_it; ++it) {
      const int b = it & 1, cs = it % kCsColStages;
      const bool need_mask = it < n_mask;  // (the leading tiles, see n_mask)
      // K-slot form: the row holds positions only and exists for mask tiles only
      if (!kCsKslot || need_mask) mbar_wait(&bars->c_full[cs], (it / kCsColStages) & 1);
      const uint32_t col = smem_u32(col_sm + cs * kCsColRow) + hf * 256;  // this thread's 64 columns: lse (+512:
                                                                          // positions), or positions alone
      mbar_wait(&bars->d_full[b], (it >> 1) & 1);
      tc_fence_after();
      uint32_t d[2][32];
      tmem_ld32(tmem + lane_addr + b * 128 + hf * 64, d[0]);
      tmem_ld32(tmem + lane_addr + b * 128 + hf * 64 + 32, d[1]);
      tmem_wait_ld();
      tc_fence_before();
      mbar_arrive(&bars->d_empty[b]);  // D[b] is in registers: the next-but-one tile may overwrite it
      // (two copies of the loop: a per-element `if (need_mask)` would be predicated compares and selects that
      // take issue slots on every tile, and only the few tiles on the causal diagonal need them)
      if (need_mask) acc2 = cs_consume<true>(d, col, sc2, j, acc2);
      else acc2 = cs_consume<false>(d, col, sc2, j, acc2);
    }
    // the two halves of a key add up in a fixed order
    float *xch = reinterpret_cast<float *>(col_sm);  // every column row has been consumed
    named_bar_sync(1, 256);
    const float acc = acc2.x + acc2.y;
    if (hf == 1) xch[row] = acc;
    named_bar_sync(1, 256);
    if (hf == 0 && j < T) p.partial[(size_t)kvh * p.total_tokens + tok0 + j] = acc + xch[row];
  }

  tc_fence_before();
  __syncthreads();
  if (warp == kWarpMma) tmem_dealloc(tmem, 256);
}

size_t colsum_tab_bytes(const sx_pool *pool, const sx_batch *b) {
  const int g = pool->num_q_heads / pool->num_kv_heads;
  const int rpt = kTile / (g > 0 ? g : 1) > 0 ? kTile / (g > 0 ? g : 1) : 1;
  const size_t entries = (size_t)(b->total_new / rpt + b->num_reqs) * pool->num_kv_heads * kCsTabEntry;
  const size_t plan = (size_t)(b->total_tokens / kTile + b->num_reqs) * pool->num_kv_heads * 2 * sizeof(int4);
  return entries + plan;  // column entries, then one 32-byte work record per colsum CTA
}

sx_status launch_colsum(const sx_pool *pool, const sx_batch *b, const void *q_new, const float *lse_new,
                        int lse_by_token, int lse_splits, float *partial, float2 *col_tab, const ZcArgs &zc,
                        cudaStream_t st) {
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
  p.lse_splits = lse_splits;
  p.lse_stride = (size_t)b->total_new * pool->num_q_heads;
  p.partial = partial;
  p.col_tab = col_tab;
  p.num_reqs = b->num_reqs;
  p.max_pages = b->max_pages_per_req;
  p.num_q_heads = pool->num_q_heads;
  p.num_kv_heads = pool->num_kv_heads;
  p.group = g;
  p.rows_per_tile = rpt;
  p.total_tokens = b->total_tokens;
  p.scale_log2 = (float)(kLog2e / sqrt((double)kHeadDim));
  p.zc_table = zc.table;
  p.zc_page_seg = zc.page_seg;
  const int grid = (b->total_tokens / kTile + b->num_reqs) * pool->num_kv_heads;
  auto kern = zc.style < 0 ? colsum_kernel<0> : (zc.style == 0 ? colsum_kernel<1> : colsum_kernel<2>);
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kCsSmemBytes);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "colsum smem attr: %s", cudaGetErrorString(e));
  const int n_qt = b->total_new / rpt + b->num_reqs;  // >= sum_r ceil(|I_nr(r)| / rpt)
  p.plan = reinterpret_cast<int4 *>(reinterpret_cast<uint8_t *>(col_tab) + (size_t)n_qt * pool->num_kv_heads * kCsTabEntry);
  p.n_qt_blocks = n_qt;
  p.cs_grid = grid;
  const int plan_blocks = (grid + 128 * pool->num_kv_heads - 1) / (128 * pool->num_kv_heads);
  e = launch_pdl(coltab_kernel, dim3(n_qt + plan_blocks, pool->num_kv_heads), dim3(128), 0, st, 1, p);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "coltab launch: %s", cudaGetErrorString(e));
  s = check_launch("coltab_kernel");
  if (s != SX_OK) return s;
  e = launch_pdl(kern, dim3(grid), dim3(kCsThreads), kCsSmemBytes, st, 1, tm_q, tm_k, p);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "colsum launch: %s", cudaGetErrorString(e));
  return check_launch("colsum_kernel");
}

}  // namespace sx
