// sx_attn_small.cu -- stage (c) when GQA packing gives FEWER than 64 query rows per KV head:
//   O[R] = SparseAttn(Q[R], K_cur[1:T], V_cur[1:T], M_causal)          Alg. 1 l.546-548
// on the CUDA cores (BASELINE.json north_star: tensor-core tiles only where at least 64 (row, head) pairs
// share a KV head; below that the work is a K/V stream with a handful of dot products per key, bound by
// HBM for up to ~10 pairs and by the FMA pipe beyond).
//
// Split-KV ("flash-decoding") design, no tensor cores:
//   * a CTA owns one (request, chunk of rows, KV head, split of the key range); the m <= 64 (row, head)
//     pairs of the chunk share every K/V row it streams. Key tiles of 128 keys = 8 pages arrive through
//     16-byte cp.async copies (coalesced: 256 B per (page, head, row)) into a two-stage ring with a padded
//     row pitch of 272 B, so that "one thread per key" reads are free of bank conflicts.
//   * phase 1 (QK^T): thread = (key, half of the pairs); the K row is unpacked from bf16 once per 8 pairs,
//     the fp32 queries (pre-multiplied by log2(e)/sqrt(d)) are broadcast reads from shared memory.
//   * phase 2 (softmax): one warp per pair: row maximum / sum by warp shuffles, running (m, l) per pair.
//   * phase 3 (PV): thread = (8 output dims, pairs p = pg mod 16): V rows unpacked once per thread and
//     reused by its pairs, P read as 4-key vectors.
//   * every split writes (m, l, unnormalised O) to the workspace; a merge kernel combines the splits in a
//     fixed order (deterministic), normalises and writes bf16 O and the natural-log LSE.
#include <math.h>

#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

constexpr int kSmThreads = 256;
constexpr int kSmPairs = 64;     // pair slots per CTA (at most 63 are used by the dispatch rule, 64 by chunking)
constexpr int kSmRowB = 272;     // bytes between consecutive K (or V) rows in shared memory (256 + 16 pad)
constexpr int kSmPPitch = 132;   // floats between consecutive rows of the S/P tile
constexpr int kSmOffQ = 0;                                        // float [64][128]
constexpr int kSmOffKV = kSmOffQ + kSmPairs * kHeadDim * 4;       // 2 stages x (K, V) x 128 rows x 272 B
constexpr int kSmStageB = 2 * kTile * kSmRowB;
constexpr int kSmOffP = kSmOffKV + 2 * kSmStageB;                 // float [64][132]
constexpr int kSmOffStat = kSmOffP + kSmPairs * kSmPPitch * 4;    // m[64], l[64], alpha[64] float; pos[64] int
constexpr int kSmSmemBytes = kSmOffStat + 4 * kSmPairs * 4;
constexpr int kSmPartFloats = kSmPairs * (kHeadDim + 2);          // per (slot, kv head, split): O, m, l

struct SmallParams {
  const __nv_bfloat16 *q;   // [total_rows][Hq][128]
  const uint4 *pool_k, *pool_v;
  const int32_t *rows;      // positions, or nullptr (full mode)
  const int32_t *rows_off, *seq_len, *k_table, *v_table;
  float *part;              // [slots][Hkv][splits][kSmPartFloats]
  __nv_bfloat16 *out;
  float *lse;
  int num_reqs, max_pages, num_q_heads, num_kv_heads, group, rows_per_chunk, splits;
  float scale_log2;
};

// slot -> (request, chunk of rows). Returns false if the slot is beyond the last chunk.
__device__ __forceinline__ bool small_decode(const SmallParams &p, int slot, int &req, int &r0, int &nr) {
  int base = 0;
  for (req = 0; req < p.num_reqs; ++req) {
    const int n_r = p.rows_off[req + 1] - p.rows_off[req];
    const int chunks = (n_r + p.rows_per_chunk - 1) / p.rows_per_chunk;
    if (slot < base + chunks) {
      const int c = slot - base;
      r0 = p.rows_off[req] + c * p.rows_per_chunk;
      nr = min(p.rows_per_chunk, n_r - c * p.rows_per_chunk);
      return true;
    }
    base += chunks;
  }
  return false;
}

__device__ __forceinline__ void cp_async16(void *dst, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

__device__ __forceinline__ float bf_lo_f(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf_hi_f(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

__global__ void __launch_bounds__(kSmThreads, 1)
attn_small_kernel(const SmallParams p) {
  extern __shared__ __align__(16) uint8_t sm[];
  float *Qs = reinterpret_cast<float *>(sm + kSmOffQ);
  float *Ps = reinterpret_cast<float *>(sm + kSmOffP);
  float *m_s = reinterpret_cast<float *>(sm + kSmOffStat);
  float *l_s = m_s + kSmPairs;
  float *a_s = l_s + kSmPairs;
  int *pos_s = reinterpret_cast<int *>(a_s + kSmPairs);

  const int split = blockIdx.x, kvh = blockIdx.y, slot = blockIdx.z;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = p.group;
  int req, r0, nr;
  if (!small_decode(p, slot, req, r0, nr)) return;
  const int m = nr * g;  // (row, head) pairs of this CTA, pair index = row * g + head
  const int T = p.seq_len[req];
  const int n_pages = (T + kPage - 1) / kPage;
  const int pos_max = p.rows ? p.rows[r0 + nr - 1] : (r0 + nr - 1 - p.rows_off[req]);
  const int nt = pos_max / kTile + 1;
  const int per = (nt + p.splits - 1) / p.splits;
  const int t_begin = split * per, t_end = min(nt, t_begin + per);
  float *part = p.part + ((size_t)(slot * p.num_kv_heads + kvh) * p.splits + split) * kSmPartFloats;

  if (t_begin >= t_end) {  // nothing to do for this split: neutral partial
    for (int i = tid; i < kSmPairs; i += kSmThreads) {
      part[kSmPairs * kHeadDim + i] = -INFINITY;
      part[kSmPairs * kHeadDim + kSmPairs + i] = 0.f;
    }
    return;
  }

  // ---- queries (fp32, pre-scaled), per-pair state
  for (int i = tid; i < kSmPairs * 16; i += kSmThreads) {
    const int pr = i >> 4, c = i & 15;
    float4 lo = make_float4(0.f, 0.f, 0.f, 0.f), hi = lo;
    if (pr < m) {
      const int ri = pr / g, hh = pr - ri * g;
      const uint4 v = *reinterpret_cast<const uint4 *>(p.q + ((size_t)(r0 + ri) * p.num_q_heads + kvh * g + hh) * kHeadDim + c * 8);
      lo = make_float4(bf_lo_f(v.x) * p.scale_log2, bf_hi_f(v.x) * p.scale_log2, bf_lo_f(v.y) * p.scale_log2,
                       bf_hi_f(v.y) * p.scale_log2);
      hi = make_float4(bf_lo_f(v.z) * p.scale_log2, bf_hi_f(v.z) * p.scale_log2, bf_lo_f(v.w) * p.scale_log2,
                       bf_hi_f(v.w) * p.scale_log2);
    }
    *reinterpret_cast<float4 *>(Qs + pr * kHeadDim + c * 8) = lo;
    *reinterpret_cast<float4 *>(Qs + pr * kHeadDim + c * 8 + 4) = hi;
  }
  if (tid < kSmPairs) {
    m_s[tid] = -INFINITY;
    l_s[tid] = 0.f;
    a_s[tid] = 1.f;
    int ps = -1;  // unused pair slots see no key
    if (tid < m) {
      const int ri = tid / g;
      ps = p.rows ? p.rows[r0 + ri] : (r0 + ri - p.rows_off[req]);
    }
    pos_s[tid] = ps;
  }

  // K/V tile t -> stage: thread copies chunk (tid & 15) of row (tid >> 4) + 16 j of page j, j = 0..7
  auto load_tile = [&](int t, int stage) {
    uint8_t *ks = sm + kSmOffKV + stage * kSmStageB;
    uint8_t *vs = ks + kTile * kSmRowB;
    const int r16 = tid >> 4, c = tid & 15;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      int lp = t * 8 + j;
      if (lp > n_pages - 1) lp = n_pages - 1;  // beyond the sequence: any valid page (those keys are masked)
      const size_t e = (size_t)req * p.max_pages + lp;
      const size_t ko = ((size_t)p.k_table[e] * p.num_kv_heads + kvh) * (kPage * 16) + r16 * 16 + c;
      const size_t vo = ((size_t)p.v_table[e] * p.num_kv_heads + kvh) * (kPage * 16) + r16 * 16 + c;
      cp_async16(ks + (j * 16 + r16) * kSmRowB + c * 16, p.pool_k + ko);
      cp_async16(vs + (j * 16 + r16) * kSmRowB + c * 16, p.pool_v + vo);
    }
    cp_async_commit();
  };

  // phase-3 ownership: 8 output dims x pairs pg, pg + 16, pg + 32, pg + 48
  const int oc = tid & 15, pg = tid >> 4;
  float acc[4][8];
#pragma unroll
  for (int j = 0; j < 4; ++j)
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[j][i] = 0.f;

  load_tile(t_begin, 0);
  for (int t = t_begin; t < t_end; ++t) {
    const int stage = (t - t_begin) & 1;
    if (t + 1 < t_end) {
      load_tile(t + 1, stage ^ 1);
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    const uint8_t *ks = sm + kSmOffKV + stage * kSmStageB;
    const uint8_t *vs = ks + kTile * kSmRowB;
    const int nkeys = min(kTile, pos_max + 1 - t * kTile);  // keys of this tile any pair can see (< T)

    // ---- phase 1: S[pair][key] = <q_pair, k_key> (log2 domain), causal mask
    {
      const int key = tid & 127, half = tid >> 7;
      const int cnt0 = (m + 1) >> 1;
      const int p_lo = half ? cnt0 : 0, p_hi = half ? m : cnt0;
      const uint4 *krow = reinterpret_cast<const uint4 *>(ks + key * kSmRowB);
      const int kpos = t * kTile + key;
      for (int pb = p_lo; pb < p_hi; pb += 8) {
        float s[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) s[i] = 0.f;
#pragma unroll 4
        for (int c = 0; c < 16; ++c) {
          const uint4 kv = krow[c];
          const float k0 = bf_lo_f(kv.x), k1 = bf_hi_f(kv.x), k2 = bf_lo_f(kv.y), k3 = bf_hi_f(kv.y);
          const float k4 = bf_lo_f(kv.z), k5 = bf_hi_f(kv.z), k6 = bf_lo_f(kv.w), k7 = bf_hi_f(kv.w);
#pragma unroll
          for (int i = 0; i < 8; ++i) {  // rows past p_hi read valid (zero or foreign) queries; never stored
            const float4 qa = *reinterpret_cast<const float4 *>(Qs + ((pb + i) & (kSmPairs - 1)) * kHeadDim + c * 8);
            const float4 qb = *reinterpret_cast<const float4 *>(Qs + ((pb + i) & (kSmPairs - 1)) * kHeadDim + c * 8 + 4);
            s[i] = fmaf(qa.x, k0, s[i]);
            s[i] = fmaf(qa.y, k1, s[i]);
            s[i] = fmaf(qa.z, k2, s[i]);
            s[i] = fmaf(qa.w, k3, s[i]);
            s[i] = fmaf(qb.x, k4, s[i]);
            s[i] = fmaf(qb.y, k5, s[i]);
            s[i] = fmaf(qb.z, k6, s[i]);
            s[i] = fmaf(qb.w, k7, s[i]);
          }
        }
#pragma unroll
        for (int i = 0; i < 8; ++i)
          if (pb + i < p_hi) Ps[(pb + i) * kSmPPitch + key] = (kpos <= pos_s[pb + i]) ? s[i] : -INFINITY;
      }
    }
    __syncthreads();

    // ---- phase 2: online softmax statistics, one warp per pair
    for (int pr = warp; pr < m; pr += kSmThreads / 32) {
      float4 sv = *reinterpret_cast<float4 *>(Ps + pr * kSmPPitch + lane * 4);
      float mx = fmaxf(fmaxf(sv.x, sv.y), fmaxf(sv.z, sv.w));
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, d));
      const float m_old = m_s[pr];
      const float m_new = fmaxf(m_old, mx);
      float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
      float alpha = 1.f;
      if (m_new > -INFINITY) {
        e.x = ex2_approx(sv.x - m_new);
        e.y = ex2_approx(sv.y - m_new);
        e.z = ex2_approx(sv.z - m_new);
        e.w = ex2_approx(sv.w - m_new);
        alpha = ex2_approx(m_old - m_new);
      }
      float sum = (e.x + e.y) + (e.z + e.w);
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
      *reinterpret_cast<float4 *>(Ps + pr * kSmPPitch + lane * 4) = e;
      if (lane == 0) {
        m_s[pr] = m_new;
        l_s[pr] = l_s[pr] * alpha + sum;
        a_s[pr] = alpha;
      }
    }
    __syncthreads();

    // ---- phase 3: O[pair][8 dims] = alpha * O + sum_key P[pair][key] * V[key][8 dims]
    {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const float al = a_s[pg + 16 * j];
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[j][i] *= al;
      }
      const int np = (m - pg + 15) >> 4;  // pairs pg + 16 j < m
      for (int k4 = 0; k4 < nkeys; k4 += 4) {
        float v[4][8];
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          uint4 vv = make_uint4(0, 0, 0, 0);  // keys past the visible range may hold anything: P = 0 there
          if (k4 + kk < nkeys) vv = *reinterpret_cast<const uint4 *>(vs + (k4 + kk) * kSmRowB + oc * 16);
          v[kk][0] = bf_lo_f(vv.x); v[kk][1] = bf_hi_f(vv.x); v[kk][2] = bf_lo_f(vv.y); v[kk][3] = bf_hi_f(vv.y);
          v[kk][4] = bf_lo_f(vv.z); v[kk][5] = bf_hi_f(vv.z); v[kk][6] = bf_lo_f(vv.w); v[kk][7] = bf_hi_f(vv.w);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (j < np) {
            const float4 pv = *reinterpret_cast<const float4 *>(Ps + (pg + 16 * j) * kSmPPitch + k4);
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              acc[j][i] = fmaf(pv.x, v[0][i], acc[j][i]);
              acc[j][i] = fmaf(pv.y, v[1][i], acc[j][i]);
              acc[j][i] = fmaf(pv.z, v[2][i], acc[j][i]);
              acc[j][i] = fmaf(pv.w, v[3][i], acc[j][i]);
            }
          }
        }
      }
    }
    __syncthreads();  // the stage and the P tile are free again
  }

  // ---- partial result of this split
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    float *o = part + (pg + 16 * j) * kHeadDim + oc * 8;
    *reinterpret_cast<float4 *>(o) = make_float4(acc[j][0], acc[j][1], acc[j][2], acc[j][3]);
    *reinterpret_cast<float4 *>(o + 4) = make_float4(acc[j][4], acc[j][5], acc[j][6], acc[j][7]);
  }
  if (tid < kSmPairs) {
    part[kSmPairs * kHeadDim + tid] = m_s[tid];
    part[kSmPairs * kHeadDim + kSmPairs + tid] = l_s[tid];
  }
}

// Combine the splits of one (slot, KV head) in the fixed order 0..splits-1, normalise, write bf16 O and LSE.
__global__ void __launch_bounds__(kSmThreads)
attn_small_merge_kernel(const SmallParams p) {
  const int slot = blockIdx.x, kvh = blockIdx.y;
  int req, r0, nr;
  if (!small_decode(p, slot, req, r0, nr)) return;
  const int g = p.group;
  const int pr = threadIdx.x >> 2, qd = threadIdx.x & 3;  // pair, quarter of the head dim
  if (pr >= nr * g) return;
  const float *part = p.part + (size_t)(slot * p.num_kv_heads + kvh) * p.splits * kSmPartFloats;
  float mx = -INFINITY;
  for (int s = 0; s < p.splits; ++s) mx = fmaxf(mx, part[(size_t)s * kSmPartFloats + kSmPairs * kHeadDim + pr]);
  float l = 0.f;
  float o[32];
#pragma unroll
  for (int i = 0; i < 32; ++i) o[i] = 0.f;
  for (int s = 0; s < p.splits; ++s) {
    const float *ps = part + (size_t)s * kSmPartFloats;
    const float ls = ps[kSmPairs * kHeadDim + kSmPairs + pr];
    if (ls == 0.f) continue;  // this split saw no key of the row
    const float w = ex2_approx(ps[kSmPairs * kHeadDim + pr] - mx);
    l = fmaf(ls, w, l);
    const float4 *src = reinterpret_cast<const float4 *>(ps + pr * kHeadDim + qd * 32);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float4 v = src[i];
      o[4 * i + 0] = fmaf(v.x, w, o[4 * i + 0]);
      o[4 * i + 1] = fmaf(v.y, w, o[4 * i + 1]);
      o[4 * i + 2] = fmaf(v.z, w, o[4 * i + 2]);
      o[4 * i + 3] = fmaf(v.w, w, o[4 * i + 3]);
    }
  }
  const int ri = pr / g, hh = pr - ri * g;
  const size_t out_row = (size_t)(r0 + ri) * p.num_q_heads + kvh * g + hh;
  const float inv = 1.f / l;
  uint4 *dst = reinterpret_cast<uint4 *>(p.out + out_row * kHeadDim + qd * 32);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint4 v;
    v.x = pack_bf16x2(o[8 * i + 0] * inv, o[8 * i + 1] * inv);
    v.y = pack_bf16x2(o[8 * i + 2] * inv, o[8 * i + 3] * inv);
    v.z = pack_bf16x2(o[8 * i + 4] * inv, o[8 * i + 5] * inv);
    v.w = pack_bf16x2(o[8 * i + 6] * inv, o[8 * i + 7] * inv);
    dst[i] = v;
  }
  // m is in the log2 domain of s * log2(e) / sqrt(d): natural-log normaliser = m * ln 2 + ln l
  if (p.lse && qd == 0) p.lse[out_row] = mx * 0.6931471805599453f + logf(l);
}

// Host-side plan shared by the workspace query and the launcher.
void small_plan(int total_rows, int num_reqs, int num_kv_heads, int group, int *rows_per_chunk, int *slots,
                int *splits) {
  const int rc = (kSmPairs - 1) / group > 0 ? (kSmPairs - 1) / group : 1;
  const int sl = (total_rows + rc - 1) / rc + num_reqs;  // >= sum_r ceil(n_r / rc)
  int sp = (2 * 148 + sl * num_kv_heads - 1) / (sl * num_kv_heads);  // about two CTAs per SM in total
  if (sp < 1) sp = 1;
  if (sp > 64) sp = 64;
  *rows_per_chunk = rc;
  *slots = sl;
  *splits = sp;
}

size_t small_ws_bytes(int num_reqs, int num_kv_heads, int group) {
  // the CUDA-core path is taken only when total_rows * group < 64 * num_reqs (see sx_sparse_attn):
  // slots <= total_rows + num_reqs, slots * Hkv * splits <= 2 * 148 + slots * Hkv
  const size_t rows_max = (size_t)64 * num_reqs / (group > 0 ? group : 1) + 1;
  const size_t slots = rows_max + num_reqs;
  return (2 * 148 + slots * num_kv_heads) * (size_t)kSmPartFloats * sizeof(float);
}

sx_status launch_attn_small(const sx_pool *pool, const sx_batch *b, const void *q, const int32_t *rows,
                            const int32_t *rows_off, int32_t total_rows, void *out, float *lse, float *part,
                            cudaStream_t st) {
  SmallParams p;
  p.q = reinterpret_cast<const __nv_bfloat16 *>(q);
  p.pool_k = reinterpret_cast<const uint4 *>(pool->k);
  p.pool_v = reinterpret_cast<const uint4 *>(pool->v);
  p.rows = rows;
  p.rows_off = rows_off;
  p.seq_len = b->seq_len;
  p.k_table = b->k_block_table;
  p.v_table = b->v_block_table;
  p.part = part;
  p.out = reinterpret_cast<__nv_bfloat16 *>(out);
  p.lse = lse;
  p.num_reqs = b->num_reqs;
  p.max_pages = b->max_pages_per_req;
  p.num_q_heads = pool->num_q_heads;
  p.num_kv_heads = pool->num_kv_heads;
  p.group = pool->num_q_heads / pool->num_kv_heads;
  p.scale_log2 = (float)(kLog2e / sqrt((double)kHeadDim));
  int slots;
  small_plan(total_rows, b->num_reqs, pool->num_kv_heads, p.group, &p.rows_per_chunk, &slots, &p.splits);
  cudaError_t e = cudaFuncSetAttribute(attn_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmSmemBytes);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "attn_small smem attr: %s", cudaGetErrorString(e));
  attn_small_kernel<<<dim3(p.splits, pool->num_kv_heads, slots), kSmThreads, kSmSmemBytes, st>>>(p);
  sx_status s = check_launch("attn_small_kernel");
  if (s != SX_OK) return s;
  attn_small_merge_kernel<<<dim3(slots, pool->num_kv_heads), kSmThreads, 0, st>>>(p);
  return check_launch("attn_small_merge_kernel");
}

}  // namespace sx
