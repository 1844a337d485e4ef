// sx_attn_small.cu -- stage (c) when GQA packing gives FEWER than 64 query rows per KV head:
//   O[R] = SparseAttn(Q[R], K_cur[1:T], V_cur[1:T], M_causal)          Alg. 1 l.546-548
// on the CUDA cores (BASELINE.json north_star: tensor-core tiles only where at least 64 (row, head) pairs
// share a KV head; below that the work is a K/V stream with a handful of dot products per key, bound by
// HBM for up to ~10 pairs and by the FMA pipe beyond).
//
// Split-KV ("flash-decoding") design, no tensor cores:
//   * a CTA owns one (request, chunk of rows, KV head, split of the key range); the m <= 64 (row, head)
//     pairs of the chunk share every K/V row it streams. Key tiles of 64 keys = 4 pages arrive through
//     16-byte cp.async copies (coalesced: 256 B per (page, head, row)) into a four-stage ring (three tiles,
//     ~100 KB, in flight per SM) with a padded row pitch of 272 B, so that "one thread per key" reads are
//     free of bank conflicts.
//   * phase 1 (QK^T): thread = (key, quarter of the pairs); the K row is unpacked from bf16 once per group
//     of 1/2/4/8 pairs, the fp32 queries (pre-multiplied by log2(e)/sqrt(d)) are broadcast reads.
//   * phase 2 (softmax): one warp per pair: row maximum / sum by warp shuffles, running (m, l) per pair.
//   * phase 3 (PV): thread = (8 output dims, group of 4 pairs, key slice): with few pairs the thread rows
//     that would idle split the keys of the tile instead; their partial O rows are added once at the end.
//   * every split writes (m, l, unnormalised O) to the workspace; a merge kernel combines the splits in a
//     fixed order (deterministic), normalises and writes bf16 O and the natural-log LSE.
#include <math.h>

#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

constexpr int kSmThreads = 256;
constexpr int kSmPairs = 64;     // pair slots per CTA (at most 63 are used by the dispatch rule, 64 by chunking)
constexpr int kSmKeys = 64;      // keys per tile = 4 pages
constexpr int kSmStages = 4;     // K/V ring: three tiles in flight while one is consumed
constexpr int kSmRowB = 272;     // bytes between consecutive K (or V) rows in shared memory (256 + 16 pad)
constexpr int kSmPPitch = 68;    // floats between consecutive KEYS of the S/P tile (layout [key][pair])
constexpr int kSmOffQ = 0;                                        // float [64 pairs][128]
constexpr int kSmOffKV = kSmOffQ + kSmPairs * kHeadDim * 4;       // stages x (K, V) x 64 rows x 272 B
constexpr int kSmStageB = 2 * kSmKeys * kSmRowB;
constexpr int kSmOffP = kSmOffKV + kSmStages * kSmStageB;         // float [64 keys][68]
constexpr int kSmOffStat = kSmOffP + kSmKeys * kSmPPitch * 4;     // m[64], l[64], alpha[64] float; pos[64] int
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
  int pairs_cap;            // pair slots per partial: 64 (attn_small_kernel) or 4 / 8 (attn_tiny_kernel)
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

// phase 1 for one thread: scores of G consecutive pairs against the thread's key (K row in shared memory)
template <int G>
__device__ __forceinline__ void small_qk(const uint4 *krow, const float *Qs, float *Pk, const int *pos_s, int pb,
                                         int p_hi, int kpos) {
  float s[G], s2[G];  // two accumulation chains per pair (dims 0-3 / 4-7 of every chunk)
#pragma unroll
  for (int i = 0; i < G; ++i) s[i] = s2[i] = 0.f;
#pragma unroll 4
  for (int c = 0; c < 16; ++c) {
    const uint4 kv = krow[c];
    const float k0 = bf_lo_f(kv.x), k1 = bf_hi_f(kv.x), k2 = bf_lo_f(kv.y), k3 = bf_hi_f(kv.y);
    const float k4 = bf_lo_f(kv.z), k5 = bf_hi_f(kv.z), k6 = bf_lo_f(kv.w), k7 = bf_hi_f(kv.w);
#pragma unroll
    for (int i = 0; i < G; ++i) {  // slots past p_hi read valid (zero or foreign) queries; never stored
      const float *qp = Qs + ((pb + i) & (kSmPairs - 1)) * kHeadDim + c * 8;
      const float4 qa = *reinterpret_cast<const float4 *>(qp);
      const float4 qb = *reinterpret_cast<const float4 *>(qp + 4);
      s[i] = fmaf(qa.x, k0, s[i]);
      s2[i] = fmaf(qb.x, k4, s2[i]);
      s[i] = fmaf(qa.y, k1, s[i]);
      s2[i] = fmaf(qb.y, k5, s2[i]);
      s[i] = fmaf(qa.z, k2, s[i]);
      s2[i] = fmaf(qb.z, k6, s2[i]);
      s[i] = fmaf(qa.w, k3, s[i]);
      s2[i] = fmaf(qb.w, k7, s2[i]);
    }
  }
#pragma unroll
  for (int i = 0; i < G; ++i) s[i] += s2[i];
#pragma unroll
  for (int i = 0; i < G; ++i)
    if (pb + i < p_hi) Pk[pb + i] = (kpos <= pos_s[pb + i]) ? s[i] : -INFINITY;
}

__global__ void __launch_bounds__(kSmThreads, 1)
attn_small_kernel(const SmallParams p) {
  extern __shared__ __align__(16) uint8_t sm[];
  float *Qs = reinterpret_cast<float *>(sm + kSmOffQ);
  float *Ps = reinterpret_cast<float *>(sm + kSmOffP);  // [key][pair], pitch kSmPPitch
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
  const int nt = pos_max / kSmKeys + 1;
  const int per = (nt + p.splits - 1) / p.splits;
  const int t_begin = split * per, t_end = min(nt, t_begin + per);
  float *part = p.part + ((size_t)(slot * p.num_kv_heads + kvh) * p.splits + split) * kSmPartFloats;

  if (t_begin >= t_end) {  // nothing to do for this split: neutral partial (O = 0 too: the merge reads it)
    for (int i = tid; i < kSmPairs * kHeadDim / 4; i += kSmThreads)
      reinterpret_cast<float4 *>(part)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
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

  // K/V tile t -> stage: thread copies chunk (tid & 15) of row (tid >> 4) of page j, j = 0..3.
  // Exactly one commit group per call (possibly empty) keeps the wait_group arithmetic uniform.
  auto load_tile = [&](int t) {
    if (t < t_end) {
      uint8_t *ks = sm + kSmOffKV + ((t - t_begin) % kSmStages) * kSmStageB;
      uint8_t *vs = ks + kSmKeys * kSmRowB;
      const int r16 = tid >> 4, c = tid & 15;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        int lp = t * 4 + j;
        if (lp > n_pages - 1) lp = n_pages - 1;  // beyond the sequence: any valid page (those keys are masked)
        const size_t e = (size_t)req * p.max_pages + lp;
        const size_t ko = ((size_t)p.k_table[e] * p.num_kv_heads + kvh) * (kPage * 16) + r16 * 16 + c;
        const size_t vo = ((size_t)p.v_table[e] * p.num_kv_heads + kvh) * (kPage * 16) + r16 * 16 + c;
        cp_async16(ks + (j * 16 + r16) * kSmRowB + c * 16, p.pool_k + ko);
        cp_async16(vs + (j * 16 + r16) * kSmRowB + c * 16, p.pool_v + vo);
      }
    }
    cp_async_commit();
  };

  // phase-3 ownership: 8 output dims (chunk oc) x 4 consecutive pairs (group pgrp) x every nks-th key (slice ks).
  // With few pairs the 16 thread rows split the KEYS of a tile instead of idling; their partial O rows are
  // added up once, after the last tile.
  const int oc = tid & 15, rest = tid >> 4;
  int npg = 1;
  while (npg * 4 < m) npg <<= 1;  // pair groups of 4, power of two <= 16
  const int nks = 16 / npg;
  const int pgrp = rest % npg, ks_id = rest / npg;
  float acc[4][8];
#pragma unroll
  for (int j = 0; j < 4; ++j)
#pragma unroll
    for (int i = 0; i < 8; ++i) acc[j][i] = 0.f;

  // phase-1 ownership: one key of the tile x one quarter of the pairs
  const int key1 = tid & 63, qtr = tid >> 6;
  const int cntq = (m + 3) >> 2;
  const int p_lo = min(m, qtr * cntq), p_hi = min(m, p_lo + cntq);

  load_tile(t_begin);
  load_tile(t_begin + 1);
  load_tile(t_begin + 2);
  for (int t = t_begin; t < t_end; ++t) {
    load_tile(t + 3);      // its stage was consumed at iteration t - 1
    cp_async_wait<3>();    // tile t has landed (groups complete in order)
    __syncthreads();
    const uint8_t *ks = sm + kSmOffKV + ((t - t_begin) % kSmStages) * kSmStageB;
    const uint8_t *vs = ks + kSmKeys * kSmRowB;
    const int nkeys = min(kSmKeys, pos_max + 1 - t * kSmKeys);  // keys of this tile any pair can see (< T)

    // ---- phase 1: S[key][pair] = <q_pair, k_key> (log2 domain), causal mask
    {
      const uint4 *krow = reinterpret_cast<const uint4 *>(ks + key1 * kSmRowB);
      float *Pk = Ps + key1 * kSmPPitch;
      const int kpos = t * kSmKeys + key1;
      const int cnt = p_hi - p_lo;
      if (cnt > 4) {
        for (int pb = p_lo; pb < p_hi; pb += 8) small_qk<8>(krow, Qs, Pk, pos_s, pb, p_hi, kpos);
      } else if (cnt > 2) {
        small_qk<4>(krow, Qs, Pk, pos_s, p_lo, p_hi, kpos);
      } else if (cnt > 1) {
        small_qk<2>(krow, Qs, Pk, pos_s, p_lo, p_hi, kpos);
      } else if (cnt > 0) {
        small_qk<1>(krow, Qs, Pk, pos_s, p_lo, p_hi, kpos);
      }
    }
    __syncthreads();

    // ---- phase 2: online softmax statistics, one warp per pair (lane = keys lane and lane + 32)
    for (int pr = warp; pr < m; pr += kSmThreads / 32) {
      const float s0 = Ps[lane * kSmPPitch + pr], s1 = Ps[(lane + 32) * kSmPPitch + pr];
      float mx = fmaxf(s0, s1);
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, d));
      const float m_old = m_s[pr];
      const float m_new = fmaxf(m_old, mx);
      float e0 = 0.f, e1 = 0.f, alpha = 1.f;
      if (m_new > -INFINITY) {
        e0 = ex2_approx(s0 - m_new);
        e1 = ex2_approx(s1 - m_new);
        alpha = ex2_approx(m_old - m_new);
      }
      float sum = e0 + e1;
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
      Ps[lane * kSmPPitch + pr] = e0;
      Ps[(lane + 32) * kSmPPitch + pr] = e1;
      if (lane == 0) {
        m_s[pr] = m_new;
        l_s[pr] = l_s[pr] * alpha + sum;
        a_s[pr] = alpha;
      }
    }
    __syncthreads();

    // ---- phase 3: O[pair][8 dims] = alpha * O + sum_key P[key][pair] * V[key][8 dims]
    {
      const float4 al = *reinterpret_cast<const float4 *>(a_s + pgrp * 4);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        acc[0][i] *= al.x;
        acc[1][i] *= al.y;
        acc[2][i] *= al.z;
        acc[3][i] *= al.w;
      }
      if (pgrp * 4 < m) {
        for (int k = ks_id; k < nkeys; k += nks) {  // keys past nkeys may hold anything (P = 0 there): skipped
          const uint4 vv = *reinterpret_cast<const uint4 *>(vs + k * kSmRowB + oc * 16);
          const float4 pv = *reinterpret_cast<const float4 *>(Ps + k * kSmPPitch + pgrp * 4);
          float v[8];
          v[0] = bf_lo_f(vv.x); v[1] = bf_hi_f(vv.x); v[2] = bf_lo_f(vv.y); v[3] = bf_hi_f(vv.y);
          v[4] = bf_lo_f(vv.z); v[5] = bf_hi_f(vv.z); v[6] = bf_lo_f(vv.w); v[7] = bf_hi_f(vv.w);
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            acc[0][i] = fmaf(pv.x, v[i], acc[0][i]);
            acc[1][i] = fmaf(pv.y, v[i], acc[1][i]);
            acc[2][i] = fmaf(pv.z, v[i], acc[2][i]);
            acc[3][i] = fmaf(pv.w, v[i], acc[3][i]);
          }
        }
      }
    }
    __syncthreads();  // the stage and the P tile are free again
  }
  cp_async_wait<0>();

  // ---- partial result of this split: add the key slices of a pair group in a fixed order
  float *red = reinterpret_cast<float *>(sm + kSmOffKV);  // [ks][4 npg pairs][128] fp32 = 32 KB, the ring is idle now
  if (nks > 1) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      float *o = red + ((size_t)ks_id * (npg * 4) + pgrp * 4 + j) * kHeadDim + oc * 8;
      *reinterpret_cast<float4 *>(o) = make_float4(acc[j][0], acc[j][1], acc[j][2], acc[j][3]);
      *reinterpret_cast<float4 *>(o + 4) = make_float4(acc[j][4], acc[j][5], acc[j][6], acc[j][7]);
    }
    __syncthreads();
  }
  if (ks_id == 0) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int pr = pgrp * 4 + j;
      float4 a = make_float4(acc[j][0], acc[j][1], acc[j][2], acc[j][3]);
      float4 b = make_float4(acc[j][4], acc[j][5], acc[j][6], acc[j][7]);
      for (int s = 1; s < nks; ++s) {
        const float *o = red + ((size_t)s * (npg * 4) + pr) * kHeadDim + oc * 8;
        const float4 x = *reinterpret_cast<const float4 *>(o), y = *reinterpret_cast<const float4 *>(o + 4);
        a.x += x.x; a.y += x.y; a.z += x.z; a.w += x.w;
        b.x += y.x; b.y += y.y; b.z += y.z; b.w += y.w;
      }
      float *o = part + pr * kHeadDim + oc * 8;
      *reinterpret_cast<float4 *>(o) = a;
      *reinterpret_cast<float4 *>(o + 4) = b;
    }
  }
  // pair groups beyond npg do not exist as threads: their (unused) O rows stay unwritten; the merge kernel
  // reads only pairs < m, all of which belong to a group < npg
  if (tid < kSmPairs) {
    part[kSmPairs * kHeadDim + tid] = m_s[tid];
    part[kSmPairs * kHeadDim + kSmPairs + tid] = l_s[tid];
  }
}

// Combine the splits of one (slot, KV head) in the fixed order 0..splits-1, normalise, write bf16 O and LSE.
__global__ void __launch_bounds__(kSmThreads)
attn_small_merge_kernel(const SmallParams p) {
  __shared__ float red_mx[kSmThreads];
  __shared__ float red_o[kSmThreads][33];  // o[32] + l per thread, padded
  const int slot = blockIdx.x, kvh = blockIdx.y;
  int req, r0, nr;
  if (!small_decode(p, slot, req, r0, nr)) return;
  const int g = p.group, cap = p.pairs_cap;
  const int part_floats = cap * (kHeadDim + 2);  // O[cap][128], m[cap], l[cap]
  // thread = (split group sg, pair pr, quarter qd of the head dim): with few pair slots the spare threads
  // walk the splits in parallel (nsg groups), so the chain of dependent loads stays short
  const int lanes = cap * 4, nsg = kSmThreads / lanes;
  const int sg = threadIdx.x / lanes, pq = threadIdx.x - sg * lanes;
  const int pr = pq >> 2, qd = pq & 3;
  const bool active = pr < nr * g;
  const float *part = p.part + (size_t)(slot * p.num_kv_heads + kvh) * p.splits * part_floats;
  float mx = -INFINITY;
  if (active)
    for (int s = sg; s < p.splits; s += nsg) mx = fmaxf(mx, part[(size_t)s * part_floats + cap * kHeadDim + pr]);
  red_mx[threadIdx.x] = mx;
  __syncthreads();
  for (int k = 0; k < nsg; ++k) mx = fmaxf(mx, red_mx[k * lanes + pq]);
  float l = 0.f;
  float o[32];
#pragma unroll
  for (int i = 0; i < 32; ++i) o[i] = 0.f;
  if (active) {
#pragma unroll 2
    for (int s = sg; s < p.splits; s += nsg) {  // no data-dependent branch: the loads of several splits overlap
      const float *ps = part + (size_t)s * part_floats;
      const float ls = ps[cap * kHeadDim + cap + pr];
      const float w = (ls == 0.f) ? 0.f : ex2_approx(ps[cap * kHeadDim + pr] - mx);  // 0: no key of the row seen
      l = fmaf(ls, w, l);
      const float4 *src = reinterpret_cast<const float4 *>(ps + pr * kHeadDim + qd * 32);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float4 v = __ldg(src + i);
        o[4 * i + 0] = fmaf(v.x, w, o[4 * i + 0]);
        o[4 * i + 1] = fmaf(v.y, w, o[4 * i + 1]);
        o[4 * i + 2] = fmaf(v.z, w, o[4 * i + 2]);
        o[4 * i + 3] = fmaf(v.w, w, o[4 * i + 3]);
      }
    }
  }
  if (nsg > 1) {  // add the split groups in a fixed order
#pragma unroll
    for (int i = 0; i < 32; ++i) red_o[threadIdx.x][i] = o[i];
    red_o[threadIdx.x][32] = l;
    __syncthreads();
    if (sg == 0) {
      for (int k = 1; k < nsg; ++k) {
#pragma unroll
        for (int i = 0; i < 32; ++i) o[i] += red_o[k * lanes + pq][i];
        l += red_o[k * lanes + pq][32];
      }
    }
  }
  if (!active || sg != 0) return;
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

// ---------------------------------------------------------------------------------------------------
// At most 8 (row, head) pairs per KV head (decode-like row sets): pure streaming, bound by HBM.
// No shared-memory staging and no block barriers in the loop: a warp reads two K rows per instruction
// (16 lanes x 16 B each), every lane keeps the 8 dims it loads of all M queries and M output rows in
// registers, dot products are finished by 4 shuffles inside the 16-lane half, and each half-warp runs its
// own online softmax. Warps of a CTA take alternate pages of the CTA's key split; half-warps, warps and
// splits are merged at the end (same partial format as above, pairs_cap = M).
// One CTA per SM (12 warps for M = 4, 8 for M = 8: the register file is the limit), one wave, so that the
// number of key splits - partials the merge kernel walks through - stays around 148 / Hkv.
template <int M>
__global__ void __launch_bounds__((M <= 4 ? 384 : 256), 1)
attn_tiny_kernel(const SmallParams p) {
  constexpr int kWarps = (M <= 4 ? 12 : 8), kTinyThreads = kWarps * 32;
  extern __shared__ __align__(16) uint8_t tiny_sm[];
  float (*red_o)[M][kHeadDim] = reinterpret_cast<float (*)[M][kHeadDim]>(tiny_sm);
  float (*red_m)[M] = reinterpret_cast<float (*)[M]>(tiny_sm + sizeof(float) * kWarps * M * kHeadDim);
  float (*red_l)[M] = red_m + kWarps;
  const int split = blockIdx.x, kvh = blockIdx.y, slot = blockIdx.z;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int hw = lane >> 4, c = lane & 15;  // half-warp = row of the pair of keys; 16-byte chunk of the row
  const int g = p.group;
  int req, r0, nr;
  if (!small_decode(p, slot, req, r0, nr)) return;
  const int m = nr * g;
  const int pos_max = p.rows ? p.rows[r0 + nr - 1] : (r0 + nr - 1 - p.rows_off[req]);
  const int n_pages = pos_max / kPage + 1;  // pages that hold a visible key
  const int per = (n_pages + p.splits - 1) / p.splits;
  const int pg_begin = split * per, pg_end = min(n_pages, pg_begin + per);
  float *part = p.part + ((size_t)(slot * p.num_kv_heads + kvh) * p.splits + split) * (M * (kHeadDim + 2));

  float q[M][8], acc[M][8], mr[M], lr[M];
  int pos[M];
#pragma unroll
  for (int i = 0; i < M; ++i) {
    mr[i] = -INFINITY;
    lr[i] = 0.f;
    pos[i] = -1;
#pragma unroll
    for (int d = 0; d < 8; ++d) q[i][d] = acc[i][d] = 0.f;
    if (i < m) {
      const int ri = i / g, hh = i - ri * g;
      pos[i] = p.rows ? p.rows[r0 + ri] : (r0 + ri - p.rows_off[req]);
      const uint4 v = *reinterpret_cast<const uint4 *>(p.q + ((size_t)(r0 + ri) * p.num_q_heads + kvh * g + hh) * kHeadDim + c * 8);
      q[i][0] = bf_lo_f(v.x) * p.scale_log2; q[i][1] = bf_hi_f(v.x) * p.scale_log2;
      q[i][2] = bf_lo_f(v.y) * p.scale_log2; q[i][3] = bf_hi_f(v.y) * p.scale_log2;
      q[i][4] = bf_lo_f(v.z) * p.scale_log2; q[i][5] = bf_hi_f(v.z) * p.scale_log2;
      q[i][6] = bf_lo_f(v.w) * p.scale_log2; q[i][7] = bf_hi_f(v.w) * p.scale_log2;
    }
  }

  for (int pg = pg_begin + warp; pg < pg_end; pg += kTinyThreads / 32) {
    const size_t e = (size_t)req * p.max_pages + pg;
    const uint4 *kp = p.pool_k + ((size_t)p.k_table[e] * p.num_kv_heads + kvh) * (kPage * 16);
    const uint4 *vp = p.pool_v + ((size_t)p.v_table[e] * p.num_kv_heads + kvh) * (kPage * 16);
#pragma unroll
    for (int r4 = 0; r4 < 2; ++r4) {  // 8 rows (4 instructions of 2 rows) per batch of loads
      uint4 kk[4], vv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int row = r4 * 8 + u * 2 + hw;
        kk[u] = __ldg(kp + row * 16 + c);
        vv[u] = __ldg(vp + row * 16 + c);
      }
      // scores of the 4 keys of this half-warp for every pair, then ONE online-softmax step per pair
      float sc[M][4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        float kf[8];
        kf[0] = bf_lo_f(kk[u].x); kf[1] = bf_hi_f(kk[u].x); kf[2] = bf_lo_f(kk[u].y); kf[3] = bf_hi_f(kk[u].y);
        kf[4] = bf_lo_f(kk[u].z); kf[5] = bf_hi_f(kk[u].z); kf[6] = bf_lo_f(kk[u].w); kf[7] = bf_hi_f(kk[u].w);
#pragma unroll
        for (int i = 0; i < M; ++i) {
          float s = 0.f;
#pragma unroll
          for (int d = 0; d < 8; ++d) s = fmaf(q[i][d], kf[d], s);
          sc[i][u] = s;
        }
      }
#pragma unroll
      for (int sh = 8; sh > 0; sh >>= 1)  // finish the dot products inside the half-warp
#pragma unroll
        for (int i = 0; i < M; ++i)
#pragma unroll
          for (int u = 0; u < 4; ++u) sc[i][u] += __shfl_xor_sync(0xffffffffu, sc[i][u], sh);
      const int kpos0 = pg * kPage + r4 * 8 + hw;  // key u of this half-warp sits at kpos0 + 2 u
      float vf[4][8];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        vf[u][0] = bf_lo_f(vv[u].x); vf[u][1] = bf_hi_f(vv[u].x); vf[u][2] = bf_lo_f(vv[u].y); vf[u][3] = bf_hi_f(vv[u].y);
        vf[u][4] = bf_lo_f(vv[u].z); vf[u][5] = bf_hi_f(vv[u].z); vf[u][6] = bf_lo_f(vv[u].w); vf[u][7] = bf_hi_f(vv[u].w);
      }
#pragma unroll
      for (int i = 0; i < M; ++i) {
        float mx = -INFINITY;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          if (kpos0 + 2 * u > pos[i]) sc[i][u] = -INFINITY;  // causal mask (also hides rows past the sequence)
          mx = fmaxf(mx, sc[i][u]);
        }
        if (mx > -INFINITY) {  // uniform inside a half-warp
          const float m_new = fmaxf(mr[i], mx);
          const float alpha = ex2_approx(mr[i] - m_new);
          mr[i] = m_new;
          float pe[4], ps = 0.f;
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            pe[u] = ex2_approx(sc[i][u] - m_new);
            ps += pe[u];
          }
          lr[i] = fmaf(lr[i], alpha, ps);
#pragma unroll
          for (int d = 0; d < 8; ++d) {
            float a = acc[i][d] * alpha;
#pragma unroll
            for (int u = 0; u < 4; ++u) a = fmaf(pe[u], (pe[u] == 0.f) ? 0.f : vf[u][d], a);
            acc[i][d] = a;
          }
        }
      }
    }
  }

  // ---- merge the two half-warps, then the 4 warps, in fixed order
#pragma unroll
  for (int i = 0; i < M; ++i) {
    const float mo = __shfl_xor_sync(0xffffffffu, mr[i], 16), lo = __shfl_xor_sync(0xffffffffu, lr[i], 16);
    const float mn = fmaxf(mr[i], mo);
    const float wa = (mr[i] == -INFINITY) ? 0.f : ex2_approx(mr[i] - mn);
    const float wb = (mo == -INFINITY) ? 0.f : ex2_approx(mo - mn);
#pragma unroll
    for (int d = 0; d < 8; ++d) {
      const float ao = __shfl_xor_sync(0xffffffffu, acc[i][d], 16);
      acc[i][d] = acc[i][d] * wa + ao * wb;
    }
    lr[i] = lr[i] * wa + lo * wb;
    mr[i] = mn;
    if (hw == 0) {
#pragma unroll
      for (int d = 0; d < 8; ++d) red_o[warp][i][c * 8 + d] = acc[i][d];
      if (c == 0) {
        red_m[warp][i] = mr[i];
        red_l[warp][i] = lr[i];
      }
    }
  }
  __syncthreads();
  for (int idx = threadIdx.x; idx < M * kHeadDim; idx += kTinyThreads) {
    const int i = idx / kHeadDim, d = idx - i * kHeadDim;
    float mn = -INFINITY;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) mn = fmaxf(mn, red_m[w][i]);
    float o = 0.f, l = 0.f;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
      const float wt = (red_m[w][i] == -INFINITY) ? 0.f : ex2_approx(red_m[w][i] - mn);
      o = fmaf(red_o[w][i][d], wt, o);
      l = fmaf(red_l[w][i], wt, l);
    }
    part[i * kHeadDim + d] = o;
    if (d == 0) {
      part[M * kHeadDim + i] = mn;
      part[M * kHeadDim + M + i] = l;
    }
  }
}

// Host-side plan shared by the workspace query and the launcher.
void small_plan(int total_rows, int num_reqs, int num_kv_heads, int group, int *rows_per_chunk, int *slots,
                int *splits) {
  const int rc = (kSmPairs - 1) / group > 0 ? (kSmPairs - 1) / group : 1;
  const int sl = (total_rows + rc - 1) / rc + num_reqs;  // >= sum_r ceil(n_r / rc)
  // one CTA per SM (190 KB of shared memory): the working CTAs should fill ONE wave of 148 SMs, never spill
  // a few CTAs into a second one. The host does not know how many slots are non-empty; estimate from the rows.
  const int est = (total_rows + rc - 1) / rc > num_reqs ? (total_rows + rc - 1) / rc : num_reqs;
  int sp = 148 / (est * num_kv_heads);
  if (sp < 1) sp = 1;
  if (sp > 64) sp = 64;
  *rows_per_chunk = rc;
  *slots = sl;
  *splits = sp;
}

constexpr int kTinyTargetCtas = 148;  // one CTA per SM, one wave

size_t small_ws_bytes(int num_reqs, int num_kv_heads, int group) {
  // the CUDA-core path is taken only when total_rows * group < 64 * num_reqs (see sx_sparse_attn):
  // grid slots <= 2 * est (est >= rows / rc and est >= num_reqs) and splits <= 148 / (est * Hkv), so
  // slots * Hkv * splits <= max(2 * 148, slots * Hkv)
  const size_t rows_max = (size_t)64 * num_reqs / (group > 0 ? group : 1) + 1;
  const size_t slots = rows_max + num_reqs;
  const size_t general = (2 * 148 + slots * num_kv_heads) * (size_t)kSmPartFloats * sizeof(float);
  // attn_tiny_kernel: at most kTinyTargetCtas + slots * Hkv partials of 8 pairs
  const size_t tiny = ((size_t)kTinyTargetCtas + slots * num_kv_heads) * 8 * (kHeadDim + 2) * sizeof(float);
  return general > tiny ? general : tiny;
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
  // Decode-like row sets (on average at most 8 pairs per KV head): streaming kernel, registers only.
  if (p.group <= 8 && (int64_t)total_rows * p.group <= (int64_t)8 * b->num_reqs) {
    const int M = (p.group <= 4 && (int64_t)total_rows * p.group <= (int64_t)4 * b->num_reqs) ? 4 : 8;
    p.pairs_cap = M;
    p.rows_per_chunk = M / p.group;
    const int est = (total_rows + p.rows_per_chunk - 1) / p.rows_per_chunk > b->num_reqs
                        ? (total_rows + p.rows_per_chunk - 1) / p.rows_per_chunk : b->num_reqs;
    const int slots_t = (total_rows + p.rows_per_chunk - 1) / p.rows_per_chunk + b->num_reqs;
    int sp = kTinyTargetCtas / (est * pool->num_kv_heads);
    const int sp_max = (b->max_seq_len / kPage) / 16 > 1 ? (b->max_seq_len / kPage) / 16 : 1;  // >= 16 pages per split
    if (sp > sp_max) sp = sp_max;
    if (sp < 1) sp = 1;
    p.splits = sp;
    const dim3 grid(p.splits, pool->num_kv_heads, slots_t);
    const int warps = M == 4 ? 12 : 8;
    const int smem = warps * M * (kHeadDim + 2) * (int)sizeof(float);
    cudaError_t e = M == 4 ? cudaFuncSetAttribute(attn_tiny_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)
                           : cudaFuncSetAttribute(attn_tiny_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "attn_tiny smem attr: %s", cudaGetErrorString(e));
    if (M == 4)
      attn_tiny_kernel<4><<<grid, warps * 32, smem, st>>>(p);
    else
      attn_tiny_kernel<8><<<grid, warps * 32, smem, st>>>(p);
    sx_status s = check_launch("attn_tiny_kernel");
    if (s != SX_OK) return s;
    attn_small_merge_kernel<<<dim3(slots_t, pool->num_kv_heads), kSmThreads, 0, st>>>(p);
    return check_launch("attn_small_merge_kernel");
  }
  p.pairs_cap = kSmPairs;
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
