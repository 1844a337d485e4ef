// sx_select.cu -- stage (b), second half: head aggregation of the column sums,
// S_key = TopK({s_j}, k) over the cached positions (Eq. 3; DESIGN.md readings
// A7/A8: candidates = I_reuse, order = score descending then position ascending) and the
// recompute set R = I_nr U S_key (Alg. 1 l.537-539), both emitted in ascending position order.
//
// One CTA per request. Scores are non-negative fp32, so their bit patterns order like unsigned
// integers: 4-pass 8-bit radix select finds the k-th largest pattern, one ordered pass with block
// scans then emits S_key and R. Integer atomics only (deterministic).
#include <cooperative_groups.h>

#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

constexpr int kSelThreads = 1024;
constexpr int kSelWarps = kSelThreads / 32;

// exclusive block scan of three small counters at once; returns exclusive prefixes, adds totals to base
struct Scan3 {
  int a, b, c;
};

__device__ __forceinline__ Scan3 block_scan3(bool fa, bool fb, bool fc, int (*warp_tot)[kSelWarps], int *tot) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const unsigned ba = __ballot_sync(0xffffffffu, fa), bb = __ballot_sync(0xffffffffu, fb),
                 bc = __ballot_sync(0xffffffffu, fc);
  const unsigned lt = (1u << lane) - 1u;
  if (lane == 0) {
    warp_tot[0][w] = __popc(ba);
    warp_tot[1][w] = __popc(bb);
    warp_tot[2][w] = __popc(bc);
  }
  __syncthreads();
  if (w < 3) {  // warp w scans counter w over the 32 warp totals
    int v = warp_tot[w][lane];
    int x = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      int y = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += y;
    }
    warp_tot[w][lane] = x - v;  // exclusive
    if (lane == 31) tot[w] = x;
  }
  __syncthreads();
  Scan3 r;
  r.a = warp_tot[0][w] + __popc(ba & lt);
  r.b = warp_tot[1][w] + __popc(bb & lt);
  r.c = warp_tot[2][w] + __popc(bc & lt);
  return r;
}

// Head aggregation: scores[j] = sum over KV heads of the per-head column sums, fixed order.
__global__ void __launch_bounds__(256)
score_sum_kernel(int num_kv_heads, int total_tokens, const float *__restrict__ partial, float *__restrict__ scores) {
  griddep_launch();  // programmatic dependent launch: the next kernel may become resident now ...
  griddep_wait();    // ... and this one touches global memory only after its predecessor has completed
  const int j = blockIdx.x * 256 + threadIdx.x;
  if (j >= total_tokens) return;
  float s = 0.f;
  for (int h = 0; h < num_kv_heads; ++h) s += ld_dep(partial + (size_t)h * total_tokens + j);  // (colsum's output)
  scores[j] = s;
}

__global__ void __launch_bounds__(kSelThreads)
select_kernel(int num_kv_heads, int total_tokens, const int32_t *__restrict__ seq_len,
              const int32_t *__restrict__ tok_off, const int32_t *__restrict__ new_off,
              const int32_t *__restrict__ new_idx, const float *__restrict__ partial,
              const int32_t *__restrict__ sel_off, const int32_t *__restrict__ rows_off, float *__restrict__ scores,
              int32_t *__restrict__ sel_idx, int32_t *__restrict__ rows_R, int ov_tokens, int tail_tokens,
              const sx_segment *__restrict__ segs, int num_segments, int32_t *__restrict__ rows_cnt,
              int *__restrict__ scratch) {
  // gridDim.y > 1 (cooperative launch, long requests): the positions of a request are cut into gridDim.y
  // slices, one CTA each; digit histograms and the per-slice counts of the ordered emission meet in `scratch`
  // (zeroed by the launcher) and the CTAs of the grid synchronise between the phases.
  namespace cg = cooperative_groups;
  griddep_launch();
  griddep_wait();  // (a no-op under the cooperative launch, which does not use programmatic serialisation)
  const int ns = gridDim.y, sl = blockIdx.y;
  int *ghist = scratch + (size_t)blockIdx.x * (4 * 256 + 4 * 64);  // [4 passes][256] then [4 counters][64 slices]
  int *gcnt = ghist + 4 * 256;
  extern __shared__ uint32_t is_new[];  // bitmaps over positions: I_nr, forced rows (S_ov U S_tail), candidates
  __shared__ int hist[256];
  __shared__ int warp_tot[3][kSelWarps];
  __shared__ int tot[3];
  __shared__ uint32_t sh_prefix;
  __shared__ int sh_remaining;
  __shared__ int sh_ncand;

  const int req = blockIdx.x;
  const int T = seq_len[req];
  const int off = tok_off[req];
  // slice [jb, je) of this CTA, a multiple of 128 positions long (the emission walks 4 x 32 at a time)
  const int slen = (((T + ns - 1) / ns) + 127) & ~127;
  const int jb = min(T, sl * slen), je = min(T, jb + slen);
  const int n0 = new_off[req], nn = new_off[req + 1] - n0;
  const int words = (T + 31) >> 5;
  int k = sel_off[req + 1] - sel_off[req];
  // Candidates of Eq. (3) = I_reuse = the positions covered by this request's segments. Positions that are neither
  // new nor in a segment are prefix-cache hits (Alg. 1 l.501: "excluded from the current prefill computation"):
  // visible as keys, never candidates, never in S_ov / S_tail, never query rows.
  uint32_t *forced = is_new + words;  // S_ov U S_tail (Alg. 1 l.535-536), cached positions only
  uint32_t *cand = forced + words;    // I_reuse
  for (int i = threadIdx.x; i < 3 * words; i += kSelThreads) is_new[i] = 0u;
  if (threadIdx.x == 0) {
    sh_ncand = 0;
    sh_prefix = 0u;
    sh_remaining = 0;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < nn; i += kSelThreads) {
    int p = new_idx[n0 + i];
    atomicOr(&is_new[p >> 5], 1u << (p & 31));
  }
  for (int m = 0; m < num_segments; ++m) {  // segment bounds are multiples of 16: half a bitmap word per page
    if (segs[m].req != req) continue;
    const int p0 = segs[m].new_pos;
    for (int c = threadIdx.x; c < segs[m].len / kPage; c += kSelThreads) {
      const int q = p0 + c * kPage;
      if (q < T) atomicOr(&cand[q >> 5], 0xFFFFu << (q & 31));
    }
  }
  // k is clamped to the number of candidates that really exist: bits of the candidate bitmap below T (a segment
  // whose last page straddles seq_len, or overlapping segments, make sum(len) an overestimate)
  __syncthreads();
  {
    int c = 0;
    for (int i = threadIdx.x; i < words; i += kSelThreads) {
      uint32_t wv = cand[i];
      if (i == words - 1 && (T & 31)) wv &= (1u << (T & 31)) - 1u;
      c += __popc(wv);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(&sh_ncand, c);
  }
  __syncthreads();
  if (k > sh_ncand) k = sh_ncand;
  if (k < 0) k = 0;
  if (ov_tokens > 0 || tail_tokens > 0) {
    __syncthreads();
    // overflow (Alg. 1 l.535): every maximal interval [a, b] of I_nr grows by one block
    // on both sides; only positions that are not new themselves are recorded
    for (int i = threadIdx.x; i < nn; i += kSelThreads) {
      const int p = new_idx[n0 + i];
      if (i == 0 || new_idx[n0 + i - 1] != p - 1)
        for (int q = max(0, p - ov_tokens); q < p; ++q)
          if ((cand[q >> 5] >> (q & 31)) & 1u) atomicOr(&forced[q >> 5], 1u << (q & 31));
      if (i == nn - 1 || new_idx[n0 + i + 1] != p + 1)
        for (int q = p + 1; q <= min(T - 1, p + ov_tokens); ++q)
          if ((cand[q >> 5] >> (q & 31)) & 1u) atomicOr(&forced[q >> 5], 1u << (q & 31));
    }
    // tail fallback (Alg. 1 l.536): the prompt ends inside a reused segment -> its last
    // tail_tokens positions are recomputed
    if (tail_tokens > 0 && ((cand[(T - 1) >> 5] >> ((T - 1) & 31)) & 1u)) {
      int seg_start = 0;  // start of the reused segment that contains position T - 1
      for (int m = 0; m < num_segments; ++m)
        if (segs[m].req == req && segs[m].new_pos <= T - 1 && T - 1 < segs[m].new_pos + segs[m].len)
          seg_start = segs[m].new_pos;
      for (int q = max(seg_start, T - tail_tokens) + threadIdx.x; q < T; q += kSelThreads)
        atomicOr(&forced[q >> 5], 1u << (q & 31));
    }
  }
  // head aggregation in fixed order kvh = 0..Hkv-1 (global score across heads)
  // (the head sum of PAPER.md:225 was formed by score_sum_kernel, all SMs, before this launch)
  __syncthreads();

  // ---- radix select: bit pattern of the k-th largest candidate score
  uint32_t prefix = 0, mask = 0;
  int remaining = k;
  for (int pass = 3; pass >= 0; --pass) {  // (every CTA of the grid runs every pass: the grid syncs are collective)
    const int shift = pass * 8;
    for (int i = threadIdx.x; i < 256; i += kSelThreads) hist[i] = 0;
    __syncthreads();
    if (k > 0) {
      // all 32 lanes stay in the loop (warp-aggregated histogram: the top digits of the scores take few
      // distinct values, a plain shared-memory atomic per lane would serialise 32-fold)
      for (int j0 = jb; j0 < je; j0 += 8 * kSelThreads) {
        uint32_t u[8];  // eight independent loads in flight per thread: the pass is bound by load latency
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const int j = j0 + q * kSelThreads + threadIdx.x;
          u[q] = j < je ? __float_as_uint(ld_dep(scores + off + j)) : 0u;  // (score_sum's output)
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const int j = j0 + q * kSelThreads + threadIdx.x;
          int bin = -1;
          if (j < je && ((cand[j >> 5] >> (j & 31)) & 1u) && (u[q] & mask) == prefix)
            bin = (int)((u[q] >> shift) & 255u);
          const unsigned peers = __match_any_sync(0xffffffffu, bin);
          if (bin >= 0 && (threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&hist[bin], __popc(peers));
        }
      }
    }
    __syncthreads();
    if (ns > 1) {  // add up the slices of the request (integer atomics: order does not matter), then read the sum
      for (int i = threadIdx.x; i < 256; i += kSelThreads)
        if (hist[i]) atomicAdd(&ghist[pass * 256 + i], hist[i]);
      __threadfence();
      cg::this_grid().sync();
      for (int i = threadIdx.x; i < 256; i += kSelThreads) hist[i] = __ldcg(&ghist[pass * 256 + i]);
      __syncthreads();
    }
    if (k > 0) {
      if (threadIdx.x < 32) {
        // bins from high to low; lane l owns bins [255-8l-7, 255-8l]
        const int lane = threadIdx.x;
        int c[8], sum = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          c[i] = hist[255 - (lane * 8 + i)];
          sum += c[i];
        }
        int incl = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          int y = __shfl_up_sync(0xffffffffu, incl, d);
          if (lane >= d) incl += y;
        }
        int before = incl - sum;  // candidates in bins above this lane's bins
        if (before < remaining && remaining <= incl) {
          int acc = before;
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            if (acc < remaining && remaining <= acc + c[i]) {
              sh_prefix = prefix | ((uint32_t)(255 - (lane * 8 + i)) << shift);
              sh_remaining = remaining - acc;
            }
            acc += c[i];
          }
        }
      }
      __syncthreads();
      prefix = sh_prefix;
      remaining = sh_remaining;
      mask |= 255u << shift;
    }
    __syncthreads();
  }
  // prefix = threshold pattern; `remaining` = how many candidates equal to it are taken (lowest positions)
  const uint32_t thr = prefix;
  const int take_eq = (k > 0) ? remaining : 0;

  // ---- ordered emission. Every warp owns one contiguous range of positions and walks it 32 at a time
  // (coalesced); ranks inside a warp come from ballots, ranks across warps from one 32-entry scan per phase:
  //   A: equals of the threshold per warp -> which of them are taken (lowest positions first, reading A8)
  //   B: |S_key| and |R| per warp          C: write S_key and R in ascending position order
  // (three cheap passes over L2-resident scores instead of a block-wide scan per 1024 positions)
  // (extended selection: rows_R is the workspace array rows_tmp [total_tokens], where request r owns the T_r
  // slots behind tok_off[r] -- always enough, whatever capacities the caller passed)
  const int so = sel_off[req], ro = rows_cnt ? off : rows_off[req];
  const int cap_r = min(rows_off[req + 1] - rows_off[req], T);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  const int seg = ((((je - jb) + kSelWarps - 1) / kSelWarps) + 127) & ~127;  // positions per warp, multiple of 32 * kB
  const int j_lo = min(je, jb + w * seg), j_hi = min(je, j_lo + seg);
  // counter c of the slices before this one (slice totals meet in gcnt[c][slice]); the grid sync is collective
  auto slice_base = [&](int c, int mine_total, int *all_total) -> int {
    if (ns == 1) {
      if (all_total) *all_total = mine_total;
      return 0;
    }
    if (threadIdx.x == 0) gcnt[c * 64 + sl] = mine_total;
    __threadfence();
    cg::this_grid().sync();
    int b0 = 0, all = 0;
    for (int i = 0; i < ns; ++i) {
      const int v = __ldcg(&gcnt[c * 64 + i]);
      if (i < sl) b0 += v;
      all += v;
    }
    if (all_total) *all_total = all;
    return b0;
  };
  constexpr int kB = 4;  // groups of 32 positions whose score loads are issued together
  auto load4 = [&](int j0, uint32_t (&u)[kB]) {
#pragma unroll
    for (int q = 0; q < kB; ++q) {
      const int j = j0 + q * 32 + lane;
      u[q] = j < j_hi ? __float_as_uint(ld_dep(scores + off + j)) : 0u;
    }
  };
  auto flags = [&](int j, uint32_t u, bool &isn, bool &gt, bool &eq, bool &frc) {
    isn = gt = eq = frc = false;
    if (j < j_hi) {
      isn = (is_new[j >> 5] >> (j & 31)) & 1u;
      frc = (forced[j >> 5] >> (j & 31)) & 1u;
      if (k > 0 && ((cand[j >> 5] >> (j & 31)) & 1u)) {
        gt = u > thr;
        eq = u == thr;
      }
    }
  };
  // exclusive scan of one per-warp counter over the 32 warps (all threads get their warp's base)
  auto warp_base = [&](int mine, int *total) -> int {
    __syncthreads();
    if (lane == 0) warp_tot[0][w] = mine;
    __syncthreads();
    if (w == 0) {
      const int v = warp_tot[0][lane];
      int x = v;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, d);
        if (lane >= d) x += y;
      }
      warp_tot[1][lane] = x - v;
      if (lane == 31) tot[0] = x;
    }
    __syncthreads();
    if (total) *total = tot[0];
    return warp_tot[1][w];
  };
  bool isn, gt, eq, frc;
  int n_eq = 0;
  uint32_t ub[kB];
  for (int j0 = j_lo; j0 < j_hi; j0 += 32 * kB) {
    load4(j0, ub);
#pragma unroll
    for (int q = 0; q < kB; ++q) {
      flags(j0 + q * 32 + lane, ub[q], isn, gt, eq, frc);
      n_eq += __popc(__ballot_sync(0xffffffffu, eq));
    }
  }
  int cta_eq = 0;
  int eq_base = warp_base(n_eq, &cta_eq);
  eq_base += slice_base(0, cta_eq, nullptr);
  int n_sel = 0, n_r = 0, run_eq = eq_base;
  for (int j0 = j_lo; j0 < j_hi; j0 += 32 * kB) {
    load4(j0, ub);
#pragma unroll
    for (int q = 0; q < kB; ++q) {
      flags(j0 + q * 32 + lane, ub[q], isn, gt, eq, frc);
      const unsigned be = __ballot_sync(0xffffffffu, eq);
      const bool sel = gt || (eq && run_eq + __popc(be & lt) < take_eq);
      run_eq += __popc(be);
      n_sel += __popc(__ballot_sync(0xffffffffu, sel));
      n_r += __popc(__ballot_sync(0xffffffffu, sel || isn || frc));  // R = I_nr U S_key U S_ov U S_tail
    }
  }
  int cta_sel = 0, cta_r = 0, total_r = 0;
  int sel_base = warp_base(n_sel, &cta_sel);
  int r_base = warp_base(n_r, &cta_r);
  if (ns > 1 && threadIdx.x == 0) gcnt[1 * 64 + sl] = cta_sel;  // rides on the grid sync of the next call
  r_base += slice_base(2, cta_r, &total_r);
  if (ns > 1)
    for (int i = 0; i < sl; ++i) sel_base += __ldcg(&gcnt[1 * 64 + i]);
  int run_sel = sel_base, run_r = r_base;
  run_eq = eq_base;
  for (int j0 = j_lo; j0 < j_hi; j0 += 32 * kB) {
    load4(j0, ub);
#pragma unroll
    for (int q = 0; q < kB; ++q) {
      const int j = j0 + q * 32 + lane;
      flags(j, ub[q], isn, gt, eq, frc);
      const unsigned be = __ballot_sync(0xffffffffu, eq);
      const bool sel = gt || (eq && run_eq + __popc(be & lt) < take_eq);
      run_eq += __popc(be);
      const bool in_r = sel || isn || frc;
      const unsigned bs = __ballot_sync(0xffffffffu, sel), br = __ballot_sync(0xffffffffu, in_r);
      if (sel) sel_idx[so + run_sel + __popc(bs & lt)] = j;
      const int rr = run_r + __popc(br & lt);
      if (in_r && rr < cap_r) rows_R[ro + rr] = j;
      run_sel += __popc(bs);
      run_r += __popc(br);
    }
  }
  if (rows_cnt && threadIdx.x == 0 && sl == 0) rows_cnt[req] = min(total_r, cap_r);
}

// Extended selection only: per-request row lists sit in the T_r-sized slots of `tmp` (at tok_off[r]); pack them into one
// CSR (rows_R, rows_off_out) so that the scatter and attention stages take them unchanged.
__global__ void __launch_bounds__(kSelThreads)
compact_rows_kernel(int num_reqs, const int32_t *__restrict__ tok_off, const int32_t *__restrict__ cnt,
                    const int32_t *__restrict__ tmp, int32_t *__restrict__ rows_R, int32_t *__restrict__ rows_off_out) {
  griddep_launch();
  griddep_wait();
  int out = 0;
  for (int r = 0; r < num_reqs; ++r) {
    const int n = ld_dep(cnt + r), src = tok_off[r];  // (cnt, tmp: select_kernel's outputs)
    for (int i = threadIdx.x; i < n; i += kSelThreads) rows_R[out + i] = ld_dep(tmp + src + i);
    if (threadIdx.x == 0) rows_off_out[r] = out;
    out += n;
  }
  if (threadIdx.x == 0) rows_off_out[num_reqs] = out;
}

size_t select_scratch_bytes(const sx_batch *b) { return sizeof(int) * (size_t)b->num_reqs * (4 * 256 + 4 * 64); }

sx_status launch_select(const sx_pool *pool, const sx_batch *b, const float *partial, const int32_t *sel_off,
                        const int32_t *rows_off, float *scores, int32_t *sel_idx, int32_t *rows_R, int ov_blocks,
                        int tail_tokens, int32_t *rows_tmp, int32_t *rows_cnt, int32_t *rows_off_out, int *scratch,
                        cudaStream_t st) {
  size_t smem = 3 * sizeof(uint32_t) * (size_t)((b->max_seq_len + 31) / 32);
  if (smem > 200 * 1024) return set_error(SX_ERR_UNSUPPORTED, "max_seq_len %d too large for the select bitmaps", b->max_seq_len);
  if (smem > 40 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "select smem attr: %s", cudaGetErrorString(e));
  }
  cudaError_t le = launch_pdl(score_sum_kernel, dim3((b->total_tokens + 255) / 256), dim3(256), 0, st, 1,
                              pool->num_kv_heads, b->total_tokens, partial, scores);
  if (le != cudaSuccess) return set_error(SX_ERR_CUDA, "score_sum launch: %s", cudaGetErrorString(le));
  sx_status s0 = check_launch("score_sum_kernel");
  if (s0 != SX_OK) return s0;
  const bool ex = rows_off_out != nullptr;  // extended: variable |R|, slots of capacity rows_off, then compaction
  // Long requests: several CTAs per request (cooperative launch: every CTA must be resident, one per SM).
  int ns = 1;
  if (b->max_seq_len >= 4096 && b->num_reqs <= 74) {
    ns = (b->max_seq_len + 4095) / 4096;
    if (ns > 148 / b->num_reqs) ns = 148 / b->num_reqs;
    if (ns > 32) ns = 32;
  }
  int num_kv = pool->num_kv_heads, total_tokens = b->total_tokens, ov_tokens = ov_blocks * kPage, nseg = b->num_segments;
  const int32_t *seq_len = b->seq_len, *tok_off = b->tok_off, *new_off = b->new_off, *new_idx = b->new_idx;
  int32_t *rows_dst = ex ? rows_tmp : rows_R, *cnt = ex ? rows_cnt : nullptr;
  const sx_segment *segs = b->segments;
  if (ns > 1) {
    cudaError_t e = cudaMemsetAsync(scratch, 0, select_scratch_bytes(b), st);
    if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "select scratch memset: %s", cudaGetErrorString(e));
    void *args[] = {&num_kv, &total_tokens, &seq_len, &tok_off, &new_off, &new_idx, &partial, &sel_off, &rows_off,
                    &scores, &sel_idx, &rows_dst, &ov_tokens, &tail_tokens, &segs, &nseg, &cnt, &scratch};
    e = cudaLaunchCooperativeKernel(reinterpret_cast<void *>(select_kernel), dim3(b->num_reqs, ns), dim3(kSelThreads),
                                    args, smem, st);
    if (e != cudaSuccess) {
      cudaGetLastError();
      ns = 1;  // cooperative launch not possible here (e.g. too few free SMs): one CTA per request
    }
  }
  if (ns == 1) {
    le = launch_pdl(select_kernel, dim3(b->num_reqs, 1), dim3(kSelThreads), smem, st, 1, num_kv, total_tokens, seq_len,
                    tok_off, new_off, new_idx, partial, sel_off, rows_off, scores, sel_idx, rows_dst, ov_tokens,
                    tail_tokens, segs, nseg, cnt, scratch);
    if (le != cudaSuccess) return set_error(SX_ERR_CUDA, "select launch: %s", cudaGetErrorString(le));
  }
  sx_status s = check_launch("select_kernel");
  if (s != SX_OK || !ex) return s;
  le = launch_pdl(compact_rows_kernel, dim3(1), dim3(kSelThreads), 0, st, 1, b->num_reqs, b->tok_off,
                  (const int32_t *)rows_cnt, (const int32_t *)rows_tmp, rows_R, rows_off_out);
  if (le != cudaSuccess) return set_error(SX_ERR_CUDA, "compact launch: %s", cudaGetErrorString(le));
  return check_launch("compact_rows_kernel");
}

}  // namespace sx
