// sx_split_merge.cuh -- key-split bookkeeping shared by the attention kernels that cut the key range of a row set
// into splits (sx_attn.cu, sx_attn_stream.cu): arrival words in the workspace and the fixed-order merge.
#pragma once
#include <math.h>

#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

// Rendezvous of the key splits of one (request, KV head, row pair) on a workspace word that the host never
// zeroes. The word holds (kSplitTag << 8 | count); anything else is memory that no launch has used yet and counts
// as zero. Every split ARRIVES once its partial result is written (count 1 .. splits), waits until all have
// arrived, merges its share of the (row, head) pairs -- each pair in the fixed order 0 .. splits-1, so who merges
// what does not change the result -- and DEPARTS (count splits+1 .. 2 splits); the last one to depart puts the
// word back to count 0. The protocol therefore depends on nothing but the word itself: it is safe under CUDA-graph
// replay (same kernel parameters every time) and needs no memset. The splits of a launch are sized for one wave
// (at most one CTA per SM), so the CTAs that wait here are all resident.
constexpr unsigned long long kSplitTag = 0x53784d65726765ull;  // 56 bits

__device__ __forceinline__ void split_arrive(unsigned long long *w) {
  unsigned long long old = atomicAdd(w, 1ull);  // fast path: one atomic
  if ((old >> 8) == kSplitTag) return;
  // first use of this memory: install the tag. The add above (and any other add on the untagged word) is overwritten
  // by the install and repeated through this loop; an add that lands after the install already counts.
  unsigned long long cur = old + 1ull;
  for (;;) {
    const unsigned long long cnt = ((cur >> 8) == kSplitTag) ? (cur & 255ull) : 0ull;
    const unsigned long long prev = atomicCAS(w, cur, (kSplitTag << 8) | (cnt + 1ull));
    if (prev == cur) return;
    cur = prev;
  }
}
__device__ __forceinline__ void split_wait_all(const unsigned long long *w, int splits) {
  uint32_t polls = 0;
  for (;;) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(w) : "memory");
    if ((v >> 8) == kSplitTag && (int)(v & 255ull) >= splits) return;
    __nanosleep(20);
    if (++polls > (1u << 24)) __trap();  // a protocol bug traps instead of hanging the GPU
  }
}
__device__ __forceinline__ void split_depart(unsigned long long *w, int splits) {
  const unsigned long long old = atomicAdd(w, 1ull);
  if ((int)(old & 255ull) == 2 * splits - 1) atomicExch(w, kSplitTag << 8);  // everyone has left: count 0 again
}

// Combine the key splits of one (row, head) pair: out = sum_s exp(lse_s - lse) O_s in the fixed order 0..splits-1.
// One warp per pair, lane = 4 output dims. The partial log-sum-exps (lane s holds split s, two rounds for more than
// 32 splits) and the first partial O rows are requested together, so the merge costs about one trip to L2.
__device__ __forceinline__ void merge_splits(const float *part_o, const float *part_lse, int splits, size_t stride,
                                             size_t rh, int lane, __nv_bfloat16 *out, float *lse) {
  const float ls0 = lane < splits ? __ldcg(part_lse + (size_t)lane * stride + rh) : -INFINITY;
  const float ls1 = lane + 32 < splits ? __ldcg(part_lse + (size_t)(lane + 32) * stride + rh) : -INFINITY;
  const float4 *po = reinterpret_cast<const float4 *>(part_o + rh * kHeadDim) + lane;
  const size_t ostride = stride * (kHeadDim / 4);  // float4 units between consecutive splits
  constexpr int kB = 8;
  float4 v[kB];
#pragma unroll
  for (int i = 0; i < kB; ++i)
    if (i < splits) v[i] = __ldcg(po + (size_t)i * ostride);
  float mx = fmaxf(ls0, ls1);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, d));
  // a split without a visible key of the row (-inf) holds an undefined O: weight 0
  const float w0 = ls0 == -INFINITY ? 0.f : __expf(ls0 - mx), w1 = ls1 == -INFINITY ? 0.f : __expf(ls1 - mx);
  float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
  float den = 0.f;
  for (int s0 = 0; s0 < splits; s0 += kB) {
    float4 nx[kB];
#pragma unroll
    for (int i = 0; i < kB; ++i)
      if (s0 + kB + i < splits) nx[i] = __ldcg(po + (size_t)(s0 + kB + i) * ostride);
#pragma unroll
    for (int i = 0; i < kB; ++i) {
      const int sidx = s0 + i;  // (warp-uniform)
      if (sidx < splits) {
        const float w = __shfl_sync(0xffffffffu, sidx < 32 ? w0 : w1, sidx & 31);
        if (w != 0.f) {
          den += w;
          o.x = fmaf(v[i].x, w, o.x);
          o.y = fmaf(v[i].y, w, o.y);
          o.z = fmaf(v[i].z, w, o.z);
          o.w = fmaf(v[i].w, w, o.w);
        }
      }
    }
#pragma unroll
    for (int i = 0; i < kB; ++i) v[i] = nx[i];
  }
  const float inv = 1.f / den;
  uint2 pk;
  pk.x = pack_bf16x2(o.x * inv, o.y * inv);
  pk.y = pack_bf16x2(o.z * inv, o.w * inv);
  reinterpret_cast<uint2 *>(out + rh * kHeadDim)[lane] = pk;
  if (lse && lane == 0) lse[rh] = mx + logf(den);
}

}  // namespace sx
