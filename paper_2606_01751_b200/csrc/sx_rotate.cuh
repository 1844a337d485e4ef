// sx_rotate.cuh -- the Delta-RoPE arithmetic of stage (a), shared by every kernel that applies
// it: the copy kernel of sx_realign.cu, and -- in zero-copy mode (sx_batch::zero_copy, include/sparsex.h) -- the
// kernels that rotate cached K on the fly (a K tile in shared memory before the MMA reads it; a page during
// copy-on-write). One definition, so that a key rotated on the fly has exactly the bits sx_rope_realign would have
// stored: angles in fp64, (cos, sin) rounded to fp32 once, the rotation in fp32 with one fused multiply-add per
// component, one RNE rounding to bf16.
#pragma once
#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

// (cos, sin)(delta * theta^(-2i/128)), i in [0, 64)
__device__ __forceinline__ float2 rope_cos_sin(double theta, int delta, int i) {
  const double inv_freq = pow(theta, -2.0 * (double)i / (double)kHeadDim);
  double s, c;
  sincos((double)delta * inv_freq, &s, &c);
  return make_float2((float)c, (float)s);
}

__device__ __forceinline__ float bf_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf_hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }

// half-split pairing: element i of `a` (columns [8c, 8c+8)) pairs with element i of `b`
// (columns [64+8c, 64+8c+8)); cs[e] = (cos, sin) of pair index 8c+e.
__device__ __forceinline__ void rotate_split(uint4 &a, uint4 &b, const float2 *cs) {
  uint32_t *pa = reinterpret_cast<uint32_t *>(&a);
  uint32_t *pb = reinterpret_cast<uint32_t *>(&b);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float x0 = bf_lo(pa[w]), x1 = bf_hi(pa[w]);
    float y0 = bf_lo(pb[w]), y1 = bf_hi(pb[w]);
    float2 c0 = cs[2 * w], c1 = cs[2 * w + 1];
    float xr0 = fmaf(x0, c0.x, -(y0 * c0.y)), yr0 = fmaf(x0, c0.y, y0 * c0.x);
    float xr1 = fmaf(x1, c1.x, -(y1 * c1.y)), yr1 = fmaf(x1, c1.y, y1 * c1.x);
    pa[w] = pack_bf16x2(xr0, xr1);
    pb[w] = pack_bf16x2(yr0, yr1);
  }
}
// interleaved pairing: the 4 pairs (2i, 2i+1) of one 16-byte chunk; cs[e] = pair 4c+e.
__device__ __forceinline__ void rotate_inter(uint4 &a, const float2 *cs) {
  uint32_t *pa = reinterpret_cast<uint32_t *>(&a);
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    float x = bf_lo(pa[w]), y = bf_hi(pa[w]);
    float2 c = cs[w];
    pa[w] = pack_bf16x2(fmaf(x, c.x, -(y * c.y)), fmaf(x, c.y, y * c.x));
  }
}

// Segment of request `req` that covers position `pos`, or -1. Segments are sorted by (req, new_pos) and do not
// overlap (sx_check_batch verifies it).
__device__ __forceinline__ int find_segment(const sx_segment *__restrict__ segs, int num_segments, int req, int pos) {
  int lo = 0, hi = num_segments;  // first segment with (req, new_pos) > (req, pos)
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    const int r = segs[mid].req, np = segs[mid].new_pos;
    if (r < req || (r == req && np <= pos)) lo = mid + 1; else hi = mid;
  }
  const int m = lo - 1;
  if (m < 0 || segs[m].req != req || pos >= segs[m].new_pos + segs[m].len) return -1;
  return m;
}

// Zero-copy mode: rotate in place the rows of one K tile in shared memory whose page still is the cached source
// page. Tile layout (what the TMA boxes of the tensor-core kernels produce): [2 halves of 64 columns][128 rows]
// [128 B], 128-B swizzle (16-byte chunk c of row r sits at chunk c ^ (r & 7)), the halves `half_bytes` apart, the
// tile 1024-B aligned. page_seg8[pg] = segment of page pg (16 rows) of the tile or -1 (private / fresh / prefix
// page: stored at its position already); pages >= n_valid lie past the sequence. table = (cos, sin) per segment.
// Called by NTHREADS threads with tid in [0, NTHREADS); the caller orders it between the TMA completion and the
// MMA (fence.proxy.async + barrier).
template <int STYLE, int NTHREADS>
__device__ __forceinline__ void rotate_k_tile(uint8_t *tile, int half_bytes, const int32_t *__restrict__ page_seg8,
                                              int n_valid, const float2 *__restrict__ table, int tid) {
  int m_prev = -1;
  if (STYLE == 0) {
    const int c = tid & 7;
    float2 cs[8];
    for (int r = tid >> 3; r < kTile; r += NTHREADS / 8) {
      const int pg = r >> 4;
      const int m = pg < n_valid ? ld_dep(page_seg8 + pg) : -1;
      if (m < 0) continue;
      if (m != m_prev) {
        const float4 *tp = reinterpret_cast<const float4 *>(table + m * 64 + c * 8);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const float4 f = ld_dep(tp + i);
          cs[2 * i] = make_float2(f.x, f.y);
          cs[2 * i + 1] = make_float2(f.z, f.w);
        }
        m_prev = m;
      }
      uint4 *pa = reinterpret_cast<uint4 *>(tile + r * 128 + ((c ^ (r & 7)) << 4));
      uint4 *pb = reinterpret_cast<uint4 *>(reinterpret_cast<uint8_t *>(pa) + half_bytes);
      uint4 a = *pa, b = *pb;
      rotate_split(a, b, cs);
      *pa = a;
      *pb = b;
    }
  } else {
    const int c16 = tid & 15;  // 16-byte chunk of the 256-B row: pairs 4 c16 .. 4 c16 + 3
    float2 cs[4];
    for (int r = tid >> 4; r < kTile; r += NTHREADS / 16) {
      const int pg = r >> 4;
      const int m = pg < n_valid ? ld_dep(page_seg8 + pg) : -1;
      if (m < 0) continue;
      if (m != m_prev) {
        const float4 *tp = reinterpret_cast<const float4 *>(table + m * 64 + c16 * 4);
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const float4 f = ld_dep(tp + i);
          cs[2 * i] = make_float2(f.x, f.y);
          cs[2 * i + 1] = make_float2(f.z, f.w);
        }
        m_prev = m;
      }
      uint4 *pa = reinterpret_cast<uint4 *>(tile + (c16 >> 3) * half_bytes + r * 128 + (((c16 & 7) ^ (r & 7)) << 4));
      uint4 a = *pa;
      rotate_inter(a, cs);
      *pa = a;
    }
  }
}

}  // namespace sx
