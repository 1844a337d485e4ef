// sx_realign.cu -- stage (a): fused page copy + Delta-RoPE on K + V copy (PAPER.md:151-165 S3.1,
// "fused copy-Delta-RoPE kernel" PAPER.md:165/331; Alg. 1 l.502-504).
//
//   k^_{p'+j} <- R_{p'-p} k^_{p+j},  v^_{p'+j} <- v^_{p+j}
//
// HBM-bound: per cached token 8*Hkv*128 bytes (read K,V + write K,V). One CTA per source page
// (all KV heads, K and V): 16-byte coalesced loads issued up front, rotation in fp32 on
// (cos, sin)(Delta_m * theta_i) taken from a per-segment table that a tiny first kernel builds in
// fp64 (an fp32 product Delta*theta_i loses ~3e-3 in the sine at Delta ~ 1.3e5), one RNE to bf16.
#include "sx_internal.h"
#include "sx_ptx.cuh"

namespace sx {

// table[m][i] = (cos, sin)(Delta_m * theta^(-2i/128)), i in [0, 64)
__global__ void rope_table_kernel(const sx_segment *__restrict__ segs, int num_segments, double theta,
                                  float2 *__restrict__ table) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= num_segments * 64) return;
  int m = idx >> 6, i = idx & 63;
  double delta = (double)(segs[m].new_pos - segs[m].old_pos);
  double inv_freq = pow(theta, -2.0 * (double)i / (double)kHeadDim);
  double s, c;
  sincos(delta * inv_freq, &s, &c);
  table[idx] = make_float2((float)c, (float)s);
}

__device__ __forceinline__ uint4 ld_stream(const uint4 *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(uint4 *p, const uint4 &v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
               "r"(v.w)
               : "memory");
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

constexpr int kRealignThreads = 256;

template <int STYLE>
__global__ void __launch_bounds__(kRealignThreads)
realign_kernel(const uint4 *pool_k_src, uint4 *pool_k_dst, const uint4 *pool_v_src, uint4 *pool_v_dst, int num_kv_heads, const sx_segment *__restrict__ segs, int num_segments,
               const int32_t *__restrict__ src_blocks, const int32_t *__restrict__ k_table,
               const int32_t *__restrict__ v_table, int max_pages, const float2 *__restrict__ table) {
  __shared__ float2 cs_sm[64];
  __shared__ int sh[4];
  const int page = blockIdx.x;  // index into src_blocks
  if (threadIdx.x == 0) {
    // segment m with src_off[m] <= page < src_off[m] + len/16 (src_off ascending: binary search)
    int lo = 0, hi = num_segments - 1;
    while (lo < hi) {
      int mid = (lo + hi + 1) >> 1;
      if (segs[mid].src_off <= page) lo = mid; else hi = mid - 1;
    }
    const sx_segment s = segs[lo];
    int pg = page - s.src_off;
    int lpage = s.new_pos / kPage + pg;
    sh[0] = lo;
    sh[1] = src_blocks[page];
    sh[2] = k_table[(size_t)s.req * max_pages + lpage];
    sh[3] = v_table[(size_t)s.req * max_pages + lpage];
  }
  __syncthreads();
  const int m = sh[0], src = sh[1], dk = sh[2], dv = sh[3];
  if (threadIdx.x < 64) cs_sm[threadIdx.x] = table[m * 64 + threadIdx.x];
  __syncthreads();

  const int chunks = num_kv_heads * kPage * 16;            // 16-byte chunks of one page (all heads)
  const size_t page_chunks = (size_t)chunks;
  const uint4 *ks = pool_k_src + (size_t)src * page_chunks;
  uint4 *kd = pool_k_dst + (size_t)dk * page_chunks;
  const uint4 *vs = pool_v_src + (size_t)src * page_chunks;
  uint4 *vd = pool_v_dst + (size_t)dv * page_chunks;
  const bool copy_v = (dv != src);

  if (STYLE == 0) {
    // task = (row, c): chunks c and c+8 of one 256-B row
    const int tasks = chunks / 2;
    for (int t0 = threadIdx.x; t0 < tasks; t0 += 4 * kRealignThreads) {
      uint4 a[4], b[4], v0[4], v1[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        int t = t0 + u * kRealignThreads;
        if (t < tasks) {
          int row = t >> 3, c = t & 7;
          a[u] = ld_stream(ks + row * 16 + c);
          b[u] = ld_stream(ks + row * 16 + c + 8);
          if (copy_v) {
            v0[u] = ld_stream(vs + row * 16 + c);
            v1[u] = ld_stream(vs + row * 16 + c + 8);
          }
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        int t = t0 + u * kRealignThreads;
        if (t < tasks) {
          int row = t >> 3, c = t & 7;
          rotate_split(a[u], b[u], cs_sm + c * 8);
          st_stream(kd + row * 16 + c, a[u]);
          st_stream(kd + row * 16 + c + 8, b[u]);
          if (copy_v) {
            st_stream(vd + row * 16 + c, v0[u]);
            st_stream(vd + row * 16 + c + 8, v1[u]);
          }
        }
      }
    }
  } else {
    for (int t0 = threadIdx.x; t0 < chunks; t0 += 4 * kRealignThreads) {
      uint4 a[4], v0[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        int t = t0 + u * kRealignThreads;
        if (t < chunks) {
          a[u] = ld_stream(ks + t);
          if (copy_v) v0[u] = ld_stream(vs + t);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        int t = t0 + u * kRealignThreads;
        if (t < chunks) {
          rotate_inter(a[u], cs_sm + (t & 15) * 4);
          st_stream(kd + t, a[u]);
          if (copy_v) st_stream(vd + t, v0[u]);
        }
      }
    }
  }
}

sx_status launch_realign(const sx_pool *pool, const sx_batch *b, float2 *table, cudaStream_t st) {
  int n = b->num_segments * 64;
  rope_table_kernel<<<(n + 127) / 128, 128, 0, st>>>(b->segments, b->num_segments, b->rope_theta, table);
  sx_status s = check_launch("rope_table_kernel");
  if (s != SX_OK) return s;
  const uint4 *k = reinterpret_cast<const uint4 *>(pool->k);
  const uint4 *v = reinterpret_cast<const uint4 *>(pool->v);
  if (b->rope_style == 0)
    realign_kernel<0><<<b->total_seg_pages, kRealignThreads, 0, st>>>(
        k, reinterpret_cast<uint4 *>(pool->k), v, reinterpret_cast<uint4 *>(pool->v), pool->num_kv_heads, b->segments,
        b->num_segments, b->src_blocks, b->k_block_table, b->v_block_table, b->max_pages_per_req, table);
  else
    realign_kernel<1><<<b->total_seg_pages, kRealignThreads, 0, st>>>(
        k, reinterpret_cast<uint4 *>(pool->k), v, reinterpret_cast<uint4 *>(pool->v), pool->num_kv_heads, b->segments,
        b->num_segments, b->src_blocks, b->k_block_table, b->v_block_table, b->max_pages_per_req, table);
  return check_launch("realign_kernel");
}

}  // namespace sx
