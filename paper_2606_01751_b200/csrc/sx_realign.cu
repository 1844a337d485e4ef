// sx_realign.cu -- stage (a): fused page copy + Delta-RoPE on K + V copy (PAPER.md:151-165 S3.1,
// "fused copy-Delta-RoPE kernel" PAPER.md:165/331; Alg. 1 l.502-504).
//
//   k^_{p'+j} <- R_{p'-p} k^_{p+j},  v^_{p'+j} <- v^_{p+j}
//
// HBM-bound: per cached token 8*Hkv*128 bytes (read K,V + write K,V). One CTA per (source page, KV head)
// = 4 KB of K and of V: 16-byte coalesced loads issued up front, rotation in fp32 on
// (cos, sin)(Delta_m * theta_i) taken from a per-segment table that a tiny first kernel builds in
// fp64 (an fp32 product Delta*theta_i loses ~3e-3 in the sine at Delta ~ 1.3e5), one RNE to bf16.
#include "sx_internal.h"
#include "sx_ptx.cuh"
#include "sx_rotate.cuh"

namespace sx {

// One preparatory launch per call: thread idx < num_segments * 64 builds the rotation table
// table[m][i] = (cos, sin)(Delta_m * theta^(-2i/128)), i in [0, 64), in fp64; thread idx < total pages
// resolves its page once: (segment, source page, destination K page, destination V page), so that the
// copy kernel starts streaming after a single 16-byte load instead of a chain of dependent lookups.
__global__ void rope_table_kernel(const sx_segment *__restrict__ segs, int num_segments, double theta,
                                  float2 *__restrict__ table, int total_pages,
                                  const int32_t *__restrict__ src_blocks, const int32_t *__restrict__ k_table,
                                  const int32_t *__restrict__ v_table, int max_pages, int4 *__restrict__ page_desc) {
  griddep_launch();  // programmatic dependent launch: the copy kernel may become resident now ...
  griddep_wait();    // ... and the block tables may be outputs of the previous kernel in the stream
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < num_segments * 64) {
    int m = idx >> 6, i = idx & 63;
    table[idx] = rope_cos_sin(theta, segs[m].new_pos - segs[m].old_pos, i);
  }
  if (idx < total_pages) {
    // segment m with src_off[m] <= page < src_off[m] + len/16 (src_off ascending: binary search)
    int lo = 0, hi = num_segments - 1;
    while (lo < hi) {
      int mid = (lo + hi + 1) >> 1;
      if (segs[mid].src_off <= idx) lo = mid; else hi = mid - 1;
    }
    const sx_segment sg = segs[lo];
    const int lpage = sg.new_pos / kPage + (idx - sg.src_off);
    page_desc[idx] = make_int4(lo, src_blocks[idx], ld_dep(k_table + (size_t)sg.req * max_pages + lpage),
                               ld_dep(v_table + (size_t)sg.req * max_pages + lpage));  // (tables: a scatter may just have flipped them)
  }
}

__device__ __forceinline__ uint4 ld_stream(const uint4 *p) {
  uint4 r;
  asm volatile("ld.global.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void st_stream(uint4 *p, const uint4 &v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z),
               "r"(v.w)
               : "memory");
}

constexpr int kRealignThreads = 128;

// One CTA per (source page, KV head): 4 KB of K and 4 KB of V in, the same out. Every thread issues its
// four 16-byte loads (and the rotation coefficients of its column pair) right after the descriptor.
constexpr int kRealignMaxLayers = 64;
struct LayerPools {  // K and V pools of the layers of one launch (blockIdx.z = layer), passed by value
  uint4 *k[kRealignMaxLayers];
  uint4 *v[kRealignMaxLayers];
};

template <int STYLE>
__global__ void __launch_bounds__(kRealignThreads)
realign_kernel(const __grid_constant__ LayerPools pools, int num_kv_heads, const int4 *__restrict__ page_desc,
               const float2 *__restrict__ table) {
  griddep_launch();
  griddep_wait();  // page descriptors and rotation table come from the preparation kernel
  const int page = blockIdx.x, h = blockIdx.y;
  const uint4 *pool_k_src = pools.k[blockIdx.z], *pool_v_src = pools.v[blockIdx.z];
  uint4 *pool_k_dst = pools.k[blockIdx.z], *pool_v_dst = pools.v[blockIdx.z];
  const int4 d = ld_dep(page_desc + page);  // (segment, source page, destination K page, destination V page)
  const size_t tile = (size_t)kPage * 16;  // 16-byte chunks of one (page, head) tile
  const uint4 *ks = pool_k_src + ((size_t)d.y * num_kv_heads + h) * tile;
  uint4 *kd = pool_k_dst + ((size_t)d.z * num_kv_heads + h) * tile;
  const uint4 *vs = pool_v_src + ((size_t)d.y * num_kv_heads + h) * tile;
  uint4 *vd = pool_v_dst + ((size_t)d.w * num_kv_heads + h) * tile;
  const bool copy_v = (d.w != d.y);
  const int t = threadIdx.x;
  if (STYLE == 0) {
    // chunks c and c + 8 of row t >> 3: columns [8c, 8c+8) pair with [64+8c, 64+8c+8)
    const int row = t >> 3, c = t & 7;
    uint4 a = ld_stream(ks + row * 16 + c);
    uint4 b = ld_stream(ks + row * 16 + c + 8);
    uint4 v0, v1;
    if (copy_v) {
      v0 = ld_stream(vs + row * 16 + c);
      v1 = ld_stream(vs + row * 16 + c + 8);
    }
    float2 cs[8];
    const float4 *tp = reinterpret_cast<const float4 *>(table + d.x * 64 + c * 8);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float4 f = ld_dep(tp + i);
      cs[2 * i] = make_float2(f.x, f.y);
      cs[2 * i + 1] = make_float2(f.z, f.w);
    }
    rotate_split(a, b, cs);
    st_stream(kd + row * 16 + c, a);
    st_stream(kd + row * 16 + c + 8, b);
    if (copy_v) {
      st_stream(vd + row * 16 + c, v0);
      st_stream(vd + row * 16 + c + 8, v1);
    }
  } else {
    // chunks t and t + 128: the 4 interleaved pairs (2i, 2i+1) of each 16-byte chunk
    uint4 a0 = ld_stream(ks + t), a1 = ld_stream(ks + t + 128);
    uint4 v0, v1;
    if (copy_v) {
      v0 = ld_stream(vs + t);
      v1 = ld_stream(vs + t + 128);
    }
    float2 cs[4];
    const float4 *tp = reinterpret_cast<const float4 *>(table + d.x * 64 + (t & 15) * 4);
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const float4 f = ld_dep(tp + i);
      cs[2 * i] = make_float2(f.x, f.y);
      cs[2 * i + 1] = make_float2(f.z, f.w);
    }
    rotate_inter(a0, cs);
    rotate_inter(a1, cs);  // (t + 128) & 15 == t & 15: same column group
    st_stream(kd + t, a0);
    st_stream(kd + t + 128, a1);
    if (copy_v) {
      st_stream(vd + t, v0);
      st_stream(vd + t + 128, v1);
    }
  }
}

// Zero-copy mode (sx_batch::zero_copy): nothing is copied; the stage kernels rotate cached K on the fly. They need,
// per request and logical page, whether the page still IS the cached source page of a segment (then its keys are
// stored at their old positions: rotate by that segment's Delta) or a private page (already at its position):
//   page_seg[req][lp] = m if a segment m covers lp and k_block_table[req][lp] == the source page of m for lp, else -1
// and the same per-segment (cos, sin) table as the copy kernel.
__global__ void zc_prepare_kernel(const sx_segment *__restrict__ segs, int num_segments, double theta,
                                  float2 *__restrict__ table, const int32_t *__restrict__ src_blocks,
                                  const int32_t *__restrict__ k_table, int num_reqs, int max_pages,
                                  const int32_t *__restrict__ seq_len, int32_t *__restrict__ page_seg) {
  griddep_launch();
  griddep_wait();  // the block tables may have been flipped by the previous kernel (a scatter)
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < num_segments * 64) {
    const int m = idx >> 6, i = idx & 63;
    table[idx] = rope_cos_sin(theta, segs[m].new_pos - segs[m].old_pos, i);
  }
  if (idx < num_reqs * max_pages) {
    const int req = idx / max_pages, lp = idx - req * max_pages;
    int m = -1;
    if (lp * kPage < seq_len[req]) {
      m = find_segment(segs, num_segments, req, lp * kPage);
      if (m >= 0 && ld_dep(k_table + idx) != src_blocks[segs[m].src_off + lp - segs[m].new_pos / kPage]) m = -1;
    }
    page_seg[idx] = m;
  }
}

sx_status launch_zc_prepare(const sx_batch *b, float2 *table, int32_t *page_seg, cudaStream_t st) {
  const int a = b->num_segments * 64, c = b->num_reqs * b->max_pages_per_req;
  const int n = a > c ? a : c;
  cudaError_t e = launch_pdl(zc_prepare_kernel, dim3((n + 127) / 128), dim3(128), 0, st, 1, b->segments, b->num_segments,
                             b->rope_theta, table, b->src_blocks, (const int32_t *)b->k_block_table, b->num_reqs,
                             b->max_pages_per_req, b->seq_len, page_seg);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "zc_prepare launch: %s", cudaGetErrorString(e));
  return check_launch("zc_prepare_kernel");
}

sx_status launch_realign(const sx_pool *pools, int num_layers, const sx_batch *b, float2 *table, int4 *page_desc,
                         cudaStream_t st) {
  const int n = b->num_segments * 64 > b->total_seg_pages ? b->num_segments * 64 : b->total_seg_pages;
  cudaError_t e = launch_pdl(rope_table_kernel, dim3((n + 127) / 128), dim3(128), 0, st, 1, b->segments, b->num_segments,
                             b->rope_theta, table, b->total_seg_pages, b->src_blocks, (const int32_t *)b->k_block_table,
                             (const int32_t *)b->v_block_table, b->max_pages_per_req, page_desc);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "rope_table launch: %s", cudaGetErrorString(e));
  sx_status s = check_launch("rope_table_kernel");
  if (s != SX_OK) return s;
  for (int l0 = 0; l0 < num_layers; l0 += kRealignMaxLayers) {
    const int nl = num_layers - l0 < kRealignMaxLayers ? num_layers - l0 : kRealignMaxLayers;
    LayerPools lp;
    for (int l = 0; l < nl; ++l) {
      lp.k[l] = reinterpret_cast<uint4 *>(pools[l0 + l].k);
      lp.v[l] = reinterpret_cast<uint4 *>(pools[l0 + l].v);
    }
    const dim3 grid(b->total_seg_pages, pools[0].num_kv_heads, nl);
    e = launch_pdl(b->rope_style == 0 ? realign_kernel<0> : realign_kernel<1>, grid, dim3(kRealignThreads), 0, st, 1, lp,
                   pools[0].num_kv_heads, (const int4 *)page_desc, (const float2 *)table);
    if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "realign launch: %s", cudaGetErrorString(e));
    s = check_launch("realign_kernel");
    if (s != SX_OK) return s;
  }
  return SX_OK;
}

}  // namespace sx
