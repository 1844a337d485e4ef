// sx_attn_noalloc.cu -- sx_sparse_attn_noalloc (include/sparsex.h): stage (c) for small row sets with NO
// caller-provided workspace and no allocation of any kind. Some callers cannot allocate device memory where
// they call from (code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc); the
// small-row regime (a handful of query rows against a long context: the tail fallback of PAPER.md:235, decode-like
// steps) is exactly where they live, and it is the regime in which the attention kernel NEEDS scratch: the key
// range is cut into splits whose fp32 partial (O, log-sum-exp) meet in memory before they merge themselves
// (sx_attn.cu, sx_split_merge.cuh).
//
// Here that scratch is a file-scope device array of a fixed, modest size (below): every GPU that loads the library
// holds it until the process exits. The kernel is the one sx_sparse_attn launches (attn_kernel<false> with key
// splits); only where its scratch lives differs, and -- because the array is smaller than the caller-sized
// workspace -- the largest row set it takes.
//
// Shared state, stated once: every call on a device uses THE SAME array.
//   * Nothing in it has to start at zero: the partial (O, lse) slots of a launch are all written before any of
//     them is read, and the rendezvous words are tagged and return to their rest state (tag | count 0) when the
//     last split of a row pair departs (split_arrive / split_depart); a zero word (the array's initial content) is
//     "untagged" and is installed by the first arrival. So no clearing launch is needed between calls.
//   * Calls that OVERLAP on the GPU (different streams, or graph branches without an edge between them) race on
//     the array and give wrong results or hang at the rendezvous; calls on one stream, or ordered by events /
//     graph edges, are safe. sx_sparse_attn with its own workspace is the entry point for concurrent callers.
#include <mutex>

#include "sx_internal.h"

namespace sx {

// Sizes (include/sparsex.h states them for the caller):
//   kNoallocMaxPairs   largest row set: total_rows * num_q_heads (row, query head) pairs
//   kNoallocSlots      (split, row, head) partial slots: the number of key splits is reduced until
//                      splits * total_rows * num_q_heads fits (18 splits at the largest row set, up to 64 below 288 pairs)
//   per slot           128 fp32 of normalised partial O + 1 fp32 partial log-sum-exp
//   kNoallocTickets    one 64-bit rendezvous word per (request, KV head, row pair): fewer than 148 whenever splits exist
constexpr int kNoallocMaxPairs = SX_NOALLOC_MAX_PAIRS;
constexpr size_t kNoallocSlots = 18432;
constexpr size_t kNoallocPartBytes = kNoallocSlots * (kHeadDim + 1) * sizeof(float);  // 9 510 912 B
constexpr int kNoallocTickets = 148;
constexpr size_t kNoallocBytes = kNoallocPartBytes + kNoallocTickets * sizeof(unsigned long long);
static_assert(kNoallocPartBytes % 256 == 0, "the rendezvous words follow the partials, 256-B aligned");
static_assert(kNoallocBytes == SX_NOALLOC_SCRATCH_BYTES, "include/sparsex.h states the size of the array");

// In HOST code this name is a host-side stand-in for the symbol, not a device address: it is only ever handed to
// cudaGetSymbolAddress (below). Device code of this file could name it directly; the kernel lives in sx_attn.cu and
// receives the address as a parameter.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoallocBytes];

// Device address of the array on the CURRENT device: looked up once per device (the array exists once per device
// that has loaded the library's module), with that device current, return code checked.
constexpr int kNoallocMaxDevices = 64;
static sx_status noalloc_scratch(unsigned char **out) {
  static std::mutex mu;
  static unsigned char *ptr[kNoallocMaxDevices] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return set_error(SX_ERR_CUDA, "noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kNoallocMaxDevices) return set_error(SX_ERR_UNSUPPORTED, "noalloc: device ordinal %d", dev);
  std::lock_guard<std::mutex> lk(mu);
  if (!ptr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return set_error(SX_ERR_CUDA, "noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    }
    ptr[dev] = static_cast<unsigned char *>(p);
  }
  *out = ptr[dev];
  return SX_OK;
}

sx_status launch_attn_noalloc(const sx_pool *pool, const sx_batch *b, const void *q, const int32_t *rows,
                              const int32_t *rows_off, int32_t total_rows, void *out, float *lse, cudaStream_t st) {
  const size_t pairs = (size_t)total_rows * pool->num_q_heads;
  if (pairs > (size_t)kNoallocMaxPairs)
    return set_error(SX_ERR_UNSUPPORTED,
                     "sx_sparse_attn_noalloc: %d rows x %d query heads = %zu (row, head) pairs exceed the built-in "
                     "scratch (SX_NOALLOC_MAX_PAIRS = %d); use sx_sparse_attn with a workspace",
                     total_rows, pool->num_q_heads, pairs, kNoallocMaxPairs);
  // the split rule of sx_sparse_attn, then fewer splits until the partials fit the array
  int splits = attn_pv_splits(pool, b, total_rows, 2);
  while (splits > 1 && (size_t)splits * pairs > kNoallocSlots) --splits;
  float *part = nullptr;
  unsigned long long *tickets = nullptr;
  if (splits > 1) {
    // one rendezvous word per block of the un-split grid (launch_attn's grid bound)
    const int g = pool->num_q_heads / pool->num_kv_heads;
    const int grid = (total_rows / (2 * (kTile / g)) + b->num_reqs) * pool->num_kv_heads;
    if (grid > kNoallocTickets)
      return set_error(SX_ERR_UNSUPPORTED, "sx_sparse_attn_noalloc: %d row-pair blocks exceed the built-in scratch", grid);
    unsigned char *base = nullptr;
    sx_status s = noalloc_scratch(&base);
    if (s != SX_OK) return s;
    part = reinterpret_cast<float *>(base);
    tickets = reinterpret_cast<unsigned long long *>(base + kNoallocPartBytes);
  }
  return launch_attn(pool, b, q, rows, rows_off, total_rows, out, lse, splits, part, /*cta_pair=*/false, ZcArgs(), st,
                     tickets);
}

}  // namespace sx
