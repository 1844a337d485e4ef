// sx_index.cu -- host-side segment index (include/sparsex_index.h): virtual-block hash with namespace keys,
// frozen-block pool with reference counts and utilisation-triggered eviction, and the planner that turns a
// prompt with candidate reuse segments into the segment map / source pages / Sparse-Q mask of sx_batch
// (PAPER.md:285-337 S4; Alg. 1 l.500-501). Host code only: no kernel, no CUDA call.
#include <stdint.h>
#include <string.h>

#include <algorithm>
#include <unordered_map>
#include <vector>

#include "../../include/sparsex_index.h"

namespace {

struct Entry {                 // one virtual block
  std::vector<int32_t> tokens; // the block's token ids (a hash match alone is not a hit)
  uint64_t key;                // namespace ("extra") key e
  int32_t block;               // physical KV block
  int32_t old_pos;             // position of the block's first token when it was cached
  int32_t refs;                // requests currently copying from it
  int64_t hits;                // how often it was handed out ("least-referenced" eviction order)
  int64_t serial;              // insertion order
  bool frozen;
};

// H(B, e): 64-bit FNV-1a over the key bytes, then the token bytes (reading A25; the paper leaves H open)
uint64_t virt_hash(const int32_t *tok, int n, uint64_t key) {
  uint64_t h = 1469598103934665603ull;
  auto mix = [&](uint64_t v, int bytes) {
    for (int i = 0; i < bytes; ++i) {
      h ^= (v >> (8 * i)) & 0xffu;
      h *= 1099511628211ull;
    }
  };
  mix(key, 8);
  for (int i = 0; i < n; ++i) mix((uint32_t)tok[i], 4);
  return h;
}

}  // namespace

struct sx_index {
  int32_t bs;
  int64_t next_serial = 0;
  std::unordered_multimap<uint64_t, Entry> map;  // hash -> entries (collisions resolved by comparing tokens + key)
  std::unordered_multimap<int32_t, uint64_t> by_block;  // physical block -> hashes of the virtual blocks on it

  using It = std::unordered_multimap<uint64_t, Entry>::iterator;
  It find(const int32_t *tok, uint64_t key) {
    auto range = map.equal_range(virt_hash(tok, bs, key));
    for (auto it = range.first; it != range.second; ++it)
      if (it->second.key == key && memcmp(it->second.tokens.data(), tok, sizeof(int32_t) * bs) == 0) return it;
    return map.end();
  }
  void unlink(int32_t block, uint64_t h) {
    auto r = by_block.equal_range(block);
    for (auto it = r.first; it != r.second; ++it)
      if (it->second == h) {
        by_block.erase(it);
        return;
      }
  }
  void erase(It it) {
    unlink(it->second.block, it->first);
    map.erase(it);
  }
};

extern "C" {

sx_index *sx_index_create(int32_t block_size) {
  if (block_size <= 0) return nullptr;
  sx_index *ix = new sx_index();
  ix->bs = block_size;
  return ix;
}

void sx_index_destroy(sx_index *ix) { delete ix; }

int32_t sx_index_size(const sx_index *ix) { return ix ? (int32_t)ix->map.size() : SX_ERR_INVALID_ARG; }

int32_t sx_index_insert(sx_index *ix, const int32_t *tokens, int32_t len, uint64_t extra_key, int32_t old_pos,
                        const int32_t *blocks, int32_t frozen) {
  if (!ix || !tokens || !blocks || len <= 0 || len % ix->bs || old_pos < 0 || old_pos % ix->bs)
    return SX_ERR_INVALID_ARG;
  const int n = len / ix->bs;
  for (int j = 0; j < n; ++j) {
    const int32_t *tok = tokens + (size_t)j * ix->bs;
    auto it = ix->find(tok, extra_key);
    if (it == ix->map.end()) {
      Entry e;
      e.tokens.assign(tok, tok + ix->bs);
      e.key = extra_key;
      e.refs = 0;
      e.hits = 0;
      e.serial = ix->next_serial++;
      e.block = -1;
      it = ix->map.emplace(virt_hash(tok, ix->bs, extra_key), std::move(e));
    }
    if (it->second.block != blocks[j]) {
      if (it->second.block >= 0) ix->unlink(it->second.block, it->first);
      ix->by_block.emplace(blocks[j], it->first);
    }
    it->second.block = blocks[j];
    it->second.old_pos = old_pos + j * ix->bs;
    it->second.frozen = frozen != 0;
  }
  return n;
}

int32_t sx_index_erase(sx_index *ix, const int32_t *tokens, int32_t len, uint64_t extra_key) {
  if (!ix || !tokens || len <= 0 || len % ix->bs) return SX_ERR_INVALID_ARG;
  int removed = 0;
  for (int j = 0; j < len / ix->bs; ++j) {
    auto it = ix->find(tokens + (size_t)j * ix->bs, extra_key);
    if (it != ix->map.end()) {
      ix->erase(it);
      ++removed;
    }
  }
  return removed;
}

int32_t sx_index_plan_request(sx_index *ix, int32_t req, const int32_t *tokens, int32_t seq_len,
                              const int32_t *cand, int32_t num_cand, uint64_t extra_key,
                              sx_segment *segments_out, int32_t *src_blocks_out, int32_t *new_idx_out,
                              int32_t *counts_out) {
  if (!ix || !tokens || seq_len <= 0 || num_cand < 0 || (num_cand > 0 && !cand) || !segments_out ||
      !src_blocks_out || !new_idx_out || !counts_out)
    return SX_ERR_INVALID_ARG;
  const int bs = ix->bs;
  int prev_end = 0;
  for (int c = 0; c < num_cand; ++c) {
    const int start = cand[2 * c], len = cand[2 * c + 1];
    if (start < prev_end || len <= 0 || start % bs || len % bs || start + len > seq_len) return SX_ERR_INVALID_ARG;
    prev_end = start + len;
  }
  int n_seg = 0, n_src = 0, n_new = 0, n_hit = 0, pos = 0;
  std::vector<sx_index::It> found;
  for (int c = 0; c <= num_cand; ++c) {
    const int start = c < num_cand ? cand[2 * c] : seq_len;
    for (; pos < start; ++pos) new_idx_out[n_new++] = pos;  // uncovered positions are Sparse-Q tokens
    if (c == num_cand) break;
    const int len = cand[2 * c + 1], nb = len / bs;
    found.clear();
    for (int j = 0; j < nb; ++j) {
      auto it = ix->find(tokens + start + (size_t)j * bs, extra_key);
      if (it == ix->map.end()) break;
      found.push_back(it);
    }
    if ((int)found.size() < nb) {  // a partial hit is a miss: the whole candidate is recomputed
      for (; pos < start + len; ++pos) new_idx_out[n_new++] = pos;
      continue;
    }
    ++n_hit;
    for (int j = 0; j < nb; ++j) {
      Entry &e = found[j]->second;
      const bool extend = j > 0 && e.old_pos == found[j - 1]->second.old_pos + bs;
      if (!extend) {  // a new run of constant delta = new_pos - old_pos
        sx_segment &s = segments_out[n_seg++];
        s.req = req;
        s.len = 0;
        s.old_pos = e.old_pos;
        s.new_pos = start + j * bs;
        s.src_off = n_src;
      }
      segments_out[n_seg - 1].len += bs;
      src_blocks_out[n_src++] = e.block;
      ++e.refs;
      ++e.hits;
    }
    pos = start + len;
  }
  counts_out[0] = n_seg;
  counts_out[1] = n_src;
  counts_out[2] = n_new;
  return n_hit;
}

int32_t sx_index_release(sx_index *ix, const int32_t *src_blocks, int32_t n) {
  if (!ix || (n > 0 && !src_blocks) || n < 0) return SX_ERR_INVALID_ARG;
  int removed = 0;
  for (int i = 0; i < n; ++i) {
    auto r = ix->by_block.equal_range(src_blocks[i]);
    sx_index::It hit = ix->map.end();
    for (auto b = r.first; b != r.second && hit == ix->map.end(); ++b) {
      auto er = ix->map.equal_range(b->second);
      for (auto it = er.first; it != er.second; ++it)
        if (it->second.block == src_blocks[i] && it->second.refs > 0 &&
            (hit == ix->map.end() || it->second.serial < hit->second.serial))
          hit = it;  // several namespaces may view the same block: the oldest referenced view gives back first
    }
    if (hit == ix->map.end()) continue;
    if (--hit->second.refs == 0 && !hit->second.frozen) {
      ix->erase(hit);
      ++removed;
    }
  }
  return removed;
}

int32_t sx_index_evict(sx_index *ix, int32_t used_blocks, int32_t total_blocks, double threshold,
                       int32_t *evicted_out, int32_t max_out) {
  if (!ix || total_blocks <= 0 || used_blocks < 0 || max_out < 0 || (max_out > 0 && !evicted_out))
    return SX_ERR_INVALID_ARG;
  // Eviction frees PHYSICAL blocks, and several virtual blocks (other namespaces, other token views) may sit on
  // one physical block: a block is evictable only if EVERY view of it is frozen and unreferenced; it is ranked by
  // the hand-outs of all its views (sum of hits, then its oldest view), all its views leave the index together and
  // the block is reported once.
  struct Blk {
    int32_t block;
    int64_t hits, serial;
    std::vector<sx_index::It> views;
  };
  std::unordered_map<int32_t, Blk> blocks;
  std::unordered_map<int32_t, bool> pinned;  // some view of the block is referenced or not frozen
  for (auto it = ix->map.begin(); it != ix->map.end(); ++it) {
    const Entry &e = it->second;
    if (!e.frozen || e.refs > 0) pinned[e.block] = true;
    auto ins = blocks.emplace(e.block, Blk{e.block, 0, e.serial, {}});
    Blk &b = ins.first->second;
    b.hits += e.hits;
    b.serial = std::min(b.serial, e.serial);
    b.views.push_back(it);
  }
  std::vector<Blk *> cand;
  for (auto &kv : blocks)
    if (!pinned.count(kv.first)) cand.push_back(&kv.second);
  std::sort(cand.begin(), cand.end(), [](const Blk *a, const Blk *b) {
    if (a->hits != b->hits) return a->hits < b->hits;
    return a->serial < b->serial;
  });
  int n = 0;
  for (Blk *b : cand) {
    if (n >= max_out || (double)(used_blocks - n) / (double)total_blocks <= threshold) break;
    evicted_out[n++] = b->block;
    for (auto &it : b->views) ix->erase(it);
  }
  return n;
}

}  // extern "C"
