"""Plain Python reference of the host-side segment index (PAPER.md:285-337 S4; Alg. 1 l.500-501).

TEST INFRASTRUCTURE ONLY: imported by tests/ alone; the package never imports it. It shares no code with
csrc/sx_index.cu: where that one hashes, this one keys a dict by the (namespace key, token tuple) itself, which is
the definition "reusable only when both token IDs and the extra key match" with no hash at all.

  virtual block: physical block id + position of the block's first token when cached.
  frozen block: survives reference count 0; leaves through erase or eviction only.
  eviction: above the utilisation threshold free the least-referenced physical blocks whose
                  views are ALL frozen and unreferenced (ties: older first); every view of a freed block leaves,
                  the block is reported once (a block that another namespace still references is never freed).
"""
from __future__ import annotations


class IndexOracle:
    def __init__(self, block_size=16):
        self.bs = block_size
        self.d = {}          # (key, tokens tuple) -> dict(block, old_pos, refs, hits, serial, frozen)
        self.serial = 0

    def __len__(self):
        return len(self.d)

    def _blocks(self, tokens):
        assert len(tokens) % self.bs == 0 and len(tokens) > 0
        return [tuple(int(x) for x in tokens[j:j + self.bs]) for j in range(0, len(tokens), self.bs)]

    def insert(self, tokens, key, old_pos, blocks, frozen=False):
        for j, tb in enumerate(self._blocks(tokens)):
            e = self.d.get((key, tb))
            if e is None:
                e = dict(refs=0, hits=0, serial=self.serial)
                self.serial += 1
                self.d[(key, tb)] = e
            e.update(block=int(blocks[j]), old_pos=old_pos + j * self.bs, frozen=bool(frozen))
        return len(tokens) // self.bs

    def erase(self, tokens, key):
        n = 0
        for tb in self._blocks(tokens):
            if self.d.pop((key, tb), None) is not None:
                n += 1
        return n

    def plan_request(self, req, tokens, candidates, key):
        """Alg. 1 l.500-501: full-candidate hits only; one segment per run of contiguous cached positions."""
        segs, src, new_idx, hits, pos = [], [], [], 0, 0
        for (start, ln) in candidates:
            new_idx.extend(range(pos, start))
            ents = [self.d.get((key, tb)) for tb in self._blocks(tokens[start:start + ln])]
            if any(e is None for e in ents):
                new_idx.extend(range(start, start + ln))
            else:
                hits += 1
                for j, e in enumerate(ents):
                    if j == 0 or e["old_pos"] != ents[j - 1]["old_pos"] + self.bs:
                        segs.append([req, 0, e["old_pos"], start + j * self.bs, len(src)])
                    segs[-1][1] += self.bs
                    src.append(e["block"])
                    e["refs"] += 1
                    e["hits"] += 1
            pos = start + ln
        new_idx.extend(range(pos, len(tokens)))
        return hits, segs, src, new_idx

    def release(self, src_blocks):
        removed = 0
        for b in src_blocks:
            live = [(e["serial"], k) for k, e in self.d.items() if e["block"] == b and e["refs"] > 0]
            if not live:
                continue
            k = min(live)[1]
            e = self.d[k]
            e["refs"] -= 1
            if e["refs"] == 0 and not e["frozen"]:
                del self.d[k]
                removed += 1
        return removed

    def evict(self, used, total, threshold=0.9, max_out=1 << 16):
        by_block = {}
        for k, e in self.d.items():
            by_block.setdefault(e["block"], []).append(k)
        cand = []
        for b, keys in by_block.items():
            ents = [self.d[k] for k in keys]
            if all(e["frozen"] and e["refs"] == 0 for e in ents):
                cand.append((sum(e["hits"] for e in ents), min(e["serial"] for e in ents), b))
        out = []
        for _, _, b in sorted(cand):
            if len(out) >= max_out or (used - len(out)) / total <= threshold:
                break
            for k in by_block[b]:
                del self.d[k]
            out.append(b)
        return out
