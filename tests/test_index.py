"""Host-side segment index (include/sparsex_index.h): oracle pinned by hand cases, C++
implementation against the oracle on seeded random traffic, and the planner reproducing a known layout.
CPU only (the index makes no CUDA call)."""
import os
import re

import numpy as np
import pytest

from oracle.sx_index_oracle import IndexOracle
from paper_2606_01751_b200 import build as sxbuild
from paper_2606_01751_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BS = 16


@pytest.fixture(scope="module")
def idx_mod():
    sxbuild.build()
    from paper_2606_01751_b200 import index
    return index


def _tok(rng, n):
    return rng.integers(0, 50000, size=n).astype(np.int32)


# ----------------------------------------------------------------------------- oracle pins (hand cases)

def test_oracle_hand_cases():
    """Expected values typed from the paper's definitions, not computed by the oracle."""
    o = IndexOracle(BS)
    a = np.arange(100, 148)            # 3 blocks, cached at positions 32..79 in blocks 7, 8, 9
    o.insert(a, key=1, old_pos=32, blocks=[7, 8, 9], frozen=True)
    # same text under another namespace key is a different entry
    assert o.plan_request(0, a, [(0, 48)], key=2) == (0, [], [], list(range(48)))
    # prompt: 16 new | the segment | 16 new -> one segment, delta = 16 - 32, I_nr = the 32 uncovered positions
    prompt = np.concatenate([np.arange(16), a, np.arange(16)])
    hits, segs, src, new_idx = o.plan_request(3, prompt, [(16, 48)], key=1)
    assert hits == 1 and segs == [[3, 48, 32, 16, 0]] and src == [7, 8, 9]
    assert new_idx == list(range(16)) + list(range(64, 80))
    # a candidate with one unknown block is a miss as a whole (block-granular lookup, all blocks must hit)
    broken = prompt.copy()
    broken[40] += 1
    assert o.plan_request(3, broken, [(16, 48)], key=1)[0] == 0
    # blocks cached at non-contiguous positions -> one segment per run of constant delta
    o.insert(np.arange(500, 516), key=1, old_pos=0, blocks=[20])
    o.insert(np.arange(516, 532), key=1, old_pos=160, blocks=[21])
    hits, segs, src, _ = o.plan_request(0, np.arange(500, 532), [(0, 32)], key=1)
    assert hits == 1 and segs == [[0, 16, 0, 0, 0], [0, 16, 160, 16, 1]] and src == [20, 21]
    # release: non-frozen entries disappear at reference count 0, frozen ones stay
    assert o.release([20, 21]) == 2 and len(o) == 3
    assert o.release([7, 8, 9]) == 0 and len(o) == 3          # first plan's references; still referenced once...
    # eviction order: least referenced first, older first among equals; stops at the threshold
    o2 = IndexOracle(BS)
    for i in range(4):
        o2.insert(np.arange(i * 16, i * 16 + 16), key=9, old_pos=0, blocks=[100 + i], frozen=True)
    o2.plan_request(0, np.arange(16, 32), [(0, 16)], key=9)   # block 101 referenced (refs 1, hits 1)
    o2.plan_request(0, np.arange(32, 48), [(0, 16)], key=9)
    o2.release([102])                                         # block 102: hits 1, unreferenced
    assert o2.evict(used=95, total=100, threshold=0.9) == [100, 103, 102]   # 101 is referenced: never evicted
    assert o2.evict(used=92, total=100, threshold=0.9) == []


def test_oracle_eviction_with_two_namespaces_on_one_block():
    """Several virtual blocks may sit on one physical block (other namespace keys). Eviction
    frees PHYSICAL blocks: one referenced or non-frozen view pins the block; an evictable block is reported once
    and all its views leave together. Expected lists typed by hand."""
    o = IndexOracle(BS)
    a, b, c = np.arange(0, 16), np.arange(16, 32), np.arange(32, 48)
    o.insert(a, key=1, old_pos=0, blocks=[50], frozen=True)
    o.insert(a, key=2, old_pos=0, blocks=[50], frozen=True)    # second namespace, same physical block 50
    o.insert(b, key=1, old_pos=16, blocks=[51], frozen=True)
    o.insert(b, key=2, old_pos=16, blocks=[51], frozen=False)  # block 51 also carries a NON-frozen view
    o.insert(c, key=1, old_pos=32, blocks=[52], frozen=True)
    o.plan_request(0, a, [(0, 16)], key=2)                     # namespace 2 references block 50
    # 50: view (key 2) referenced -> pinned; 51: one view not frozen -> pinned; 52: free to go
    assert o.evict(used=100, total=100, threshold=0.5) == [52]
    assert len(o) == 4
    o.release([50])                                            # now every view of 50 is frozen and unreferenced
    assert o.evict(used=100, total=100, threshold=0.5) == [50]  # reported ONCE, both views gone
    assert len(o) == 2
    assert o.plan_request(1, a, [(0, 16)], key=1)[0] == 0 and o.plan_request(1, a, [(0, 16)], key=2)[0] == 0
    assert o.evict(used=100, total=100, threshold=0.5) == []   # 51 stays pinned by its non-frozen view


def test_eviction_with_two_namespaces_matches_oracle(idx_mod):
    ix, o = idx_mod.SegmentIndex(BS), IndexOracle(BS)
    a, b, c = (np.arange(i * 16, i * 16 + 16, dtype=np.int32) for i in range(3))
    for (t, key, old, blk, fr) in [(a, 1, 0, 50, True), (a, 2, 0, 50, True), (b, 1, 16, 51, True),
                                   (b, 2, 16, 51, False), (c, 1, 32, 52, True)]:
        assert ix.insert(t, key, old, np.asarray([blk], np.int32), fr) == o.insert(t, key, old, [blk], fr)
    h1 = ix.plan_request(0, a, [(0, 16)], 2)
    h2 = o.plan_request(0, a, [(0, 16)], key=2)
    assert h1[0] == h2[0] == 1
    assert ix.evict(100, 100, 0.5).tolist() == o.evict(100, 100, 0.5) == [52]
    assert ix.release(np.asarray([50], np.int32)) == o.release([50]) == 0
    assert ix.evict(100, 100, 0.5).tolist() == o.evict(100, 100, 0.5) == [50]
    assert len(ix) == len(o) == 2
    assert ix.evict(100, 100, 0.5).tolist() == o.evict(100, 100, 0.5) == []


# ----------------------------------------------------------------------------- C++ against the oracle

def test_header_symbols(idx_mod):
    hdr = open(os.path.join(ROOT, "include", "sparsex_index.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sx_index_[a-z_]+)\s*\(", hdr))
    assert declared == set(idx_mod.EXPORTS), declared ^ set(idx_mod.EXPORTS)
    lib = idx_mod._lib()
    for name in declared:
        assert getattr(lib, name) is not None


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_random_traffic_matches_oracle(idx_mod, seed):
    rng = np.random.default_rng(260601751 + seed)
    ix, o = idx_mod.SegmentIndex(BS), IndexOracle(BS)
    lib_docs = []
    next_block = 0
    outstanding = []
    for step in range(300):
        op = rng.choice(["insert", "plan", "plan", "release", "erase", "evict"])
        if op == "insert" or not lib_docs:
            n = int(rng.integers(1, 9)) * BS
            toks = lib_docs[int(rng.integers(len(lib_docs)))][0] if (lib_docs and rng.random() < 0.2) else _tok(rng, n)
            key = int(rng.integers(1, 4))
            blocks = np.arange(next_block, next_block + len(toks) // BS, dtype=np.int32)
            next_block += len(blocks)
            old = int(rng.integers(0, 64)) * BS
            frozen = bool(rng.random() < 0.5)
            assert ix.insert(toks, key, old, blocks, frozen) == o.insert(toks, key, old, blocks, frozen)
            lib_docs.append((toks, key))
            if rng.random() < 0.3:     # a second namespace viewing the SAME physical blocks
                key2 = key % 3 + 1
                fr2 = bool(rng.random() < 0.7)
                assert ix.insert(toks, key2, old, blocks, fr2) == o.insert(toks, key2, old, blocks, fr2)
                lib_docs.append((toks, key2))
        elif op == "plan":
            parts, cands, pos = [], [], 0
            for _ in range(int(rng.integers(1, 5))):
                gap = int(rng.integers(0, 3)) * BS
                parts.append(_tok(rng, gap))
                pos += gap
                toks, key0 = lib_docs[int(rng.integers(len(lib_docs)))]
                if rng.random() < 0.3:                         # partial reuse of a document: a block-aligned slice
                    a = int(rng.integers(0, len(toks) // BS)) * BS
                    toks = toks[a:]
                if rng.random() < 0.15:                        # corrupt one token: must miss
                    toks = toks.copy()
                    toks[int(rng.integers(len(toks)))] ^= 1
                parts.append(toks)
                cands.append((pos, len(toks)))
                pos += len(toks)
            parts.append(_tok(rng, int(rng.integers(0, 2)) * BS + int(rng.integers(0, 5))))
            prompt = np.concatenate(parts).astype(np.int32)
            key = int(rng.integers(1, 4))
            h1, s1, b1, n1 = ix.plan_request(step, prompt, cands, key)
            h2, s2, b2, n2 = o.plan_request(step, prompt, cands, key)
            assert h1 == h2 and s1.tolist() == s2 and b1.tolist() == b2 and n1.tolist() == n2
            if len(b1):
                outstanding.append(b1)
        elif op == "release" and outstanding:
            b = outstanding.pop(int(rng.integers(len(outstanding))))
            assert ix.release(b) == o.release(b.tolist())
        elif op == "erase":
            toks, key = lib_docs[int(rng.integers(len(lib_docs)))]
            assert ix.erase(toks, key) == o.erase(toks, key)
        elif op == "evict":
            used, total = int(rng.integers(80, 101)), 100
            assert ix.evict(used, total, 0.9).tolist() == o.evict(used, total, 0.9)
        assert len(ix) == len(o)


def test_planner_reproduces_the_c1_layout(idx_mod):
    """Tokens in, descriptor out: indexing the three cached segments of C1 (cached at position 0) and planning
    the prompt new128|A|new128|B|new128|C|new128 must give the segment map and Sparse-Q mask of
    workloads.config_c1 (BASELINE.json configs[0])."""
    lay = wl.config_c1()
    rng = np.random.default_rng(7)
    ix = idx_mod.SegmentIndex(BS)
    docs = [_tok(rng, 512) for _ in range(3)]
    for s, d in enumerate(docs):
        ix.insert(d, 42, 0, lay.pool_seg_pages[s], frozen=True)
    new = [_tok(rng, 128) for _ in range(4)]
    prompt = np.concatenate([new[0], docs[0], new[1], docs[1], new[2], docs[2], new[3]])
    cands = [(128, 512), (768, 512), (1408, 512)]
    hits, segs, src, new_idx = ix.plan_request(0, prompt, cands, 42)
    assert hits == 3
    assert np.array_equal(segs, lay.segments)
    assert np.array_equal(src, lay.src_blocks)
    assert np.array_equal(new_idx, lay.new_idx)
    with pytest.raises(Exception):
        ix.plan_request(0, prompt, [(100, 512)], 42)           # unaligned candidate: SX_ERR_INVALID_ARG
