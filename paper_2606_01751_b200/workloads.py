"""Seeded synthetic workloads for the Sparse-KV recomputation step (numpy only).

This module serves BOTH the fp64 oracle (through tests/) and the CUDA path. It
holds none of the method's arithmetic: no RoPE, no softmax, no top-k, no page
scatter. It only draws random tensors, rounds them to bf16 bit patterns and lays
out block tables / segment maps for the five BASELINE.json configs (C1..C5) and
scaled-down versions of them.

Recipe:
  * RNG: numpy PCG64(SeedSequence([260601751, cfg, layer, tensor_id, index])),
    float32 standard normals, round-to-nearest-even to bf16.
  * tensor_id: 0 layout, 1 cached K, 2 cached V, 3 Q_full, 4 K_fresh, 5 V_fresh,
    6 salient permutation, 7 physical page permutation.
  * Cached keys are stored "as cached": the bf16 values ARE the keys rotated at
    their old positions. A RoPE rotation of an isotropic N(0,1) vector is again
    N(0,1), so drawing the rotated key directly is the same distribution as
    drawing a base key and rotating it (BASELINE.json C1 "K/V generated with RoPE
    ... at positions 0..511"); this keeps the method's arithmetic out of here.
  * Salient tokens (BASELINE.json C1 "5% of cached tokens per segment get key
    norm scaled x4"): round_half_up(frac*len) tokens per pool segment, seeded
    permutation, key row multiplied by 4 before bf16 rounding; K_fresh of the
    same token carries the same x4.
  * All segment lengths and positions are multiples of the page size 16
    (reuse-segment boundaries are padded to the block size).
  * Physical page ids are a seeded permutation (gathers are never contiguous).

Pool layout (one layer): K and V pools, each uint16[num_blocks][Hkv][16][128]
holding bf16 bit patterns.
"""
from __future__ import annotations

import dataclasses
from concurrent.futures import ThreadPoolExecutor
from typing import List, Optional, Sequence, Tuple

import numpy as np

ROOT_SEED = 260601751
PAGE = 16
HEAD_DIM = 128

T_LAYOUT, T_KC, T_VC, T_Q, T_KF, T_VF, T_SAL, T_PERM = range(8)


def _rng(cfg: int, layer: int, tensor_id: int, index: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence(
        [ROOT_SEED, cfg, layer, tensor_id, index])))


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even float32 -> bf16 bit pattern (uint16). Finite inputs."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + r) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    return bf16_bits_to_f32(b).astype(np.float64)


def _normal_bf16(rng: np.random.Generator, shape, row_scale: Optional[np.ndarray] = None) -> np.ndarray:
    x = rng.standard_normal(shape, dtype=np.float32)
    if row_scale is not None:
        x *= row_scale.astype(np.float32).reshape((-1,) + (1,) * (x.ndim - 1))
    return f32_to_bf16_bits(x)


@dataclasses.dataclass
class PoolSegment:
    length: int
    old_pos: int


@dataclasses.dataclass
class Layout:
    """Block-table / segment-map descriptor of one batch (host mirror; shared by all layers)."""
    name: str
    cfg_id: int
    num_q_heads: int
    num_kv_heads: int
    rope_theta: float
    rope_style: int
    num_blocks: int
    num_reqs: int
    max_pages_per_req: int
    seq_len: np.ndarray            # int32 [num_reqs]
    tok_off: np.ndarray            # int32 [num_reqs+1] prefix sum of seq_len
    k_block_table: np.ndarray      # int32 [num_reqs][max_pages_per_req]; -1 = unused
    v_block_table: np.ndarray      # int32, same shape
    cow_private: np.ndarray        # int32, same shape; -1 = no COW for that page
    segments: np.ndarray           # int32 [num_segments][5] = (req, len, old_pos, new_pos, src_off)
    seg_pool_id: np.ndarray        # int32 [num_segments] which pool segment it came from
    src_blocks: np.ndarray         # int32 concatenated source page ids
    new_off: np.ndarray            # int32 [num_reqs+1]
    new_idx: np.ndarray            # int32 sorted positions of I_nr, per request
    k_per_req: np.ndarray          # int32 [num_reqs] top-k budget
    pool_segments: List[PoolSegment]
    pool_seg_pages: List[np.ndarray]   # physical source pages of each pool segment
    salient_frac: float
    pool_salient: List[np.ndarray]     # bool [len] per pool segment
    cow: bool
    zero_copy: bool = False            # K tables alias the cached source pages too (include/sparsex.h, zero-copy mode)

    @property
    def num_segments(self) -> int:
        return int(self.segments.shape[0])

    @property
    def total_tokens(self) -> int:
        return int(self.tok_off[-1])

    @property
    def total_new(self) -> int:
        return int(self.new_off[-1])

    @property
    def total_cached(self) -> int:
        return self.total_tokens - self.total_new

    @property
    def total_seg_pages(self) -> int:
        return int(self.segments[:, 1].sum() // PAGE) if self.num_segments else 0

    def cached_mask(self, req: int) -> np.ndarray:
        """bool [T_req]: position is covered by a reused segment (I_reuse, the top-k candidates)."""
        m = np.zeros(int(self.seq_len[req]), dtype=bool)
        for s in range(self.num_segments):
            r, ln, _, new_pos, _ = (int(v) for v in self.segments[s])
            if r == req:
                m[new_pos:new_pos + ln] = True
        return m

    def prefix_mask(self, req: int) -> np.ndarray:
        """bool [T_req]: prefix-cache hit (neither new nor in a segment)."""
        return ~(self.cached_mask(req) | self.is_new_mask(req))

    def is_new_mask(self, req: int) -> np.ndarray:
        m = np.zeros(int(self.seq_len[req]), dtype=bool)
        m[self.new_idx[self.new_off[req]:self.new_off[req + 1]]] = True
        return m

    def salient_mask(self, req: int) -> np.ndarray:
        """bool [T_req]: position holds a salient cached token."""
        m = np.zeros(int(self.seq_len[req]), dtype=bool)
        for s in range(self.num_segments):
            r, ln, _, new_pos, _ = (int(v) for v in self.segments[s])
            if r == req:
                n = len(m[new_pos:new_pos + ln])     # a trimmed request ends inside its last segment
                m[new_pos:new_pos + ln] = self.pool_salient[int(self.seg_pool_id[s])][:n]
        return m


@dataclasses.dataclass
class LayerTensors:
    """bf16 bit patterns (uint16) of one layer's pool and per-token inputs."""
    layer: int
    pool_k: np.ndarray   # [num_blocks][Hkv][16][128]; source pages filled, others 0
    pool_v: np.ndarray
    q_full: np.ndarray   # [sum T][Hq][128]    queries, already rotated at their positions
    k_fresh: np.ndarray  # [sum T][Hkv][128]   recomputed keys (rotated at new positions)
    v_fresh: np.ndarray  # [sum T][Hkv][128]


# ("new", length) | ("seg", pool_segment_id) | ("prefix", length): positions whose K/V the request's own pages
# already hold at the right positions (prefix-cache hits, Alg. 1 l.501): keys only, no queries, never candidates
ReqSpec = Sequence[Tuple[str, int]]


def build_layout(name: str, cfg_id: int, num_q_heads: int, num_kv_heads: int, rope_theta: float,
                 pool_segments: Sequence[PoolSegment], requests: Sequence[ReqSpec],
                 ratios: Sequence[float], salient_frac: float, cow: bool = False,
                 rope_style: int = 0, k_override: Optional[Sequence[int]] = None,
                 trim: Optional[Sequence[int]] = None) -> Layout:
    """trim[r] (< 16): tokens cut from the END of request r, whose last item must then be a segment: the
    segment's last page straddles seq_len (ragged tail inside a reused segment, reading A19)."""
    pool_segments = list(pool_segments)
    for ps in pool_segments:
        assert ps.length % PAGE == 0 and ps.old_pos % PAGE == 0 and ps.length > 0
    num_reqs = len(requests)
    seq_len = np.zeros(num_reqs, dtype=np.int32)
    for r, spec in enumerate(requests):
        t = 0
        for kind, val in spec:
            t += val if kind in ("new", "prefix") else pool_segments[val].length
        seq_len[r] = t
    if trim is not None:
        for r, cut in enumerate(trim):
            assert 0 <= cut < PAGE and (cut == 0 or requests[r][-1][0] == "seg")
            seq_len[r] -= cut
    pages_per_req = (seq_len + PAGE - 1) // PAGE
    max_pages = int(pages_per_req.max())
    n_src = sum(ps.length // PAGE for ps in pool_segments)
    num_blocks = n_src + int(pages_per_req.sum())
    perm = _rng(cfg_id, 0, T_PERM, 0).permutation(num_blocks).astype(np.int32)
    cur = 0
    pool_seg_pages = []
    for ps in pool_segments:
        n = ps.length // PAGE
        pool_seg_pages.append(perm[cur:cur + n].copy())
        cur += n
    kbt = np.full((num_reqs, max_pages), -1, dtype=np.int32)
    for r in range(num_reqs):
        n = int(pages_per_req[r])
        kbt[r, :n] = perm[cur:cur + n]
        cur += n
    vbt = kbt.copy()
    cowp = np.full_like(kbt, -1)
    segs, seg_pool_id, src_blocks, new_idx, new_off = [], [], [], [], [0]
    for r, spec in enumerate(requests):
        pos = 0
        for kind, val in spec:
            if kind == "new":
                assert val % PAGE == 0 or pos + val == seq_len[r]
                new_idx.append(np.arange(pos, pos + val, dtype=np.int32))
                pos += val
            elif kind == "prefix":
                assert pos % PAGE == 0 and val % PAGE == 0
                pos += val
            else:
                ps = pool_segments[val]
                assert pos % PAGE == 0
                segs.append((r, ps.length, ps.old_pos, pos, sum(len(b) for b in src_blocks)))
                seg_pool_id.append(val)
                src_blocks.append(pool_seg_pages[val])
                if cow:   # V pages alias the shared source pages until written
                    p0 = pos // PAGE
                    n = ps.length // PAGE
                    cowp[r, p0:p0 + n] = kbt[r, p0:p0 + n]
                    vbt[r, p0:p0 + n] = pool_seg_pages[val]
                pos += ps.length
        new_off.append(sum(len(a) for a in new_idx))
    tok_off = np.concatenate([[0], np.cumsum(seq_len)]).astype(np.int32)
    n_new = np.diff(np.asarray(new_off))
    n_cached = np.zeros(num_reqs, dtype=np.int64)       # |I_reuse|: segment tokens (prefix hits are not candidates)
    for (r, ln, _old, _new, _off) in segs:
        n_cached[r] += ln
    if k_override is not None:
        k_per_req = np.asarray(k_override, dtype=np.int32)
    else:
        k_per_req = np.asarray([int(np.floor(ratios[r] * int(n_cached[r]) + 1e-9))
                                for r in range(num_reqs)], dtype=np.int32)
    pool_salient = []
    for s, ps in enumerate(pool_segments):
        n_sal = int(np.floor(salient_frac * ps.length + 0.5))
        m = np.zeros(ps.length, dtype=bool)
        m[_rng(cfg_id, 0, T_SAL, s).permutation(ps.length)[:n_sal]] = True
        pool_salient.append(m)
    return Layout(
        name=name, cfg_id=cfg_id, num_q_heads=num_q_heads, num_kv_heads=num_kv_heads,
        rope_theta=float(rope_theta), rope_style=rope_style, num_blocks=num_blocks, num_reqs=num_reqs,
        max_pages_per_req=max_pages, seq_len=seq_len, tok_off=tok_off, k_block_table=kbt,
        v_block_table=vbt, cow_private=cowp,
        segments=np.asarray(segs, dtype=np.int32).reshape(-1, 5),
        seg_pool_id=np.asarray(seg_pool_id, dtype=np.int32),
        src_blocks=(np.concatenate(src_blocks).astype(np.int32) if src_blocks else np.zeros(0, np.int32)),
        new_off=np.asarray(new_off, dtype=np.int32),
        new_idx=(np.concatenate(new_idx).astype(np.int32) if new_idx else np.zeros(0, np.int32)),
        k_per_req=k_per_req, pool_segments=pool_segments, pool_seg_pages=pool_seg_pages,
        salient_frac=salient_frac, pool_salient=pool_salient, cow=cow)


def zero_copy_layout(lay: Layout) -> Layout:
    """The same batch described for zero-copy mode (include/sparsex.h): the K and V table entries of every reused
    page point at the shared source page, the request's own page becomes the reserved private page (cow_private)
    that the first scatter into the page fills."""
    kbt, cowp = lay.k_block_table.copy(), np.full_like(lay.k_block_table, -1)
    for (r, ln, _old, new_pos, src_off) in (tuple(int(v) for v in s) for s in lay.segments):
        p0, n = new_pos // PAGE, ln // PAGE
        cowp[r, p0:p0 + n] = lay.k_block_table[r, p0:p0 + n]
        kbt[r, p0:p0 + n] = lay.src_blocks[src_off:src_off + n]
    return dataclasses.replace(lay, name=lay.name + "-zc", k_block_table=kbt, v_block_table=kbt.copy(),
                               cow_private=cowp, cow=True, zero_copy=True)


def build_layer(lay: Layout, layer: int = 0, threads: int = 8, need_q: bool = True) -> LayerTensors:
    """Draw one layer's tensors. Every chunk has its own seed, so chunks are drawn in parallel."""
    hq, hkv, d = lay.num_q_heads, lay.num_kv_heads, HEAD_DIM
    pool_k = np.zeros((lay.num_blocks, hkv, PAGE, d), dtype=np.uint16)
    pool_v = np.zeros_like(pool_k)
    total = lay.total_tokens
    q_full = np.zeros((total if need_q else 0, hq, d), dtype=np.uint16)
    k_fresh = np.zeros((total, hkv, d), dtype=np.uint16)
    v_fresh = np.zeros((total, hkv, d), dtype=np.uint16)

    def do_pool_seg(s: int):
        ps = lay.pool_segments[s]
        scale = np.where(lay.pool_salient[s], 4.0, 1.0)
        kc = _normal_bf16(_rng(lay.cfg_id, layer, T_KC, s), (ps.length, hkv, d), scale)
        vc = _normal_bf16(_rng(lay.cfg_id, layer, T_VC, s), (ps.length, hkv, d))
        pages = lay.pool_seg_pages[s]
        # [len][Hkv][D] -> [pages][16][Hkv][D] -> [pages][Hkv][16][D]
        pool_k[pages] = kc.reshape(-1, PAGE, hkv, d).transpose(0, 2, 1, 3)
        pool_v[pages] = vc.reshape(-1, PAGE, hkv, d).transpose(0, 2, 1, 3)

    # token chunks of <= 8192 tokens, each with its own seed index
    CH = 8192

    def do_tok_chunk(args):
        r, c = args
        t = int(lay.seq_len[r])
        lo, hi = c * CH, min(t, (c + 1) * CH)
        o = int(lay.tok_off[r])
        idx = r * 4096 + c
        scale = np.where(lay.salient_mask(r)[lo:hi], 4.0, 1.0)
        if need_q:
            q_full[o + lo:o + hi] = _normal_bf16(_rng(lay.cfg_id, layer, T_Q, idx), (hi - lo, hq, d))
        k_fresh[o + lo:o + hi] = _normal_bf16(_rng(lay.cfg_id, layer, T_KF, idx), (hi - lo, hkv, d), scale)
        v_fresh[o + lo:o + hi] = _normal_bf16(_rng(lay.cfg_id, layer, T_VF, idx), (hi - lo, hkv, d))

    chunks = [(r, c) for r in range(lay.num_reqs) for c in range((int(lay.seq_len[r]) + CH - 1) // CH)]
    with ThreadPoolExecutor(max_workers=max(1, threads)) as ex:
        list(ex.map(do_pool_seg, range(len(lay.pool_segments))))
        list(ex.map(do_tok_chunk, chunks))
    # prefix-cache hits: the request's own pages already hold their K/V (here: the fresh rows of those positions)
    for r in range(lay.num_reqs):
        o = int(lay.tok_off[r])
        for pos in np.nonzero(lay.prefix_mask(r))[0]:
            pool_k[lay.k_block_table[r, pos // PAGE], :, pos % PAGE, :] = k_fresh[o + pos]
            pool_v[lay.v_block_table[r, pos // PAGE], :, pos % PAGE, :] = v_fresh[o + pos]
    return LayerTensors(layer=layer, pool_k=pool_k, pool_v=pool_v, q_full=q_full,
                        k_fresh=k_fresh, v_fresh=v_fresh)


# --------------------------------------------------------------------------------------
# The five configs of BASELINE.json (C1..C5), each with a `scale` knob for small test cases.
# --------------------------------------------------------------------------------------

def _r16(x: float, lo: int = PAGE) -> int:
    return max(lo, int(round(x / PAGE)) * PAGE)


def _split_gaps(rng: np.random.Generator, total: int, n: int) -> List[int]:
    """Split `total` tokens (multiple of 16) into n gaps, each a multiple of 16 and >= 16 (Dirichlet(1))."""
    units = total // PAGE
    assert units >= n
    w = rng.dirichlet(np.ones(n))
    extra = np.floor(w * (units - n)).astype(np.int64)
    rem = (units - n) - int(extra.sum())
    extra[:rem] += 1
    return [int((1 + e) * PAGE) for e in extra]


def _interleave(rng, seg_ids, n_new_total):
    gaps = _split_gaps(rng, n_new_total, len(seg_ids) + 1)
    spec = [("new", gaps[0])]
    for i, s in enumerate(seg_ids):
        spec.append(("seg", int(s)))
        spec.append(("new", gaps[i + 1]))
    return spec


def config_c1(scale: float = 1.0, ratio: float = 0.15) -> Layout:
    """C1: 1 request, 8Q/2KV heads, new128|segA|new128|segB|new128|segC|new128, theta 1e4, 5% salient."""
    seg = _r16(512 * scale)
    new = _r16(128 * scale)
    pool = [PoolSegment(seg, 0) for _ in range(3)]
    spec = [("new", new), ("seg", 0), ("new", new), ("seg", 1), ("new", new), ("seg", 2), ("new", new)]
    return build_layout("C1", 1, 8, 2, 10000.0, pool, [spec], [ratio], 0.05)


def config_c2(scale: float = 1.0, num_reqs: int = 4, ratio: float = 0.15) -> Layout:
    """C2: Llama-3-8B shape 32Q/8KV, 4 requests x 8K = 6 segments of 1024 from a pool of 16 + 2048 new."""
    rng = _rng(2, 0, T_LAYOUT, 0)
    seg = _r16(1024 * scale)
    pool = [PoolSegment(seg, int(rng.integers(0, 449)) * PAGE) for _ in range(16)]
    reqs = []
    for _ in range(num_reqs):
        ids = rng.permutation(16)[:6]
        reqs.append(_interleave(rng, ids, _r16(2048 * scale, 7 * PAGE)))
    return build_layout("C2", 2, 32, 8, 500000.0, pool, reqs, [ratio] * num_reqs, 0.05)


def config_c3(scale: float = 1.0, ratio: float = 0.10, turns: int = 10) -> Layout:
    """C3: one 32K request, 10 cached history turns of 2-4K (sum 30208) interleaved with 10 new turns of 256."""
    rng = _rng(3, 0, T_LAYOUT, 0)
    new = _r16(256 * scale)
    target = _r16(30208 * scale * turns / 10)
    lo, hi = max(1, int(128 * scale)), max(1, int(256 * scale))
    units = rng.integers(lo, hi + 1, size=turns).astype(np.int64)
    # adjust to the exact total, staying inside [lo, hi]
    need = target // PAGE - int(units.sum())
    i = 0
    while need != 0:
        step = 1 if need > 0 else -1
        if lo <= units[i % turns] + step <= hi:
            units[i % turns] += step
            need -= step
        i += 1
        if i > 100000:
            raise RuntimeError("cannot reach the C3 history total")
    pool, spec, old = [], [], 0
    for t in range(turns):
        ln = int(units[t]) * PAGE
        pool.append(PoolSegment(ln, old))       # history cached back-to-back in earlier rounds
        old += ln
        spec += [("seg", t), ("new", new)]
    return build_layout("C3", 3, 32, 8, 500000.0, pool, [spec], [ratio], 0.03)


def config_c4(scale: float = 1.0, num_reqs: int = 16, cow: bool = False) -> Layout:
    """C4: 16 requests over a shared pool of 64 segments of 1-4K; 4-8 segments each + 512 new; ratio U[0.1,0.3]."""
    rng = _rng(4, 0, T_LAYOUT, 0)
    lo, hi = max(1, int(64 * scale)), max(1, int(256 * scale))
    pool = [PoolSegment(int(rng.integers(lo, hi + 1)) * PAGE, int(rng.integers(0, 1024)) * PAGE)
            for _ in range(64)]
    reqs, ratios = [], []
    for _ in range(num_reqs):
        n_seg = int(rng.integers(4, 9))
        ids = rng.permutation(64)[:n_seg]
        reqs.append(_interleave(rng, ids, _r16(512 * scale, (n_seg + 1) * PAGE)))
        ratios.append(float(rng.uniform(0.10, 0.30)))
    return build_layout("C4-cow" if cow else "C4", 4, 32, 8, 500000.0, pool, reqs, ratios, 0.05, cow=cow)


def config_c5(scale: float = 1.0, ratio: float = 0.05) -> Layout:
    """C5: 128K of 32 cached 4K segments + 2K new, 28Q/4KV heads, 1% salient; all segments cached at 0."""
    seg = _r16(4096 * scale)
    pool = [PoolSegment(seg, 0) for _ in range(32)]
    news = [_r16(512 * scale), _r16(256 * scale), _r16(256 * scale), _r16(256 * scale), _r16(768 * scale)]
    spec = [("new", news[0])]
    for grp in range(4):
        spec += [("seg", grp * 8 + i) for i in range(8)]
        spec.append(("new", news[grp + 1]))
    return build_layout("C5", 5, 28, 4, 500000.0, pool, [spec], [ratio], 0.01)


CONFIGS = {"C1": config_c1, "C2": config_c2, "C3": config_c3, "C4": config_c4, "C5": config_c5}


def config_tail(seed_id: int = 15, prefix: int = 0, trim: Optional[Sequence[int]] = None,
                k_override: Sequence[int] = (8, 4, 19)) -> Layout:
    """Requests that END inside a reused segment (tail fallback) and whose new-token intervals
    touch reused segments on both sides (overflow): request 0 ends with a 96-token segment
    (tail = its last 64 tokens), request 1 with a 32-token one (tail = all of it), request 2 ends with new
    tokens (no tail) and starts with new tokens (no block before the first interval)."""
    pool = [PoolSegment(32, 64), PoolSegment(48, 0), PoolSegment(16, 160), PoolSegment(96, 32)]
    reqs = [[("new", 16), ("seg", 0), ("new", 16), ("seg", 1), ("seg", 3)],
            [("seg", 2), ("new", 32), ("seg", 0)],
            [("new", 32), ("seg", 1), ("new", 16), ("seg", 2), ("new", 16)]]
    if prefix:  # prefix-cache hits in front of every request: the first new interval of requests 0 and 2 then has a
        # prefix-hit block before it, which the overflow must NOT pull in
        reqs = [[("prefix", prefix)] + spec for spec in reqs]
    # budgets below the number of cached tokens that some new query can see (the tokens behind the last new
    # token score exactly 0 and would turn the cut into a pure position tie)
    return build_layout("tail", seed_id, 4, 2, 10000.0, pool, reqs, [0.2, 0.25, 0.3], 0.1, k_override=list(k_override),
                        trim=trim)


def config_tiny(seed_id: int = 9, num_q_heads: int = 4, num_kv_heads: int = 2, tail: int = 0,
                rope_style: int = 0, cow: bool = False, prefix: int = 0) -> Layout:
    """Two small requests with uneven segments, negative and zero deltas; optional ragged tail (T % 16 != 0);
    prefix > 0: both requests start with prefix-cache hits (2 * prefix and prefix tokens, multiples of 16)."""
    pool = [PoolSegment(32, 64), PoolSegment(48, 0), PoolSegment(16, 160)]
    reqs = [[("new", 16), ("seg", 0), ("new", 32), ("seg", 1), ("new", 16 + tail)],
            [("seg", 2), ("new", 16), ("seg", 0), ("new", 16)]]
    if prefix:
        reqs = [[("prefix", 2 * prefix)] + reqs[0], [("prefix", prefix)] + reqs[1]]
    return build_layout("tiny", seed_id, num_q_heads, num_kv_heads, 10000.0, pool, reqs, [0.25, 0.5], 0.1,
                        cow=cow, rope_style=rope_style)
