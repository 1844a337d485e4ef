"""Pins of the fp64 oracle against what the paper and the mathematics fix (CPU only).

The paper prints no worked numeric example for this path, so the pins are: closed forms, invariants,
special cases that reduce to a library routine written independently (fp64 torch SDPA, numpy sort),
and brute-force python loops on tiny inputs. Each pin is chosen so a plausible mistake (dropped term,
wrong sign/index, transposed operand, wrong head mapping, off-by-one causal mask) fails it.
"""
import math

import numpy as np
import pytest
import torch

from oracle import sx_oracle as orc
from paper_2606_01751_b200 import workloads as wl

from helpers import oracle_layer

D = 128


def rbits(rng, shape, scale=1.0):
    return wl.f32_to_bf16_bits(rng.standard_normal(shape).astype(np.float32) * scale)


# ------------------------------------------------------------------ bf16 rounding

def test_f64_to_bf16_is_single_rne():
    # exactly representable values survive; ties go to even; no double rounding through fp32
    x = np.array([1.0, 1.0 + 2.0 ** -8, 1.0 + 3 * 2.0 ** -8, -2.5, 0.0, 1.0 + 2.0 ** -8 + 2.0 ** -40])
    got = orc.bf16_to_f64(orc.f64_to_bf16(x))
    # 1+2^-8 is a tie between 1 and 1+2^-7 -> even mantissa (1.0); 1+3*2^-8 tie -> 1+2^-6 (even)
    assert got.tolist() == [1.0, 1.0, 1.0 + 2.0 ** -6, -2.5, 0.0, 1.0 + 2.0 ** -7]
    # a value that double rounding (fp64->fp32->bf16) gets wrong: just below a bf16 tie, within half an
    # fp32 ulp of it -> fp32 rounds up onto the tie, the tie then rounds to even (up); single RNE rounds down
    y = np.array([1.0 + 2.0 ** -8 + 2.0 ** -7 - 2.0 ** -30])   # just below the tie 1+3*2^-8
    assert orc.bf16_to_f64(orc.f64_to_bf16(y))[0] == 1.0 + 2.0 ** -7
    rng = np.random.default_rng(1)
    b = rbits(rng, 4096, 3.0)
    assert np.array_equal(orc.f64_to_bf16(orc.bf16_to_f64(b)), b)   # round trip on representable values


# ------------------------------------------------------------------ O-a: RoPE re-alignment

@pytest.mark.parametrize("style", [0, 1])
@pytest.mark.parametrize("theta", [1e4, 5e5])
def test_rope_composition(style, theta):
    # PAPER.md:147  R_{n'} k = R_{n'-n} R_n k ; positions up to the C5 range
    rng = np.random.default_rng(2)
    k = rng.standard_normal((7, D))
    for p1, p2 in [(0, 512), (511, 2047), (64, 0), (4096, 133104), (131071, 3)]:
        a = orc.rope_rotate(orc.rope_rotate(k, p1, theta, style), p2 - p1, theta, style)
        b = orc.rope_rotate(k, p2, theta, style)
        assert np.max(np.abs(a - b)) < 1e-9


def test_rope_hand_case_d2():
    # D = 2, theta_0 = base^0 = 1: k = (1, 0) -> (cos delta, sin delta); k = (0, 1) -> (-sin, cos)
    for delta in [1, -3, 7]:
        for style in (0, 1):
            got = orc.rope_rotate(np.array([[1.0, 0.0], [0.0, 1.0]]), delta, 10000.0, style)
            assert np.allclose(got[0], [math.cos(delta), math.sin(delta)], atol=1e-15)
            assert np.allclose(got[1], [-math.sin(delta), math.cos(delta)], atol=1e-15)


def test_rope_frequencies_and_pairing():
    # D = 4, base 10000: theta = (1, 1/100). style 0 pairs (0,2),(1,3); style 1 pairs (0,1),(2,3)
    delta = 5
    x = np.array([1.0, 2.0, 3.0, 4.0])
    c0, s0, c1, s1 = math.cos(5.0), math.sin(5.0), math.cos(0.05), math.sin(0.05)
    want0 = [1 * c0 - 3 * s0, 2 * c1 - 4 * s1, 1 * s0 + 3 * c0, 2 * s1 + 4 * c1]
    want1 = [1 * c0 - 2 * s0, 1 * s0 + 2 * c0, 3 * c1 - 4 * s1, 3 * s1 + 4 * c1]
    assert np.allclose(orc.rope_rotate(x, delta, 10000.0, 0), want0, atol=1e-14)
    assert np.allclose(orc.rope_rotate(x, delta, 10000.0, 1), want1, atol=1e-14)


def test_rope_norm_and_relative_position_identity():
    # PAPER.md:143  <R_m q, R_n k> = q^T R_{n-m} k, applied to a re-aligned key:
    # <R_m q, Align_delta(R_n k)> = <q, R_{n+delta-m} k>
    rng = np.random.default_rng(3)
    q, k = rng.standard_normal(D), rng.standard_normal(D)
    th = 5e5
    for m, n, delta in [(900, 100, 650), (70000, 5, 60000), (50, 300, -280)]:
        lhs = orc.rope_rotate(q, m, th) @ orc.rope_rotate(orc.rope_rotate(k, n, th), delta, th)
        rhs = q @ orc.rope_rotate(k, n + delta - m, th)
        assert abs(lhs - rhs) < 1e-9
    r = orc.rope_rotate(k, 12345, th)
    pair = k[:64] ** 2 + k[64:] ** 2
    assert np.allclose(r[:64] ** 2 + r[64:] ** 2, pair, rtol=1e-13)     # per-pair norm preserved


def test_realign_pages_v_bitcopy_delta0_and_destination():
    lay = wl.config_tiny()
    lt = wl.build_layer(lay)
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    ref = orc.realign(pk, pv, lay.k_block_table, lay.v_block_table, lay.segments, lay.src_blocks,
                      lay.rope_theta, 0)
    off = 0
    for s in range(lay.num_segments):
        req, ln, old, new, so = (int(v) for v in lay.segments[s])
        for j in range(ln):
            src = lay.src_blocks[so + j // 16]
            dst = lay.k_block_table[req, (new + j) // 16]
            # V: bit-identical copy
            assert np.array_equal(pv[dst, :, (new + j) % 16], lt.pool_v[src, :, j % 16])
            want = orc.rope_rotate(orc.bf16_to_f64(lt.pool_k[src, :, j % 16]), new - old, lay.rope_theta)
            assert np.array_equal(ref[off + j], want)
            assert np.array_equal(pk[dst, :, (new + j) % 16], orc.f64_to_bf16(want))
        off += ln
    # source pages never written
    for pages in lay.pool_seg_pages:
        assert np.array_equal(pk[pages], lt.pool_k[pages]) and np.array_equal(pv[pages], lt.pool_v[pages])
    # delta = 0 -> K pages bit-identical
    seg0 = lay.segments.copy()
    seg0[:, 2] = seg0[:, 3]
    pk2, pv2 = lt.pool_k.copy(), lt.pool_v.copy()
    orc.realign(pk2, pv2, lay.k_block_table, lay.v_block_table, seg0, lay.src_blocks, lay.rope_theta, 0)
    req, ln, old, new, so = (int(v) for v in seg0[0])
    assert np.array_equal(pk2[lay.k_block_table[req, new // 16]], lt.pool_k[lay.src_blocks[so]])


# ------------------------------------------------------------------ O-d: scatter

def test_scatter_untouched_idempotent_roundtrip_and_cow():
    lay = wl.config_tiny(cow=True)
    lt = wl.build_layer(lay)
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta)
    # under COW realign leaves V pages aliased: no private V page was written
    assert np.array_equal(pv, lt.pool_v)
    r = 0
    t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
    before_k = orc.gather_tokens(pk, kt[r], t).copy()
    before_v = orc.gather_tokens(pv, vt[r], t).copy()
    rows = np.array([3, 17, 18, 40, 95], dtype=np.int32)   # 17, 18, 40 lie in cached (aliased) pages
    kf, vf = lt.k_fresh[o + rows], lt.v_fresh[o + rows]
    orc.scatter_kv(pk, pv, kt, vt, lay.cow_private, r, rows, kf, vf)
    after_k = orc.gather_tokens(pk, kt[r], t)
    after_v = orc.gather_tokens(pv, vt[r], t)
    assert np.array_equal(after_k[rows], kf) and np.array_equal(after_v[rows], vf)   # gather o scatter = id
    keep = np.setdiff1d(np.arange(t), rows)
    assert np.array_equal(after_k[keep], before_k[keep]) and np.array_equal(after_v[keep], before_v[keep])
    # shared source pages are unchanged, touched V pages flipped to the host-reserved private ids
    for pages in lay.pool_seg_pages:
        assert np.array_equal(pv[pages], lt.pool_v[pages]) and np.array_equal(pk[pages], lt.pool_k[pages])
    touched = np.unique(rows // 16)
    for pg in range(kt.shape[1]):
        if lay.cow_private[r, pg] >= 0 and pg in touched:
            assert vt[r, pg] == lay.cow_private[r, pg]
        else:
            assert vt[r, pg] == lay.v_block_table[r, pg]
    assert np.array_equal(vt[1], lay.v_block_table[1])
    # idempotent
    pk2, pv2, kt2, vt2 = pk.copy(), pv.copy(), kt.copy(), vt.copy()
    orc.scatter_kv(pk2, pv2, kt2, vt2, lay.cow_private, r, rows, kf, vf)
    assert np.array_equal(pk2, pk) and np.array_equal(pv2, pv) and np.array_equal(vt2, vt)


# ------------------------------------------------------------------ O-b: scores and top-k

def _tiny_problem(seed, t=45, hq=4, hkv=2, d=D, zero_q=False, new=(0, 1, 2, 3, 20, 21, 22, 44)):
    rng = np.random.default_rng(seed)
    nblk = (t + 15) // 16
    pool_k = rbits(rng, (nblk + 2, hkv, 16, d))
    pool_v = rbits(rng, (nblk + 2, hkv, 16, d))
    table = rng.permutation(nblk + 2)[:nblk].astype(np.int32)
    new_idx = np.asarray(new, dtype=np.int32)
    q = rbits(rng, (len(new_idx), hq, d))
    if zero_q:
        q[:] = 0
    return pool_k, pool_v, table, new_idx, q


def _brute_scores(pool_k, table, t, q, new_idx, hq):
    """Eq. (1)-(2) by explicit python loops (independent of the C code)."""
    hkv, d = pool_k.shape[1], pool_k.shape[3]
    g = hq // hkv
    K = orc.bf16_to_f64(orc.gather_tokens(pool_k, table, t))
    Q = orc.bf16_to_f64(q)
    s = [0.0] * t
    lse = np.zeros((len(new_idx), hq))
    for h in range(hq):
        for n, i in enumerate(new_idx.tolist()):
            logits = [sum(Q[n, h, x] * K[j, h // g, x] for x in range(d)) / math.sqrt(d) for j in range(i + 1)]
            m = max(logits)
            e = [math.exp(v - m) for v in logits]
            z = sum(e)
            for j in range(i + 1):
                s[j] += e[j] / z
            lse[n, h] = m + math.log(z)
    return np.asarray(s), lse


def test_scores_bruteforce_tiny():
    pool_k, _, table, new_idx, q = _tiny_problem(5, d=16)
    t = 45
    s, lse = orc.scores(pool_k, table, t, q, new_idx, 4, want_lse=True)
    bs, blse = _brute_scores(pool_k, table, t, q, new_idx, 4)
    assert np.max(np.abs(s - bs)) < 1e-12 and np.max(np.abs(lse - blse)) < 1e-12


def test_scores_sum_invariant_and_harmonic_closed_form():
    t, hq = 45, 4
    pool_k, _, table, new_idx, q = _tiny_problem(6)
    s = orc.scores(pool_k, table, t, q, new_idx, hq)
    # softmax rows sum to 1 (Eq. 1) => sum_j s_j = N_n * Hq (Eq. 2 + head sum)
    assert abs(s.sum() - len(new_idx) * hq) < 1e-10
    assert np.all(s[int(new_idx.max()) + 1:] == 0.0)     # keys after the last query are never seen
    # Q = 0 => A[i, j] = 1/(i+1) => s_j = Hq * sum_{i in I_nr, i >= j} 1/(i+1)
    pool_k, _, table, new_idx, q = _tiny_problem(7, zero_q=True)
    s0 = orc.scores(pool_k, table, t, q, new_idx, hq)
    want = np.array([hq * sum(1.0 / (i + 1) for i in new_idx.tolist() if i >= j) for j in range(t)])
    assert np.max(np.abs(s0 - want)) < 1e-12


def test_scores_gqa_head_mapping():
    # query head h must read KV head h // g: zero all queries but head 3 (-> kv head 1 with g = 2),
    # then changing kv head 0's keys must not change the scores, changing kv head 1's must.
    t, hq = 45, 4
    pool_k, _, table, new_idx, q = _tiny_problem(8)
    q[:, :3] = 0
    base = orc.scores(pool_k, table, t, q, new_idx, hq)
    p2 = pool_k.copy()
    p2[:, 0] = p2[::-1, 0]
    assert np.array_equal(orc.scores(p2, table, t, q, new_idx, hq), base)
    p3 = pool_k.copy()
    p3[:, 1] = p3[::-1, 1]
    assert not np.allclose(orc.scores(p3, table, t, q, new_idx, hq), base)


def test_topk_matches_full_sort_ties_and_edges():
    rng = np.random.default_rng(9)
    t = 64
    s = rng.random(t)
    s[[10, 11, 30, 31, 32]] = 0.5          # exact ties: lower position wins (reading A8)
    is_new = np.zeros(t, bool)
    is_new[[0, 1, 2, 40, 41, 63]] = True
    s[40] = 99.0                           # new tokens are never candidates (reading A7)
    cand = [j for j in range(t) if not is_new[j]]
    ranked = sorted(cand, key=lambda j: (-s[j], j))
    for k in [0, 1, 5, 29, len(cand), len(cand) + 7]:
        sel, rows = orc.select_topk(s, is_new, k)
        kk = min(k, len(cand))
        assert sel.tolist() == sorted(ranked[:kk])
        assert rows.tolist() == sorted(set(ranked[:kk]) | set(np.nonzero(is_new)[0].tolist()))
    # cut inside the tie group {10, 11, 30, 31, 32}
    n_above = int((s[cand] > 0.5).sum())
    sel, _ = orc.select_topk(s, is_new, n_above + 2)
    assert 10 in sel and 11 in sel and 30 not in sel


# ------------------------------------------------------------------ O-c: attention

def _sdpa_reference(pool_k, pool_v, table, t, q_all, hq):
    """Dense causal attention by fp64 torch SDPA with KV heads repeated g times (library special case)."""
    hkv = pool_k.shape[1]
    g = hq // hkv
    K = torch.from_numpy(orc.bf16_to_f64(orc.gather_tokens(pool_k, table, t)))   # [T][Hkv][D]
    V = torch.from_numpy(orc.bf16_to_f64(orc.gather_tokens(pool_v, table, t)))
    Q = torch.from_numpy(orc.bf16_to_f64(q_all))                                   # [T][Hq][D]
    K = K.repeat_interleave(g, dim=1).permute(1, 0, 2)
    V = V.repeat_interleave(g, dim=1).permute(1, 0, 2)
    o = torch.nn.functional.scaled_dot_product_attention(Q.permute(1, 0, 2)[None], K[None], V[None],
                                                         is_causal=True)
    return o[0].permute(1, 0, 2).numpy()


def test_attention_dense_equals_torch_sdpa_and_subset_rows():
    t, hq = 45, 4
    pool_k, pool_v, table, _, _ = _tiny_problem(10)
    rng = np.random.default_rng(11)
    q_all = rbits(rng, (t, hq, D))
    allrows = np.arange(t, dtype=np.int32)
    full, lse = orc.attention(pool_k, pool_v, table, table, t, q_all, allrows, hq, want_lse=True)
    want = _sdpa_reference(pool_k, pool_v, table, t, q_all, hq)
    assert np.max(np.abs(full - want)) < 1e-12
    # sparse rows == full attention restricted to those rows (Alg. 1 line 21)
    rows = np.array([0, 7, 16, 31, 44], dtype=np.int32)
    sub, lse_sub = orc.attention(pool_k, pool_v, table, table, t, q_all[rows], rows, hq, want_lse=True)
    assert np.array_equal(sub, full[rows]) and np.array_equal(lse_sub, lse[rows])
    # lse agrees with the score pass's normaliser on the same rows
    _, lse_b = orc.scores(pool_k, table, t, q_all[rows], rows, hq, want_lse=True)
    assert np.max(np.abs(lse_b - lse_sub)) < 1e-12


def test_attention_closed_forms():
    t, hq = 37, 4
    pool_k, pool_v, table, _, _ = _tiny_problem(12, t=37)
    allrows = np.arange(t, dtype=np.int32)
    # Q = 0 -> uniform weights -> O_r = mean of V[0..r]
    q0 = np.zeros((t, hq, D), dtype=np.uint16)
    o = orc.attention(pool_k, pool_v, table, table, t, q0, allrows, hq)
    V = orc.bf16_to_f64(orc.gather_tokens(pool_v, table, t))       # [T][Hkv][D]
    for r in (0, 1, 15, 16, 36):
        for h in range(hq):
            assert np.allclose(o[r, h], V[: r + 1, h // 2].mean(axis=0), atol=1e-13)
    # T = 1 -> O = V[0]
    assert np.array_equal(o[0, 3], V[0, 1])
    # constant V -> constant O whatever Q is; V and K tables are independent arguments
    rng = np.random.default_rng(13)
    q = rbits(rng, (t, hq, D))
    pv = pool_v.copy()
    pv[:] = wl.f32_to_bf16_bits(np.float32(1.5))
    o = orc.attention(pool_k, pv, table, table, t, q, allrows, hq)
    assert np.allclose(o, 1.5, atol=1e-13)


# ------------------------------------------------------------------ whole layer

def test_layer_ratio_100_equals_dense_attention_on_fresh_tensors():
    """k = N_c (ratio 100%) => every row recomputed: the output equals dense causal attention over
    (Q_full, K_fresh, V_fresh), whatever the cached pool and the deltas are (reading A13: this holds
    only with scatter BEFORE attention, the order of Alg. 1 lines 19 -> 21)."""
    lay = wl.config_tiny()
    lt = wl.build_layer(lay)
    n_c = lay.seq_len - np.diff(lay.new_off)
    res, pk, pv, kt, vt = oracle_layer(lay, lt, k_per_req=n_c)
    for r in range(lay.num_reqs):
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        assert res.rows[r].tolist() == list(range(t))
        # dense reference on a pool that only ever held the fresh tensors
        nblk = (t + 15) // 16
        fk = np.zeros((nblk, lay.num_kv_heads, 16, D), np.uint16)
        fv = np.zeros_like(fk)
        tab = np.arange(nblk, dtype=np.int32)
        pos = np.arange(t)
        fk[pos // 16, :, pos % 16] = lt.k_fresh[o:o + t]
        fv[pos // 16, :, pos % 16] = lt.v_fresh[o:o + t]
        want = _sdpa_reference(fk, fv, tab, t, lt.q_full[o:o + t], lay.num_q_heads)
        assert np.max(np.abs(res.out[r] - want)) < 1e-12
    # and the full-mode layer gives the same thing
    res_full, *_ = oracle_layer(lay, lt, mode="full")
    for r in range(lay.num_reqs):
        assert np.array_equal(res_full.out[r], res.out[r])


def test_layer_sparse_structure():
    lay = wl.config_tiny(tail=5)          # ragged last page
    lt = wl.build_layer(lay)
    res, pk, pv, kt, vt = oracle_layer(lay, lt)
    for r in range(lay.num_reqs):
        is_new = lay.is_new_mask(r)
        k = int(lay.k_per_req[r])
        assert len(res.sel[r]) == k and not is_new[res.sel[r]].any()
        assert len(res.rows[r]) == k + is_new.sum() and np.all(np.diff(res.rows[r]) > 0)
        # rows not in R keep the aligned cached K (bit-unchanged by the scatters)
        t = int(lay.seq_len[r])
        pk0, pv0 = lt.pool_k.copy(), lt.pool_v.copy()
        orc.realign(pk0, pv0, lay.k_block_table, lay.v_block_table, lay.segments, lay.src_blocks,
                    lay.rope_theta)
        keep = np.setdiff1d(np.arange(t), res.rows[r])
        a = orc.gather_tokens(pk, kt[r], t)[keep]
        b = orc.gather_tokens(pk0, lay.k_block_table[r], t)[keep]
        assert np.array_equal(a, b)


# ----------------------------------------------------------------------------- overflow / tail fallback

def test_recompute_set_hand_cases():
    """Alg. 1 l.535-539 on hand-written cases (block 16): expected lists typed from the definitions of
    PAPER.md:235 (tail: last 64 tokens of the final reused segment) and PAPER.md:241 (one block on each
    side of every Sparse-Q interval)."""
    # T = 96: cached [0,32), new [32,48), cached segment [48,96) which also ends the prompt
    is_new = np.zeros(96, dtype=bool)
    is_new[32:48] = True
    rows = orc.recompute_set(is_new, np.asarray([3]), [(0, 32), (48, 96)], overflow_blocks=1, tail_tokens=64)
    # S_ov = [16,32) U [48,64); S_tail = last 64 of segment [48,96) -> only 48 long -> [48,96); S_key = {3}
    assert rows.tolist() == [3] + list(range(16, 96))
    # tail segment longer than 64: only its last 64 positions
    is_new = np.zeros(160, dtype=bool)
    is_new[0:16] = True
    rows = orc.recompute_set(is_new, np.asarray([], dtype=np.int32), [(16, 160)], overflow_blocks=1, tail_tokens=64)
    assert rows.tolist() == list(range(0, 32)) + list(range(96, 160))     # new + one block after + tail
    # prompt ends with new tokens: no tail; interval at position 0 has no block before it
    is_new = np.zeros(96, dtype=bool)
    is_new[0:16] = True
    is_new[80:96] = True
    rows = orc.recompute_set(is_new, np.asarray([40, 41]), [(16, 80)], overflow_blocks=1, tail_tokens=64)
    assert rows.tolist() == list(range(0, 32)) + [40, 41] + list(range(64, 96))
    # two intervals 16 apart share the block between them; overflow 0 and tail 0 reduce to R = I_nr U S_key
    is_new = np.zeros(80, dtype=bool)
    is_new[16:32] = True
    is_new[48:64] = True
    rows = orc.recompute_set(is_new, np.asarray([70]), [(0, 16), (32, 48), (64, 80)], 1, 0)
    assert rows.tolist() == list(range(0, 80))
    rows = orc.recompute_set(is_new, np.asarray([70]), [(0, 16), (32, 48), (64, 80)], 0, 0)
    assert rows.tolist() == list(range(16, 32)) + list(range(48, 64)) + [70]
    _, plain = orc.select_topk(np.arange(80, dtype=np.float64), is_new, 0)
    assert np.array_equal(orc.recompute_set(is_new, np.asarray([], dtype=np.int32), [], 0, 0), plain)


def test_prefix_hits_are_never_candidates_nor_recomputed():
    """Alg. 1 l.501: "Prefix-cache hits, if present, are excluded from the current prefill computation."
    Hand case, T = 64: prefix hits [0,16), new [16,32), reused segment [32,64). The prefix positions carry
    the LARGEST scores and must still not be selected; overflow stops at the prefix (expected lists typed by hand)."""
    is_new = np.zeros(64, dtype=bool)
    is_new[16:32] = True
    cand = np.zeros(64, dtype=bool)
    cand[32:64] = True
    s = np.zeros(64)
    s[0:16] = 100.0                       # prefix hits: high scores, not candidates
    s[40], s[50], s[33] = 3.0, 2.0, 1.0
    sel, rows = orc.select_topk(s, is_new, 2, cand)
    assert sel.tolist() == [40, 50]
    assert rows.tolist() == list(range(16, 32)) + [40, 50]
    sel, _ = orc.select_topk(s, is_new, 1000, cand)      # the budget is clamped to |I_reuse| = 32
    assert sel.tolist() == list(range(32, 64))
    # default (no mask) = every position that is not new, as before
    sel, _ = orc.select_topk(s, is_new, 2)
    assert sel.tolist() == [0, 1]
    # overflow: one block after the interval (reused), none before it (prefix hit); tail: last position is reused
    rows = orc.recompute_set(is_new, np.asarray([40]), [(32, 64)], overflow_blocks=1, tail_tokens=8, cand_mask=cand)
    assert rows.tolist() == list(range(16, 48)) + list(range(56, 64))
    # a prompt that ENDS in prefix-hit tokens has no tail fallback
    cand2 = np.zeros(64, dtype=bool)
    cand2[0:16] = True                    # reused [0,16), new [16,32), prefix-like [32,64) (not candidates)
    rows = orc.recompute_set(is_new, np.asarray([], dtype=np.int32), [(0, 16)], 1, 8, cand_mask=cand2)
    assert rows.tolist() == list(range(0, 32))
