"""GPU parity: every stage of libsparsex.so against the fp64 oracle on identical seeded inputs,
element by element, through the C ABI (paper_2606_01751_b200.binding).

Bars (BASELINE.json north_star): selected index sets, R, block tables and scattered pages bit-exact;
re-rotated keys and attention outputs within max-abs 2e-2 / mean-abs 2e-3 of fp64 (keys: per-element
bound max(2e-2, 2^-7 |ref|), reading A12). Inputs get their top-k margin carved
(helpers.carve_margins, reading A10) so that the fp32 scorer and the fp64 oracle agree on the set.
"""
import numpy as np
import pytest
import torch

from oracle import sx_oracle as orc
from paper_2606_01751_b200 import workloads as wl

from helpers import carve_margins, carve_margins_fresh, check_close, oracle_layer

pytestmark = pytest.mark.gpu

SCORE_RTOL = 5e-3   # fp32 tensor-core scores vs fp64 (measured ~1e-5); carved margin is 1e-3 each side


def _gpu():
    from paper_2606_01751_b200 import binding as sx   # noqa: F401  (fails loudly if the .so is missing)
    from paper_2606_01751_b200.layer import GpuLayer, dev_to_bits
    return GpuLayer, dev_to_bits


CASES = {
    "tiny": lambda: wl.config_tiny(),
    "tiny-ragged": lambda: wl.config_tiny(seed_id=10, tail=5),
    "tiny-interleaved": lambda: wl.config_tiny(seed_id=11, rope_style=1),
    "tiny-g7": lambda: wl.config_tiny(seed_id=12, num_q_heads=7, num_kv_heads=1, tail=3),
    "tiny-g1": lambda: wl.config_tiny(seed_id=13, num_q_heads=2, num_kv_heads=2),
    "tiny-cow": lambda: wl.config_tiny(seed_id=14, cow=True),
    "tiny-prefix": lambda: wl.config_tiny(seed_id=15, prefix=16, tail=7),   # prefix-cache hits: keys only
    "C1": lambda: wl.config_c1(),
    "C2-quarter": lambda: wl.config_c2(scale=0.25),
    "C3-eighth": lambda: wl.config_c3(scale=0.125),
    "C4-eighth": lambda: wl.config_c4(scale=0.125, num_reqs=6),
    "C4-eighth-cow": lambda: wl.config_c4(scale=0.125, num_reqs=6, cow=True),
    "C5-1/16": lambda: wl.config_c5(scale=1.0 / 16),
}

_cache = {}


def prepared(name):
    """(layout, carved layer tensors, oracle sparse-layer result and final pool/tables)."""
    if name not in _cache:
        lay = CASES[name]()
        lt = wl.build_layer(lay, 0)
        carve_margins(lay, lt)
        res, pk, pv, kt, vt = oracle_layer(lay, lt, mode="sparse")
        _cache[name] = (lay, lt, res, pk, pv, kt, vt)
    return _cache[name]


def _logical_view(pool_bits, table, seq_len):
    return [orc.gather_tokens(pool_bits, table[r], int(seq_len[r])) for r in range(len(seq_len))]


@pytest.mark.parametrize("name", list(CASES))
def test_realign_stage(name):
    GpuLayer, dev_to_bits = _gpu()
    lay, lt = prepared(name)[:2]
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    ref64 = orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    g = GpuLayer(lay, lt)
    g.realign()
    torch.cuda.synchronize()
    gk, gv = dev_to_bits(g.pool_k), dev_to_bits(g.pool_v)
    # V pages: bit copies; every page the oracle did not touch is unchanged
    assert np.array_equal(gv, pv)
    touched = np.zeros(lay.num_blocks, dtype=bool)
    got = []
    for (req, ln, old, new, so) in lay.segments.tolist():
        for pg in range(ln // 16):
            blk = int(kt[req][new // 16 + pg])
            touched[blk] = True
            got.append(np.transpose(orc.bf16_to_f64(gk[blk]), (1, 0, 2)))
    assert np.array_equal(gk[~touched], lt.pool_k[~touched])
    got = np.concatenate(got, axis=0)
    worst, mean = check_close(name + " realigned K", got, ref64, ulp_floor=True)
    # the GPU result may differ from the oracle's own bf16 rounding by one ulp only
    exact = np.mean(gk[touched] == pk[touched])
    assert exact > 0.995, exact
    # delta = 0 segments must come out bit-identical (PAPER.md:147 with n' = n)
    for (req, ln, old, new, so) in lay.segments.tolist():
        if old == new:
            for pg in range(ln // 16):
                assert np.array_equal(gk[int(kt[req][new // 16 + pg])], lt.pool_k[int(lay.src_blocks[so + pg])])


@pytest.mark.parametrize("name", list(CASES))
def test_scatter_stage(name):
    GpuLayer, dev_to_bits = _gpu()
    lay, lt = prepared(name)[:2]
    # oracle: realign then scatter the new tokens then an arbitrary strided subset of cached rows
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    cow = lay.cow_private if lay.cow else None
    orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    g = GpuLayer(lay, lt)
    # start the GPU from the ORACLE's realigned pool so the comparison below is bit-exact
    g.pool_k.copy_(torch.from_numpy(pk.view(np.int16)))
    g.pool_v.copy_(torch.from_numpy(pv.view(np.int16)))
    rows_all, off = [], [0]
    for r in range(lay.num_reqs):
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        nidx = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]
        orc.scatter_kv(pk, pv, kt, vt, cow, r, nidx, lt.k_fresh[o + nidx], lt.v_fresh[o + nidx])
        extra = np.nonzero(~lay.is_new_mask(r))[0][::3].astype(np.int32)
        orc.scatter_kv(pk, pv, kt, vt, cow, r, extra, lt.k_fresh[o + extra], lt.v_fresh[o + extra])
        rows_all.append(extra)
        off.append(off[-1] + len(extra))
    g.scatter_new()
    sel = torch.from_numpy(np.concatenate(rows_all)).to(g.dev)
    g.sel_off = torch.tensor(off, dtype=torch.int32, device=g.dev)
    g.rows_off = g.sel_off   # only used for index staging below
    g.stage_rows(sel, sel)
    g.scatter_sel()
    torch.cuda.synchronize()
    assert np.array_equal(dev_to_bits(g.pool_k), pk)
    assert np.array_equal(dev_to_bits(g.pool_v), pv)
    assert np.array_equal(g.batch.k_block_table.cpu().numpy(), kt)
    assert np.array_equal(g.batch.v_block_table.cpu().numpy(), vt)


@pytest.mark.parametrize("pair", [False, True], ids=["1cta", "cta-pair"])
@pytest.mark.parametrize("name", list(CASES))
def test_sparse_layer_chained(name, pair):
    """Whole sparse layer on the GPU (its own outputs feed the next stage) vs the oracle layer driver.
    cta-pair: stage (c) with SX_ATTN_CTA_PAIR (2-CTA clusters, odd pair counts and ragged tails included)."""
    GpuLayer, dev_to_bits = _gpu()
    lay, lt, res, pk, pv, kt, vt = prepared(name)
    g = GpuLayer(lay, lt)
    g.cta_pair = pair
    g.step_sparse()
    torch.cuda.synchronize()
    sc = g.scores.cpu().numpy().astype(np.float64)
    sel = g.sel_idx.cpu().numpy()
    rows = g.rows_R.cpu().numpy()
    out = orc.bf16_to_f64(dev_to_bits(g.out))
    lse = g.lse.cpu().numpy().astype(np.float64)
    for r in range(lay.num_reqs):
        o, t = int(lay.tok_off[r]), int(lay.seq_len[r])
        ref_s = res.scores[r]
        rel = np.abs(sc[o:o + t] - ref_s) / (np.abs(ref_s) + 1e-2)
        assert rel.max() < SCORE_RTOL, (name, r, rel.max())
        assert abs(sc[o:o + t].sum() - (lay.new_off[r + 1] - lay.new_off[r]) * lay.num_q_heads) < 1e-2 * t ** 0.5
        s0, s1 = g.sel_off_h[r], g.sel_off_h[r + 1]
        r0, r1 = g.rows_off_h[r], g.rows_off_h[r + 1]
        assert np.array_equal(sel[s0:s1], res.sel[r]), (name, r)           # bit-exact index set
        assert np.array_equal(rows[r0:r1], res.rows[r]), (name, r)
        check_close("%s req %d O" % (name, r), out[r0:r1], res.out[r])
        assert np.max(np.abs(lse[r0:r1] - res.lse[r])) < 2e-3
    # pool and tables after the layer: logical K/V views of every request
    gk, gv = dev_to_bits(g.pool_k), dev_to_bits(g.pool_v)
    gkt, gvt = g.batch.k_block_table.cpu().numpy(), g.batch.v_block_table.cpu().numpy()
    assert np.array_equal(gkt, kt) and np.array_equal(gvt, vt)
    assert np.array_equal(gv, pv)                                           # V: copies and fresh rows only
    src = np.concatenate(lay.pool_seg_pages)
    assert np.array_equal(gk[src], lt.pool_k[src]) and np.array_equal(gv[src], lt.pool_v[src])  # shared pages
    for r in range(lay.num_reqs):
        t = int(lay.seq_len[r])
        a = orc.bf16_to_f64(orc.gather_tokens(gk, gkt[r], t))
        b = orc.bf16_to_f64(orc.gather_tokens(pk, kt[r], t))
        fresh = np.zeros(t, dtype=bool)
        fresh[res.rows[r]] = True
        assert np.array_equal(a[fresh], b[fresh])                           # scattered rows bit-exact
        # re-rotated rows: at most one bf16 ulp from the oracle's rounding (+ the fp32 rotation's absolute
        # error ~2^-23 (|x|+|y|), which exceeds an ulp only for results that cancel to ~1e-5)
        assert np.all(np.abs(a - b) <= 2.0 ** -7 * np.abs(b) + 1e-5)


@pytest.mark.parametrize("pair", [False, True], ids=["1cta", "cta-pair"])
@pytest.mark.parametrize("name", ["tiny", "tiny-ragged", "tiny-g7", "C1", "C3-eighth"])
def test_full_layer(name, pair):
    """Full-attention layer (layers below the threshold, Alg. 1 l.507-511): R = all positions."""
    GpuLayer, dev_to_bits = _gpu()
    lay, lt = prepared(name)[:2]
    res, pk, pv, kt, vt = oracle_layer(lay, lt, mode="full")
    g = GpuLayer(lay, lt)
    g.cta_pair = pair
    g.step_full()
    torch.cuda.synchronize()
    out = orc.bf16_to_f64(dev_to_bits(g.out))
    lse = g.lse.cpu().numpy().astype(np.float64)
    for r in range(lay.num_reqs):
        o, t = int(lay.tok_off[r]), int(lay.seq_len[r])
        check_close("%s full O" % name, out[o:o + t], res.out[r])
        assert np.max(np.abs(lse[o:o + t] - res.lse[r])) < 2e-3
    assert np.array_equal(dev_to_bits(g.pool_k)[kt[kt >= 0]], pk[kt[kt >= 0]])
    assert np.array_equal(dev_to_bits(g.pool_v), pv)


def test_paper_mode_boundary_selection():
    """A11/A16: select once on the boundary layer after its full attention (LSE supplied -> one sweep),
    reuse R in the next (sparse) layer."""
    GpuLayer, dev_to_bits = _gpu()
    from paper_2606_01751_b200 import binding as sx
    lay = wl.config_c3(scale=0.125)
    l3, l4 = wl.build_layer(lay, 3), wl.build_layer(lay, 4)
    # the boundary selection reads an all-fresh pool: the margin at the rank-k cut is carved into K_fresh of
    # layer 3 (helpers.carve_margins_fresh), then S_key and R must be bit-exact
    carve_margins_fresh(lay, l3)
    res3, pk3, pv3, kt3, vt3 = oracle_layer(lay, l3, mode="full")
    g3 = GpuLayer(lay, l3)
    g3.step_full()
    g3.select(lse_new=g3.lse, lse_by_token=True)      # full-mode LSE indexed by token: single sweep
    torch.cuda.synchronize()
    sel = g3.sel_idx.cpu().numpy()
    s = orc.scores(pk3, kt3[0], int(lay.seq_len[0]), l3.q_full[lay.new_idx], lay.new_idx, lay.num_q_heads)
    ref_sel, ref_rows = orc.select_topk(s, lay.is_new_mask(0), int(lay.k_per_req[0]))
    assert np.array_equal(sel, ref_sel)
    assert np.array_equal(g3.rows_R.cpu().numpy(), ref_rows)
    gsc = g3.scores.cpu().numpy().astype(np.float64)
    assert np.max(np.abs(gsc - s) / (np.abs(s) + 1e-2)) < SCORE_RTOL
    # layer 4 reuses the ORACLE's R (so both sides attend the same rows)
    res4, pk4, pv4, kt4, vt4 = oracle_layer(lay, l4, mode="sparse", rows_given=[(ref_sel, ref_rows)])
    g4 = GpuLayer(lay, l4)
    g4.step_sparse(rows_given=(torch.from_numpy(ref_sel).to(g4.dev), torch.from_numpy(ref_rows).to(g4.dev)))
    torch.cuda.synchronize()
    check_close("paper-mode layer 4 O", orc.bf16_to_f64(dev_to_bits(g4.out)), res4.out[0])


def test_degenerate_budgets():
    """k = 0 (S_key empty, R = I_nr) and k = N_c (ratio 100 %: every output row equals dense causal
    attention over the fresh tensors, independent of the cached pool)."""
    GpuLayer, dev_to_bits = _gpu()
    for k_over in ("zero", "all"):
        lay = wl.config_tiny(seed_id=21)
        n_c = lay.seq_len - np.diff(lay.new_off)
        lay.k_per_req = (np.zeros_like(n_c) if k_over == "zero" else n_c).astype(np.int32)
        lt = wl.build_layer(lay, 0)
        res, pk, pv, kt, vt = oracle_layer(lay, lt, mode="sparse")
        g = GpuLayer(lay, lt)
        g.step_sparse()
        torch.cuda.synchronize()
        rows = g.rows_R.cpu().numpy()
        out = orc.bf16_to_f64(dev_to_bits(g.out))
        for r in range(lay.num_reqs):
            r0, r1 = g.rows_off_h[r], g.rows_off_h[r + 1]
            assert np.array_equal(rows[r0:r1], res.rows[r])
            check_close("degenerate %s" % k_over, out[r0:r1], res.out[r])
        if k_over == "all":
            assert np.array_equal(dev_to_bits(g.pool_k)[kt[kt >= 0]], pk[kt[kt >= 0]])


@pytest.mark.parametrize("name", ["C2-quarter", "C5-1/16"])   # the second one takes the multi-CTA select
def test_determinism(name):
    GpuLayer, dev_to_bits = _gpu()
    lay, lt = prepared(name)[:2]
    outs = []
    for _ in range(2):
        g = GpuLayer(lay, lt)
        g.step_sparse()
        torch.cuda.synchronize()
        outs.append((g.scores.cpu().numpy().copy(), dev_to_bits(g.out).copy(), g.rows_R.cpu().numpy().copy()))
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a, b)


SMALL_CASES = {
    # name: (prepared case, rows per request as a function of (T, request index))
    "tiny-last3": ("tiny", lambda t, r: np.arange(t - 3, t)),
    "tiny-ragged-mixed": ("tiny-ragged", lambda t, r: np.asarray([0, 1, t // 2, t - 1])),
    "tiny-g7-5rows": ("tiny-g7", lambda t, r: np.asarray([0, 17, t // 3, t - 2, t - 1])),
    "tiny-g1": ("tiny-g1", lambda t, r: np.arange(t - 9, t)),
    "C1-last8": ("C1", lambda t, r: np.arange(t - 8, t)),                   # 32 pairs per KV head
    "C1-15-scattered": ("C1", lambda t, r: np.unique(np.linspace(0, t - 1, 15).astype(np.int64))),
    "C2q-chunked": ("C2-quarter", lambda t, r: np.arange(t - (7 if r == 0 else 1), t) if r else
                    np.unique(np.linspace(5, t - 1, 7).astype(np.int64))),
    "C4e-one-row-each": ("C4-eighth", lambda t, r: np.asarray([t - 1])),    # decode-like: 4 pairs per KV head
    "C5-last2": ("C5-1/16", lambda t, r: np.arange(t - 2, t)),               # g = 7: 14 pairs per KV head
}


@pytest.mark.parametrize("path", ["cuda-core", "tcgen05-splits"])
@pytest.mark.parametrize("case", list(SMALL_CASES))
def test_small_row_sets(case, path):
    """Fewer than 64 (row, head) pairs per KV head: with SX_ATTN_CUDA_CORE sx_sparse_attn takes the CUDA-core
    split-KV kernels (the north_star rule), by default the padded tensor-core tile with key splits that merge
    themselves in one launch (measured faster on B200); same definition O-c, same tolerance on both."""
    GpuLayer, dev_to_bits = _gpu()
    cuda_core = path == "cuda-core"
    name, pick = SMALL_CASES[case]
    lay, lt, res, pk, pv, kt, vt = prepared(name)
    g = GpuLayer(lay, lt)
    g.step_sparse()
    rows, off = [], [0]
    for r in range(lay.num_reqs):
        rr = np.asarray(pick(int(lay.seq_len[r]), r), dtype=np.int32)
        rows.append(rr)
        off.append(off[-1] + len(rr))
    gq = lay.num_q_heads // lay.num_kv_heads
    assert off[-1] * gq < 64 * lay.num_reqs          # the dispatch rule of include/sparsex.h
    g.rows_off = torch.tensor(off, dtype=torch.int32, device=g.dev)
    g.sel_off = torch.zeros(lay.num_reqs + 1, dtype=torch.int32, device=g.dev)
    g.stage_rows(torch.zeros(0, dtype=torch.int32, device=g.dev), torch.from_numpy(np.concatenate(rows)).to(g.dev))
    g.attend(cuda_core=cuda_core)
    torch.cuda.synchronize()
    out = orc.bf16_to_f64(dev_to_bits(g.out))
    lse = g.lse.cpu().numpy().astype(np.float64)
    for r in range(lay.num_reqs):
        o, t = int(lay.tok_off[r]), int(lay.seq_len[r])
        ref_o, ref_l = orc.attention(pk, pv, kt[r], vt[r], t, lt.q_full[o + rows[r]], rows[r], lay.num_q_heads,
                                     want_lse=True)
        check_close("%s req %d O" % (case, r), out[off[r]:off[r + 1]], ref_o)
        assert np.max(np.abs(lse[off[r]:off[r + 1]] - ref_l)) < 2e-3


def test_realign_all_layers_in_one_launch():
    """sx_rope_realign_layers (alignment of the whole scheduling batch at once) must give,
    layer by layer, exactly the bits of the per-layer call."""
    GpuLayer, dev_to_bits = _gpu()
    from paper_2606_01751_b200 import binding as sx
    lay = wl.config_c3(scale=0.125)
    lts = [wl.build_layer(lay, l) for l in range(3)]
    single = []
    for lt in lts:
        g = GpuLayer(lay, lt)
        g.realign()
        torch.cuda.synchronize()
        single.append((dev_to_bits(g.pool_k).copy(), dev_to_bits(g.pool_v).copy()))
    gs = [GpuLayer(lay, lt) for lt in lts]
    sx.rope_realign_layers([g.pool for g in gs], gs[0].batch)
    torch.cuda.synchronize()
    for g, (k, v) in zip(gs, single):
        assert np.array_equal(dev_to_bits(g.pool_k), k)
        assert np.array_equal(dev_to_bits(g.pool_v), v)


@pytest.mark.parametrize("ov,tail,prefix", [(1, 64, 0), (1, 0, 0), (0, 64, 0), (2, 16, 0), (1, 64, 32), (2, 16, 16)])
def test_overflow_and_tail_fallback(ov, tail, prefix):
    """sx_score_select_ex: R = I_nr U S_key U S_ov U S_tail (Alg. 1 l.535-539) bit-exact against the oracle,
    then scatter + attention on that (data-dependent) row list. prefix > 0: every request starts with prefix-cache
    hits (visible keys that are never candidates and never pulled in by the overflow)."""
    GpuLayer, dev_to_bits = _gpu()
    lay = wl.config_tail(prefix=prefix)
    lt = wl.build_layer(lay, 0)
    carve_margins(lay, lt)
    g = GpuLayer(lay, lt)
    g.realign()
    g.scatter_new()
    g.select_ex(overflow_blocks=ov, tail_tokens=tail)
    g.stage_rows(g.sel_idx, g.rows_R)
    sx_rows_total = int(g.rows_off_h[-1])
    from paper_2606_01751_b200 import binding as sx
    sx.scatter_kv(g.pool, g.batch, g.kf_R, g.vf_R, g.rows_R, g.rows_off, max_rows=g.rows_cap)
    g.attend()
    torch.cuda.synchronize()
    # oracle
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    sel_g, rows_g = g.sel_idx.cpu().numpy(), g.rows_R.cpu().numpy()
    out = orc.bf16_to_f64(dev_to_bits(g.out))
    total = 0
    for r in range(lay.num_reqs):
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        nidx = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]
        orc.scatter_kv(pk, pv, kt, vt, None, r, nidx, lt.k_fresh[o + nidx], lt.v_fresh[o + nidx])
        s = orc.scores(pk, kt[r], t, lt.q_full[o + nidx], nidx, lay.num_q_heads)
        is_new = lay.is_new_mask(r)
        cand = lay.cached_mask(r)
        sel, _ = orc.select_topk(s, is_new, int(lay.k_per_req[r]), cand)
        segr = [(int(n), int(n + ln)) for (rq, ln, _, n, _) in lay.segments.tolist() if rq == r]
        rows = orc.recompute_set(is_new, sel, segr, ov, tail, cand_mask=cand)
        r0, r1 = int(g.rows_off_h[r]), int(g.rows_off_h[r + 1])
        assert np.array_equal(sel_g[g.sel_off_h[r]:g.sel_off_h[r + 1]], sel), (r, ov, tail)
        assert np.array_equal(rows_g[r0:r1], rows), (r, ov, tail)
        orc.scatter_kv(pk, pv, kt, vt, None, r, rows, lt.k_fresh[o + rows], lt.v_fresh[o + rows])
        ref = orc.attention(pk, pv, kt[r], vt[r], t, lt.q_full[o + rows], rows, lay.num_q_heads)
        check_close("overflow/tail req %d O" % r, out[r0:r1], ref)
        total += len(rows)
    assert total == sx_rows_total
    # tokens behind the last new token have score exactly 0 and are reached only through S_tail / S_key
    assert np.array_equal(dev_to_bits(g.pool_v), pv)


@pytest.mark.parametrize("name,nlast", [("C5-1/16", 16), ("C1", 40), ("C3-eighth", 24)])
def test_few_rows_tensor_core_path_with_key_splits(name, nlast):
    """At least 64 (row, head) pairs per KV head but only a few query tiles against a long context: the tcgen05
    kernel cuts the key range into splits (partial O and LSE in the workspace) that merge themselves in fixed order
    once all splits of a row pair have arrived."""
    GpuLayer, dev_to_bits = _gpu()
    lay, lt, res, pk, pv, kt, vt = prepared(name)
    g = GpuLayer(lay, lt)
    g.step_sparse()
    rows, off = [], [0]
    for r in range(lay.num_reqs):
        t = int(lay.seq_len[r])
        rr = np.unique(np.concatenate([np.arange(t - nlast, t), [3, t // 2]])).astype(np.int32)
        rows.append(rr)
        off.append(off[-1] + len(rr))
    assert off[-1] * (lay.num_q_heads // lay.num_kv_heads) >= 64 * lay.num_reqs
    g.rows_off = torch.tensor(off, dtype=torch.int32, device=g.dev)
    g.sel_off = torch.zeros(lay.num_reqs + 1, dtype=torch.int32, device=g.dev)
    g.stage_rows(torch.zeros(0, dtype=torch.int32, device=g.dev), torch.from_numpy(np.concatenate(rows)).to(g.dev))
    g.attend()
    torch.cuda.synchronize()
    out = orc.bf16_to_f64(dev_to_bits(g.out))
    lse = g.lse.cpu().numpy().astype(np.float64)
    for r in range(lay.num_reqs):
        o, t = int(lay.tok_off[r]), int(lay.seq_len[r])
        ref_o, ref_l = orc.attention(pk, pv, kt[r], vt[r], t, lt.q_full[o + rows[r]], rows[r], lay.num_q_heads,
                                     want_lse=True)
        check_close("%s req %d O" % (name, r), out[off[r]:off[r + 1]], ref_o)
        assert np.max(np.abs(lse[off[r]:off[r + 1]] - ref_l)) < 2e-3


def test_paper_mode_boundary_selection_uncarved_band():
    """Second, explicitly labelled case (reading A10 fallback): the same boundary selection WITHOUT a carved margin.
    The rank-k cut then falls among near-tied ordinary tokens, so the GPU set is compared modulo the tau band
    (NOT a bit-exact claim): everything clearly above the cut is selected, nothing clearly below it, and the GPU's
    own fp32 scores reproduce its set exactly under the tie rule."""
    GpuLayer, dev_to_bits = _gpu()
    lay = wl.config_c3(scale=0.125)
    l3 = wl.build_layer(lay, 3)
    res3, pk3, pv3, kt3, vt3 = oracle_layer(lay, l3, mode="full")
    g3 = GpuLayer(lay, l3)
    g3.step_full()
    g3.select(lse_new=g3.lse, lse_by_token=True)
    torch.cuda.synchronize()
    sel = g3.sel_idx.cpu().numpy()
    s = orc.scores(pk3, kt3[0], int(lay.seq_len[0]), l3.q_full[lay.new_idx], lay.new_idx, lay.num_q_heads)
    ref_sel, _ = orc.select_topk(s, lay.is_new_mask(0), int(lay.k_per_req[0]))
    k = int(lay.k_per_req[0])
    cand = np.nonzero(~lay.is_new_mask(0))[0]
    srt = np.sort(s[cand])[::-1]
    c = 0.5 * (srt[k - 1] + srt[k])
    tau = 1e-3
    must = cand[s[cand] > c * (1 + tau)]
    never = cand[s[cand] < c * (1 - tau)]
    assert len(sel) == k and np.all(np.diff(sel) > 0)
    assert np.all(np.isin(must, sel)) and not np.any(np.isin(never, sel))
    band = int(np.sum(np.abs(s[cand] - c) <= tau * c))
    assert len(np.setdiff1d(sel, ref_sel)) <= band
    own_sel, own_rows = orc.select_topk(g3.scores.cpu().numpy().astype(np.float64), lay.is_new_mask(0), k)
    assert np.array_equal(sel, own_sel) and np.array_equal(g3.rows_R.cpu().numpy(), own_rows)


def test_check_batch_and_rows_reject_bad_device_descriptors():
    """sx_check_batch / sx_check_rows (include/sparsex.h): the device-resident arrays that the stage calls cannot
    see from the host mirrors. A misaligned segment must give SX_ERR_INVALID_ARG, not corrupt pages."""
    GpuLayer, dev_to_bits = _gpu()
    from paper_2606_01751_b200 import binding as sx
    import copy
    lay = wl.config_tiny()
    lt = wl.build_layer(lay, 0)
    g = GpuLayer(lay, lt)
    sx.check_batch(g.pool, g.batch)                                   # a good descriptor passes

    def broken(mutate, needle):
        bad = copy.deepcopy(lay)
        mutate(bad)
        gb = GpuLayer(bad, lt)
        with pytest.raises(sx.SparseXError) as ei:
            sx.check_batch(gb.pool, gb.batch)
        assert "(-1)" in str(ei.value) and needle in str(ei.value), str(ei.value)

    def seg_set(m, col, val):
        def f(bad):
            bad.segments = bad.segments.copy()
            bad.segments[m, col] = val
        return f
    broken(seg_set(1, 3, int(lay.segments[1, 3]) + 8), "multiple of block_size")      # new_pos misaligned
    broken(seg_set(0, 2, int(lay.segments[0, 2]) + 4), "multiple of block_size")      # old_pos misaligned
    broken(seg_set(2, 4, int(lay.segments[2, 4]) + 1), "running sum")                 # src_off
    broken(seg_set(1, 3, int(lay.segments[0, 3])), "sorted")                          # overlaps segment 0

    def bad_new_idx(bad):
        bad.new_idx = bad.new_idx.copy()
        bad.new_idx[3], bad.new_idx[4] = bad.new_idx[4], bad.new_idx[3]
    broken(bad_new_idx, "new_idx")

    def bad_page(bad):
        bad.src_blocks = bad.src_blocks.copy()
        bad.src_blocks[1] = bad.num_blocks + 7
    broken(bad_page, "src_blocks")

    def bad_table(bad):
        bad.k_block_table = bad.k_block_table.copy()
        bad.k_block_table[1, 0] = -3
    broken(bad_table, "k_block_table")

    # row lists
    rows = torch.tensor([0, 5, 9, 2, 3], dtype=torch.int32, device=g.dev)
    off = torch.tensor([0, 3, 5], dtype=torch.int32, device=g.dev)
    sx.check_rows(g.pool, g.batch, rows, off)
    with pytest.raises(sx.SparseXError):
        sx.check_rows(g.pool, g.batch, torch.tensor([0, 9, 5, 2, 3], dtype=torch.int32, device=g.dev), off)
    with pytest.raises(sx.SparseXError):
        sx.check_rows(g.pool, g.batch, torch.tensor([0, 5, 9, 2, 4000], dtype=torch.int32, device=g.dev), off)
    with pytest.raises(sx.SparseXError):
        sx.check_rows(g.pool, g.batch, rows, torch.tensor([0, 4, 3], dtype=torch.int32, device=g.dev))


@pytest.mark.parametrize("extended", [False, True], ids=["select", "select_ex"])
def test_budget_clamped_to_real_candidates_and_unclipped_capacities(extended):
    """Two requests END inside a reused segment whose last page straddles seq_len (reading A19), and ask for more
    cached tokens than exist: k must be clamped to the candidates below seq_len (sum of segment lengths
    overestimates them). The extended call additionally gets capacities far above T_r, as a C caller might pass."""
    GpuLayer, dev_to_bits = _gpu()
    from paper_2606_01751_b200 import binding as sx
    lay = wl.config_tail(trim=[5, 3, 0], k_override=[200, 200, 19])
    lt = wl.build_layer(lay, 0)
    carve_margins(lay, lt)
    res, pk, pv, kt, vt = oracle_layer(lay, lt, mode="sparse")
    g = GpuLayer(lay, lt)
    g.realign()
    g.scatter_new()
    if not extended:
        g.select()
        sel, rows = g.sel_idx.cpu().numpy(), g.rows_R.cpu().numpy()
        for r in range(lay.num_reqs):
            n_sel, n_rows = len(res.sel[r]), len(res.rows[r])
            s0, r0 = int(g.sel_off_h[r]), int(g.rows_off_h[r])
            assert np.array_equal(sel[s0:s0 + n_sel], res.sel[r]), r
            assert np.array_equal(rows[r0:r0 + n_rows], res.rows[r]), r
    else:
        cap = np.concatenate([[0], np.cumsum(10 * lay.seq_len)]).astype(np.int32)      # NOT clipped to T_r
        n_sel = int(g.sel_off_h[-1])
        sel = torch.full((n_sel,), -1, dtype=torch.int32, device=g.dev)
        rows = torch.full((int(cap[-1]),), -1, dtype=torch.int32, device=g.dev)
        off_out = torch.zeros(lay.num_reqs + 1, dtype=torch.int32, device=g.dev)
        sx.score_select_ex(g.pool, g.batch, g.q_new, g.sel_off, torch.from_numpy(cap).to(g.dev), sel, rows, off_out,
                           overflow_blocks=0, tail_tokens=0)
        torch.cuda.synchronize()
        off_h, rows_h, sel_h = off_out.cpu().numpy(), rows.cpu().numpy(), sel.cpu().numpy()
        for r in range(lay.num_reqs):
            assert np.array_equal(rows_h[off_h[r]:off_h[r + 1]], res.rows[r]), r
            s0 = int(g.sel_off_h[r])
            assert np.array_equal(sel_h[s0:s0 + len(res.sel[r])], res.sel[r]), r
        assert np.all(rows_h[off_h[-1]:] == -1)                                       # nothing written past the end


def test_copy_on_write_two_layers_each_with_its_own_tables():
    """COW state (v_block_table) is per layer. Two layers of one request batch, each with its own
    descriptor, both end with the oracle's tables and pools; the all-layer realign refuses the COW descriptor."""
    GpuLayer, dev_to_bits = _gpu()
    from paper_2606_01751_b200 import binding as sx
    lay = wl.config_c4(scale=0.125, num_reqs=3, cow=True)
    gs = []
    for layer in range(2):
        lt = wl.build_layer(lay, layer)
        carve_margins(lay, lt)
        res, pk, pv, kt, vt = oracle_layer(lay, lt, mode="sparse")
        g = GpuLayer(lay, lt)                       # own DeviceBatch -> own block tables
        g.step_sparse()
        torch.cuda.synchronize()
        assert np.array_equal(g.batch.v_block_table.cpu().numpy(), vt) and np.array_equal(dev_to_bits(g.pool_v), pv)
        assert np.array_equal(g.batch.k_block_table.cpu().numpy(), kt)
        out = orc.bf16_to_f64(dev_to_bits(g.out))
        for r in range(lay.num_reqs):
            r0, r1 = g.rows_off_h[r], g.rows_off_h[r + 1]
            assert np.array_equal(g.rows_R.cpu().numpy()[r0:r1], res.rows[r])
            check_close("cow layer %d req %d" % (layer, r), out[r0:r1], res.out[r])
        gs.append(g)
    with pytest.raises(sx.SparseXError):
        sx.rope_realign_layers([g.pool for g in gs], gs[0].batch)


@pytest.mark.parametrize("nrows", [3, 14, 30])
def test_reference_moves_and_rescales_with_key_splits(nrows):
    """The attention kernel rescales O lazily (only when a row maximum grows by more than 2^24). Keys whose norm
    grows with the position (x1 ... x8) make later tiles exceed the reference of earlier ones many times over, in
    every row and in every key split; rows in the middle of the context exercise the causal mask inside a tile."""
    GpuLayer, dev_to_bits = _gpu()
    lay, lt, res, pk, pv, kt, vt = prepared("C1")
    t = int(lay.seq_len[0])
    pk = pk.copy()
    for pos in range(t):                       # key norm grows stepwise with the position
        scale = 1.0 + 7.0 * (pos // 256) / (t // 256 - 1)
        blk, off = int(kt[0][pos // 16]), pos % 16
        pk[blk, :, off, :] = orc.f64_to_bf16(orc.bf16_to_f64(pk[blk, :, off, :]) * scale)
    g = GpuLayer(lay, lt)
    g.pool_k.copy_(torch.from_numpy(pk.view(np.int16)))
    g.pool_v.copy_(torch.from_numpy(pv.view(np.int16)))
    rows = np.unique(np.concatenate([np.arange(t - nrows + 2, t), [700, t // 2 + 5]])).astype(np.int32)
    assert len(rows) == nrows
    g.rows_off = torch.tensor([0, len(rows)], dtype=torch.int32, device=g.dev)
    g.sel_off = torch.zeros(2, dtype=torch.int32, device=g.dev)
    g.stage_rows(torch.zeros(0, dtype=torch.int32, device=g.dev), torch.from_numpy(rows).to(g.dev))
    g.attend()
    torch.cuda.synchronize()
    ref_o, ref_l = orc.attention(pk, pv, kt[0], vt[0], t, lt.q_full[rows], rows, lay.num_q_heads, want_lse=True)
    check_close("key splits, growing key norms", orc.bf16_to_f64(dev_to_bits(g.out)), ref_o)
    assert np.max(np.abs(g.lse.cpu().numpy().astype(np.float64) - ref_l)) < 2e-3


def test_key_split_path_under_cuda_graph_replay():
    """The self-merging key splits meet on a workspace word that no memset prepares; the rendezvous must come back to
    its initial state by itself, so that a captured launch (identical kernel parameters on every replay) works any
    number of times and keeps giving the bits of the eager call."""
    GpuLayer, dev_to_bits = _gpu()
    from paper_2606_01751_b200 import binding as sx
    lay, lt, res, pk, pv, kt, vt = prepared("C1")
    g = GpuLayer(lay, lt)
    g.step_sparse()
    t = int(lay.seq_len[0])
    rows = torch.arange(t - 6, t, dtype=torch.int32, device=g.dev)
    off = torch.tensor([0, 6], dtype=torch.int32, device=g.dev)
    q = g.q_full[t - 6:t].contiguous()
    out = torch.zeros((6, lay.num_q_heads, 128), dtype=torch.int16, device=g.dev)
    sx.sparse_attn(g.pool, g.batch, q, out, rows_R=rows, rows_off=off, total_rows=6)
    torch.cuda.synchronize()
    eager = out.clone()
    gr = torch.cuda.CUDAGraph()
    with torch.cuda.graph(gr):
        sx.sparse_attn(g.pool, g.batch, q, out, rows_R=rows, rows_off=off, total_rows=6)
    for _ in range(4):
        out.zero_()
        gr.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, eager)
    out.zero_()
    sx.sparse_attn(g.pool, g.batch, q, out, rows_R=rows, rows_off=off, total_rows=6)   # and eager again afterwards
    torch.cuda.synchronize()
    assert torch.equal(out, eager)


def test_pipe_probe_reports_plausible_rates():
    """sx_probe_pipe (diagnostic; the denominator of stage (b)'s roofline in bench.py): MUFU.EX2 retires 16 lane-ops
    per clock and SM on sm_100, FFMA about 128; the probe must land near both on any healthy B200."""
    from paper_2606_01751_b200 import binding as sx
    mufu = sx.probe_pipe(0, iters=2048)
    ffma = sx.probe_pipe(1, iters=2048)
    mix = sx.probe_pipe(3, iters=2048)
    assert 14.0 < mufu < 16.5, mufu
    assert 100.0 < ffma < 130.0, ffma
    assert mufu < mix < 2.0 * mufu, (mufu, mix)          # the polynomial share adds to what MUFU alone retires
    with pytest.raises(sx.SparseXError):
        sx.probe_pipe(9)


def test_attention_output_pointer_aligned_to_16_bytes_only():
    """The ABI asks for 16-byte alignment of `out`; the epilogue of the tensor-core kernel stores 32 bytes per lane
    when the pointer allows it and falls back to 16-byte stores otherwise: same bits either way."""
    GpuLayer, dev_to_bits = _gpu()
    from paper_2606_01751_b200 import binding as sx
    lay, lt, res, pk, pv, kt, vt = prepared("C2-quarter")
    g = GpuLayer(lay, lt)
    g.step_sparse()
    n, hq = int(g.rows_R.numel()), lay.num_q_heads
    buf = torch.zeros(n * hq * 128 + 8, dtype=torch.int16, device=g.dev)
    shifted = buf[8:].view(n, hq, 128)
    assert shifted.data_ptr() % 32 == 16 and shifted.is_contiguous()
    for pair in (False, True):
        buf.zero_()
        sx.sparse_attn(g.pool, g.batch, g.q_R, shifted, rows_R=g.rows_R, rows_off=g.rows_off, total_rows=n, cta_pair=pair)
        ref = torch.zeros((n, hq, 128), dtype=torch.int16, device=g.dev)
        sx.sparse_attn(g.pool, g.batch, g.q_R, ref, rows_R=g.rows_R, rows_off=g.rows_off, total_rows=n, cta_pair=pair)
        torch.cuda.synchronize()
        assert torch.equal(shifted, ref) and int(buf[:8].abs().sum()) == 0


def test_one_workspace_reused_by_different_batches_back_to_back():
    """Two batches of the same shape but different content (other deltas, other positions of the new tokens, other
    block tables) take turns on ONE workspace without any synchronisation in between. Every intermediate a kernel
    reads from the workspace (rotation table, page descriptors, work records, column tables, partial scores, row
    lists) was written moments earlier by the preceding kernel at an address that still holds the OTHER batch's
    values in some SM's read-only cache: under programmatic dependent launch a kernel that read them through the
    read-only path (ld.global.nc) got the stale ones (found with the colsum work records; include/sparsex.h, ld_dep
    in sx_ptx.cuh). Both batches must keep giving their own oracle results."""
    GpuLayer, dev_to_bits = _gpu()
    # four requests of 1.5-3K tokens (about 700 column-sum CTAs: every SM sees several work records per call); batch B
    # = the requests of A in reverse order over a pool with other old positions: same sizes, other content everywhere
    lens = [512, 768, 256, 1024, 384, 640]
    pool_a = [wl.PoolSegment(n, 16 * (7 * i + 3)) for i, n in enumerate(lens)]
    pool_b = [wl.PoolSegment(n, 16 * (5 * i + 40)) for i, n in enumerate(lens)]
    reqs_a = [[("seg", 0), ("new", 128), ("seg", 3), ("new", 256), ("seg", 1), ("new", 64)],
              [("new", 64), ("seg", 2), ("seg", 4), ("new", 512), ("seg", 5), ("new", 37)],
              [("seg", 5), ("new", 256), ("seg", 0), ("new", 128)],
              [("new", 192), ("seg", 1), ("new", 64), ("seg", 3), ("seg", 2), ("new", 320)]]
    reqs_b = reqs_a[::-1]
    ratios = [0.1, 0.25, 0.15, 0.2]
    lays = [wl.build_layout("ws-a", 41, 8, 2, 500000.0, pool_a, reqs_a, ratios, 0.05),
            wl.build_layout("ws-b", 42, 8, 2, 500000.0, pool_b, reqs_b, ratios[::-1], 0.05)]
    cases = []
    for lay in lays:
        lt = wl.build_layer(lay, 0)
        carve_margins(lay, lt)
        cases.append((lay, lt, oracle_layer(lay, lt, mode="sparse")[0]))
    gs = [GpuLayer(lay, lt) for lay, lt, _ in cases]
    ws = gs[0].batch.workspace(gs[0].pool)
    assert gs[1].batch.workspace(gs[1].pool).numel() == ws.numel()      # same shape, same workspace layout
    gs[1].batch._ws = ws
    pools0 = [(g.pool_k.clone(), g.pool_v.clone()) for g in gs]
    for rep in range(4):
        for g, (pk0, pv0) in zip(gs, pools0):
            g.pool_k.copy_(pk0)
            g.pool_v.copy_(pv0)
            g.step_sparse()                 # no synchronisation between the two batches
        torch.cuda.synchronize()
        for g, (lay, lt, res) in zip(gs, cases):
            sel, rows = g.sel_idx.cpu().numpy(), g.rows_R.cpu().numpy()
            out = orc.bf16_to_f64(dev_to_bits(g.out))
            for r in range(lay.num_reqs):
                assert np.array_equal(sel[g.sel_off_h[r]:g.sel_off_h[r + 1]], res.sel[r]), (rep, lay.name, r)
                assert np.array_equal(rows[g.rows_off_h[r]:g.rows_off_h[r + 1]], res.rows[r]), (rep, lay.name, r)
                check_close("%s rep %d req %d O" % (lay.name, rep, r), out[g.rows_off_h[r]:g.rows_off_h[r + 1]], res.out[r])
