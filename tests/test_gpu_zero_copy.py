"""GPU parity of zero-copy mode (include/sparsex.h, sx_batch::zero_copy; S9 NEXT-3): the block tables
of reused pages point at the shared cached pages, nothing is re-aligned up front, the stage kernels rotate K while
they read it and the scatter copies-on-write (rotating) only the pages it writes.

What must hold: the rotation done on the fly has the bits sx_rope_realign would have stored, so scores, S_key and R
are those of the copy path (and of the fp64 oracle, bit-exact sets); attention within the same tolerance against
fp64; every page written is a private page whose content equals the copy path's page bit for bit; every page not
written still is the shared source page, unmodified; V is never rotated.
"""
import numpy as np
import pytest
import torch

from oracle import sx_oracle as orc
from paper_2606_01751_b200 import workloads as wl

from helpers import check_close, oracle_layer
from test_gpu_parity import SCORE_RTOL, _gpu, prepared

pytestmark = pytest.mark.gpu

ZC_CASES = ["tiny", "tiny-ragged", "tiny-interleaved", "tiny-g7", "tiny-g1", "tiny-prefix", "C1", "C2-quarter",
            "C3-eighth", "C4-eighth", "C5-1/16"]


def _seg_page_mask(lay):
    """bool [num_reqs][max_pages]: logical page is covered by a reused segment."""
    m = np.zeros(lay.k_block_table.shape, dtype=bool)
    for (req, ln, _old, new, _so) in lay.segments.tolist():
        m[req, new // 16:(new + ln) // 16] = True
    return m


@pytest.mark.parametrize("name", ZC_CASES)
def test_zero_copy_sparse_layer(name):
    GpuLayer, dev_to_bits = _gpu()
    lay, lt, res, pk, pv, kt, vt = prepared(name)
    g0 = GpuLayer(lay, lt)                    # copy path: realign, then the same stages
    g0.step_sparse()
    zlay = wl.zero_copy_layout(lay)
    g = GpuLayer(zlay, lt)
    g.step_sparse(do_realign=False)
    torch.cuda.synchronize()
    # scores: same kernels, same decomposition, K bits identical -> identical to the copy path
    assert np.array_equal(g.scores.cpu().numpy(), g0.scores.cpu().numpy())
    sc = g.scores.cpu().numpy().astype(np.float64)
    sel, rows = g.sel_idx.cpu().numpy(), g.rows_R.cpu().numpy()
    out = orc.bf16_to_f64(dev_to_bits(g.out))
    lse = g.lse.cpu().numpy().astype(np.float64)
    for r in range(lay.num_reqs):
        o, t = int(lay.tok_off[r]), int(lay.seq_len[r])
        rel = np.abs(sc[o:o + t] - res.scores[r]) / (np.abs(res.scores[r]) + 1e-2)
        assert rel.max() < SCORE_RTOL
        s0, s1 = g.sel_off_h[r], g.sel_off_h[r + 1]
        r0, r1 = g.rows_off_h[r], g.rows_off_h[r + 1]
        assert np.array_equal(sel[s0:s1], res.sel[r]), (name, r)
        assert np.array_equal(rows[r0:r1], res.rows[r]), (name, r)
        check_close("%s zero-copy req %d O" % (name, r), out[r0:r1], res.out[r])
        assert np.max(np.abs(lse[r0:r1] - res.lse[r])) < 2e-3
    # ---- pages and tables
    gk, gv = dev_to_bits(g.pool_k), dev_to_bits(g.pool_v)
    gk0 = dev_to_bits(g0.pool_k)
    gkt, gvt = g.batch.k_block_table.cpu().numpy(), g.batch.v_block_table.cpu().numpy()
    in_seg = _seg_page_mask(lay)
    written = np.zeros_like(in_seg)
    for r in range(lay.num_reqs):
        written[r, np.unique(res.rows[r] // 16)] = True
    priv = lay.k_block_table                  # the request's own pages = the reserved private pages
    flipped = in_seg & written
    assert np.array_equal(gkt[flipped], priv[flipped]) and np.array_equal(gvt[flipped], priv[flipped])
    still = in_seg & ~written
    assert np.array_equal(gkt[still], zlay.k_block_table[still]) and np.array_equal(gvt[still], zlay.v_block_table[still])
    assert np.array_equal(gkt[~in_seg], priv[~in_seg])
    # written pages: bit-identical to the copy path's pages (rotated copy + fresh rows); V to the oracle's
    pages = priv[flipped | (~in_seg & written)]
    assert np.array_equal(gk[pages], gk0[pages])
    assert np.array_equal(gv[pages], pv[pages])
    # shared source pages untouched; private pages of unwritten reused pages never filled (the memory not spent)
    src = np.concatenate(lay.pool_seg_pages)
    assert np.array_equal(gk[src], lt.pool_k[src]) and np.array_equal(gv[src], lt.pool_v[src])
    assert not gk[priv[still]].any() and not gv[priv[still]].any()
    # V through the final tables = the oracle's logical V everywhere
    for r in range(lay.num_reqs):
        t = int(lay.seq_len[r])
        assert np.array_equal(orc.gather_tokens(gv, gvt[r], t), orc.gather_tokens(pv, vt[r], t))


@pytest.mark.parametrize("name", ["tiny", "tiny-interleaved", "tiny-ragged", "C1"])
def test_zero_copy_full_layer(name):
    """Full-attention layer in zero-copy mode: every page is written, so every reused page goes through the rotating
    copy-on-write before its rows are overwritten; attention then reads private pages only."""
    GpuLayer, dev_to_bits = _gpu()
    lay, lt = prepared(name)[:2]
    res, pk, pv, kt, vt = oracle_layer(lay, lt, mode="full")
    g = GpuLayer(wl.zero_copy_layout(lay), lt)
    g.step_full(do_realign=False)
    torch.cuda.synchronize()
    out = orc.bf16_to_f64(dev_to_bits(g.out))
    lse = g.lse.cpu().numpy().astype(np.float64)
    for r in range(lay.num_reqs):
        o, t = int(lay.tok_off[r]), int(lay.seq_len[r])
        check_close("%s zero-copy full O" % name, out[o:o + t], res.out[r])
        assert np.max(np.abs(lse[o:o + t] - res.lse[r])) < 2e-3
    assert np.array_equal(g.batch.k_block_table.cpu().numpy(), lay.k_block_table)
    gk = dev_to_bits(g.pool_k)
    # rows of a ragged last page beyond seq_len keep the rotated copy; everything else is fresh: compare the tokens
    for r in range(lay.num_reqs):
        t = int(lay.seq_len[r])
        assert np.array_equal(orc.gather_tokens(gk, lay.k_block_table[r], t), orc.gather_tokens(pk, kt[r], t))


@pytest.mark.parametrize("name,nlast", [("C5-1/16", 16), ("C1", 40), ("C3-eighth", 24), ("tiny-interleaved", 8)])
def test_zero_copy_attention_reads_rotated_pages(name, nlast):
    """Attention over an arbitrary small row set on a pool where NOTHING has been made private yet (only the new
    tokens are scattered): every reused key the rows see is rotated in shared memory, key splits included."""
    GpuLayer, dev_to_bits = _gpu()
    lay, lt = prepared(name)[:2]
    # oracle state: realign + scatter(I_nr)
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    g = GpuLayer(wl.zero_copy_layout(lay), lt)
    g.scatter_new()
    rows, off = [], [0]
    for r in range(lay.num_reqs):
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        nidx = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]
        orc.scatter_kv(pk, pv, kt, vt, None, r, nidx, lt.k_fresh[o + nidx], lt.v_fresh[o + nidx])
        rr = np.unique(np.concatenate([np.arange(max(t - nlast, 0), t), [3, t // 2]])).astype(np.int32)
        rows.append(rr)
        off.append(off[-1] + len(rr))
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
        check_close("%s zero-copy req %d O" % (name, r), out[off[r]:off[r + 1]], ref_o)
        assert np.max(np.abs(lse[off[r]:off[r + 1]] - ref_l)) < 2e-3
    # the tables still alias the source pages: attention wrote nothing
    assert np.array_equal(g.batch.k_block_table.cpu().numpy(), wl.zero_copy_layout(lay).k_block_table)


def test_zero_copy_refusals():
    from paper_2606_01751_b200 import binding as sx
    GpuLayer, _ = _gpu()
    lay, lt = prepared("tiny")[:2]
    g = GpuLayer(wl.zero_copy_layout(lay), lt)
    with pytest.raises(sx.SparseXError, match="zero-copy"):
        g.realign()
    g.scatter_new()
    g.select()
    g.stage_rows(g.sel_idx, g.rows_R)
    with pytest.raises(sx.SparseXError, match="zero-copy"):
        g.attend(cuda_core=True)
    g.cta_pair = True
    with pytest.raises(sx.SparseXError, match="zero-copy"):
        g.attend()
    # scatter without reserved private pages would have to write the shared source pages
    nocow = sx.DeviceBatch(wl.zero_copy_layout(lay), cow=False)
    with pytest.raises(sx.SparseXError, match="cow_private"):
        sx.scatter_kv(g.pool, nocow, g.kf_sel, g.vf_sel, g.sel_idx, g.sel_off, max_rows=int(g.sel_idx.numel()))


@pytest.mark.parametrize("name", ["C4", "C3"])
def test_zero_copy_fullsize(name):
    """Zero-copy mode at BASELINE.json's full sizes (C4: 16 requests, 208K context tokens; C3: one 32K request), on
    the carved inputs of test_gpu_fullsize.py. Scores / S_key / R must equal the copy path's bit for bit (that path is
    held against the oracle at full size in test_gpu_fullsize.py); attention is compared with the fp64 oracle on
    the seam-aware row sample; written pages are bit-identical to the copy path's, unwritten ones still shared."""
    import os
    from helpers import apply_carve, edge_rows, load_carve
    GpuLayer, dev_to_bits = _gpu()
    gold = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    lay = wl.CONFIGS[name]()
    lt = wl.build_layer(lay, 0)
    apply_carve(lt, load_carve(os.path.join(gold, "carve_%s.txt" % name)))
    hq, g_sz = lay.num_q_heads, lay.num_q_heads // lay.num_kv_heads
    g0 = GpuLayer(lay, lt)
    g0.step_sparse()
    zlay = wl.zero_copy_layout(lay)
    g = GpuLayer(zlay, lt)
    g.step_sparse(do_realign=False)
    torch.cuda.synchronize()
    assert np.array_equal(g.scores.cpu().numpy(), g0.scores.cpu().numpy())
    sel, rows = g.sel_idx.cpu().numpy(), g.rows_R.cpu().numpy()
    assert np.array_equal(sel, g0.sel_idx.cpu().numpy()) and np.array_equal(rows, g0.rows_R.cpu().numpy())
    # ---- oracle state after the layer's scatters, attention on sampled rows
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    lse = g.lse.cpu().numpy().astype(np.float64)
    written = np.zeros(lay.k_block_table.shape, dtype=bool)
    for r in range(lay.num_reqs):
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        r0, r1 = g.rows_off_h[r], g.rows_off_h[r + 1]
        rr = rows[r0:r1]
        orc.scatter_kv(pk, pv, kt, vt, None, r, rr, lt.k_fresh[o + rr], lt.v_fresh[o + rr])
        written[r, np.unique(rr // 16)] = True
        n = 12 if name == "C4" else 256
        pick = edge_rows(rr, n, 128 // g_sz) if len(rr) > n else np.arange(len(rr))   # a zero-copy CTA owns ONE tile
        ref_o, ref_l = orc.attention(pk, pv, kt[r], vt[r], t, lt.q_full[o + rr[pick]], rr[pick], hq, want_lse=True)
        got = orc.bf16_to_f64(dev_to_bits(g.out[r0:r1][torch.from_numpy(pick).to(g.dev)]))
        check_close("%s zero-copy req %d O (sampled rows)" % (name, r), got, ref_o)
        assert np.max(np.abs(lse[r0:r1][pick] - ref_l)) < 2e-3
    # ---- pages and tables
    gk, gv, gk0 = dev_to_bits(g.pool_k), dev_to_bits(g.pool_v), dev_to_bits(g0.pool_k)
    gkt = g.batch.k_block_table.cpu().numpy()
    in_seg = _seg_page_mask(lay)
    priv = lay.k_block_table
    assert np.array_equal(gkt[in_seg & written], priv[in_seg & written])
    assert np.array_equal(gkt[in_seg & ~written], zlay.k_block_table[in_seg & ~written])
    pages = priv[written]
    assert np.array_equal(gk[pages], gk0[pages])
    assert np.array_equal(gv[pages], pv[pages])
    src = np.concatenate(lay.pool_seg_pages)
    assert np.array_equal(gk[src], lt.pool_k[src])
    saved = int((in_seg & ~written).sum())
    assert saved > 0 and not gk[priv[in_seg & ~written]].any()


def test_check_batch_wants_a_private_page_behind_every_shared_entry():
    """sx_check_batch: a table entry that still is its segment's shared source page (zero-copy K / V, copy-on-write V)
    must have a reserved private page, or the first scatter into it would write the shared cache."""
    import dataclasses
    from paper_2606_01751_b200 import binding as sx
    GpuLayer, _ = _gpu()
    lay, lt = prepared("tiny")[:2]
    z = wl.zero_copy_layout(lay)
    g = GpuLayer(z, lt)
    sx.check_batch(g.pool, g.batch)                       # a good zero-copy descriptor passes
    _req, _ln, _old, new, so = (int(v) for v in lay.segments[1])
    cowp = z.cow_private.copy()
    cowp[_req, new // 16 + 1] = -1                        # no private page behind a shared entry
    gb = GpuLayer(dataclasses.replace(z, cow_private=cowp), lt)
    with pytest.raises(sx.SparseXError, match="reserved private page"):
        sx.check_batch(gb.pool, gb.batch)
    cowp = z.cow_private.copy()
    cowp[_req, new // 16] = int(lay.src_blocks[so])       # "private" page IS the shared page
    gb = GpuLayer(dataclasses.replace(z, cow_private=cowp), lt)
    with pytest.raises(sx.SparseXError, match="reserved private page"):
        sx.check_batch(gb.pool, gb.batch)
    # the copy-on-write layout of round 1 (V aliases, K private) and the plain layout still pass
    for other in (wl.config_tiny(seed_id=14, cow=True), lay):
        go = GpuLayer(other, wl.build_layer(other, 0))
        sx.check_batch(go.pool, go.batch)


@pytest.mark.parametrize("ov,tail,prefix", [(1, 64, 0), (2, 16, 16)])
def test_zero_copy_extended_selection_and_cuda_graph(ov, tail, prefix):
    """sx_score_select_ex (overflow + tail fallback: a data-dependent row list whose rows sit on page boundaries of
    reused segments) and the stages after it in zero-copy mode, against the copy path on the same inputs: same
    S_key and R bit for bit, same written pages, outputs within a few bf16 ulps of each other (the two modes cut the
    attention into different CTAs). Then the whole zero-copy layer once more from a CUDA graph: same results."""
    from helpers import carve_margins
    from paper_2606_01751_b200 import binding as sx
    GpuLayer, dev_to_bits = _gpu()
    lay = wl.config_tail(prefix=prefix)
    lt = wl.build_layer(lay, 0)
    carve_margins(lay, lt)

    def layer(g, realign):
        if realign:
            g.realign()
        g.scatter_new()
        g.select_ex(overflow_blocks=ov, tail_tokens=tail)
        g.stage_rows(g.sel_idx, g.rows_R)
        sx.scatter_kv(g.pool, g.batch, g.kf_R, g.vf_R, g.rows_R, g.rows_off, max_rows=g.rows_cap)
        g.attend()
        torch.cuda.synchronize()
    g0 = GpuLayer(lay, lt)
    layer(g0, True)
    zlay = wl.zero_copy_layout(lay)
    g = GpuLayer(zlay, lt)
    layer(g, False)
    assert np.array_equal(g.scores.cpu().numpy(), g0.scores.cpu().numpy())
    assert np.array_equal(g.sel_idx.cpu().numpy(), g0.sel_idx.cpu().numpy())
    assert np.array_equal(g.rows_R.cpu().numpy(), g0.rows_R.cpu().numpy())
    a, b = orc.bf16_to_f64(dev_to_bits(g.out)), orc.bf16_to_f64(dev_to_bits(g0.out))
    assert np.max(np.abs(a - b)) < 2e-2 and np.mean(np.abs(a - b)) < 5e-4
    rows, off = g.rows_R.cpu().numpy(), g.rows_off_h
    gk, gk0 = dev_to_bits(g.pool_k), dev_to_bits(g0.pool_k)
    for r in range(lay.num_reqs):
        pages = lay.k_block_table[r, np.unique(rows[off[r]:off[r + 1]] // 16)]
        assert np.array_equal(gk[pages], gk0[pages])
    # ---- the same zero-copy stages replayed from a CUDA graph (tables reset first: the scatter flips them)
    out_eager, lse_eager = g.out.clone(), g.lse.clone()
    kt0 = torch.from_numpy(zlay.k_block_table).to(g.dev)
    g.batch.k_block_table.copy_(kt0)
    g.batch.v_block_table.copy_(kt0)
    g.pool_k.copy_(torch.from_numpy(lt.pool_k.view(np.int16)))
    g.pool_v.copy_(torch.from_numpy(lt.pool_v.view(np.int16)))
    g.scatter_new()
    cap = torch.from_numpy(sx.rows_capacity(lay, ov, tail)).to(g.dev)
    sel = torch.full_like(g.sel_idx, -1)
    rows_d = torch.full((g.rows_cap,), -1, dtype=torch.int32, device=g.dev)
    off_out = torch.zeros(lay.num_reqs + 1, dtype=torch.int32, device=g.dev)
    torch.cuda.synchronize()

    def stages():
        sx.score_select_ex(g.pool, g.batch, g.q_new, g.sel_off, cap, sel, rows_d, off_out, overflow_blocks=ov,
                           tail_tokens=tail)
        sx.scatter_kv(g.pool, g.batch, g.kf_R, g.vf_R, rows_d, off_out, max_rows=g.rows_cap)
        sx.sparse_attn(g.pool, g.batch, g.q_R, g.out, rows_R=rows_d, rows_off=off_out, total_rows=int(g.out.shape[0]),
                       lse=g.lse)

    def reset():
        g.batch.k_block_table.copy_(kt0)
        g.batch.v_block_table.copy_(kt0)
        g.out.zero_()
        torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        stages()
    for _ in range(2):
        reset()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(g.out, out_eager) and torch.equal(g.lse, lse_eager)
        assert np.array_equal(rows_d[:len(rows)].cpu().numpy(), rows)
