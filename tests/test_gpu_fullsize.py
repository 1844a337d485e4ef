"""GPU parity at BASELINE.json's FULL sizes, in the launch configurations bench.py times.

The oracle cannot finish a whole full-size layer in seconds, so (tier rule 3):
  * realigned keys, V copies, scattered rows, block tables: compared on EVERY element (bit level / one bf16 ulp);
  * scores, the selected set S_key and R: compared in full (the oracle's score pass takes seconds to a minute);
  * attention outputs and LSE: on the headline config C3 EVERY row of the sparse layer (5 580) and >= 1 024 rows
    of the 32K full layer; on C2 / C4 / C5 a spread of rows; in every case the sample is built by
    helpers.edge_rows so that it contains, for every seventh CTA and for the last cluster, the CTA's first / last row,
    the rows on its query-tile seam and the rows whose position sits on a 128-key tile edge (128k-1, 128k, 128k+1).
Index sets must be bit-exact; the top-k margin of the inputs is the replayed carve log
tests/golden/carve_<cfg>.txt (written by tests/golden/make_carve.py from the oracle alone; readings A9/A10),
and the test re-checks on the oracle's own scores that the margin really holds. The boundary-layer selection of
C3 in paper mode (all keys fresh) has its own carve log, carve_C3_L3.txt, applied to K_fresh of layer 3.
"""
import os

import numpy as np
import pytest
import torch

from oracle import sx_oracle as orc
from paper_2606_01751_b200 import workloads as wl

from helpers import apply_carve, apply_carve_fresh, check_close, edge_rows, load_carve, load_carve_fresh

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
TAU = 1e-3
SCORE_RTOL = 5e-3
ROWS_PER_REQ = {"C2": 64, "C3": 1 << 30, "C4": 12, "C5": 128}   # spread rows per request (C3: every row)


def _gpu():
    from paper_2606_01751_b200 import binding as sx   # noqa: F401  (fails loudly if the .so is missing)
    from paper_2606_01751_b200.layer import GpuLayer, dev_to_bits
    return GpuLayer, dev_to_bits


def _sample(rows: np.ndarray, n: int, lay) -> np.ndarray:
    """Indices into `rows` (one request): n rows spread over the whole range plus the rows that sit on the launch
    geometry's seams (helpers.edge_rows; a CTA of stage (c) owns 2 * (128 / g) rows of R)."""
    if len(rows) <= n:
        return np.arange(len(rows))
    g = lay.num_q_heads // lay.num_kv_heads
    return edge_rows(rows, n, 2 * (128 // g))


def _check_keys(name, lay, lt, gk, pk, kt, kref):
    """Re-rotated keys of every destination page: <= 1 bf16 ulp from the oracle's rounding everywhere,
    and within the north_star tolerance of the unrounded fp64 value (reading A12)."""
    dst = []
    for (req, ln, old, new, so) in lay.segments.tolist():
        dst.append(kt[req][new // 16:(new + ln) // 16])
    dst = np.concatenate(dst)
    a = orc.bf16_to_f64(gk[dst])
    b = orc.bf16_to_f64(pk[dst])
    assert np.all(np.abs(a - b) <= 2.0 ** -7 * np.abs(b) + 1e-5), name
    assert np.mean(gk[dst] == pk[dst]) > 0.995, name
    got = np.transpose(a, (0, 2, 1, 3)).reshape(-1, a.shape[1], a.shape[3])   # [token][head][d]
    check_close(name + " realigned K vs fp64", got, kref, ulp_floor=True)
    untouched = np.ones(lay.num_blocks, dtype=bool)
    untouched[dst] = False
    assert np.array_equal(gk[untouched], lt.pool_k[untouched]), name


@pytest.mark.parametrize("name", ["C2", "C2-pair", "C3", "C3-1cta", "C4", "C4-cow", "C5"])
def test_fullsize_sparse_layer(name):
    """One sparse-mode layer with its own two-sweep selection (what bench.py --config <name> times).
    C4-cow: the copy-on-write variant of C4 (V pages alias the shared source pages until a row is written,
    reading A14); keys, scores and index sets are those of C4, so the same carve log applies.
    C2-pair: stage (c) with SX_ATTN_CTA_PAIR (the 2-CTA cluster kernel; 47 row pairs per request = an odd count).
    C3: one sparse layer of the headline config at T = 32 768 with its own two-sweep selection (k = 3 020,
    |R| = 5 580; bench.py's C3_select_every_layer), every output row checked; the library picks the 2-CTA cluster
    kernel for it (one request); C3-1cta forces the single-CTA kernel on the same inputs."""
    GpuLayer, dev_to_bits = _gpu()
    cta_pair = True if name.endswith("-pair") else (False if name.endswith("-1cta") else None)
    lay = wl.config_c4(cow=True) if name == "C4-cow" else wl.CONFIGS[name.split("-")[0]]()
    name = name.split("-")[0]
    lt = wl.build_layer(lay, 0)
    apply_carve(lt, load_carve(os.path.join(GOLD, "carve_%s.txt" % name)))
    hq = lay.num_q_heads

    # ---- GPU: whole layer, chained
    g = GpuLayer(lay, lt)
    g.cta_pair = cta_pair
    g.realign()
    torch.cuda.synchronize()
    gk_re, gv_re = dev_to_bits(g.pool_k).copy(), dev_to_bits(g.pool_v).copy()
    g.scatter_new()
    g.select()
    g.stage_rows(g.sel_idx, g.rows_R)
    g.scatter_sel()
    g.attend()
    torch.cuda.synchronize()
    g_sc = g.scores.cpu().numpy().astype(np.float64)
    g_sel, g_rows = g.sel_idx.cpu().numpy(), g.rows_R.cpu().numpy()
    g_lse = g.lse.cpu().numpy().astype(np.float64)

    # ---- oracle: stage (a) on everything
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    cow = lay.cow_private if lay.cow else None
    kref = orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    _check_keys(name, lay, lt, gk_re, pk, kt, kref)
    del kref
    assert np.array_equal(gv_re, pv), name                     # V pages: bit copies

    # ---- oracle: stages (d), (b), (d), (c) per request
    for r in range(lay.num_reqs):
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        nidx = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]
        orc.scatter_kv(pk, pv, kt, vt, cow, r, nidx, lt.k_fresh[o + nidx], lt.v_fresh[o + nidx])
        s = orc.scores(pk, kt[r], t, lt.q_full[o + nidx], nidx, hq)
        is_new = lay.is_new_mask(r)
        k = int(lay.k_per_req[r])
        sel, rows = orc.select_topk(s, is_new, k)
        cand = np.nonzero(~is_new)[0]
        srt = np.sort(s[cand])[::-1]
        if 0 < k < len(cand):                                  # the replayed carve still gives the margin
            c = 0.5 * (srt[k - 1] + srt[k])
            assert srt[k - 1] - srt[k] >= 2 * TAU * c * 0.999, (name, r, srt[k - 1], srt[k])
        rel = np.abs(g_sc[o:o + t] - s) / (np.abs(s) + 1e-2)
        assert rel.max() < SCORE_RTOL, (name, r, rel.max())
        s0, s1 = g.sel_off_h[r], g.sel_off_h[r + 1]
        r0, r1 = g.rows_off_h[r], g.rows_off_h[r + 1]
        assert np.array_equal(g_sel[s0:s1], sel), (name, r)    # bit-exact index sets
        assert np.array_equal(g_rows[r0:r1], rows), (name, r)
        orc.scatter_kv(pk, pv, kt, vt, cow, r, sel, lt.k_fresh[o + sel], lt.v_fresh[o + sel])
        pick = _sample(rows, ROWS_PER_REQ[name], lay)
        ref_o, ref_l = orc.attention(pk, pv, kt[r], vt[r], t, lt.q_full[o + rows[pick]], rows[pick], hq,
                                     want_lse=True)
        got = orc.bf16_to_f64(dev_to_bits(g.out[r0:r1][torch.from_numpy(pick).to(g.dev)]))
        check_close("%s req %d O (sampled rows)" % (name, r), got, ref_o)
        assert np.max(np.abs(g_lse[r0:r1][pick] - ref_l)) < 2e-3

    # ---- pool and tables after the layer
    gk, gv = dev_to_bits(g.pool_k), dev_to_bits(g.pool_v)
    gkt, gvt = g.batch.k_block_table.cpu().numpy(), g.batch.v_block_table.cpu().numpy()
    assert np.array_equal(gkt, kt) and np.array_equal(gvt, vt)
    assert np.array_equal(gv, pv)
    src = np.concatenate(lay.pool_seg_pages)
    assert np.array_equal(gk[src], lt.pool_k[src]) and np.array_equal(gv[src], lt.pool_v[src])   # shared pages
    for r in range(lay.num_reqs):                              # scattered rows bit-exact
        t = int(lay.seq_len[r])
        rows = g_rows[g.rows_off_h[r]:g.rows_off_h[r + 1]]
        a = gk[gkt[r][rows // 16], :, rows % 16, :]
        b = pk[kt[r][rows // 16], :, rows % 16, :]
        assert np.array_equal(a, b), (name, r)


def test_fullsize_c3_paper_mode():
    """C3 as bench.py runs it: boundary layer 3 in full mode (32K rows), single-sweep selection fed with that
    layer's LSE, layer 4 in sparse mode on the selected R (one scatter of the fresh K,V of R)."""
    GpuLayer, dev_to_bits = _gpu()
    lay = wl.CONFIGS["C3"]()
    hq = lay.num_q_heads
    t = int(lay.seq_len[0])
    l3 = wl.build_layer(lay, 3)
    apply_carve_fresh(l3, load_carve_fresh(os.path.join(GOLD, "carve_C3_L3.txt")))   # margin at the rank-k cut

    g3 = GpuLayer(lay, l3)
    g3.step_full()
    g3.select(lse_new=g3.lse, lse_by_token=True)
    torch.cuda.synchronize()

    # oracle layer 3: realign, scatter every row, attention on sampled rows
    pk, pv = l3.pool_k.copy(), l3.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    allrows = np.arange(t, dtype=np.int32)
    orc.scatter_kv(pk, pv, kt, vt, None, 0, allrows, l3.k_fresh, l3.v_fresh)
    assert np.array_equal(dev_to_bits(g3.pool_k)[kt[kt >= 0]], pk[kt[kt >= 0]])
    assert np.array_equal(dev_to_bits(g3.pool_v), pv)
    pick = np.unique(np.concatenate([_sample(allrows, 1024, lay), [0, 1, 127, 128, 129, t - 1]]))
    assert len(pick) >= 1024
    ref_o, ref_l = orc.attention(pk, pv, kt[0], vt[0], t, l3.q_full[pick], pick.astype(np.int32), hq, want_lse=True)
    pick_d = torch.from_numpy(pick).to(g3.dev)
    check_close("C3 layer 3 full O (sampled rows)", orc.bf16_to_f64(dev_to_bits(g3.out[pick_d])), ref_o)
    assert np.max(np.abs(g3.lse[pick_d].cpu().numpy().astype(np.float64) - ref_l)) < 2e-3

    # boundary selection (Alg. 1 l.515-531): all keys of layer 3 are fresh; the margin at the cut was carved into
    # K_fresh of layer 3 (carve_C3_L3.txt), so S_key and R must be bit-exact
    s = orc.scores(pk, kt[0], t, l3.q_full[lay.new_idx], lay.new_idx, hq)
    is_new = lay.is_new_mask(0)
    k = int(lay.k_per_req[0])
    ref_sel, ref_rows = orc.select_topk(s, is_new, k)
    g_sc = g3.scores.cpu().numpy().astype(np.float64)
    assert np.max(np.abs(g_sc - s) / (np.abs(s) + 1e-2)) < SCORE_RTOL
    sel = g3.sel_idx.cpu().numpy()
    rows = g3.rows_R.cpu().numpy()
    cand = np.nonzero(~is_new)[0]
    srt = np.sort(s[cand])[::-1]
    c = 0.5 * (srt[k - 1] + srt[k])
    assert srt[k - 1] - srt[k] >= 2 * TAU * c * 0.999, (srt[k - 1], srt[k])   # the replayed carve gives the margin
    assert np.array_equal(sel, ref_sel)                                       # bit-exact index sets
    assert np.array_equal(rows, ref_rows)

    # layer 4 (sparse) on the GPU's R
    l4 = wl.build_layer(lay, 4)
    g4 = GpuLayer(lay, l4)
    g4.step_sparse(rows_given=(g3.sel_idx, g3.rows_R))
    torch.cuda.synchronize()
    pk, pv = l4.pool_k.copy(), l4.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    kref = orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    orc.scatter_kv(pk, pv, kt, vt, None, 0, rows, l4.k_fresh[rows], l4.v_fresh[rows])
    gk = dev_to_bits(g4.pool_k)
    assert np.array_equal(dev_to_bits(g4.pool_v), pv)
    a = orc.bf16_to_f64(orc.gather_tokens(gk, kt[0], t))
    b = orc.bf16_to_f64(orc.gather_tokens(pk, kt[0], t))
    assert np.array_equal(a[rows], b[rows])
    assert np.all(np.abs(a - b) <= 2.0 ** -7 * np.abs(b) + 1e-5)
    del kref
    pick = np.arange(len(rows))                                               # every row of R
    ref_o, ref_l = orc.attention(pk, pv, kt[0], vt[0], t, l4.q_full[rows[pick]], rows[pick], hq, want_lse=True)
    got = orc.bf16_to_f64(dev_to_bits(g4.out[torch.from_numpy(pick).to(g4.dev)]))
    check_close("C3 layer 4 sparse O (all rows of the boundary R)", got, ref_o)
    assert np.max(np.abs(g4.lse.cpu().numpy().astype(np.float64)[pick] - ref_l)) < 2e-3
