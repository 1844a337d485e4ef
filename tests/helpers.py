"""Test-side glue: feeds the seeded workloads to the fp64 oracle, carves top-k margins, compares.

Lives in tests/ because it calls oracle/ (only tests, smoke() and bench.py's CPU legs may).
"""
from __future__ import annotations

import copy

import numpy as np

from oracle import sx_oracle as orc
from paper_2606_01751_b200 import workloads as wl

# tolerances fixed by BASELINE.json north_star (bf16 in / fp32 accumulate vs fp64)
MAX_ABS = 2e-2
MEAN_ABS = 2e-3
# reading A12: on rows whose |value| exceeds 2.56 one bf16 ulp is already > 2e-2; per-element bound
# max(2e-2, 2^-7 |ref|) (2^-7 |ref| >= one bf16 ulp of ref).
BF16_ULP_REL = 2.0 ** -7


def oracle_layer(lay: wl.Layout, lt: wl.LayerTensors, mode="sparse", rows_given=None, tables=None,
                 k_per_req=None):
    """Run the oracle layer driver on COPIES of the pool/tables. Returns (result, pool_k, pool_v, kt, vt)."""
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    if tables is None:
        kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    else:
        kt, vt = tables[0].copy(), tables[1].copy()
    res = orc.layer_step(pk, pv, kt, vt, lay.cow_private if lay.cow else None, lay.segments,
                         lay.src_blocks, lay.rope_theta, lay.rope_style, lay.seq_len, lay.tok_off,
                         lay.new_off, lay.new_idx, lay.k_per_req if k_per_req is None else k_per_req,
                         lay.num_q_heads, lt.q_full, lt.k_fresh, lt.v_fresh, mode=mode,
                         rows_given=rows_given)
    return res, pk, pv, kt, vt


def oracle_scores_after_realign(lay: wl.LayerTensors, lt: wl.LayerTensors):
    """fp64 scores of every request on the pool state stage (b) sees: realign + scatter(I_nr)."""
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    out = []
    for r in range(lay.num_reqs):
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        nidx = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]
        orc.scatter_kv(pk, pv, kt, vt, None, r, nidx, lt.k_fresh[o + nidx], lt.v_fresh[o + nidx])
        out.append(orc.scores(pk, kt[r], t, lt.q_full[o + nidx], nidx, lay.num_q_heads))
    return out


def carve_margins(lay: wl.Layout, lt: wl.LayerTensors, tau: float = 1e-3, max_iter: int = 12, log=None,
                  widen_later: float = 1.5):
    """Reading A9/A10: the x4 salient tokens alone do not make the rank-k cut unambiguous
    (ratio > salient fraction, the cut falls among ordinary tokens). Enforce a relative margin at the
    cut: every cached token whose fp64 score lies within tau of the midpoint c between ranks k and k+1
    has its SOURCE key row rescaled (x1.25 above the cut, x0.8 below), re-rounded to bf16; repeat until
    the band is empty and the gap is >= 2 tau. Modifies lt.pool_k in place; returns per-iteration band
    sizes. Uses the oracle, hence lives in tests/. `log` (a list) receives every (block, row, scale)
    applied, in order, so that the result can be replayed with apply_carve (tests/golden/carve_*.txt).
    """
    hist = []
    bs = wl.PAGE
    for it in range(max_iter):
        # every rescaled key also moves the softmax normalisers, hence the cut itself, by a few 1e-4
        # relative: clear a wider band (3 tau first, 1.5 tau later) than the one that must end up empty
        widen = 3.0 if it == 0 else widen_later
        sc = oracle_scores_after_realign(lay, lt)
        band_total = 0
        touched = set()     # a source row shared by two requests is moved once per iteration (else a row that
                            # sits above one request's cut and below another's is scaled x1.25 x0.8 = x1)
        for r in range(lay.num_reqs):
            k = int(lay.k_per_req[r])
            is_new = lay.is_new_mask(r)
            cand = np.nonzero(lay.cached_mask(r))[0]    # I_reuse (prefix-cache hits are not candidates)
            if k <= 0 or k >= len(cand):
                continue
            s = sc[r][cand]
            order = np.lexsort((cand, -s))
            c = 0.5 * (s[order[k - 1]] + s[order[k]])
            gap_ok = (s[order[k - 1]] - s[order[k]]) >= 2 * tau * c
            if gap_ok and not np.any(np.abs(s - c) <= tau * c):
                continue
            band = np.nonzero(np.abs(s - c) <= widen * tau * c)[0]
            if len(band) == 0:          # gap too small but nobody inside the band: push the two neighbours
                band = np.asarray([order[k - 1], order[k]])
            band_total += len(band)
            # map position -> (segment, offset) -> source page row
            for bi in band.tolist():
                pos = int(cand[bi])
                scale = 1.25 if s[bi] > c else 0.8
                for sidx in range(lay.num_segments):
                    rq, ln, _, new_pos, src_off = (int(v) for v in lay.segments[sidx])
                    if rq == r and new_pos <= pos < new_pos + ln:
                        j = pos - new_pos
                        blk = int(lay.src_blocks[src_off + j // bs])
                        if (blk, j % bs) in touched:
                            break
                        touched.add((blk, j % bs))
                        row = orc.bf16_to_f64(lt.pool_k[blk, :, j % bs, :]) * scale
                        lt.pool_k[blk, :, j % bs, :] = orc.f64_to_bf16(row)
                        if log is not None:
                            log.append((blk, j % bs, scale))
                        break
        hist.append(band_total)
        if band_total == 0:
            return hist
    raise RuntimeError("margin carving did not converge: %r" % hist)


def oracle_scores_full_layer(lay: wl.Layout, lt: wl.LayerTensors):
    """fp64 scores of every request on the pool state the BOUNDARY-layer selection sees (Alg. 1 l.507-531,
    readings A11/A16): the layer ran in full mode, so every position holds its fresh key."""
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    orc.realign(pk, pv, kt, vt, lay.segments, lay.src_blocks, lay.rope_theta, lay.rope_style)
    out = []
    for r in range(lay.num_reqs):
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        orc.scatter_kv(pk, pv, kt, vt, None, r, np.arange(t, dtype=np.int32), lt.k_fresh[o:o + t], lt.v_fresh[o:o + t])
        nidx = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]
        out.append(orc.scores(pk, kt[r], t, lt.q_full[o + nidx], nidx, lay.num_q_heads))
    return out


def carve_margins_fresh(lay: wl.Layout, lt: wl.LayerTensors, tau: float = 1e-3, max_iter: int = 20, log=None,
                        widen_later: float = 1.5):
    """carve_margins for the boundary-layer selection of paper mode (readings A10/A11/A16): that selection
    reads a pool in which every key is FRESH (the layer ran full attention), so the margin at the rank-k cut is
    carved into lt.k_fresh: the fresh key row of every cached position whose fp64 score lies within tau of the
    cut is rescaled (x1.25 above, x0.8 below) and re-rounded to bf16, until the band is empty and the gap is
    >= 2 tau. `log` receives (batch token index, scale) in application order (replay: apply_carve_fresh)."""
    hist = []
    for it in range(max_iter):
        widen = 3.0 if it == 0 else widen_later
        sc = oracle_scores_full_layer(lay, lt)
        band_total = 0
        for r in range(lay.num_reqs):
            k = int(lay.k_per_req[r])
            cand = np.nonzero(lay.cached_mask(r))[0]
            if k <= 0 or k >= len(cand):
                continue
            s = sc[r][cand]
            order = np.lexsort((cand, -s))
            c = 0.5 * (s[order[k - 1]] + s[order[k]])
            gap_ok = (s[order[k - 1]] - s[order[k]]) >= 2 * tau * c
            if gap_ok and not np.any(np.abs(s - c) <= tau * c):
                continue
            band = np.nonzero(np.abs(s - c) <= widen * tau * c)[0]
            if len(band) == 0:
                band = np.asarray([order[k - 1], order[k]])
            band_total += len(band)
            o = int(lay.tok_off[r])
            for bi in band.tolist():
                tok = o + int(cand[bi])
                scale = 1.25 if s[bi] > c else 0.8
                lt.k_fresh[tok] = orc.f64_to_bf16(orc.bf16_to_f64(lt.k_fresh[tok]) * scale)
                if log is not None:
                    log.append((tok, scale))
        hist.append(band_total)
        if band_total == 0:
            return hist
    raise RuntimeError("margin carving (fresh keys) did not converge: %r" % hist)


def apply_carve_fresh(lt: wl.LayerTensors, ops):
    """Replay a fresh-key carve log: k_fresh[token] (every KV head) times scale, re-rounded to bf16, in order."""
    for tok, scale in ops:
        lt.k_fresh[tok] = orc.f64_to_bf16(orc.bf16_to_f64(lt.k_fresh[tok]) * scale)


def load_carve_fresh(path):
    ops = []
    with open(path) as f:
        for ln in f:
            if ln.startswith("#") or not ln.strip():
                continue
            a, b = ln.split()
            ops.append((int(a), float(b)))
    return ops


def edge_rows(rows: np.ndarray, n_spread: int, rows_per_pair: int, every: int = 7) -> np.ndarray:
    """Indices into the sorted row list `rows` (one request) chosen to hit the launch geometry of stage (c) at
    full size: a spread of n_spread rows, plus -- for every `every`-th CTA (rows_per_pair rows of R per CTA; an odd
    stride, so that both CTAs of a 2-CTA cluster and both parities of 64-row CTAs against 128-key tiles occur) and
    for the last two CTAs (the last cluster, whose odd pair may be empty) -- the CTA's first row, the last row
    of its first query tile, the first row of its second tile and its last row, plus every listed row whose
    POSITION is 128k-1, 128k or 128k+1 for the key-tile edges k of that CTA's last row."""
    n = len(rows)
    if n == 0:
        return np.zeros(0, np.int64)
    pick = set(np.unique(np.linspace(0, n - 1, min(n, n_spread)).astype(np.int64)).tolist())
    n_cta = (n + rows_per_pair - 1) // rows_per_pair
    ctas = sorted(set(list(range(0, n_cta, every)) + [max(0, n_cta - 2), n_cta - 1]))
    half = rows_per_pair // 2
    for c in ctas:
        lo, hi = c * rows_per_pair, min(n, (c + 1) * rows_per_pair)
        for i in (lo, lo + half - 1, lo + half, hi - 1):
            if lo <= i < hi:
                pick.add(int(i))
        # rows of this CTA sitting on a 128-key tile edge
        pos = rows[lo:hi].astype(np.int64)
        m = ((pos % 128) == 127) | ((pos % 128) == 0) | ((pos % 128) == 1)
        for i in np.nonzero(m)[0][:6].tolist() + np.nonzero(m)[0][-3:].tolist():
            pick.add(int(lo + i))
    return np.asarray(sorted(pick), dtype=np.int64)


def apply_carve(lt: wl.LayerTensors, ops):
    """Replay a carve log: key row (block, row) of every KV head times scale, re-rounded to bf16, in order."""
    for blk, row, scale in ops:
        v = orc.bf16_to_f64(lt.pool_k[blk, :, row, :]) * scale
        lt.pool_k[blk, :, row, :] = orc.f64_to_bf16(v)


def load_carve(path):
    ops = []
    with open(path) as f:
        for ln in f:
            if ln.startswith("#") or not ln.strip():
                continue
            a, b, c = ln.split()
            ops.append((int(a), int(b), float(c)))
    return ops


def check_close(name, got, ref64, max_abs=MAX_ABS, mean_abs=MEAN_ABS, ulp_floor=False):
    """Tolerance of BASELINE.json north_star. With ulp_floor the per-element bound is
    max(max_abs, 2^-7 |ref|) (reading A12: one bf16 ulp on the x4 salient key rows)."""
    got = np.asarray(got, dtype=np.float64)
    ref64 = np.asarray(ref64, dtype=np.float64)
    assert got.shape == ref64.shape, (name, got.shape, ref64.shape)
    if got.size == 0:
        return 0.0, 0.0
    err = np.abs(got - ref64)
    bound = np.full_like(err, max_abs)
    if ulp_floor:
        bound = np.maximum(bound, BF16_ULP_REL * np.abs(ref64))
    worst = float(err.max())
    mean = float(err.mean())
    assert np.all(np.isfinite(got)), name + ": non-finite output"
    assert np.all(err <= bound), "%s: max-abs %.4g exceeds bound (n_bad=%d)" % (
        name, worst, int((err > bound).sum()))
    assert mean <= mean_abs, "%s: mean-abs %.4g > %.4g" % (name, mean, mean_abs)
    return worst, mean


def clone_layer(lt: wl.LayerTensors) -> wl.LayerTensors:
    return copy.deepcopy(lt)
