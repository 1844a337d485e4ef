"""CPU checks of the test-side glue itself (tests/helpers.py): the fresh-key margin carve used for the
boundary-layer selection of paper mode, its replay, and the row sampler that targets the launch geometry."""
import os

import numpy as np

from oracle import sx_oracle as orc
from paper_2606_01751_b200 import workloads as wl

from helpers import (apply_carve_fresh, carve_margins_fresh, edge_rows, load_carve_fresh, oracle_scores_full_layer)

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_carve_fresh_gives_margin_and_replays():
    lay = wl.config_c3(scale=1.0 / 16)
    lt = wl.build_layer(lay, 3)
    ref = wl.build_layer(lay, 3)
    log = []
    hist = carve_margins_fresh(lay, lt, log=log)
    assert hist[-1] == 0
    s = oracle_scores_full_layer(lay, lt)[0]
    cand = np.nonzero(lay.cached_mask(0))[0]
    k = int(lay.k_per_req[0])
    srt = np.sort(s[cand])[::-1]
    c = 0.5 * (srt[k - 1] + srt[k])
    assert srt[k - 1] - srt[k] >= 2e-3 * c
    assert not np.any(np.abs(s[cand] - c) <= 1e-3 * c)
    # only K_fresh rows of cached positions moved; the replay reproduces the carved tensor bit for bit
    assert np.array_equal(lt.pool_k, ref.pool_k) and np.array_equal(lt.q_full, ref.q_full)
    changed = np.nonzero(np.any(lt.k_fresh != ref.k_fresh, axis=(1, 2)))[0]
    assert set(changed.tolist()) <= set(t for t, _ in log) and np.all(lay.cached_mask(0)[changed])
    apply_carve_fresh(ref, log)
    assert np.array_equal(ref.k_fresh, lt.k_fresh)


def test_committed_c3_boundary_carve_is_well_formed():
    ops = load_carve_fresh(os.path.join(GOLD, "carve_C3_L3.txt"))
    lay = wl.CONFIGS["C3"]()
    assert len(ops) > 0
    toks = np.asarray([t for t, _ in ops])
    assert toks.min() >= 0 and toks.max() < lay.total_tokens
    assert np.all(lay.cached_mask(0)[toks])                    # only cached positions are candidates
    assert set(sc for _, sc in ops) <= {1.25, 0.8}


def test_edge_rows_hits_the_seams():
    rows = np.sort(np.random.default_rng(0).choice(32768, 5580, replace=False)).astype(np.int32)
    rpp = 2 * (128 // 4)       # g = 4: 64 rows of R per CTA
    pick = edge_rows(rows, 128, rpp)
    assert np.all(np.diff(pick) > 0) and pick[0] == 0 and pick[-1] == len(rows) - 1
    n_cta = (len(rows) + rpp - 1) // rpp
    for c in list(range(0, n_cta, 7)) + [n_cta - 2, n_cta - 1]:
        lo, hi = c * rpp, min(len(rows), (c + 1) * rpp)
        assert lo in pick and hi - 1 in pick
        if lo + rpp // 2 < hi:
            assert lo + rpp // 2 - 1 in pick and lo + rpp // 2 in pick
    # full mode: consecutive rows -> every sampled CTA contributes its 128k-1 / 128k / 128k+1 rows
    allrows = np.arange(32768, dtype=np.int32)
    pick = edge_rows(allrows, 1024, rpp)
    assert len(pick) >= 1024
    pos = allrows[pick]
    assert np.sum(pos % 128 == 127) > 20 and np.sum(pos % 128 == 0) > 20 and np.sum(pos % 128 == 1) > 20
    assert len(edge_rows(allrows[:5], 128, rpp)) == 5
