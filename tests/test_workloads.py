"""Host-side checks of the seeded workload generator (CPU only)."""
import numpy as np
import pytest

from paper_2606_01751_b200 import workloads as wl


def _check_layout(lay):
    assert lay.seq_len.sum() == lay.total_tokens
    used = []
    for r in range(lay.num_reqs):
        t = int(lay.seq_len[r])
        n_pages = (t + 15) // 16
        assert np.all(lay.k_block_table[r, :n_pages] >= 0) and np.all(lay.k_block_table[r, n_pages:] == -1)
        used.append(lay.k_block_table[r, :n_pages])
        cover = np.zeros(t, dtype=np.int32)
        cover[lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]] += 1
        for s in range(lay.num_segments):
            rq, ln, old, new, so = (int(v) for v in lay.segments[s])
            assert ln % 16 == 0 and old % 16 == 0 and new % 16 == 0
            if rq == r:
                cover[new:new + ln] += 1
        assert np.all(cover == 1)                                         # I_nr and I_reuse partition 1..T
        nn = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]
        assert np.all(np.diff(nn) > 0)
    used = np.concatenate(used + [np.concatenate(lay.pool_seg_pages)])
    assert len(np.unique(used)) == len(used) == lay.num_blocks           # pages are disjoint
    assert np.all(np.diff(lay.segments[:, 0] * (1 << 20) + lay.segments[:, 3]) > 0)   # sorted by (req, new_pos)


def test_c1_matches_baseline_config():
    lay = wl.config_c1()
    _check_layout(lay)
    assert (lay.num_q_heads, lay.num_kv_heads, lay.rope_theta) == (8, 2, 10000.0)
    assert lay.seq_len.tolist() == [2048] and lay.total_new == 512
    assert (lay.segments[:, 3] - lay.segments[:, 2]).tolist() == [128, 768, 1408]
    assert lay.k_per_req.tolist() == [230]
    assert [int(m.sum()) for m in lay.pool_salient] == [26, 26, 26]


def test_full_size_totals():
    c2, c3, c5 = wl.config_c2(), wl.config_c3(), wl.config_c5()
    for lay in (c2, c3, c5):
        _check_layout(lay)
    assert c2.seq_len.tolist() == [8192] * 4 and c2.k_per_req.tolist() == [921] * 4
    assert c3.seq_len.tolist() == [32768] and c3.total_new == 2560 and c3.k_per_req.tolist() == [3020]
    assert (c3.segments[:, 3] - c3.segments[:, 2]).tolist() == [256 * i for i in range(10)]
    assert all(2048 <= ps.length <= 4096 for ps in c3.pool_segments)
    assert c5.seq_len.tolist() == [133120] and c5.total_new == 2048 and c5.k_per_req.tolist() == [6553]
    assert (c5.num_q_heads, c5.num_kv_heads) == (28, 4)
    c4 = wl.config_c4()
    _check_layout(c4)
    assert c4.num_reqs == 16 and np.all(np.diff(c4.new_off) == 512)
    assert all(4 <= (c4.segments[:, 0] == r).sum() <= 8 for r in range(16))
    c4c = wl.config_c4(cow=True)
    assert np.array_equal(c4c.k_block_table, c4.k_block_table)
    cached_pages = c4c.cow_private >= 0
    assert np.array_equal(c4c.cow_private[cached_pages], c4c.k_block_table[cached_pages])
    assert np.all(c4c.v_block_table[cached_pages] != c4c.k_block_table[cached_pages])


@pytest.mark.parametrize("name,scale", [("C2", 1 / 8), ("C3", 1 / 16), ("C4", 1 / 8), ("C5", 1 / 32)])
def test_scaled_configs(name, scale):
    _check_layout(wl.CONFIGS[name](scale=scale))


def test_layer_tensors_seeded_and_salient():
    lay = wl.config_c1(scale=0.25)
    a, b = wl.build_layer(lay, 0), wl.build_layer(lay, 0, threads=1)
    assert np.array_equal(a.pool_k, b.pool_k) and np.array_equal(a.q_full, b.q_full)
    c = wl.build_layer(lay, 1)
    assert not np.array_equal(a.pool_k, c.pool_k)
    # salient rows carry ~4x the key norm, in the cached pool and in K_fresh
    pages = lay.pool_seg_pages[0]
    k = wl.bf16_bits_to_f32(a.pool_k[pages]).transpose(0, 2, 1, 3).reshape(-1, lay.num_kv_heads, 128)
    nrm = np.linalg.norm(k.reshape(len(k), -1), axis=1)
    sal = lay.pool_salient[0]
    assert nrm[sal].min() > 2.5 * nrm[~sal].max() / 1.5 and abs(nrm[sal].mean() / nrm[~sal].mean() - 4) < 0.3
    m = lay.salient_mask(0)
    kf = np.linalg.norm(wl.bf16_bits_to_f32(a.k_fresh).reshape(len(m), -1), axis=1)
    assert abs(kf[m].mean() / kf[~m].mean() - 4) < 0.3
    assert not m[lay.is_new_mask(0)].any()


def test_tail_layout_and_row_capacity():
    """config_tail ends two requests inside a reused segment; the capacity offsets handed to sx_score_select_ex
    must cover R = I_nr U S_key U S_ov U S_tail for ANY S_key of size k (checked with the oracle's set builder)."""
    import pytest
    torch = pytest.importorskip("torch")  # noqa: F841  (binding imports torch)
    from oracle import sx_oracle as orc
    from paper_2606_01751_b200 import binding as sx
    lay = wl.config_tail()
    assert not lay.is_new_mask(0)[-1] and not lay.is_new_mask(1)[-1] and lay.is_new_mask(2)[-1]
    for ov, tail in [(1, 64), (2, 16), (0, 0)]:
        cap = sx.rows_capacity(lay, ov, tail)
        for r in range(lay.num_reqs):
            is_new = lay.is_new_mask(r)
            cand = np.nonzero(~is_new)[0]
            k = int(lay.k_per_req[r])
            segr = [(int(n), int(n + ln)) for (rq, ln, _, n, _) in lay.segments.tolist() if rq == r]
            for sel in (cand[:k], cand[-k:] if k else cand[:0]):
                rows = orc.recompute_set(is_new, sel, segr, ov, tail)
                assert len(rows) <= cap[r + 1] - cap[r]


def test_prefix_layout_classes_partition_the_request():
    """tiny layout with prefix-cache hits: every position is exactly one of new / reused / prefix hit, the prefix
    rows of the request's own pages hold the fresh K/V of those positions, budgets count reused tokens only."""
    lay = wl.config_tiny(seed_id=15, prefix=16, tail=7)
    lt = wl.build_layer(lay, 0)
    for r in range(lay.num_reqs):
        new, reused, pre = lay.is_new_mask(r), lay.cached_mask(r), lay.prefix_mask(r)
        assert np.all(new.astype(int) + reused.astype(int) + pre.astype(int) == 1)
        assert pre[:16 * (2 - r)].all() and pre.sum() == 16 * (2 - r)
        assert int(lay.k_per_req[r]) <= int(reused.sum())
        o = int(lay.tok_off[r])
        for pos in np.nonzero(pre)[0]:
            page, row = lay.k_block_table[r, pos // 16], pos % 16
            assert np.array_equal(lt.pool_k[page, :, row, :], lt.k_fresh[o + pos])
            assert np.array_equal(lt.pool_v[page, :, row, :], lt.v_fresh[o + pos])
