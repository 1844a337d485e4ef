"""sx_sparse_attn_noalloc (include/sparsex.h): stage (c) for small row sets with the library's built-in scratch --
no workspace argument, no allocation -- against the existing path (sx_sparse_attn with a caller workspace) on the
same inputs, two calls in a row (the scratch is shared by every call and keeps the last call's contents).

Collected last on purpose (the file name sorts behind every other test file): the suite runs with pytest -x, so a
failure here hides nothing. It builds its own inputs, so it passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest
import torch

from paper_2606_01751_b200 import workloads as wl

pytestmark = pytest.mark.gpu

# tolerances of the attention parity tests (tests/helpers.py: BASELINE.json north_star; LSE as in test_gpu_parity.py)
MAX_ABS, MEAN_ABS, LSE_ABS = 2e-2, 2e-3, 2e-3


def _bf16_bits_to_f64(t: torch.Tensor) -> np.ndarray:
    return t.view(torch.bfloat16).to(torch.float64).cpu().numpy()


def _layer(lay):
    """One layer on the GPU after realign + scatter of every fresh row: the pool a small row set attends over."""
    from paper_2606_01751_b200 import binding as sx
    from paper_2606_01751_b200.layer import GpuLayer
    lt = wl.build_layer(lay, 0)
    g = GpuLayer(lay, lt)
    g.realign()
    all_rows = torch.cat([torch.arange(int(n), dtype=torch.int32) for n in lay.seq_len]).to(g.dev)
    sx.scatter_kv(g.pool, g.batch, g.k_fresh, g.v_fresh, all_rows, g.batch.tok_off, max_rows=lay.total_tokens)
    torch.cuda.synchronize()
    return sx, g


def _rows(lay, g, picks):
    """picks[r] = positions of request r (ascending) -> (rows, rows_off, compact q) on the device."""
    off = np.concatenate([[0], np.cumsum([len(p) for p in picks])]).astype(np.int32)
    rows = np.concatenate(picks).astype(np.int32)
    tok = np.concatenate([int(lay.tok_off[r]) + np.asarray(p, dtype=np.int64) for r, p in enumerate(picks)])
    q = g.q_full[torch.from_numpy(tok).to(g.dev)].contiguous()
    return torch.from_numpy(rows).to(g.dev), torch.from_numpy(off).to(g.dev), q


def _both(sx, g, lay, picks):
    rows, off, q = _rows(lay, g, picks)
    n, hq = int(rows.numel()), lay.num_q_heads
    ref_o = torch.zeros((n, hq, 128), dtype=torch.int16, device=g.dev)
    ref_l = torch.zeros((n, hq), dtype=torch.float32, device=g.dev)
    new_o, new_l = torch.full_like(ref_o, 0x7fc0), torch.full_like(ref_l, float("nan"))
    sx.sparse_attn(g.pool, g.batch, q, ref_o, rows_R=rows, rows_off=off, total_rows=n, lse=ref_l, cta_pair=False)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    sx.sparse_attn_noalloc(g.pool, g.batch, q, new_o, rows, off, total_rows=n, lse=new_l)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    a, b = _bf16_bits_to_f64(new_o), _bf16_bits_to_f64(ref_o)
    assert np.isfinite(a).all()
    assert np.max(np.abs(a - b)) <= MAX_ABS and np.mean(np.abs(a - b)) <= MEAN_ABS
    assert np.max(np.abs(new_l.cpu().numpy().astype(np.float64) - ref_l.cpu().numpy().astype(np.float64))) <= LSE_ABS
    return torch.equal(new_o, ref_o) and torch.equal(new_l, ref_l), free_before, free_after


def test_noalloc_matches_the_workspace_path_on_two_calls_in_a_row():
    """C1 (2K context, 8 Q / 2 KV heads): the last 6 rows, then -- the scratch still holding the first call's
    partials and rendezvous words -- 11 other rows; both against sx_sparse_attn. Both take 8 key splits in either
    path (fewer than 148 blocks, 16 key tiles), so the results are not only within tolerance but the same bits."""
    lay = wl.config_c1()
    sx, g = _layer(lay)
    t = int(lay.seq_len[0])
    same1, _, _ = _both(sx, g, lay, [np.arange(t - 6, t)])
    same2, before, after = _both(sx, g, lay, [np.unique(np.concatenate([[3, 200, t // 2], np.arange(t - 40, t, 5)]))])
    assert same1 and same2                   # equal cuts give equal bits (deterministic merge order)
    assert after >= before                   # the second call took no device memory
    # and once more the first row set: a third call on the used scratch, same answer
    same3, _, _ = _both(sx, g, lay, [np.arange(t - 6, t)])
    assert same3


def test_noalloc_batch_of_requests_and_the_size_limit():
    """C4 at 1/8 scale (6 requests, 32 Q / 8 KV heads): a few rows per request (several row-pair blocks meeting on
    their own rendezvous words), twice in a row; then the limit: 33 rows x 32 heads = 1 056 pairs > 1 024 is
    refused with a clear error and nothing is launched (the output keeps its fill pattern)."""
    lay = wl.config_c4(scale=0.125, num_reqs=6)
    sx, g = _layer(lay)
    picks = [np.unique(np.concatenate([[1, int(t) // 3], np.arange(int(t) - 3, int(t))])) for t in lay.seq_len]
    assert sum(len(p) for p in picks) * lay.num_q_heads <= sx.NOALLOC_MAX_PAIRS
    _both(sx, g, lay, picks)
    _both(sx, g, lay, [p[-2:] for p in picks])
    t0 = int(lay.seq_len[0])
    # beyond it
    rows, off, q = _rows(lay, g, [np.arange(t0 - 33, t0)] + [np.zeros(0, np.int64)] * (lay.num_reqs - 1))
    out = torch.full((33, lay.num_q_heads, 128), 0x1234, dtype=torch.int16, device=g.dev)
    with pytest.raises(sx.SparseXError, match="SX_NOALLOC_MAX_PAIRS"):
        sx.sparse_attn_noalloc(g.pool, g.batch, q, out, rows, off, total_rows=33)
    torch.cuda.synchronize()
    assert bool((out == 0x1234).all())


def test_noalloc_near_the_limit_cuts_the_keys_differently_but_stays_in_tolerance():
    """C5 at 1/16 scale (8 320 keys, 28 Q / 4 KV heads, g = 7): the last 35 rows = 980 (row, head) pairs in 4 blocks.
    sx_sparse_attn cuts the keys into 32 splits; 32 x 980 partial slots do not fit the built-in scratch, so the
    no-allocation path takes 18: different rounding, same tolerance. Twice in a row."""
    lay = wl.config_c5(scale=1.0 / 16)
    sx, g = _layer(lay)
    t = int(lay.seq_len[0])
    assert 35 * lay.num_q_heads <= sx.NOALLOC_MAX_PAIRS
    _both(sx, g, lay, [np.arange(t - 35, t)])
    same, _, _ = _both(sx, g, lay, [np.arange(t - 16, t)])      # 448 pairs: 32 splits fit, equal cuts again
    assert same


def test_noalloc_under_cuda_graph_capture_and_replay():
    """The use case the entry point exists for: captured into a CUDA graph (after one eager call, which performs the
    once-per-device address lookup) and replayed; every replay gives the bits of the eager call."""
    lay = wl.config_c1()
    sx, g = _layer(lay)
    t = int(lay.seq_len[0])
    rows, off, q = _rows(lay, g, [np.arange(t - 6, t)])
    out = torch.zeros((6, lay.num_q_heads, 128), dtype=torch.int16, device=g.dev)
    lse = torch.zeros((6, lay.num_q_heads), dtype=torch.float32, device=g.dev)
    sx.sparse_attn_noalloc(g.pool, g.batch, q, out, rows, off, total_rows=6, lse=lse)
    torch.cuda.synchronize()
    eager_o, eager_l = out.clone(), lse.clone()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        sx.sparse_attn_noalloc(g.pool, g.batch, q, out, rows, off, total_rows=6, lse=lse)
    for _ in range(3):
        out.zero_()
        lse.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, eager_o) and torch.equal(lse, eager_l)
