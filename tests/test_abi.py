"""CPU-only checks of the C-ABI boundary: the library builds, loads, exports every symbol that
include/sparsex.h declares, validates arguments on the host, and fails loudly without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

from paper_2606_01751_b200 import binding as sx
from paper_2606_01751_b200 import build as sxbuild
from paper_2606_01751_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    sxbuild.build()
    return sx.load()


def test_header_symbols_are_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "sparsex.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sx_[a-z_]+)\s*\(", hdr))
    assert declared == set(sx.EXPORTS), declared ^ set(sx.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert b"sm_100a" in lib.sx_version()


def test_struct_sizes_match_header():
    # int32 x5 after two pointers; the batch struct has 7 int32, 9 pointers, a double and two int32
    assert ctypes.sizeof(sx.SxPool) == 2 * 8 + 5 * 4 + 4
    assert ctypes.sizeof(sx.SxBatch) == 7 * 4 + 4 + 9 * 8 + 8 + 8
    assert sx.SxBatch.zero_copy.offset == sx.SxBatch.rope_style.offset + 4


def _host_structs(lay):
    pool = sx.SxPool(0x1000, 0x2000, lay.num_blocks, 16, lay.num_kv_heads, lay.num_q_heads, 128)
    b = sx.SxBatch(lay.num_reqs, lay.num_segments, lay.max_pages_per_req, lay.total_tokens, lay.total_new,
                   lay.total_seg_pages, int(lay.seq_len.max()), 0x100, 0x100, 0x100, 0x100, None, 0x100, 0x100,
                   0x100, 0x100, lay.rope_theta, lay.rope_style)
    return pool, b


def test_workspace_size_is_host_only(lib):
    lay = wl.config_c1()
    pool, b = _host_structs(lay)
    n = ctypes.c_size_t(0)
    assert lib.sx_workspace_size(ctypes.byref(pool), ctypes.byref(b), ctypes.byref(n)) == 0
    # at least: rope table + page descriptors + 8 lse splits + per-head partial scores + scores + row scratch
    lo = (8 * 64 * lay.num_segments + 16 * lay.total_seg_pages + 8 * 4 * lay.total_new * 8 +
          4 * 2 * lay.total_tokens + 4 * lay.total_tokens + 4 * lay.total_tokens)
    assert lo <= n.value <= lo + (64 << 20)          # + column table and split-KV partials (bounded)
    assert n.value % 256 == 0
    assert lib.sx_workspace_size(None, ctypes.byref(b), ctypes.byref(n)) == -1


def test_argument_validation(lib):
    lay = wl.config_c1()
    pool, b = _host_structs(lay)
    ws = ctypes.c_void_p(0x10000)
    bad = sx.SxPool(0x1000, 0x2000, lay.num_blocks, 16, lay.num_kv_heads, lay.num_q_heads, 64)
    assert lib.sx_rope_realign(ctypes.byref(bad), ctypes.byref(b), ws, 1 << 30, None) == -2     # head_dim
    assert b"head_dim" in lib.sx_last_error()
    bad = sx.SxPool(0x1000, 0x2000, lay.num_blocks, 32, lay.num_kv_heads, lay.num_q_heads, 128)
    assert lib.sx_rope_realign(ctypes.byref(bad), ctypes.byref(b), ws, 1 << 30, None) == -2     # block_size
    bad = sx.SxPool(0x1000, 0x2000, lay.num_blocks, 16, 3, 8, 128)
    assert lib.sx_rope_realign(ctypes.byref(bad), ctypes.byref(b), ws, 1 << 30, None) == -2     # Hq % Hkv
    bad = sx.SxPool(0x1008, 0x2000, lay.num_blocks, 16, lay.num_kv_heads, lay.num_q_heads, 128)
    assert lib.sx_rope_realign(ctypes.byref(bad), ctypes.byref(b), ws, 1 << 30, None) == -5     # alignment
    assert lib.sx_rope_realign(ctypes.byref(pool), ctypes.byref(b), ws, 16, None) == -3         # workspace
    assert lib.sx_rope_realign(ctypes.byref(pool), ctypes.byref(b), None, 1 << 30, None) == -1  # NULL ws
    assert lib.sx_sparse_attn(ctypes.byref(pool), ctypes.byref(b), 7, ws, ws, ws, 4, ws, None, ws, 1 << 30,
                              None) == -1                                                         # mode
    assert lib.sx_scatter_kv(ctypes.byref(pool), ctypes.byref(b), None, ws, ws, ws, 4, None) == -1


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback(lib):
    # valid arguments, no device: the stage must report SX_ERR_CUDA, never compute on the host
    lay = wl.config_tiny()
    pool, b = _host_structs(lay)
    ws = ctypes.c_void_p(0x10000)
    assert lib.sx_rope_realign(ctypes.byref(pool), ctypes.byref(b), ws, 1 << 30, None) == -4
    assert len(lib.sx_last_error()) > 0


def test_selection_offsets():
    lay = wl.config_tiny()
    sel_off, rows_off = sx.selection_offsets(lay)
    n_new = np.diff(lay.new_off)
    assert np.array_equal(np.diff(sel_off), lay.k_per_req)
    assert np.array_equal(np.diff(rows_off), lay.k_per_req + n_new)


def test_cow_tables_are_per_layer(lib):
    """Copy-on-write state (v_block_table) belongs to one layer: the all-layer realign refuses a COW descriptor
    with more than one layer (include/sparsex.h) instead of leaving the other layers' private pages unfilled."""
    lay = wl.config_tiny(cow=True)
    pool, b = _host_structs(lay)
    b.cow_private = 0x100
    pools = (sx.SxPool * 2)(pool, pool)
    ws = ctypes.c_void_p(0x10000)
    assert lib.sx_rope_realign_layers(pools, 2, ctypes.byref(b), ws, 1 << 30, None) == -2
    assert b"per layer" in lib.sx_last_error()


def test_check_calls_validate_host_arguments_first(lib):
    lay = wl.config_tiny()
    pool, b = _host_structs(lay)
    ws = ctypes.c_void_p(0x10000)
    assert lib.sx_check_batch(None, ctypes.byref(b), ws, 1 << 30, None) == -1
    assert lib.sx_check_batch(ctypes.byref(pool), ctypes.byref(b), ws, 16, None) == -3
    assert lib.sx_check_rows(ctypes.byref(pool), ctypes.byref(b), ws, None, 4, ws, 1 << 30, None) == -1
    assert lib.sx_launch_count() >= 0


def test_zero_copy_mode_host_rules(lib):
    """include/sparsex.h, zero-copy mode: the re-alignment refuses the descriptor, the scatter needs reserved private
    pages, CUDA-core kernels and CTA pairs are not available -- all decided on the host, before any launch."""
    lay = wl.config_tiny()
    pool, b = _host_structs(lay)
    ws = ctypes.c_void_p(0x10000)
    b.zero_copy = 2
    assert lib.sx_check_batch(ctypes.byref(pool), ctypes.byref(b), ws, 1 << 30, None) == -1
    b.zero_copy = 1
    assert lib.sx_rope_realign(ctypes.byref(pool), ctypes.byref(b), ws, 1 << 30, None) == -1
    assert b"zero-copy" in lib.sx_last_error()
    assert lib.sx_scatter_kv(ctypes.byref(pool), ctypes.byref(b), ws, ws, ws, ws, 4, None) == -1
    assert b"cow_private" in lib.sx_last_error()
    for flag in (2, 4):
        assert lib.sx_sparse_attn(ctypes.byref(pool), ctypes.byref(b), flag, ws, ws, ws, 4, ws, None, ws, 1 << 30,
                                  None) == -2
        assert b"zero-copy" in lib.sx_last_error()


def test_zero_copy_layout_aliases_every_reused_page():
    lay = wl.config_tiny(seed_id=10, tail=5)
    z = wl.zero_copy_layout(lay)
    assert z.zero_copy and z.cow and not lay.zero_copy
    covered = np.zeros(lay.k_block_table.shape, dtype=bool)
    for (req, ln, _old, new, so) in lay.segments.tolist():
        p0, n = new // 16, ln // 16
        covered[req, p0:p0 + n] = True
        assert np.array_equal(z.k_block_table[req, p0:p0 + n], lay.src_blocks[so:so + n])
        assert np.array_equal(z.cow_private[req, p0:p0 + n], lay.k_block_table[req, p0:p0 + n])
    assert np.array_equal(z.k_block_table[~covered], lay.k_block_table[~covered])
    assert np.all(z.cow_private[~covered] == -1)
    assert np.array_equal(z.v_block_table, z.k_block_table)
    assert np.array_equal(lay.k_block_table, wl.config_tiny(seed_id=10, tail=5).k_block_table)   # input untouched
