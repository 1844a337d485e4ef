"""ctypes binding of libsparsex.so (include/sparsex.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; PyTorch is used here for device
memory and streams and nothing else. There is no fallback: if the library is missing or a call
fails, an exception is raised.

    from paper_2606_01751_b200 import binding as sx
    b = sx.DeviceBatch(layout, device)          # uploads the block-table / segment-map descriptor
    pool = sx.DevicePool(pool_k, pool_v, Hq)    # wraps two torch tensors (bf16 bits)
    sx.rope_realign(pool, b); sx.scatter_kv(...); sx.score_select(...); sx.sparse_attn(...)
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libsparsex.so")
_lib = None

SX_OK = 0
EXPORTS = ["sx_workspace_size", "sx_rope_realign", "sx_rope_realign_layers", "sx_scatter_kv", "sx_score_select",
           "sx_score_select_ex", "sx_sparse_attn", "sx_check_batch", "sx_check_rows", "sx_launch_count",
           "sx_probe_pipe", "sx_sparse_attn_noalloc", "sx_last_error", "sx_version"]
NOALLOC_MAX_PAIRS = 1024          # SX_NOALLOC_MAX_PAIRS of include/sparsex.h


class SxPool(ctypes.Structure):
    _fields_ = [("k", ctypes.c_void_p), ("v", ctypes.c_void_p), ("num_blocks", ctypes.c_int32),
                ("block_size", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32),
                ("num_q_heads", ctypes.c_int32), ("head_dim", ctypes.c_int32)]


class SxBatch(ctypes.Structure):
    _fields_ = [("num_reqs", ctypes.c_int32), ("num_segments", ctypes.c_int32),
                ("max_pages_per_req", ctypes.c_int32), ("total_tokens", ctypes.c_int32),
                ("total_new", ctypes.c_int32), ("total_seg_pages", ctypes.c_int32),
                ("max_seq_len", ctypes.c_int32),
                ("seq_len", ctypes.c_void_p), ("tok_off", ctypes.c_void_p),
                ("k_block_table", ctypes.c_void_p), ("v_block_table", ctypes.c_void_p),
                ("cow_private", ctypes.c_void_p), ("segments", ctypes.c_void_p),
                ("src_blocks", ctypes.c_void_p), ("new_off", ctypes.c_void_p), ("new_idx", ctypes.c_void_p),
                ("rope_theta", ctypes.c_double), ("rope_style", ctypes.c_int32), ("zero_copy", ctypes.c_int32)]


class SparseXError(RuntimeError):
    pass


def lib_path() -> str:
    return _LIB_PATH


def load():
    """Load libsparsex.so (built in-tree by paper_2606_01751_b200.build). Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise SparseXError("libsparsex.so not built: run `python -m paper_2606_01751_b200.build` "
                               "(there is no CPU fallback)")
        lib = ctypes.CDLL(_LIB_PATH)
        vp, i32, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_size_t
        PP, PB = ctypes.POINTER(SxPool), ctypes.POINTER(SxBatch)
        lib.sx_workspace_size.restype = ctypes.c_int
        lib.sx_workspace_size.argtypes = [PP, PB, ctypes.POINTER(sz)]
        lib.sx_rope_realign.restype = ctypes.c_int
        lib.sx_rope_realign.argtypes = [PP, PB, vp, sz, vp]
        lib.sx_rope_realign_layers.restype = ctypes.c_int
        lib.sx_rope_realign_layers.argtypes = [PP, i32, PB, vp, sz, vp]
        lib.sx_scatter_kv.restype = ctypes.c_int
        lib.sx_scatter_kv.argtypes = [PP, PB, vp, vp, vp, vp, i32, vp]
        lib.sx_score_select.restype = ctypes.c_int
        lib.sx_score_select.argtypes = [PP, PB, vp, vp, i32, vp, vp, vp, vp, vp, vp, sz, vp]
        lib.sx_score_select_ex.restype = ctypes.c_int
        lib.sx_score_select_ex.argtypes = [PP, PB, vp, vp, i32, vp, vp, i32, i32, vp, vp, vp, vp, vp, sz, vp]
        lib.sx_sparse_attn.restype = ctypes.c_int
        lib.sx_sparse_attn.argtypes = [PP, PB, i32, vp, vp, vp, i32, vp, vp, vp, sz, vp]
        lib.sx_check_batch.restype = ctypes.c_int
        lib.sx_check_batch.argtypes = [PP, PB, vp, sz, vp]
        lib.sx_check_rows.restype = ctypes.c_int
        lib.sx_check_rows.argtypes = [PP, PB, vp, vp, i32, vp, sz, vp]
        lib.sx_launch_count.restype = ctypes.c_uint64
        lib.sx_launch_count.argtypes = []
        lib.sx_sparse_attn_noalloc.restype = ctypes.c_int
        lib.sx_sparse_attn_noalloc.argtypes = [PP, PB, vp, vp, vp, i32, vp, vp, vp]
        lib.sx_probe_pipe.restype = ctypes.c_int
        lib.sx_probe_pipe.argtypes = [i32, i32, vp, i32, vp]
        lib.sx_last_error.restype = ctypes.c_char_p
        lib.sx_version.restype = ctypes.c_char_p
        _lib = lib
    return _lib


def version() -> str:
    return load().sx_version().decode()


def launch_count() -> int:
    """Kernels the library has launched in this process so far (counted inside libsparsex.so)."""
    return int(load().sx_launch_count())


def probe_pipe(pipe: int, iters: int = 4096, num_ctas: Optional[int] = None, device="cuda", stream=None) -> float:
    """sx_probe_pipe: lane-operations per clock and SM of one instruction pipe (0 MUFU.EX2, 1 FFMA, 2 FFMA2,
    3 the scoring sweeps' 6:2 MUFU / polynomial mix); median over one CTA per SM."""
    dev = torch.device(device)
    n = int(num_ctas) if num_ctas else torch.cuda.get_device_properties(dev).multi_processor_count
    cyc = torch.zeros(n + 1, dtype=torch.int64, device=dev)
    for _ in range(2):   # the first launch warms the clocks up
        _check(load().sx_probe_pipe(int(pipe), int(iters), _ptr(cyc), n, _stream(stream)), "sx_probe_pipe")
    torch.cuda.synchronize(dev)
    return 1024.0 * 8.0 * iters / float(cyc[:n].median().item())


def _check(rc: int, what: str):
    if rc != SX_OK:
        raise SparseXError("%s failed (%d): %s" % (what, rc, load().sx_last_error().decode()))


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream: Optional[torch.cuda.Stream]):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _dev_i32(a: np.ndarray, device) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(device)


class DevicePool:
    """K and V pools of one layer: torch tensors [num_blocks][Hkv][16][128] of bf16 (or int16 bits)."""

    def __init__(self, k: torch.Tensor, v: torch.Tensor, num_q_heads: int):
        assert k.is_cuda and v.is_cuda and k.is_contiguous() and v.is_contiguous()
        assert k.shape == v.shape and k.dim() == 4 and k.element_size() == 2
        self.k, self.v = k, v
        self.c = SxPool(k.data_ptr(), v.data_ptr(), k.shape[0], k.shape[2], k.shape[1], num_q_heads, k.shape[3])


class DeviceBatch:
    """Uploads a host layout (any object with the fields of workloads.Layout) once per batch."""

    def __init__(self, lay, device="cuda", cow: Optional[bool] = None):
        dev = torch.device(device)
        self.device = dev
        self.seq_len = _dev_i32(lay.seq_len, dev)
        self.tok_off = _dev_i32(lay.tok_off, dev)
        self.k_block_table = _dev_i32(lay.k_block_table, dev)
        self.v_block_table = _dev_i32(lay.v_block_table, dev)
        use_cow = bool(getattr(lay, "cow", False)) if cow is None else cow
        self.cow_private = _dev_i32(lay.cow_private, dev) if use_cow else None
        self.segments = _dev_i32(np.asarray(lay.segments).reshape(-1, 5), dev)
        self.src_blocks = _dev_i32(lay.src_blocks, dev)
        self.new_off = _dev_i32(lay.new_off, dev)
        self.new_idx = _dev_i32(lay.new_idx, dev)
        nseg = int(np.asarray(lay.segments).reshape(-1, 5).shape[0])
        seg_pages = int(np.asarray(lay.segments).reshape(-1, 5)[:, 1].sum() // 16) if nseg else 0
        self.c = SxBatch(
            int(len(lay.seq_len)), nseg, int(lay.k_block_table.shape[1]), int(lay.tok_off[-1]),
            int(lay.new_off[-1]), seg_pages, int(np.max(lay.seq_len)),
            self.seq_len.data_ptr(), self.tok_off.data_ptr(), self.k_block_table.data_ptr(),
            self.v_block_table.data_ptr(), self.cow_private.data_ptr() if use_cow else None,
            self.segments.data_ptr() if nseg else None, self.src_blocks.data_ptr() if nseg else None,
            self.new_off.data_ptr(), self.new_idx.data_ptr() if int(lay.new_off[-1]) else None,
            float(lay.rope_theta), int(lay.rope_style), int(bool(getattr(lay, "zero_copy", False))))
        self._ws = None
        self._ws_pool_key = None

    def workspace(self, pool: DevicePool) -> torch.Tensor:
        key = (pool.c.num_kv_heads, pool.c.num_q_heads)
        if self._ws is None or self._ws_pool_key != key:
            n = ctypes.c_size_t(0)
            _check(load().sx_workspace_size(ctypes.byref(pool.c), ctypes.byref(self.c), ctypes.byref(n)),
                   "sx_workspace_size")
            self._ws = torch.empty(max(int(n.value), 256), dtype=torch.uint8, device=self.device)
            assert self._ws.data_ptr() % 256 == 0
            self._ws_pool_key = key
        return self._ws


def check_batch(pool: DevicePool, batch: DeviceBatch, stream=None):
    """Validate the device-resident descriptor arrays (sx_check_batch; synchronises). Raises SparseXError."""
    ws = batch.workspace(pool)
    _check(load().sx_check_batch(ctypes.byref(pool.c), ctypes.byref(batch.c), _ptr(ws), ws.numel(), _stream(stream)),
           "sx_check_batch")


def check_rows(pool: DevicePool, batch: DeviceBatch, rows: torch.Tensor, rows_off: torch.Tensor,
               max_rows: Optional[int] = None, stream=None):
    """Validate a row list for sx_scatter_kv / sx_sparse_attn (sx_check_rows; synchronises)."""
    ws = batch.workspace(pool)
    n = int(rows.numel()) if max_rows is None else int(max_rows)
    _check(load().sx_check_rows(ctypes.byref(pool.c), ctypes.byref(batch.c), _ptr(rows), _ptr(rows_off), n, _ptr(ws),
                                ws.numel(), _stream(stream)), "sx_check_rows")


def workspace_size(pool: DevicePool, batch: DeviceBatch) -> int:
    n = ctypes.c_size_t(0)
    _check(load().sx_workspace_size(ctypes.byref(pool.c), ctypes.byref(batch.c), ctypes.byref(n)),
           "sx_workspace_size")
    return int(n.value)


def rope_realign(pool: DevicePool, batch: DeviceBatch, stream=None):
    """Stage (a): K pages rotated by R_delta into the request's pages, V copied."""
    ws = batch.workspace(pool)
    _check(load().sx_rope_realign(ctypes.byref(pool.c), ctypes.byref(batch.c), _ptr(ws), ws.numel(),
                                  _stream(stream)), "sx_rope_realign")


def rope_realign_layers(pools, batch: DeviceBatch, stream=None):
    """Stage (a) for a stack of layers in one launch (same batch descriptor for all layers)."""
    n = len(pools)
    ws = batch.workspace(pools[0])
    arr = (SxPool * n)(*[p.c for p in pools])
    _check(load().sx_rope_realign_layers(arr, n, ctypes.byref(batch.c), _ptr(ws), ws.numel(), _stream(stream)),
           "sx_rope_realign_layers")


def scatter_kv(pool: DevicePool, batch: DeviceBatch, k_fresh: torch.Tensor, v_fresh: torch.Tensor,
               rows: torch.Tensor, rows_off: torch.Tensor, max_rows: Optional[int] = None, stream=None):
    """Stage (d), Alg. 1 l.509-510/544-545: fresh K,V rows into their paged slots (COW aware)."""
    n = int(rows.numel()) if max_rows is None else int(max_rows)
    assert k_fresh.is_contiguous() and v_fresh.is_contiguous() and rows.dtype == torch.int32
    _check(load().sx_scatter_kv(ctypes.byref(pool.c), ctypes.byref(batch.c), _ptr(k_fresh), _ptr(v_fresh),
                                _ptr(rows), _ptr(rows_off), n, _stream(stream)), "sx_scatter_kv")


def score_select(pool: DevicePool, batch: DeviceBatch, q_new: torch.Tensor, sel_off: torch.Tensor,
                 rows_off: torch.Tensor, sel_idx: torch.Tensor, rows_R: torch.Tensor,
                 scores: Optional[torch.Tensor] = None, lse_new: Optional[torch.Tensor] = None,
                 lse_by_token: bool = False, stream=None):
    """Stage (b), Eq. (1)-(3): Sparse-Q scores, head/query aggregation, top-k, R = I_nr U S_key."""
    ws = batch.workspace(pool)
    _check(load().sx_score_select(ctypes.byref(pool.c), ctypes.byref(batch.c), _ptr(q_new), _ptr(lse_new),
                                  1 if lse_by_token else 0, _ptr(sel_off), _ptr(rows_off), _ptr(scores), _ptr(sel_idx), _ptr(rows_R),
                                  _ptr(ws), ws.numel(), _stream(stream)), "sx_score_select")


def score_select_ex(pool: DevicePool, batch: DeviceBatch, q_new: torch.Tensor, sel_off: torch.Tensor,
                    rows_cap_off: torch.Tensor, sel_idx: torch.Tensor, rows_R: torch.Tensor,
                    rows_off_out: torch.Tensor, overflow_blocks: int = 1, tail_tokens: int = 64,
                    scores: Optional[torch.Tensor] = None, lse_new: Optional[torch.Tensor] = None,
                    lse_by_token: bool = False, stream=None):
    """Stage (b) with overflow and tail fallback (Alg. 1 l.535-539): R = I_nr U S_key U S_ov U S_tail; the
    actual CSR offsets of the packed rows_R come back in rows_off_out (device)."""
    ws = batch.workspace(pool)
    _check(load().sx_score_select_ex(ctypes.byref(pool.c), ctypes.byref(batch.c), _ptr(q_new), _ptr(lse_new),
                                     1 if lse_by_token else 0, _ptr(sel_off), _ptr(rows_cap_off),
                                     int(overflow_blocks), int(tail_tokens), _ptr(scores), _ptr(sel_idx),
                                     _ptr(rows_R), _ptr(rows_off_out), _ptr(ws), ws.numel(), _stream(stream)),
           "sx_score_select_ex")


def rows_capacity(lay, overflow_blocks: int, tail_tokens: int) -> np.ndarray:
    """Host CSR capacity offsets for sx_score_select_ex: |I_nr| + k + 2 * 16 * overflow_blocks per interval of
    I_nr + tail_tokens per request, clipped to the request length (a sizing bound, not the set itself)."""
    sel_off, _ = selection_offsets(lay)
    cap = [0]
    for r in range(lay.num_reqs):
        idx = np.asarray(lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]])
        n_int = (1 + int(np.sum(np.diff(idx) != 1))) if len(idx) else 0
        c = len(idx) + int(sel_off[r + 1] - sel_off[r]) + 2 * 16 * overflow_blocks * n_int + tail_tokens
        cap.append(cap[-1] + min(c, int(lay.seq_len[r])))
    return np.asarray(cap, dtype=np.int32)


def sparse_attn(pool: DevicePool, batch: DeviceBatch, q: torch.Tensor, out: torch.Tensor,
                rows_R: Optional[torch.Tensor] = None, rows_off: Optional[torch.Tensor] = None,
                total_rows: Optional[int] = None, lse: Optional[torch.Tensor] = None, full: bool = False,
                cuda_core: bool = False, cta_pair: Optional[bool] = None, stream=None):
    """Stage (c), Alg. 1 l.546-548 (sparse rows) / l.507-511 (full=True). cuda_core = SX_ATTN_CUDA_CORE;
    cta_pair: None = the library's rule, True / False = SX_ATTN_CTA_PAIR / SX_ATTN_SINGLE_CTA (include/sparsex.h)."""
    ws = batch.workspace(pool)
    n = int(q.shape[0]) if total_rows is None else int(total_rows)
    assert q.is_contiguous() and out.is_contiguous()
    _check(load().sx_sparse_attn(ctypes.byref(pool.c), ctypes.byref(batch.c), (1 if full else 0) | (2 if cuda_core else 0) | (0 if cta_pair is None else (4 if cta_pair else 8)), _ptr(q),
                                 _ptr(rows_R), _ptr(rows_off), n, _ptr(out), _ptr(lse), _ptr(ws), ws.numel(),
                                 _stream(stream)), "sx_sparse_attn")


def sparse_attn_noalloc(pool: DevicePool, batch: DeviceBatch, q: torch.Tensor, out: torch.Tensor,
                        rows_R: torch.Tensor, rows_off: torch.Tensor, total_rows: Optional[int] = None,
                        lse: Optional[torch.Tensor] = None, stream=None):
    """Stage (c) for small row sets with the library's built-in scratch: no workspace, no allocation
    (sx_sparse_attn_noalloc; total_rows * Hq <= NOALLOC_MAX_PAIRS). Calls that overlap on the GPU race on that scratch."""
    n = int(q.shape[0]) if total_rows is None else int(total_rows)
    assert q.is_contiguous() and out.is_contiguous()
    _check(load().sx_sparse_attn_noalloc(ctypes.byref(pool.c), ctypes.byref(batch.c), _ptr(q), _ptr(rows_R),
                                         _ptr(rows_off), n, _ptr(out), _ptr(lse), _stream(stream)),
           "sx_sparse_attn_noalloc")


def selection_offsets(lay) -> tuple:
    """Host CSR offsets (sel_off, rows_off) for k_per_req clamped to the cached-token count."""
    n_new = np.diff(np.asarray(lay.new_off)).astype(np.int64)
    n_cached = np.zeros(len(n_new), dtype=np.int64)      # |I_reuse| = tokens covered by segments
    for seg in np.asarray(lay.segments).reshape(-1, 5):
        n_cached[int(seg[0])] += int(seg[1])
    k = np.minimum(np.asarray(lay.k_per_req, dtype=np.int64), n_cached)
    sel_off = np.concatenate([[0], np.cumsum(k)]).astype(np.int32)
    rows_off = np.concatenate([[0], np.cumsum(k + n_new)]).astype(np.int32)
    return sel_off, rows_off
