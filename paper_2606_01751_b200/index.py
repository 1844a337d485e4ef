"""ctypes binding of the host-side segment index (include/sparsex_index.h): argument marshalling only.

The index is the step BEFORE the GPU path (Alg. 1 l.500-501): it turns a prompt with
candidate reuse segments into the segment map, source pages and Sparse-Q mask that sx_batch carries.
"""
from __future__ import annotations

import ctypes
from typing import Sequence, Tuple

import numpy as np

from . import binding as sx

EXPORTS = ["sx_index_create", "sx_index_destroy", "sx_index_size", "sx_index_insert", "sx_index_erase",
           "sx_index_plan_request", "sx_index_release", "sx_index_evict"]


class SxSegment(ctypes.Structure):
    _fields_ = [("req", ctypes.c_int32), ("len", ctypes.c_int32), ("old_pos", ctypes.c_int32),
                ("new_pos", ctypes.c_int32), ("src_off", ctypes.c_int32)]


def _lib():
    lib = sx.load()
    if not getattr(lib, "_sx_index_ready", False):
        vp, i32, u64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_uint64
        ip = ctypes.POINTER(ctypes.c_int32)
        lib.sx_index_create.restype = vp
        lib.sx_index_create.argtypes = [i32]
        lib.sx_index_destroy.restype = None
        lib.sx_index_destroy.argtypes = [vp]
        lib.sx_index_size.restype = i32
        lib.sx_index_size.argtypes = [vp]
        lib.sx_index_insert.restype = i32
        lib.sx_index_insert.argtypes = [vp, ip, i32, u64, i32, ip, i32]
        lib.sx_index_erase.restype = i32
        lib.sx_index_erase.argtypes = [vp, ip, i32, u64]
        lib.sx_index_plan_request.restype = i32
        lib.sx_index_plan_request.argtypes = [vp, i32, ip, i32, ip, i32, u64, ctypes.POINTER(SxSegment), ip, ip, ip]
        lib.sx_index_release.restype = i32
        lib.sx_index_release.argtypes = [vp, ip, i32]
        lib.sx_index_evict.restype = i32
        lib.sx_index_evict.argtypes = [vp, i32, i32, ctypes.c_double, ip, i32]
        lib._sx_index_ready = True
    return lib


def _ip(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


class SegmentIndex:
    """Owns one sx_index. Methods mirror the C entry points one to one."""

    def __init__(self, block_size: int = 16):
        self._lib = _lib()
        self._h = self._lib.sx_index_create(int(block_size))
        if not self._h:
            raise sx.SparseXError("sx_index_create failed")
        self.block_size = int(block_size)

    def close(self):
        if self._h:
            self._lib.sx_index_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def __len__(self) -> int:
        return int(self._lib.sx_index_size(self._h))

    @staticmethod
    def _chk(rc: int, what: str) -> int:
        if rc < 0:
            raise sx.SparseXError("%s failed with status %d" % (what, rc))
        return rc

    def insert(self, tokens, extra_key: int, old_pos: int, blocks, frozen: bool = False) -> int:
        t, b = _i32(tokens), _i32(blocks)
        return self._chk(self._lib.sx_index_insert(self._h, _ip(t), len(t), int(extra_key), int(old_pos), _ip(b),
                                                   1 if frozen else 0), "sx_index_insert")

    def erase(self, tokens, extra_key: int) -> int:
        t = _i32(tokens)
        return self._chk(self._lib.sx_index_erase(self._h, _ip(t), len(t), int(extra_key)), "sx_index_erase")

    def plan_request(self, req: int, tokens, candidates: Sequence[Tuple[int, int]], extra_key: int):
        """-> (hits, segments int32 [n][5] = (req, len, old_pos, new_pos, src_off), src_blocks, new_idx)."""
        t = _i32(tokens)
        cand = _i32(np.asarray(candidates, dtype=np.int32).reshape(-1, 2))
        cap = max(1, len(t) // self.block_size)
        segs = (SxSegment * cap)()
        src = np.zeros(cap, dtype=np.int32)
        new_idx = np.zeros(max(1, len(t)), dtype=np.int32)
        counts = np.zeros(3, dtype=np.int32)
        hits = self._chk(self._lib.sx_index_plan_request(self._h, int(req), _ip(t), len(t), _ip(cand), len(cand),
                                                         int(extra_key), segs, _ip(src), _ip(new_idx), _ip(counts)),
                         "sx_index_plan_request")
        seg_arr = np.asarray([(s.req, s.len, s.old_pos, s.new_pos, s.src_off) for s in segs[:counts[0]]],
                             dtype=np.int32).reshape(-1, 5)
        return hits, seg_arr, src[:counts[1]].copy(), new_idx[:counts[2]].copy()

    def release(self, src_blocks) -> int:
        b = _i32(src_blocks)
        return self._chk(self._lib.sx_index_release(self._h, _ip(b), len(b)), "sx_index_release")

    def evict(self, used_blocks: int, total_blocks: int, threshold: float = 0.9, max_out: int = 1 << 16) -> np.ndarray:
        out = np.zeros(max(1, max_out), dtype=np.int32)
        n = self._chk(self._lib.sx_index_evict(self._h, int(used_blocks), int(total_blocks), float(threshold), _ip(out),
                                               int(max_out)), "sx_index_evict")
        return out[:n].copy()
