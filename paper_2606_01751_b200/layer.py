"""One layer of the Sparse-KV recomputation step on the GPU: stage sequencing only.

Order inside a layer (reading A13; Alg. 1 writes fresh K,V at l.544 before SparseAttn at l.548):
  sparse layer: realign -> scatter(I_nr) -> [score_select] -> scatter(S_key) -> sparse_attn(R)
  full layer  : realign -> scatter(all)  -> sparse_attn(full)
Every stage is a call into libsparsex.so through `binding`; torch only owns the device buffers.
Compact per-row inputs (Q[R], K_fresh[R], V_fresh[R]) stand for the projections of Alg. 1 l.544, which
the method computes for i in R only; gathering them from the full synthetic tensors is input staging.
"""
from __future__ import annotations

from typing import Optional

import numpy as np
import torch

from . import binding as sx


def _bits_to_dev(a: np.ndarray, device) -> torch.Tensor:
    """uint16 bf16 bit patterns -> int16 device tensor (same bytes)."""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(device)


def dev_to_bits(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().numpy().view(np.uint16)


class GpuLayer:
    def __init__(self, lay, lt, device="cuda", batch: Optional[sx.DeviceBatch] = None):
        self.lay = lay
        self.dev = torch.device(device)
        self.cta_pair = None    # None: library rule; True / False: SX_ATTN_CTA_PAIR / SX_ATTN_SINGLE_CTA
        self.batch = batch if batch is not None else sx.DeviceBatch(lay, self.dev)
        # lt: workloads.LayerTensors (numpy bit patterns) or any object whose pool_k / pool_v / q_full /
        # k_fresh / v_fresh are already 2-byte device tensors
        def up(a):
            if isinstance(a, torch.Tensor):
                return a if a.dtype == torch.int16 else a.view(torch.int16)
            return _bits_to_dev(a, self.dev)
        self.pool_k = up(lt.pool_k)
        self.pool_v = up(lt.pool_v)
        self.pool = sx.DevicePool(self.pool_k, self.pool_v, lay.num_q_heads)
        self.q_full = up(lt.q_full)
        self.k_fresh = up(lt.k_fresh)
        self.v_fresh = up(lt.v_fresh)
        self.tok_off_h = np.asarray(lay.tok_off, dtype=np.int64)
        # batch-wide token index of every new token, and per-request CSR of I_nr
        new_tok = []
        for r in range(lay.num_reqs):
            new_tok.append(self.tok_off_h[r] + lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]].astype(np.int64))
        self.new_tok = torch.from_numpy(np.concatenate(new_tok) if new_tok else np.zeros(0, np.int64)).to(self.dev)
        sel_off, rows_off = sx.selection_offsets(lay)
        self.sel_off_h, self.rows_off_h = sel_off, rows_off
        self.sel_off = torch.from_numpy(sel_off).to(self.dev)
        self.rows_off = torch.from_numpy(rows_off).to(self.dev)
        self.q_new = self.q_full[self.new_tok].contiguous()
        self.kf_new = self.k_fresh[self.new_tok].contiguous()
        self.vf_new = self.v_fresh[self.new_tok].contiguous()

    # ---- helpers
    def _tok_index(self, rows: torch.Tensor, off: torch.Tensor) -> torch.Tensor:
        """batch-wide token index of compact rows given per-request CSR offsets `off` (device)."""
        n = rows.numel()
        idx = torch.arange(n, device=self.dev, dtype=torch.int64)
        req = torch.searchsorted(off[1:].to(torch.int64).contiguous(), idx, right=True)
        return self.batch.tok_off.to(torch.int64)[req] + rows.to(torch.int64)

    # ---- stages
    def realign(self):
        sx.rope_realign(self.pool, self.batch)

    def scatter_new(self):
        sx.scatter_kv(self.pool, self.batch, self.kf_new, self.vf_new, self.batch.new_idx, self.batch.new_off,
                      max_rows=int(self.lay.new_off[-1]))

    def select(self, want_scores: bool = True, lse_new: Optional[torch.Tensor] = None, lse_by_token: bool = False):
        n_sel, n_rows = int(self.sel_off_h[-1]), int(self.rows_off_h[-1])
        self.sel_idx = torch.full((max(n_sel, 1),), -1, dtype=torch.int32, device=self.dev)
        self.rows_R = torch.full((max(n_rows, 1),), -1, dtype=torch.int32, device=self.dev)
        self.scores = (torch.empty(int(self.lay.tok_off[-1]), dtype=torch.float32, device=self.dev)
                       if want_scores else None)
        sx.score_select(self.pool, self.batch, self.q_new, self.sel_off, self.rows_off, self.sel_idx, self.rows_R,
                        scores=self.scores, lse_new=lse_new, lse_by_token=lse_by_token)
        self.sel_idx = self.sel_idx[:n_sel]
        self.rows_R = self.rows_R[:n_rows]

    def select_ex(self, overflow_blocks: int = 1, tail_tokens: int = 64, want_scores: bool = True):
        """Selection with overflow and tail fallback (Alg. 1 l.535-539): |R| is data dependent, so the row
        offsets are read back before the per-row inputs are staged."""
        cap = sx.rows_capacity(self.lay, overflow_blocks, tail_tokens)
        n_sel = int(self.sel_off_h[-1])
        self.sel_idx = torch.full((max(n_sel, 1),), -1, dtype=torch.int32, device=self.dev)
        rows = torch.full((max(int(cap[-1]), 1),), -1, dtype=torch.int32, device=self.dev)
        self.rows_cap = int(cap[-1])
        off_out = torch.zeros(self.lay.num_reqs + 1, dtype=torch.int32, device=self.dev)
        self.scores = (torch.empty(int(self.lay.tok_off[-1]), dtype=torch.float32, device=self.dev)
                       if want_scores else None)
        sx.score_select_ex(self.pool, self.batch, self.q_new, self.sel_off, torch.from_numpy(cap).to(self.dev),
                           self.sel_idx, rows, off_out, overflow_blocks=overflow_blocks, tail_tokens=tail_tokens,
                           scores=self.scores)
        self.sel_idx = self.sel_idx[:n_sel]
        self.rows_off = off_out
        self.rows_off_h = off_out.cpu().numpy()
        self.rows_R = rows[:int(self.rows_off_h[-1])]

    def stage_rows(self, sel_idx: torch.Tensor, rows_R: torch.Tensor):
        """Input staging for (d) and (c): compact fresh K,V of S_key and Q of R (Alg. 1 l.544)."""
        self.sel_idx, self.rows_R = sel_idx, rows_R
        ts = self._tok_index(sel_idx, self.sel_off)
        tr = self._tok_index(rows_R, self.rows_off)
        self.kf_sel = self.k_fresh[ts].contiguous()
        self.vf_sel = self.v_fresh[ts].contiguous()
        self.q_R = self.q_full[tr].contiguous()
        # all recomputed rows at once (R is known before the layer starts when an earlier boundary
        # selection is reused: one scatter of K/V_fresh[R], Alg. 1 l.544)
        self.kf_R = self.k_fresh[tr].contiguous()
        self.vf_R = self.v_fresh[tr].contiguous()

    def scatter_sel(self):
        if self.sel_idx.numel():
            sx.scatter_kv(self.pool, self.batch, self.kf_sel, self.vf_sel, self.sel_idx, self.sel_off,
                          max_rows=int(self.sel_idx.numel()))

    def attend(self, want_lse: bool = True, cuda_core: bool = False):
        n = int(self.rows_R.numel())
        hq = self.lay.num_q_heads
        self.out = torch.empty((n, hq, 128), dtype=torch.int16, device=self.dev)
        self.lse = torch.empty((n, hq), dtype=torch.float32, device=self.dev) if want_lse else None
        sx.sparse_attn(self.pool, self.batch, self.q_R, self.out, rows_R=self.rows_R, rows_off=self.rows_off,
                       total_rows=n, lse=self.lse, cuda_core=cuda_core, cta_pair=self.cta_pair)

    # ---- whole layers
    def step_sparse(self, rows_given=None, do_realign: bool = True, want_scores: bool = True):
        """rows_given: (sel_idx, rows_R) device tensors from an earlier boundary selection (paper mode)."""
        if do_realign:
            self.realign()
        if rows_given is None:
            self.scatter_new()
            self.select(want_scores=want_scores)
            self.stage_rows(self.sel_idx, self.rows_R)
            self.scatter_sel()
        else:
            self.stage_rows(*rows_given)
            sx.scatter_kv(self.pool, self.batch, self.kf_R, self.vf_R, self.rows_R, self.rows_off,
                          max_rows=int(self.rows_R.numel()))
        self.attend()

    def step_full(self, do_realign: bool = True, want_lse: bool = True):
        if do_realign:
            self.realign()
        lay = self.lay
        t = int(lay.tok_off[-1])
        all_rows = torch.cat([torch.arange(int(n), dtype=torch.int32) for n in lay.seq_len]).to(self.dev)
        sx.scatter_kv(self.pool, self.batch, self.k_fresh, self.v_fresh, all_rows, self.batch.tok_off, max_rows=t)
        self.out = torch.empty((t, lay.num_q_heads, 128), dtype=torch.int16, device=self.dev)
        self.lse = torch.empty((t, lay.num_q_heads), dtype=torch.float32, device=self.dev) if want_lse else None
        sx.sparse_attn(self.pool, self.batch, self.q_full, self.out, total_rows=t, lse=self.lse, full=True,
                       cta_pair=self.cta_pair)
        self.rows_R = all_rows
