"""fp64 CPU oracle of the SparseX per-layer Sparse-KV recomputation step.

TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this. It shares no code with paper_2606_01751_b200/ and never
imports it; inputs arrive as plain numpy arrays.

What each function is (all fp64; inputs are bf16 bit patterns widened exactly):

  realign()          O-a  PAPER.md:151-159 (k_hat_{p'+j} <- R_{p'-p} k_hat_{p+j}, v copied), Alg. 1 lines
                          502-504. Pins: composition, delta=0 identity, norm, relative-position identity
                          (PAPER.md:141-147), hand case D=2 -- tests/test_oracle_pins.py.
  scatter_kv()       O-d  Alg. 1 lines 509-510 / 544-545 (write fresh K,V of the computed positions into
                          the request's cache; slot mapping PAPER.md:333). Pins: untouched rows, idempotence,
                          gather round trip, COW leaves shared pages unchanged.
  scores()           O-b  Eq. (1)+(2), head sum PAPER.md:225 (C loops in sx_oracle.c).
                          Pins: sum_j s_j = N_n*Hq, Q=0 harmonic closed form, brute-force python loops.
  select_topk()      O-b  Eq. (3) PAPER.md:207-209 restricted to I_reuse (reading A7), ties -> lower
                          position (A8). Pins: full stable sort on tiny inputs, k=0, k=N_c.
  recompute_set()    O-b  Alg. 1 l.535-539: R = I_nr U S_key U S_ov U S_tail (overflow by
                          one block around every Sparse-Q interval, tail fallback of 64 tokens). Pins: hand-typed
                          expected lists -- tests/test_oracle_pins.py::test_recompute_set_hand_cases.
  attention()        O-c  Alg. 1 line 21 (C loops). Pins: R=all == fp64 torch SDPA,
                          Q=0 prefix mean of V, T=1, constant V, rows-subset == full on those rows.
  layer_sparse()/layer_full()  O-layer driver: order realign -> scatter(new) -> select -> scatter(S_key)
                          -> attention (reading A13: Alg. 1 writes fresh K,V at line 19 before line 21).
                          Pin: ratio 100% == dense causal attention over the fresh tensors.

(The host-side segment index has its own plain-dict reference in oracle/sx_index_oracle.py.)

No function here is "parity unpinned"; no pin comes from numbers printed in the paper (it prints none
for this path).

RoPE convention (readings A1-A3): theta_i = base^(-2i/D), i in [0, D/2); rope_style 0 pairs
(i, i + D/2) ("half-split"), rope_style 1 pairs (2i, 2i+1); rotation by angle phi = delta * theta_i:
x' = x cos(phi) - y sin(phi), y' = x sin(phi) + y cos(phi).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sx_oracle.c")
_LIB = os.path.join(_HERE, "libsx_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile sx_oracle.c with gcc (-O2 -fopenmp, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-march=native", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32p = ctypes.POINTER(ctypes.c_int32)
        u16p = ctypes.POINTER(ctypes.c_uint16)
        f64p = ctypes.POINTER(ctypes.c_double)
        lib.orc_num_threads.restype = ctypes.c_int
        lib.orc_scores.restype = ctypes.c_int
        lib.orc_scores.argtypes = [u16p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, i32p,
                                   ctypes.c_int, u16p, i32p, ctypes.c_int, f64p, f64p]
        lib.orc_attention.restype = ctypes.c_int
        lib.orc_attention.argtypes = [u16p, u16p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                      i32p, i32p, ctypes.c_int, u16p, i32p, ctypes.c_int, f64p, f64p]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().orc_num_threads())


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


# ----------------------------------------------------------------------------- bf16 <-> fp64

def bf16_to_f64(bits: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns."""
    u = np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return u.view(np.float32).astype(np.float64)


def f64_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp64 -> bf16 bit pattern in ONE rounding (no fp32 intermediate).

    bf16 has 8 significant bits: x = m * 2^e with |m| in [0.5, 1) -> rint(m * 2^8) * 2^(e-8).
    (bf16 subnormals do not occur for the N(0,1)-scale data of this path; checked.)
    """
    x = np.asarray(x, dtype=np.float64)
    m, e = np.frexp(x)
    r = np.ldexp(np.rint(np.ldexp(m, 8)), e - 8)          # np.rint rounds half to even
    assert np.all((r == 0) | (np.abs(r) >= 2.0 ** -126)), "bf16 subnormal range not supported"
    f = r.astype(np.float32)                               # exact: r has <= 8 significant bits
    return (f.view(np.uint32) >> np.uint32(16)).astype(np.uint16)


# ----------------------------------------------------------------------------- O-a realign

def rope_angles(delta: int, theta: float, head_dim: int) -> np.ndarray:
    """phi_i = delta * base^(-2i/D), i in [0, D/2) (readings A2, A3)."""
    i = np.arange(head_dim // 2, dtype=np.float64)
    return np.float64(delta) * np.power(np.float64(theta), -2.0 * i / np.float64(head_dim))


def rope_rotate(x: np.ndarray, delta: int, theta: float, rope_style: int = 0) -> np.ndarray:
    """R_delta applied to the last axis of x (fp64). PAPER.md:139, 147, 159."""
    x = np.asarray(x, dtype=np.float64)
    d = x.shape[-1]
    phi = rope_angles(delta, theta, d)
    c, s = np.cos(phi), np.sin(phi)
    out = np.empty_like(x)
    if rope_style == 0:      # pairs (i, i + D/2)
        a, b = x[..., : d // 2], x[..., d // 2:]
        out[..., : d // 2] = a * c - b * s
        out[..., d // 2:] = a * s + b * c
    else:                    # pairs (2i, 2i + 1)
        a, b = x[..., 0::2], x[..., 1::2]
        out[..., 0::2] = a * c - b * s
        out[..., 1::2] = a * s + b * c
    return out


def realign(pool_k: np.ndarray, pool_v: np.ndarray, k_table: np.ndarray, v_table: np.ndarray,
            segments: np.ndarray, src_blocks: np.ndarray, theta: float, rope_style: int = 0
            ) -> np.ndarray:
    """O-a. For every segment (req, len, old_pos, new_pos, src_off) and token j < len:
    K_dst[new_pos + j] = R_{new_pos - old_pos} K_src[old_pos + j], V_dst = V_src (bit copy).

    pool_k / pool_v: uint16 [num_blocks][Hkv][bs][D], updated IN PLACE with the RNE-bf16 of the result.
    k_table / v_table: int32 [num_reqs][max_pages] logical page -> physical page of each request.
    A V page whose table entry already IS the source page (copy-on-write aliasing) is not copied.
    Returns the unrounded fp64 keys, compact [sum len][Hkv][D] in segment order.
    """
    bs = pool_k.shape[2]
    ref = []
    for (req, ln, old_pos, new_pos, src_off) in np.asarray(segments).reshape(-1, 5).tolist():
        assert ln % bs == 0 and old_pos % bs == 0 and new_pos % bs == 0
        delta = new_pos - old_pos
        for pg in range(ln // bs):
            src = int(src_blocks[src_off + pg])
            dk = int(k_table[req][new_pos // bs + pg])
            dv = int(v_table[req][new_pos // bs + pg])
            k64 = bf16_to_f64(pool_k[src])                       # [Hkv][bs][D]
            rot = rope_rotate(k64, delta, theta, rope_style)
            pool_k[dk] = f64_to_bf16(rot)
            if dv != src:
                pool_v[dv] = pool_v[src]
            ref.append(np.transpose(rot, (1, 0, 2)))             # [bs][Hkv][D]
    if not ref:
        return np.zeros((0, pool_k.shape[1], pool_k.shape[3]))
    return np.concatenate(ref, axis=0)


# ----------------------------------------------------------------------------- O-d scatter

def scatter_kv(pool_k: np.ndarray, pool_v: np.ndarray, k_table: np.ndarray, v_table: np.ndarray,
               cow_private: Optional[np.ndarray], req: int, rows: np.ndarray,
               k_fresh: np.ndarray, v_fresh: np.ndarray) -> None:
    """O-d, one request. For each listed row r: slot = (table[req][r // bs], r % bs);
    K_pool[slot] = k_fresh[n], V_pool[slot] = v_fresh[n] (bf16 bit copy). Copy-on-write (reading A14):
    a page whose table entry differs from its reserved private page is first copied there, then the
    table entry is flipped. Pools and tables are updated IN PLACE.
    k_fresh / v_fresh: uint16 [len(rows)][Hkv][D].
    """
    bs = pool_k.shape[2]
    for n, r in enumerate(np.asarray(rows).tolist()):
        pg, off = r // bs, r % bs
        if cow_private is not None:
            for table, pool in ((k_table, pool_k), (v_table, pool_v)):
                priv = int(cow_private[req][pg])
                if priv >= 0 and int(table[req][pg]) != priv:
                    pool[priv] = pool[int(table[req][pg])]
                    table[req][pg] = priv
        pool_k[int(k_table[req][pg]), :, off, :] = k_fresh[n]
        pool_v[int(v_table[req][pg]), :, off, :] = v_fresh[n]


def gather_tokens(pool: np.ndarray, table_row: np.ndarray, seq_len: int) -> np.ndarray:
    """Logical view of one request: uint16 [seq_len][Hkv][D] read through its block table."""
    bs = pool.shape[2]
    pos = np.arange(seq_len)
    return pool[np.asarray(table_row)[pos // bs], :, pos % bs, :]


# ----------------------------------------------------------------------------- O-b scores / top-k

def scores(pool_k: np.ndarray, k_table_row: np.ndarray, seq_len: int, q_new: np.ndarray,
           new_idx: np.ndarray, num_q_heads: int, want_lse: bool = False):
    """O-b Eq. (1)-(2), one request. q_new: uint16 [N_n][Hq][D]; returns s[seq_len] (and lse[N_n][Hq])."""
    lib = _load()
    pool_k = np.ascontiguousarray(pool_k, dtype=np.uint16)
    tab = np.ascontiguousarray(k_table_row, dtype=np.int32)
    q_new = np.ascontiguousarray(q_new, dtype=np.uint16)
    new_idx = np.ascontiguousarray(new_idx, dtype=np.int32)
    _, hkv, bs, d = pool_k.shape
    assert q_new.shape == (len(new_idx), num_q_heads, d)
    s = np.zeros(seq_len, dtype=np.float64)
    lse = np.zeros((len(new_idx), num_q_heads), dtype=np.float64) if want_lse else None
    rc = lib.orc_scores(_p(pool_k, ctypes.c_uint16), hkv, num_q_heads, d, bs, _p(tab, ctypes.c_int32),
                        int(seq_len), _p(q_new, ctypes.c_uint16), _p(new_idx, ctypes.c_int32),
                        len(new_idx), _p(s, ctypes.c_double),
                        _p(lse, ctypes.c_double) if want_lse else None)
    assert rc == 0
    return (s, lse) if want_lse else s


def select_topk(s: np.ndarray, is_new: np.ndarray, k: int, cand_mask=None) -> Tuple[np.ndarray, np.ndarray]:
    """Eq. (3) over cached positions only (reading A7); order by (score desc, position asc) (A8).
    Returns (S_key sorted by position, R = I_nr U S_key sorted).
    cand_mask: I_reuse as a boolean mask (default: every position that is not new). Positions that are neither
    new nor candidates are prefix-cache hits (Alg. 1 l.501: excluded from the current prefill computation)."""
    s = np.asarray(s, dtype=np.float64)
    if cand_mask is None:
        cand_mask = ~np.asarray(is_new, dtype=bool)
    cand = np.nonzero(np.asarray(cand_mask, dtype=bool))[0]
    k = max(0, min(int(k), len(cand)))
    order = np.lexsort((cand, -s[cand]))          # primary: -score ascending, secondary: position
    sel = np.sort(cand[order[:k]]).astype(np.int32)
    rows = np.sort(np.concatenate([np.nonzero(is_new)[0], sel])).astype(np.int32)
    return sel, rows


def recompute_set(is_new: np.ndarray, sel: np.ndarray, seg_ranges, overflow_blocks: int = 1,
                  tail_tokens: int = 64, block: int = 16, cand_mask=None) -> np.ndarray:
    """Alg. 1 l.535-539, one request: R = I_nr U S_key U S_ov U S_tail, sorted.
    S_ov: every maximal contiguous interval [a, b] of I_nr expanded by `overflow_blocks` blocks of `block`
    positions on both sides (clipped to the request). S_tail: if the last position is a reused token, the
    last `tail_tokens` positions of the reused segment that contains it. seg_ranges: [(start, end)) of the
    reused segments of this request in current positions. cand_mask: I_reuse (default: not new); S_ov and
    S_tail hold reused positions only (prefix-cache hits are never recomputed)."""
    is_new = np.asarray(is_new, dtype=bool)
    t = len(is_new)
    cand_mask = ~is_new if cand_mask is None else np.asarray(cand_mask, dtype=bool)
    r = set(int(i) for i in np.nonzero(is_new)[0]) | set(int(i) for i in sel)
    a = None
    for i in range(t + 1):                       # walk the maximal intervals of I_nr
        inside = i < t and is_new[i]
        if inside and a is None:
            a = i
        if not inside and a is not None:
            b = i - 1
            r.update(q for q in range(max(0, a - overflow_blocks * block), a) if cand_mask[q])
            r.update(q for q in range(b + 1, min(t, b + 1 + overflow_blocks * block)) if cand_mask[q])
            a = None
    if tail_tokens > 0 and cand_mask[t - 1]:
        start = 0
        for (s0, s1) in seg_ranges:
            if s0 <= t - 1 < s1:
                start = s0
        r.update(range(max(start, t - tail_tokens), t))
    return np.asarray(sorted(r), dtype=np.int32)


# ----------------------------------------------------------------------------- O-c attention

def attention(pool_k: np.ndarray, pool_v: np.ndarray, k_table_row: np.ndarray, v_table_row: np.ndarray,
              seq_len: int, q_rows: np.ndarray, rows: np.ndarray, num_q_heads: int,
              want_lse: bool = False):
    """O-c, one request: out[n][h] = softmax(q_{n,h} K[0..rows[n]]^T / sqrt(D)) V[0..rows[n]] in fp64."""
    lib = _load()
    pool_k = np.ascontiguousarray(pool_k, dtype=np.uint16)
    pool_v = np.ascontiguousarray(pool_v, dtype=np.uint16)
    kt = np.ascontiguousarray(k_table_row, dtype=np.int32)
    vt = np.ascontiguousarray(v_table_row, dtype=np.int32)
    q_rows = np.ascontiguousarray(q_rows, dtype=np.uint16)
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    _, hkv, bs, d = pool_k.shape
    assert q_rows.shape == (len(rows), num_q_heads, d)
    assert len(rows) == 0 or (rows.min() >= 0 and rows.max() < seq_len)
    out = np.zeros((len(rows), num_q_heads, d), dtype=np.float64)
    lse = np.zeros((len(rows), num_q_heads), dtype=np.float64) if want_lse else None
    rc = lib.orc_attention(_p(pool_k, ctypes.c_uint16), _p(pool_v, ctypes.c_uint16), hkv, num_q_heads, d,
                           bs, _p(kt, ctypes.c_int32), _p(vt, ctypes.c_int32), int(seq_len),
                           _p(q_rows, ctypes.c_uint16), _p(rows, ctypes.c_int32), len(rows),
                           _p(out, ctypes.c_double), _p(lse, ctypes.c_double) if want_lse else None)
    assert rc == 0
    return (out, lse) if want_lse else out


# ----------------------------------------------------------------------------- O-layer driver

class LayerResult:
    """Everything one layer produced: per-request lists."""

    def __init__(self):
        self.k_ref64 = None     # realigned keys, fp64, compact in segment order
        self.scores = []        # per request: s[T]
        self.lse_new = []       # per request: lse[N_n][Hq] of the Sparse-Q rows
        self.sel = []           # per request: S_key sorted
        self.rows = []          # per request: R sorted
        self.out = []           # per request: O[|R|][Hq][D] fp64
        self.lse = []           # per request: lse[|R|][Hq]


def layer_step(pool_k, pool_v, k_table, v_table, cow_private, segments, src_blocks, theta, rope_style,
               seq_len, tok_off, new_off, new_idx, k_per_req, num_q_heads, q_full, k_fresh, v_fresh,
               mode: str = "sparse", rows_given=None, do_realign: bool = True) -> LayerResult:
    """One layer of Alg. 1, whole batch, pools/tables updated in place.

    mode "sparse": realign -> scatter(I_nr) -> [select unless rows_given] -> scatter(S_key) -> attention(R)
                   (Alg. 1 lines 6, 12-14, 17, 19-21; order = reading A13).
    mode "full":   realign -> scatter(all) -> attention(all)       (Alg. 1 lines 6, 7-10).
    rows_given: per-request (sel, rows) from an earlier boundary-layer selection (paper mode, A11).
    q_full/k_fresh/v_fresh: uint16 [sum T][H][D], token (req, pos) at tok_off[req] + pos.
    """
    res = LayerResult()
    if do_realign:
        res.k_ref64 = realign(pool_k, pool_v, k_table, v_table, segments, src_blocks, theta, rope_style)
    for r in range(len(seq_len)):
        t, o = int(seq_len[r]), int(tok_off[r])
        nidx = np.asarray(new_idx[new_off[r]:new_off[r + 1]], dtype=np.int32)
        if mode == "full":
            allrows = np.arange(t, dtype=np.int32)
            scatter_kv(pool_k, pool_v, k_table, v_table, cow_private, r, allrows,
                       k_fresh[o:o + t], v_fresh[o:o + t])
            sel, rows = np.zeros(0, np.int32), allrows
            res.scores.append(None)
            res.lse_new.append(None)
        else:
            scatter_kv(pool_k, pool_v, k_table, v_table, cow_private, r, nidx,
                       k_fresh[o + nidx], v_fresh[o + nidx])
            if rows_given is None:
                s, l = scores(pool_k, k_table[r], t, q_full[o + nidx], nidx, num_q_heads, want_lse=True)
                is_new = np.zeros(t, dtype=bool)
                is_new[nidx] = True
                cand = np.zeros(t, dtype=bool)       # I_reuse: the positions covered by the request's segments
                for (sr, slen, _old, snew, _off) in np.asarray(segments).reshape(-1, 5):
                    if int(sr) == r:
                        cand[int(snew):int(snew) + int(slen)] = True
                sel, rows = select_topk(s, is_new, int(k_per_req[r]), cand)
                res.scores.append(s)
                res.lse_new.append(l)
            else:
                sel, rows = rows_given[r]
                res.scores.append(None)
                res.lse_new.append(None)
            scatter_kv(pool_k, pool_v, k_table, v_table, cow_private, r, sel,
                       k_fresh[o + sel], v_fresh[o + sel])
        out, lse = attention(pool_k, pool_v, k_table[r], v_table[r], t, q_full[o + rows], rows,
                             num_q_heads, want_lse=True)
        res.sel.append(sel)
        res.rows.append(rows)
        res.out.append(out)
        res.lse.append(lse)
    return res
