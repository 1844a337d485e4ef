#!/usr/bin/env python
"""bench.py -- throughput of the SparseX Sparse-KV recomputation step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]

Default workload (BASELINE.json metric "... at 32K ctx" = configs[2], C3): the 32-layer multi-round
chat stack, one 32K request, layer threshold 4, paper mode (reading A11): layers 0-3 run
realign -> scatter(all) -> full attention, the boundary layer 3 also runs the single-sweep Sparse-Q
selection on its own LSE, layers 4-31 run realign -> scatter(I_nr) -> scatter(S_key) -> sparse
attention(R). A step = one pass of the whole stack. Other configs (--config C1|C2|C4|C5): a step =
one sparse layer with its own two-sweep selection.

value = context tokens x layers / second (whole job, all ranks), inputs resident in HBM.
e2e   = same metric through the C ABI with HOST (pinned) per-row inputs copied in and O copied out
        inside the timed region (the paged pool itself is the resident KV cache).
N > 1: the path has no exchange step and the headline workload is a single request, so ranks run
       independent replicas of the workload ("replicas only", weak scaling); no collective is issued.
--impl reference: the fp64 CPU oracle (oracle/), as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_01751_b200 import workloads as wl  # noqa: E402

METRIC = "sparse_recompute_context_tokens_per_s"
UNIT = "tokens/s"
CTA_PAIR = None   # None: library rule; --cta-pair / --single-cta force SX_ATTN_CTA_PAIR / SX_ATTN_SINGLE_CTA
L_STACK, THRESHOLD = 32, 4
NOMINAL_TF, NOMINAL_HBM_GBS = 2250.0, 8000.0   # BASELINE.json north_star: dense bf16 tensor peak, "~8 TB/s" HBM


def load_traffic(cfg: str):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/traffic.json, written
    when the capture is read; keyed by config). NOT measured in this run: the entry names its capture and commit."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    return json.load(open(p)).get(cfg)


# ----------------------------------------------------------------------------------------- helpers

def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "tf_burst": float(d["bf16_tflops"]),
                "tf_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "src": "measured"}
    return {"hbm_gbs": 6650.0, "tf_burst": 1590.0, "tf_sustained": 1400.0, "src": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"),
                                 f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def make_layout(cfg: str, rank: int, world: int):
    lay = wl.CONFIGS["C3" if cfg == "C3-layer" else cfg]()   # C3-layer: one sparse C3 layer with its own selection
    return lay


def attn_flops(rows_per_req, hq):
    """Algorithmic flops of stage (c): 4 * sum_{r in R} (pos_r + 1) * Hq * D (QK^T and PV, causal)."""
    return float(sum(4.0 * float(np.sum(r.astype(np.float64) + 1.0)) * hq * 128 for r in rows_per_req))


# ----------------------------------------------------------------------------------------- device inputs

class DevLayer:
    """Seeded synthetic tensors of one layer, drawn on the device with torch's Philox generator
    (same recipe as workloads.build_layer: N(0,1) bf16, x4 key norm on the salient tokens)."""

    def __init__(self, lay, layer: int, dev, torch):
        g = torch.Generator(device=dev)
        g.manual_seed(wl.ROOT_SEED * 1000 + lay.cfg_id * 100 + layer)
        hq, hkv = lay.num_q_heads, lay.num_kv_heads
        t = lay.total_tokens

        def rn(*shape):
            return torch.randn(*shape, generator=g, device=dev, dtype=torch.float32)
        pk = rn(lay.num_blocks, hkv, 16, 128)
        # salient cached tokens: (page, row) of every salient token of every pool segment
        pages, rows = [], []
        for s, pg in enumerate(lay.pool_seg_pages):
            idx = np.nonzero(lay.pool_salient[s])[0]
            pages.append(pg[idx // 16])
            rows.append(idx % 16)
        pages = torch.from_numpy(np.concatenate(pages).astype(np.int64)).to(dev)
        rows = torch.from_numpy(np.concatenate(rows).astype(np.int64)).to(dev)
        pk[pages, :, rows, :] *= 4.0
        self.pool_k = pk.to(torch.bfloat16).view(torch.int16)
        del pk
        self.pool_v = rn(lay.num_blocks, hkv, 16, 128).to(torch.bfloat16).view(torch.int16)
        self.q_full = rn(t, hq, 128).to(torch.bfloat16).view(torch.int16)
        kf = rn(t, hkv, 128)
        sal = np.concatenate([lay.salient_mask(r) for r in range(lay.num_reqs)])
        kf[torch.from_numpy(sal).to(dev)] *= 4.0
        self.k_fresh = kf.to(torch.bfloat16).view(torch.int16)
        del kf
        self.v_fresh = rn(t, hkv, 128).to(torch.bfloat16).view(torch.int16)


# ----------------------------------------------------------------------------------------- our arm

def select_flops(lay, hq, sweeps):
    """Algorithmic flops of stage (b): 2 * sum_{i in I_nr} (i + 1) * Hq * D per QK^T sweep (Eq. 1-2)."""
    w = sum(float(np.sum(lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]].astype(np.float64) + 1.0))
            for r in range(lay.num_reqs))
    return 2.0 * w * hq * 128 * sweeps


def measure(cfg, steps, warmup, ctx, want_e2e=True, want_clocks=True):
    """Times `steps` passes of config `cfg` on this rank's GPU; returns the pieces of the JSON line."""
    torch, sx, du, dev, local, rank, world, peaks, args = (ctx[k] for k in (
        "torch", "sx", "du", "dev", "local", "rank", "world", "peaks", "args"))
    from paper_2606_01751_b200.layer import GpuLayer
    stack = cfg == "C3"
    lay = make_layout(cfg, rank, world)
    n_layers = L_STACK if stack else 1
    hq, hkv = lay.num_q_heads, lay.num_kv_heads
    batch = sx.DeviceBatch(lay, dev)

    layers = []
    for l in range(n_layers):
        gl = GpuLayer(lay, DevLayer(lay, l, dev, torch), dev, batch=batch)
        gl.is_full = stack and l < THRESHOLD
        layers.append(gl)
    T = lay.total_tokens
    all_rows = torch.cat([torch.arange(int(n), dtype=torch.int32) for n in lay.seq_len]).to(dev)

    ev = {}

    def timed(name, fn):
        if ev.get("on"):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            ev.setdefault(name, []).append((a, b))
        else:
            fn()

    for gl in layers:
        n = T if gl.is_full else int(gl.rows_off_h[-1])
        gl.out = torch.empty((n, hq, 128), dtype=torch.int16, device=dev)
        gl.lse = torch.empty((n, hq), dtype=torch.float32, device=dev)
    sel_holder = {}

    def full_layer(gl, select_after):
        if not stack:
            timed("realign", lambda: sx.rope_realign(gl.pool, batch))
        timed("scatter", lambda: sx.scatter_kv(gl.pool, batch, gl.k_fresh, gl.v_fresh, all_rows, batch.tok_off,
                                               max_rows=T))
        timed("attn_full", lambda: sx.sparse_attn(gl.pool, batch, gl.q_full, gl.out, total_rows=T, lse=gl.lse,
                                                  full=True, cta_pair=CTA_PAIR))
        if select_after:
            timed("select", lambda: sx.score_select(gl.pool, batch, gl.q_new, gl.sel_off, gl.rows_off,
                                                    sel_holder["sel"], sel_holder["rows"], lse_new=gl.lse,
                                                    lse_by_token=True))

    def sparse_layer(gl, own_select):
        if not stack:
            timed("realign", lambda: sx.rope_realign(gl.pool, batch))
        n_rows = int(sel_holder["rows"].numel())
        if own_select:
            timed("scatter", lambda: sx.scatter_kv(gl.pool, batch, gl.kf_new, gl.vf_new, batch.new_idx, batch.new_off,
                                                   max_rows=lay.total_new))
            timed("select", lambda: sx.score_select(gl.pool, batch, gl.q_new, gl.sel_off, gl.rows_off,
                                                    sel_holder["sel"], sel_holder["rows"]))
            if sel_holder["sel"].numel():
                timed("scatter", lambda: sx.scatter_kv(gl.pool, batch, gl.kf_sel, gl.vf_sel, sel_holder["sel"],
                                                       gl.sel_off, max_rows=int(sel_holder["sel"].numel())))
        else:   # R fixed by the boundary layer: one scatter of the fresh K,V of all recomputed rows
            timed("scatter", lambda: sx.scatter_kv(gl.pool, batch, gl.kf_R, gl.vf_R, sel_holder["rows"], gl.rows_off,
                                                   max_rows=n_rows))
        timed("attn_sparse", lambda: sx.sparse_attn(gl.pool, batch, gl.q_R, gl.out, rows_R=sel_holder["rows"],
                                                    rows_off=gl.rows_off, total_rows=n_rows, lse=gl.lse,
                                                    cta_pair=CTA_PAIR))

    # ---- untimed pass: fixes R (deterministic) and stages the compact per-row inputs of Alg. 1 l.544
    g0 = layers[0]
    n_sel, n_rows_total = int(g0.sel_off_h[-1]), int(g0.rows_off_h[-1])
    sel_holder["sel"] = torch.zeros(max(n_sel, 1), dtype=torch.int32, device=dev)[:n_sel]
    sel_holder["rows"] = torch.zeros(n_rows_total, dtype=torch.int32, device=dev)
    pools = [gl.pool for gl in layers]
    if stack:
        sx.rope_realign_layers(pools, batch)
        for l in range(THRESHOLD):
            full_layer(layers[l], select_after=(l == THRESHOLD - 1))
    else:
        gl = layers[0]
        sx.rope_realign(gl.pool, batch)
        sx.scatter_kv(gl.pool, batch, gl.kf_new, gl.vf_new, batch.new_idx, batch.new_off, max_rows=lay.total_new)
        sx.score_select(gl.pool, batch, gl.q_new, gl.sel_off, gl.rows_off, sel_holder["sel"], sel_holder["rows"])
    torch.cuda.synchronize()
    rows_h = sel_holder["rows"].cpu().numpy()
    for gl in layers:
        if not gl.is_full:
            gl.stage_rows(sel_holder["sel"].clone(), sel_holder["rows"].clone())
            gl.q_full = None          # sparse layers only ever touch Q[R]
            if stack:
                gl.k_fresh = gl.v_fresh = None
    torch.cuda.empty_cache()

    def step():
        if stack:
            # stage (a) for the whole stack in one launch: it reads cached source pages only
            timed("realign", lambda: sx.rope_realign_layers(pools, batch))
            for l, gl in enumerate(layers):
                if gl.is_full:
                    full_layer(gl, select_after=(l == THRESHOLD - 1))
                else:
                    sparse_layer(gl, own_select=False)
        else:
            sparse_layer(layers[0], own_select=True)

    def barrier():
        du.barrier()
        torch.cuda.synchronize()

    # L2: the C3 step streams > 10 GB; for the single-layer configs a 512 MB scratch write between steps
    # evicts L2 (126 MB).
    flush = None if stack else torch.empty(512 << 20, dtype=torch.uint8, device=dev)

    for _ in range(max(warmup, 3)):
        step()
    barrier()
    # ---- timed region: K steps. C3 stack: CUDA events around every stage call inside the timed region (the
    # roofline's kernel time; 66 event pairs in a 60 ms step cost nothing). Single-layer configs: no per-stage
    # instrumentation in the timed region (two event records per stage call are a third of a launch-bound
    # 0.1 ms step); their per-stage view comes from a second pass of the same steps.
    two_pass = not stack
    ev["on"] = not two_pass
    launches0 = sx.launch_count()
    sampler = ClockSampler(local)
    if rank == 0 and want_clocks:
        sampler.start()
    step_ms = []
    for _ in range(steps):
        if flush is not None:
            flush.zero_()
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        step()
        b.record()
        barrier()
        step_ms.append(a.elapsed_time(b))
    clocks = sampler.stop() if (rank == 0 and want_clocks) else None
    launches = sx.launch_count() - launches0     # kernels launched in the timed region, counted inside libsparsex.so
    ev["on"] = False
    if two_pass:   # second pass, same steps, with CUDA events around every stage call: the per-stage view
        ev["on"] = True
        for _ in range(steps):
            if flush is not None:
                flush.zero_()
            barrier()
            step()
            barrier()
        ev["on"] = False
    t_ms = du.max_over_ranks(float(np.sum(step_ms)), dev)
    ms_per_step = t_ms / steps
    stage_ms = {k: float(sum(x.elapsed_time(y) for x, y in v)) / steps for k, v in ev.items() if k != "on"}
    stage_n = {k: len(v) // steps for k, v in ev.items() if k != "on"}

    # ---- roofline of the dominant kernel (attn_kernel<true>): algorithmic flops / event time
    rows_per_req = [rows_h[g0.rows_off_h[r]:g0.rows_off_h[r + 1]] for r in range(lay.num_reqs)]
    fl_sparse = attn_flops(rows_per_req, hq)
    fl_full = attn_flops([np.arange(int(n)) for n in lay.seq_len], hq)
    n_sparse = sum(1 for gl in layers if not gl.is_full)
    n_full = n_layers - n_sparse
    fl_total = fl_sparse * n_sparse + fl_full * n_full
    attn_ms = stage_ms.get("attn_sparse", 0.0) + stage_ms.get("attn_full", 0.0)
    achieved = fl_total / (attn_ms * 1e-3) / 1e12
    # a kernel timed alone between L2 flushes (single-layer configs) is held against the burst peak, the
    # attention launches inside the long C3 step against the sustained one (B200_PROFILING.md)
    tf_peak, tf_src = (peaks["tf_sustained"], "sustained") if stack else (peaks["tf_burst"], "burst")
    alg_bytes = float(sum(4.0 * int(n) * hkv * 128 for n in lay.seq_len) * n_layers +
                      4.0 * (n_rows_total * n_sparse + T * n_full) * hq * 128) / n_layers
    tr = load_traffic(cfg)
    roofline = {"bound": "tensor", "kernel": "attn_kernel<true%s> (sx_sparse_attn)" % (
                    ", cta pair" if (CTA_PAIR or (CTA_PAIR is None and lay.num_reqs == 1)) else ""), "achieved": round(achieved, 1),
                "peak": tf_peak, "unit": "TFLOP/s", "frac": round(achieved / tf_peak, 4),
                "peak_src": "%s bf16 %s" % (peaks["src"], tf_src),
                # every fraction against both measured peaks and the nominal one
                "frac_sustained": round(achieved / peaks["tf_sustained"], 4),
                "frac_burst": round(achieved / peaks["tf_burst"], 4),
                "frac_nominal": round(achieved / NOMINAL_TF, 4), "peak_nominal": NOMINAL_TF,
                # dram__bytes_read + dram__bytes_write per launch from the committed ncu --set full capture of this
                # kernel on this config (profiles/traffic.json); not measured in this run
                "traffic": (tr or {}).get("bytes_per_launch"), "traffic_unit": "B per launch",
                "traffic_src": ("%s @ %s (not measured in this run)" % (tr.get("capture"), tr.get("commit")) if tr else None),
                "algorithmic_bytes_per_launch": round(alg_bytes, 1),
                "traffic_over_algorithmic": (round(tr["bytes_per_launch"] / alg_bytes, 3) if tr else None),
                "launches_per_step": n_layers, "avg_launch_ms": round(attn_ms / n_layers, 4),
                "flops_per_step": fl_total}
    if "attn_sparse" in stage_ms and n_sparse:
        roofline["sparse_tflops"] = round(fl_sparse * n_sparse / (stage_ms["attn_sparse"] * 1e-3) / 1e12, 1)
    if "attn_full" in stage_ms and n_full:
        roofline["full_tflops"] = round(fl_full * n_full / (stage_ms["attn_full"] * 1e-3) / 1e12, 1)
    # HBM-bound stages: (a) 8*Hkv*128 B per cached token (read K,V + write K,V); (d) 8*Hkv*128 B per row
    row_b = 8.0 * hkv * 128
    re_bytes = row_b * lay.total_cached * n_layers
    sc_bytes = row_b * (T * n_full + n_rows_total * n_sparse)
    hbm = {"realign_gbs": round(re_bytes / (stage_ms["realign"] * 1e-3) / 1e9, 1),
           "realign_frac": round(re_bytes / (stage_ms["realign"] * 1e-3) / 1e9 / peaks["hbm_gbs"], 4),
           "scatter_gbs": round(sc_bytes / (stage_ms["scatter"] * 1e-3) / 1e9, 1),
           "scatter_frac": round(sc_bytes / (stage_ms["scatter"] * 1e-3) / 1e9 / peaks["hbm_gbs"], 4),
           "realign_frac_nominal": round(re_bytes / (stage_ms["realign"] * 1e-3) / 1e9 / NOMINAL_HBM_GBS, 4),
           "scatter_frac_nominal": round(sc_bytes / (stage_ms["scatter"] * 1e-3) / 1e9 / NOMINAL_HBM_GBS, 4),
           "peak_hbm_gbs": peaks["hbm_gbs"], "peak_hbm_nominal_gbs": NOMINAL_HBM_GBS}
    if "select" in stage_ms:
        sel_fl = select_flops(lay, hq, 1 if stack else 2)
        hbm["select_tflops"] = round(sel_fl / (stage_ms["select"] * 1e-3) / 1e12, 1)
        # stage (b) is bound by the exponentials (one per 256 flop), not by the tensor pipe: hold it against the
        # measured rate of its own MUFU / FMA-pipe mix (sx_probe_pipe), whole stage time (top-k included)
        pr = ctx.get("pipe_rates")
        if pr:
            exps = sel_fl / 256.0
            hbm["select_gexp_per_s"] = round(exps / (stage_ms["select"] * 1e-3) / 1e9, 1)
            hbm["select_alu_frac"] = round(exps / (stage_ms["select"] * 1e-3) / (pr["sweep_mix_gexp_per_s"] * 1e9), 4)

    # launch-bound single-layer configs: the same step replayed from a CUDA graph (no host launch gaps)
    graph_ms = None
    if not stack:
        try:
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr):
                step()
            for _ in range(3):
                gr.replay()
            torch.cuda.synchronize()
            gms = []
            for _ in range(max(steps, 5)):
                flush.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                gr.replay()
                b.record()
                torch.cuda.synchronize()
                gms.append(a.elapsed_time(b))
            graph_ms = float(np.median(gms))
            del gr
        except Exception as e:     # capture not possible: report the reason, keep the stream-launched number
            graph_ms = "capture failed: %s" % str(e).splitlines()[0][:120]
            torch.cuda.synchronize()

    res = {"cfg": cfg, "lay": lay, "stack": stack, "n_layers": n_layers, "T": T, "rows_R": n_rows_total,
           "graph_ms": graph_ms,
           "n_sparse": n_sparse, "ms_per_step": ms_per_step, "stage_ms": stage_ms, "stage_n": stage_n,
           "roofline": roofline, "hbm": hbm, "clocks": clocks, "launches": launches,
           "value": du.job_throughput(T * n_layers, ms_per_step, world), "bytes_per_step": re_bytes + sc_bytes,
           "e2e": None}
    if want_e2e:
        res["e2e"] = run_e2e(torch, sx, du, lay, layers, batch, all_rows, sel_holder, stack, args, dev, world, barrier)
    del layers, flush
    torch.cuda.empty_cache()
    return res


def measure_s6(ctx, reps=10):
    """Supplementary HBM-regime cases: stage (c) alone with few (row, head) pairs per KV head: K and V
    of the whole context are streamed once. Both dispatch choices are timed: the library's default (the padded
    tensor-core tile with key splits that merge themselves) and the CUDA-core kernels (SX_ATTN_CUDA_CORE, north_star's
    rule below 64 pairs per KV head).
    Achieved GB/s = 4*T*Hkv*128 B / time, L2 flushed between repetitions. "chained4": the same call on the pools of
    four consecutive layers back to back (536 MB of K/V, larger than L2, no flush): what a layer stack sees, with the
    launch of each call overlapping the tail of the previous one (programmatic dependent launch)."""
    torch, sx, dev, peaks = ctx["torch"], ctx["sx"], ctx["dev"], ctx["peaks"]
    from paper_2606_01751_b200.layer import GpuLayer
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    out = {}

    def frac(t_ms, nbytes):
        gbs = nbytes / (t_ms * 1e-3) / 1e9
        return {"ms": round(t_ms, 4), "hbm_gbs": round(gbs, 1), "hbm_frac": round(gbs / peaks["hbm_gbs"], 4),
                "hbm_frac_nominal": round(gbs / NOMINAL_HBM_GBS, 4)}
    # (i) C3 pool, last 1 / 2 / 8 positions: 4 / 8 / 32 pairs per KV head; (ii) C5 pool, last 16 positions: 112 pairs
    for cfg, layer, lasts in (("C3", 4, (1, 2, 8)), ("C5", 0, (16,))):
        lay = wl.CONFIGS[cfg]()
        n_l = 4 if cfg == "C3" else 1
        gls = [GpuLayer(lay, DevLayer(lay, layer + i, dev, torch), dev) for i in range(n_l)]
        T, hq, hkv = lay.total_tokens, lay.num_q_heads, lay.num_kv_heads
        all_rows = torch.arange(T, dtype=torch.int32, device=dev)
        for gl in gls:
            sx.rope_realign(gl.pool, gl.batch)
            sx.scatter_kv(gl.pool, gl.batch, gl.k_fresh, gl.v_fresh, all_rows, gl.batch.tok_off, max_rows=T)
        gl = gls[0]
        for n in lasts:
            rows = torch.arange(T - n, T, dtype=torch.int32, device=dev)
            off = torch.tensor([0, n], dtype=torch.int32, device=dev)
            q = gl.q_full[T - n:T].contiguous()
            o = torch.empty((n, hq, 128), dtype=torch.int16, device=dev)
            res = {}
            for label, cc, pair in (("tcgen05_splits", False, None), ("cuda_core", True, None)):
                if cc and n * hq // hkv >= 64:
                    continue                    # the CUDA-core kernels are for fewer than 64 pairs per KV head
                ms = []
                for i in range(reps + 3):
                    flush.zero_()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    sx.sparse_attn(gl.pool, gl.batch, q, o, rows_R=rows, rows_off=off, total_rows=n, cuda_core=cc,
                                   cta_pair=pair)
                    b.record()
                    torch.cuda.synchronize()
                    if i >= 3:
                        ms.append(a.elapsed_time(b))
                res[label] = frac(float(np.median(ms)), 4.0 * T * hkv * 128)
            if n_l > 1:
                ms = []
                for i in range(reps + 3):
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    for g2 in gls:
                        sx.sparse_attn(g2.pool, g2.batch, q, o, rows_R=rows, rows_off=off, total_rows=n)
                    b.record()
                    torch.cuda.synchronize()
                    if i >= 3:
                        ms.append(a.elapsed_time(b) / n_l)
                res["tcgen05_splits_chained4"] = frac(float(np.median(ms)), 4.0 * T * hkv * 128)
            out["%s_last%d_rows_%d_pairs_per_kv_head" % (cfg, n, n * hq // hkv)] = res
        del gls, gl
        torch.cuda.empty_cache()
    del flush
    torch.cuda.empty_cache()
    return out


def measure_pipes(ctx):
    """Instruction-pipe rates of this GPU (sx_probe_pipe): lane-operations per clock and SM and, with the clock the
    probe itself ran at, per second for the whole GPU. `sweep_mix` = the scoring sweeps' exponential mix (6 of 8 on
    MUFU.EX2, 2 of 8 by the FMA-pipe polynomial): the roofline of stage (b) (`select_alu_frac`)."""
    torch, sx, dev = ctx["torch"], ctx["sx"], ctx["dev"]
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    out = {"sms": n_sm}
    iters = 8192
    for name, pipe in (("mufu_ex2", 0), ("ffma", 1), ("ffma2", 2), ("sweep_mix", 3)):
        per_clk = sx.probe_pipe(pipe, iters=iters, device=dev)
        cyc = torch.zeros(n_sm + 1, dtype=torch.int64, device=dev)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        sx.load().sx_probe_pipe(pipe, iters, cyc.data_ptr(), n_sm, None)
        b.record()
        torch.cuda.synchronize()
        ms = a.elapsed_time(b)
        out[name + "_per_clk_sm"] = round(per_clk, 2)
        out[name + "_gexp_per_s" if pipe in (0, 3) else name + "_gops_per_s"] = round(
            1024.0 * 8 * iters * n_sm / (ms * 1e-3) / 1e9, 1)
        out[name + "_sm_mhz"] = round(float(cyc[:n_sm].median().item()) / (ms * 1e-3) / 1e6, 0)
    return out


def measure_zero_copy(ctx, reps=10):
    """Zero-copy mode (include/sparsex.h; S9 NEXT-3) against the copy path, same inputs, same stages:
      (i)  one sparse C4 layer (16 requests, two-sweep selection), every stage timed between events;
      (ii) the S6 row sets (stage (c) alone over a 32K / 133K context where NOTHING has been made private: every
           reused key is rotated in shared memory).
    Block tables are restored before every repetition of the zero-copy arm (its scatter flips them), L2 is flushed
    between repetitions. Memory: private pages a request holds for its reused segments after the layer."""
    torch, sx, dev = ctx["torch"], ctx["sx"], ctx["dev"]
    from paper_2606_01751_b200.layer import GpuLayer
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    out = {}

    def timed(stages):
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(len(stages) + 1)]
        evs[0].record()
        for i, (_, fn) in enumerate(stages):
            fn()
            evs[i + 1].record()
        torch.cuda.synchronize()
        return [evs[i].elapsed_time(evs[i + 1]) for i in range(len(stages))]

    # ---- (i) C4 sparse layer
    lay = wl.CONFIGS["C4"]()
    zlay = wl.zero_copy_layout(lay)
    dl = DevLayer(lay, 0, dev, torch)
    g0, g1 = GpuLayer(lay, dl, dev), GpuLayer(zlay, dl, dev)   # one pool: the arms run one after the other
    kt1, vt1 = g1.batch.k_block_table.clone(), g1.batch.v_block_table.clone()
    g0.step_sparse()                    # fixes S_key / R (identical in both arms: tests/test_gpu_zero_copy.py)
    g1.stage_rows(g0.sel_idx, g0.rows_R)
    for label, g in (("copy", g0), ("zero_copy", g1)):
        stages = [("scatter_new", g.scatter_new), ("select", lambda g=g: g.select(want_scores=False)),
                  ("scatter_sel", g.scatter_sel), ("attention", lambda g=g: g.attend(want_lse=False))]
        if label == "copy":
            stages.insert(0, ("realign", g.realign))
        acc = []
        for i in range(reps + 3):
            if label == "zero_copy":
                g.batch.k_block_table.copy_(kt1)
                g.batch.v_block_table.copy_(vt1)
            flush.zero_()
            t = timed(stages)
            if i >= 3:
                acc.append(t)
        med = np.median(np.asarray(acc), axis=0)
        out.setdefault("C4_sparse_layer", {})[label] = {
            "stage_ms": {n: round(float(v), 4) for (n, _), v in zip(stages, med)}, "ms": round(float(med.sum()), 4)}
    torch.cuda.synchronize()
    page_bytes = 2 * lay.num_kv_heads * 16 * 128 * 2    # K and V
    flipped = int((g1.batch.k_block_table != kt1).sum().item())
    out["C4_sparse_layer"]["private_pages"] = {
        "copy": lay.total_seg_pages, "zero_copy": flipped, "page_bytes": page_bytes,
        "copy_mb": round(lay.total_seg_pages * page_bytes / 1e6, 1), "zero_copy_mb": round(flipped * page_bytes / 1e6, 1)}
    del g0, g1, dl
    torch.cuda.empty_cache()

    # ---- (ii) S6 row sets over untouched shared pages
    for cfg, layer, lasts in (("C3", 4, (8,)), ("C5", 0, (16,))):
        lay = wl.CONFIGS[cfg]()
        zlay = wl.zero_copy_layout(lay)
        dl = DevLayer(lay, layer, dev, torch)
        g0, g1 = GpuLayer(lay, dl, dev), GpuLayer(zlay, dl, dev)
        T, hq, hkv = lay.total_tokens, lay.num_q_heads, lay.num_kv_heads
        g0.realign()
        g0.scatter_new()    # (new tokens live in the request's own pages in both arms)
        for n in lasts:
            rows = torch.arange(T - n, T, dtype=torch.int32, device=dev)
            off = torch.tensor([0, n], dtype=torch.int32, device=dev)
            q = g0.q_full[T - n:T].contiguous()
            o = torch.empty((n, hq, 128), dtype=torch.int16, device=dev)
            res = {}
            for label, g in (("copy", g0), ("zero_copy", g1)):
                ms = []
                for i in range(reps + 3):
                    flush.zero_()
                    ms.append(timed([("attention", lambda g=g: sx.sparse_attn(g.pool, g.batch, q, o, rows_R=rows,
                                                                                 rows_off=off, total_rows=n))])[0])
                t_ms = float(np.median(ms[3:]))
                res[label] = {"ms": round(t_ms, 4), "hbm_gbs": round(4.0 * T * hkv * 128 / (t_ms * 1e-3) / 1e9, 1)}
            out["%s_last%d_rows" % (cfg, n)] = res
        del g0, g1, dl
        torch.cuda.empty_cache()
    del flush
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    from paper_2606_01751_b200 import binding as sx
    from paper_2606_01751_b200 import build as sxbuild
    from paper_2606_01751_b200 import dist_util as du
    rank, world, local = du.env_rank()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    du.init("nccl", dev)
    if rank == 0:
        sxbuild.build()
    du.barrier()
    sx.load()
    ctx = {"torch": torch, "sx": sx, "du": du, "dev": dev, "local": local, "rank": rank, "world": world,
           "peaks": load_peaks(), "args": args}
    cfg = args.config
    if world == 1:
        ctx["pipe_rates"] = measure_pipes(ctx)
    if cfg == "S6":   # supplementary: stage (c) alone on small row sets (HBM regime); not the headline metric
        if rank == 0:
            print(json.dumps({"metric": "small_row_attention_hbm", "unit": "GB/s", "n_gpus": 1, "dtype": "bf16",
                              "data": "synthetic", "config": {"workload": "S6: last rows of a 32K / 133K context"},
                              "cases": measure_s6(ctx, reps=max(args.steps, 3))}), flush=True)
        return
    if cfg == "ZC":   # supplementary: zero-copy mode against the copy path (S9)
        if rank == 0:
            print(json.dumps({"metric": "zero_copy_vs_copy", "unit": "ms", "n_gpus": 1, "dtype": "bf16",
                              "data": "synthetic", "config": {"workload": "ZC: C4 sparse layer; S6 row sets"},
                              "cases": measure_zero_copy(ctx, reps=max(args.steps, 3))}), flush=True)
        return
    m = measure(cfg, args.steps, args.warmup, ctx)
    # the other configs of BASELINE.json (north_star: throughput of all five at 1 GPU): short runs, same code path
    others = {}
    if world == 1 and not args.no_others:
        for c in wl.CONFIGS:
            if c == cfg or c not in ("C1", "C2", "C3", "C4", "C5"):
                continue
            o = measure(c, 30 if c != "C3" else 2, 5, ctx, want_e2e=False, want_clocks=False)
            others[c] = {"context_tokens": o["T"], "rows_R": o["rows_R"], "layers": o["n_layers"],
                         "ms_per_layer": round(o["ms_per_step"] / o["n_layers"], 4),
                         "ms_per_layer_cuda_graph": (round(o["graph_ms"], 4) if isinstance(o["graph_ms"], float)
                                                     else o["graph_ms"]),
                         "context_tokens_per_s": round(o["value"], 1),
                         "stage_ms": {k: round(v, 4) for k, v in o["stage_ms"].items()},
                         "attn_tflops": o["roofline"]["achieved"], "attn_frac": o["roofline"]["frac"],
                         "attn_frac_burst": o["roofline"]["frac_burst"],
                         "attn_frac_sustained": o["roofline"]["frac_sustained"],
                         "attn_frac_nominal": o["roofline"]["frac_nominal"],
                         "attn_peak": o["roofline"]["peak_src"],
                         "attn_traffic": o["roofline"]["traffic"],
                         "attn_algorithmic_bytes": o["roofline"]["algorithmic_bytes_per_launch"],
                         "attn_traffic_over_algorithmic": o["roofline"]["traffic_over_algorithmic"],
                         "hbm_stage": o["hbm"]}
        if cfg == "C3":
            # reading A11, secondary mode: a sparse C3 layer that runs its OWN two-sweep selection (what a stack
            # costs when every sparse layer selects: 4 full layers + 28 x this)
            o = measure("C3-layer", 30, 5, ctx, want_e2e=False, want_clocks=False)
            others["C3_select_every_layer"] = {
                "ms_per_sparse_layer": round(o["ms_per_step"], 4),
                "stage_ms": {k: round(v, 4) for k, v in o["stage_ms"].items()},
                "note": "one sparse C3 layer: realign, scatter(I_nr), two-sweep selection, scatter(S_key), attention"}
        others["S6"] = measure_s6(ctx)
        others["zero_copy"] = measure_zero_copy(ctx)
    if rank != 0:
        return
    stack, n_layers, T = m["stack"], m["n_layers"], m["T"]
    line = {
        "metric": METRIC, "value": round(m["value"], 1), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": round(m["ms_per_step"], 4), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": ("C3 32-layer chat stack, 1 x 32K ctx, 32Q/8KV, threshold 4, paper mode "
                                "(select once at layer 3), ratio 10%" if stack else
                                "%s one sparse layer with two-sweep selection" % cfg),
                   "layers": n_layers, "context_tokens": T, "rows_R": m["rows_R"],
                   "ms_per_layer": round(m["ms_per_step"] / n_layers, 4),
                   "stage_ms_per_step": {k: round(v, 4) for k, v in m["stage_ms"].items()},
                   "stage_calls_per_step": m["stage_n"], "hbm_stage": m["hbm"], "parallelism": "replicas only",
                   "inputs": "drawn on the device with torch's Philox generator from the recipe of workloads.py (same "
                             "shapes, layout, salient x4 keys); NOT the numpy (PCG64) bytes the parity tests check",
                   "l2": ("step working set > L2 (%.1f GB per step)" % (m["bytes_per_step"] / 1e9) if stack
                          else "512 MB flush between steps"),
                   "recomputed_tokens_per_s": round(world * m["rows_R"] * m["n_sparse"] / (m["ms_per_step"] * 1e-3), 1)},
        "clocks": m["clocks"], "e2e": m["e2e"], "gpu_launches": m["launches"], "roofline": m["roofline"],
    }
    if "pipe_rates" in ctx:
        line["config"]["pipe_rates"] = ctx["pipe_rates"]
    if others:
        line["config"]["other_configs"] = others
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(m["lay"], cfg, stack)
    print(json.dumps(line), flush=True)


def run_e2e(torch, sx, du, lay, layers, batch, all_rows, sel_holder, stack, args, dev, world, barrier):
    """Same step with the per-row inputs in pinned HOST memory and the outputs copied back, inside the
    timed region. Host->device copies run on their own stream one or more layers ahead of the kernels
    (every layer has its own device buffers), device->host copies on a third stream behind them, so the
    two PCIe directions overlap the compute; events order copy -> kernels -> copy-out per layer."""
    hq = lay.num_q_heads
    T = lay.total_tokens

    def pin(t):
        h = torch.empty(t.shape, dtype=t.dtype, pin_memory=True)
        h.copy_(t)
        return h
    host, h2d, d2h = [], 0, 0
    for gl in layers:
        if gl.is_full:
            names = ["q_full", "k_fresh", "v_fresh"]
        elif stack:
            names = ["kf_R", "vf_R", "q_R"]
        else:
            names = ["q_new", "kf_new", "vf_new", "kf_sel", "vf_sel", "q_R"]
        d = {n: pin(getattr(gl, n)) for n in names}
        host.append(d)
        h2d += sum(v.numel() * v.element_size() for v in d.values())
        d2h += gl.out.numel() * 2
    out_host = torch.empty((T if stack else int(layers[0].rows_off_h[-1]), hq, 128), dtype=torch.int16, pin_memory=True)
    main = torch.cuda.current_stream()
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    ev_in = [torch.cuda.Event() for _ in layers]
    ev_done = [torch.cuda.Event() for _ in layers]
    for e in ev_done:
        e.record(main)

    def step():
        for l, gl in enumerate(layers):
            with torch.cuda.stream(s_in):
                s_in.wait_event(ev_done[l])        # previous step's kernels of this layer have read its buffers
                for n, h in host[l].items():
                    getattr(gl, n).copy_(h, non_blocking=True)
                ev_in[l].record(s_in)
        if stack:
            sx.rope_realign_layers([gl.pool for gl in layers], batch)
        for l, gl in enumerate(layers):
            main.wait_event(ev_in[l])
            if not stack:
                sx.rope_realign(gl.pool, batch)
            if gl.is_full:
                sx.scatter_kv(gl.pool, batch, gl.k_fresh, gl.v_fresh, all_rows, batch.tok_off, max_rows=T)
                sx.sparse_attn(gl.pool, batch, gl.q_full, gl.out, total_rows=T, lse=gl.lse, full=True,
                               cta_pair=CTA_PAIR)
                if l == THRESHOLD - 1:
                    sx.score_select(gl.pool, batch, gl.q_new, gl.sel_off, gl.rows_off, sel_holder["sel"],
                                    sel_holder["rows"], lse_new=gl.lse, lse_by_token=True)
            else:
                n_rows = int(sel_holder["rows"].numel())
                if stack:
                    sx.scatter_kv(gl.pool, batch, gl.kf_R, gl.vf_R, sel_holder["rows"], gl.rows_off, max_rows=n_rows)
                else:
                    sx.scatter_kv(gl.pool, batch, gl.kf_new, gl.vf_new, batch.new_idx, batch.new_off,
                                  max_rows=lay.total_new)
                    sx.score_select(gl.pool, batch, gl.q_new, gl.sel_off, gl.rows_off, sel_holder["sel"],
                                    sel_holder["rows"])
                    if sel_holder["sel"].numel():
                        sx.scatter_kv(gl.pool, batch, gl.kf_sel, gl.vf_sel, sel_holder["sel"], gl.sel_off,
                                      max_rows=int(sel_holder["sel"].numel()))
                sx.sparse_attn(gl.pool, batch, gl.q_R, gl.out, rows_R=sel_holder["rows"], rows_off=gl.rows_off,
                               total_rows=n_rows, lse=gl.lse, cta_pair=CTA_PAIR)
            ev_done[l].record(main)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_done[l])
                out_host[:gl.out.shape[0]].copy_(gl.out, non_blocking=True)
        main.wait_stream(s_out)   # a step ends when its last output has reached the host

    step()
    barrier()
    n = max(1, args.steps)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(n):
        step()
    b.record()
    barrier()
    ms = a.elapsed_time(b) / n
    ms = du.max_over_ranks(ms, dev)
    return {"value": round(du.job_throughput(T * len(layers), ms, world), 1), "unit": UNIT, "ms_per_step": round(ms, 3),
            "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "steps": n,
            "note": "per-row inputs (Q, fresh K/V) from pinned host memory on a copy stream ahead of the kernels, "
                    "O read back on a second copy stream; paged pool resident"}


# ----------------------------------------------------------------------------------------- CPU oracle arm
#
# The fp64 oracle (oracle/), as it stands, on the box's host cores. Two kinds of numbers, labelled:
#   "measured"  : workloads the oracle FINISHES -- the whole C1 layer and request 0 of C2 --, every stage
#                 timed by wall clock, nothing scaled ("estimated": false);
#   "estimated" : the headline config. One bounded, FIXED-SIZE sample of it is timed (realign of one segment,
#                 scatter of 1024 rows, Eq. (1)-(2) scores of 96 Sparse-Q queries, attention of 1152 rows) and
#                 scaled to the whole step by the exact algorithmic work: sum_{i in I_nr} (i+1) for the scores,
#                 sum_{r in R} (r+1) for the attention with R = the oracle's own recompute set
#                 (tests/golden/rows_C3_L3.txt for the C3 stack; k evenly spread rows otherwise), T (T+1) / 2 for
#                 full layers. value = (fraction of the step's work the sample covers) x tokens x layers / time.

SAMPLE_Q, SAMPLE_ROWS, SAMPLE_SCATTER = 96, 1152, 1024   # ~7 s of oracle time on 16 cores (10-30 s with the measured legs)


def _oracle_layer_timed(orc, lay, lt, reqs):
    """One sparse layer of `lay`, requests `reqs`, every stage timed (wall clock). Returns per-stage seconds."""
    pk, pv = lt.pool_k.copy(), lt.pool_v.copy()
    kt, vt = lay.k_block_table.copy(), lay.v_block_table.copy()
    hq = lay.num_q_heads
    segs = np.asarray([s for s in lay.segments.tolist() if s[0] in reqs], dtype=np.int32).reshape(-1, 5)
    st = {"realign": 0.0, "scatter": 0.0, "select": 0.0, "attention": 0.0}
    t0 = time.perf_counter()
    orc.realign(pk, pv, kt, vt, segs, lay.src_blocks, lay.rope_theta, lay.rope_style)
    st["realign"] = time.perf_counter() - t0
    tokens = rows_total = 0
    for r in reqs:
        t, o = int(lay.seq_len[r]), int(lay.tok_off[r])
        nidx = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]]
        t0 = time.perf_counter()
        orc.scatter_kv(pk, pv, kt, vt, None, r, nidx, lt.k_fresh[o + nidx], lt.v_fresh[o + nidx])
        t1 = time.perf_counter()
        s = orc.scores(pk, kt[r], t, lt.q_full[o + nidx], nidx, hq)
        sel, rows = orc.select_topk(s, lay.is_new_mask(r), int(lay.k_per_req[r]), lay.cached_mask(r))
        t2 = time.perf_counter()
        orc.scatter_kv(pk, pv, kt, vt, None, r, sel, lt.k_fresh[o + sel], lt.v_fresh[o + sel])
        t3 = time.perf_counter()
        orc.attention(pk, pv, kt[r], vt[r], t, lt.q_full[o + rows], rows, hq)
        t4 = time.perf_counter()
        st["scatter"] += (t1 - t0) + (t3 - t2)
        st["select"] += t2 - t1
        st["attention"] += t4 - t3
        tokens += t
        rows_total += len(rows)
    total = sum(st.values())
    return {"context_tokens": tokens, "rows_R": rows_total, "seconds": round(total, 3),
            "stage_seconds": {k: round(v, 4) for k, v in st.items()},
            "context_tokens_per_s": round(tokens / total, 1), "estimated": False}


def cpu_measured(orc):
    """Fully timed oracle runs on what it can finish: the whole C1 layer and request 0 of C2 (one sparse layer each)."""
    out = {}
    lay = wl.CONFIGS["C1"]()
    out["C1_whole_layer"] = _oracle_layer_timed(orc, lay, wl.build_layer(lay, 0), [0])
    lay = wl.CONFIGS["C2"]()
    out["C2_request_0"] = _oracle_layer_timed(orc, lay, wl.build_layer(lay, 0), [0])
    return out


def _oracle_rows_c3():
    p = os.path.join(ROOT, "tests", "golden", "rows_C3_L3.txt")
    return np.asarray([int(x) for x in open(p) if x.strip() and not x.startswith("#")], dtype=np.int64)


class CpuSample:
    """The fixed-size sample of the headline workload; prepare() builds inputs (untimed), run() is one timed step."""

    def __init__(self, lay, cfg, stack):
        from oracle import sx_oracle as orc
        orc.build()
        self.orc, self.lay, self.cfg, self.stack = orc, lay, cfg, stack
        self.cores = orc.num_threads()
        lt = wl.build_layer(lay, THRESHOLD if stack else 0, threads=max(1, self.cores))
        self.lt = lt
        self.pk, self.pv = lt.pool_k, lt.pool_v
        self.kt, self.vt = lay.k_block_table.copy(), lay.v_block_table.copy()
        o = int(lay.tok_off[0])
        nidx = lay.new_idx[lay.new_off[0]:lay.new_off[1]]
        self.nidx = nidx
        self.t_req = int(lay.seq_len[0])
        self.q_samp = nidx[np.unique(np.linspace(0, len(nidx) - 1, min(SAMPLE_Q, len(nidx))).astype(int))]
        self.sc_rows = nidx[:SAMPLE_SCATTER]
        self.o = o
        # exact algorithmic work of the whole step, in (row, key) pairs
        self.w_sel = sum(float(np.sum(lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]].astype(np.float64) + 1))
                         for r in range(lay.num_reqs))
        self.w_full = sum(int(t) * (int(t) + 1) / 2.0 for t in lay.seq_len)
        if stack:
            rr = _oracle_rows_c3()
            self.w_sparse, self.n_rows, self.rows_src = float(np.sum(rr + 1.0)), len(rr), "oracle R (tests/golden/rows_C3_L3.txt)"
        else:
            self.w_sparse, self.n_rows = 0.0, 0
            for r in range(lay.num_reqs):
                t = int(lay.seq_len[r])
                nn = lay.new_idx[lay.new_off[r]:lay.new_off[r + 1]].astype(np.float64)
                k = int(lay.k_per_req[r])
                self.w_sparse += float(np.sum(nn + 1)) + k * (t / 2.0)
                self.n_rows += len(nn) + k
            self.rows_src = "I_nr + k evenly spread cached rows (cost model)"
        # (a small config is not over-sampled: never more attention rows than one request of the step computes)
        n_samp = min(SAMPLE_ROWS, self.t_req, max(1, self.n_rows // lay.num_reqs))
        self.rows = np.unique(np.linspace(0, self.t_req - 1, n_samp).astype(np.int32))

    def run(self):
        """One timed sample. Returns (whole-step seconds extrapolated, sample seconds, per-stage estimate)."""
        orc, lay, lt = self.orc, self.lay, self.lt
        hq = lay.num_q_heads
        seg = lay.segments[:1]
        t0 = time.perf_counter()
        orc.realign(self.pk, self.pv, self.kt, self.vt, seg, lay.src_blocks, lay.rope_theta, lay.rope_style)
        t1 = time.perf_counter()
        orc.scatter_kv(self.pk, self.pv, self.kt, self.vt, None, 0, self.sc_rows, lt.k_fresh[self.o + self.sc_rows],
                       lt.v_fresh[self.o + self.sc_rows])
        t2 = time.perf_counter()
        orc.scores(self.pk, self.kt[0], self.t_req, lt.q_full[self.o + self.q_samp], self.q_samp, hq)
        t3 = time.perf_counter()
        orc.attention(self.pk, self.pv, self.kt[0], self.vt[0], self.t_req, lt.q_full[self.o + self.rows], self.rows, hq)
        t4 = time.perf_counter()
        t_re = (t1 - t0) * lay.total_cached / float(seg[0, 1])
        t_sc_row = (t2 - t1) / max(1, len(self.sc_rows))
        t_sel = (t3 - t2) * self.w_sel / float(np.sum(self.q_samp.astype(np.float64) + 1))
        per_pair = (t4 - t3) / float(np.sum(self.rows.astype(np.float64) + 1))
        t_as, t_af = per_pair * self.w_sparse, per_pair * self.w_full
        if self.stack:
            n_full, n_sparse = THRESHOLD, L_STACK - THRESHOLD
            total = (n_full * (t_re + t_sc_row * lay.total_tokens + t_af) + t_sel / 2.0 +
                     n_sparse * (t_re + t_sc_row * self.n_rows + t_as))
        else:
            total = t_re + t_sc_row * self.n_rows + t_sel + t_as
        est = {"realign": round(t_re, 2), "select": round(t_sel, 1), "attn_sparse": round(t_as, 1),
               "attn_full": round(t_af, 1)}
        return total, t4 - t0, est

    def describe(self):
        return ("fixed sample of one layer's tensors: realign of 1 segment, scatter of %d rows, Eq.(1)-(2) scores of %d "
                "Sparse-Q queries, attention of %d rows x %d heads; scaled by the exact algorithmic work of the %s; "
                "sparse rows = %s" % (len(self.sc_rows), len(self.q_samp), len(self.rows), self.lay.num_q_heads,
                                      "32-layer stack" if self.stack else "layer", self.rows_src))


def cpu_baseline(lay, cfg, stack):
    """The fp64 oracle, as it stands: measured runs on C1 / one C2 request, and the headline config estimated from a
    fixed-size sample (see the block comment above)."""
    cs = CpuSample(lay, cfg, stack)
    cs.run()                                           # warm the caches / thread pool
    total, t_sample, est = cs.run()
    layers = L_STACK if stack else 1
    return {"value": round(lay.total_tokens * layers / total, 2), "unit": UNIT, "cores": cs.cores, "kind": "oracle",
            "estimated": True, "sample": cs.describe(), "sample_seconds": round(t_sample, 2),
            "sample_fraction_of_step": t_sample / total,
            "est_seconds_per_step": round(total, 1), "est_stage_seconds": est,
            "measured": cpu_measured(cs.orc)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return
    # torchrun exports OMP_NUM_THREADS=1 for its workers; the one rank that runs the oracle uses the host's cores
    if os.environ.get("OMP_NUM_THREADS", "1") == "1":
        os.environ["OMP_NUM_THREADS"] = str(os.cpu_count() or 1)
    cfg = args.config
    stack = cfg == "C3"
    lay = wl.CONFIGS[cfg]()
    cs = CpuSample(lay, cfg, stack)
    n_layers = L_STACK if stack else 1
    # a step of this arm = one fixed-size sample of the step's work (fraction f of it, by oracle time):
    # value = f x tokens x layers / t_sample; ms_per_step is the wall clock of the sample as run
    runs = [cs.run() for _ in range(max(args.warmup, 0) + max(args.steps, 1))][max(args.warmup, 0):]
    t_sample = float(np.mean([r[1] for r in runs]))
    total = float(np.mean([r[0] for r in runs]))
    v = lay.total_tokens * n_layers / total
    line = {"impl": "reference", "metric": METRIC, "value": round(v, 2), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(t_sample * 1e3, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "estimated": True,
            "config": {"workload": "same as the CUDA arm (%s); a step of this arm is ONE fixed-size sample of the "
                                   "workload's step timed on the fp64 CPU oracle (ms_per_step = its wall clock); value = "
                                   "sample_fraction_of_step x context tokens x layers / that time" % cfg,
                       "layers": n_layers, "context_tokens": lay.total_tokens,
                       "sample_fraction_of_step": t_sample / total, "est_ms_per_whole_step": round(total * 1e3, 1)},
            "cpu_baseline": {"value": round(v, 2), "unit": UNIT, "cores": cs.cores, "kind": "oracle", "estimated": True,
                             "sample": cs.describe(), "sample_seconds": round(t_sample, 2),
                             "measured": (cpu_measured(cs.orc) if not args.no_cpu_measured else None)},
            "e2e": {"value": round(v, 2), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C3", choices=list(wl.CONFIGS) + ["S6", "ZC"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-cpu-measured", action="store_true",
                    help="reference arm: skip the fully timed oracle runs (C1 layer, C2 request)")
    ap.add_argument("--no-others", action="store_true", help="skip the short runs of the other BASELINE configs")
    ap.add_argument("--cta-pair", action="store_true",
                    help="force stage (c) onto 2-CTA clusters (SX_ATTN_CTA_PAIR, tcgen05.mma.cta_group::2)")
    ap.add_argument("--single-cta", action="store_true",
                    help="force stage (c) onto the single-CTA kernel (SX_ATTN_SINGLE_CTA); default: library rule")
    args = ap.parse_args()
    global CTA_PAIR
    CTA_PAIR = True if args.cta_pair else (False if args.single_cta else None)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
