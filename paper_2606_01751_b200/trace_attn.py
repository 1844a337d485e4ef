"""Per-CTA phase trace of the attention kernel (diagnostic; S10 quotes its numbers).

Needs a library built with the trace stamps compiled in (they compile to nothing otherwise):

    SX_NVCC_FLAGS=-DSX_ATTN_TRACE python -m paper_2606_01751_b200.build --force
    python -m paper_2606_01751_b200.trace_attn C2            # or C3 / C4 / C5 [pair|single]
    python -m paper_2606_01751_b200.build --force            # back to the product build

It runs a sparse layer of the named config three times, copies the clock64() stamps of the first 2048 CTAs of the
last attention launch back (sx_attn.cu, SX_ATTN_TRACE block) and prints the median / p10 / p90 of every phase in SM
clocks, the CTA life, and the gap between a CTA's exit and the next CTA's entry on the same SM.
"""
from __future__ import annotations

import ctypes
import sys

import numpy as np
import torch

from . import binding as sx
from . import workloads as wl
from .layer import GpuLayer


def main(argv):
    cfg = argv[1] if len(argv) > 1 else "C2"
    form = argv[2] if len(argv) > 2 else None
    lib = sx.load()
    if not hasattr(lib, "sx_attn_trace_copy"):
        raise SystemExit("this libsparsex.so was built without -DSX_ATTN_TRACE (see the module docstring)")
    dev = torch.device("cuda")
    lay = wl.CONFIGS[cfg]()
    lt = wl.build_layer(lay, 0)
    g = GpuLayer(lay, lt, dev)
    g.cta_pair = None if form is None else (form == "pair")
    for _ in range(3):
        g.step_sparse()
    torch.cuda.synchronize()
    host = torch.zeros(2048 * 16, dtype=torch.int64)
    rc = lib.sx_attn_trace_copy(ctypes.c_void_p(host.data_ptr()))
    assert rc == 0, rc
    a = host.numpy().reshape(2048, 16)
    a = a[(a[:, 0] > 0) & (a[:, 13] > 0) & (a[:, 8] > 0) & (a[:, 6] > 0)]   # CTAs with rows; cluster rank 0 holds the issuer
    print("%s: %d CTAs traced, median %d key tiles" % (cfg, len(a), int(np.median(a[:, 13]))))
    phases = [("entry -> griddepcontrol.wait", a[:, 1] - a[:, 0]), ("wait -> lookups done", a[:, 2] - a[:, 1]),
              ("lookups -> after the meeting", a[:, 3] - a[:, 2]), ("wait -> first table entries (warp 8)", a[:, 4] - a[:, 1]),
              ("issue of Q + key tile 0 (warp 8)", a[:, 5] - a[:, 4]), ("meeting -> Q landed (issuer)", a[:, 6] - a[:, 3]),
              ("Q landed -> K(0) landed", a[:, 7] - a[:, 6]), ("K(0) landed -> first S tile", a[:, 8] - a[:, 7]),
              ("first S -> key loop done", a[:, 9] - a[:, 8]), ("loop done -> output stored", a[:, 10] - a[:, 9]),
              ("stored -> exit", a[:, 11] - a[:, 10]), ("entry -> first S", a[:, 8] - a[:, 0]),
              ("loop done -> exit", a[:, 11] - a[:, 9]), ("CTA life", a[:, 11] - a[:, 0])]
    for name, v in phases:
        print("  %-38s median %8.0f   p10 %8.0f   p90 %8.0f clk" % (name, np.median(v), np.percentile(v, 10),
                                                                    np.percentile(v, 90)))
    by_sm = {}
    for row in a:
        by_sm.setdefault(int(row[12]), []).append((row[0], row[11]))
    gaps = []
    for lst in by_sm.values():
        lst.sort()
        gaps += [e1 - x0 for (_, x0), (e1, _) in zip(lst[:-1], lst[1:])]
    if gaps:
        print("  %-38s median %8.0f   p10 %8.0f   p90 %8.0f clk" % ("exit -> next CTA's entry on the SM", np.median(gaps),
                                                                    np.percentile(gaps, 10), np.percentile(gaps, 90)))


if __name__ == "__main__":
    main(sys.argv)
