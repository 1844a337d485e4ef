#!/usr/bin/env python
"""Writes tests/golden/carve_<cfg>.txt: the top-k margin carve (readings A9/A10) of the FULL-SIZE
seeded workloads C2..C5, layer 0, so that the full-size GPU parity tests replay it instead of iterating
the fp64 oracle (minutes per config). Calls only oracle/ (through tests/helpers.py) and the seeded input
generator; nothing here touches the CUDA path.

    python tests/golden/make_carve.py [C2 C3 C4 C5 C3_L3]

Each line: physical block, row in block, scale applied to that key row (all KV heads), in application order.
C3_L3: the margin of the BOUNDARY-layer selection of C3 in paper mode (layer index 3, readings A11/A16): that
selection reads a pool whose keys are all fresh, so the carve rescales rows of K_fresh of layer 3; each line is
batch token index, scale (helpers.carve_margins_fresh / apply_carve_fresh).
"""
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from helpers import carve_margins, carve_margins_fresh, oracle_scores_full_layer  # noqa: E402
from oracle import sx_oracle as orc  # noqa: E402
from paper_2606_01751_b200 import workloads as wl  # noqa: E402


def main():
    for name in (sys.argv[1:] or ["C2", "C3", "C4", "C5", "C3_L3"]):
        t0 = time.time()
        if name == "C3_L3":
            lay = wl.CONFIGS["C3"]()
            lt = wl.build_layer(lay, 3)
            log = []
            hist = carve_margins_fresh(lay, lt, log=log)
            with open(os.path.join(HERE, "carve_C3_L3.txt"), "w") as f:
                f.write("# margin carve of the boundary-layer selection: workloads.CONFIGS['C3'](), layer 3, K_fresh rows, "
                        "tau = 1e-3; band sizes per iteration %r\n" % (hist,))
                f.write("# written by tests/golden/make_carve.py (fp64 oracle only); columns: batch token index, scale\n")
                for tok, scale in log:
                    f.write("%d %.2f\n" % (tok, scale))
            # the recompute set the oracle selects on the carved boundary layer (R = I_nr U S_key, Alg. 1 l.537-539):
            # bench.py's CPU legs scale the oracle's sparse-attention time by sum_{r in R} (r + 1) of THIS set
            s = oracle_scores_full_layer(lay, lt)[0]
            sel, rows = orc.select_topk(s, lay.is_new_mask(0), int(lay.k_per_req[0]), lay.cached_mask(0))
            with open(os.path.join(HERE, "rows_C3_L3.txt"), "w") as f:
                f.write("# R = I_nr U S_key of the boundary-layer selection of C3 (layer 3, carved by carve_C3_L3.txt), "
                        "fp64 oracle; %d rows, k = %d\n" % (len(rows), len(sel)))
                f.write("# written by tests/golden/make_carve.py (fp64 oracle only); one position per line\n")
                f.write("\n".join(str(int(r)) for r in rows) + "\n")
            print(name, hist, len(log), "ops, %d rows, %.0f s" % (len(rows), time.time() - t0), flush=True)
            continue
        lay = wl.CONFIGS[name]()
        lt = wl.build_layer(lay, 0)
        log = []
        # C4: rows shared by several requests whose cuts fall in the same segment need more, wider rounds
        hist = carve_margins(lay, lt, log=log, max_iter=40, widen_later=3.0 if name == "C4" else 1.5)
        with open(os.path.join(HERE, "carve_%s.txt" % name), "w") as f:
            f.write("# margin carve of workloads.CONFIGS[%r](), layer 0, tau = 1e-3; band sizes per iteration %r\n"
                    % (name, hist))
            f.write("# written by tests/golden/make_carve.py (fp64 oracle only); columns: block row scale\n")
            for blk, row, scale in log:
                f.write("%d %d %.2f\n" % (blk, row, scale))
        print(name, hist, len(log), "ops, %.0f s" % (time.time() - t0), flush=True)


if __name__ == "__main__":
    main()
