"""Per-block timeline of the TMA stage kernels (profiling aid, not part of the product path).

    python -m paper_2603_03706_b200.probe [cfg3|cfg4|cfg5] [--steps K] [--json OUT]

Builds the profiling variant of the library (-DCAVMAG_PROBE -> libcavmag_probe.so, see build.build_probe), runs K adaptive
steps of the workload through the device-side WHILE graph and prints, for the stage kernels of the LAST step, when the
blocks entered, had their control data, saw the first tile, left the main loop and exited (microseconds from the first
block's entry, %globaltimer), and for the block that ran stage_finish its phases in SM cycles (clock64).
Numbers of this build are not bench values: the marks add a few global stores per block.
"""
from __future__ import annotations

import argparse
import ctypes as C
import json
import math
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SLOTS = 32          # per block: [0..15] %globaltimer ns, [16..31] clock64, by mark index
MARKS = {0: "entry", 1: "control data ready (consumers)", 2: "first tile acquired", 3: "main loop done",
         4: "ticket (stages 1, 7)", 5: "exit", 6: "producer: all loads issued", 13: "producer: dependency wait returned",
         15: "consumers: dependency wait returned", 9: "deferred finish: own loads landed",
         10: "deferred finish: all loads in smem"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("workload", nargs="?", default="cfg3")
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--json", default="")
    args = ap.parse_args()

    from paper_2603_03706_b200 import build
    os.environ["CAVMAG_LIB"] = build.build_probe()
    import numpy as np
    import cavmag_workloads as W
    from paper_2603_03706_b200 import api

    w = W.by_name(args.workload, dtype=np.float32) if args.workload in ("cfg3", "cfg5") else W.by_name(args.workload)
    with api.Sim(w, precision="f32") as sim:
        h = sim.h
        api.cav_run_steps(h, math.inf, tol=w.tol, max_steps=40)           # dt settles
        api.cav_run_steps(h, math.inf, tol=w.tol, max_steps=args.steps)
        api.cav_sync(h)
        buf = np.zeros(8 * 256 * SLOTS, dtype=np.uint64)
        tg = C.c_int(0)
        api._lib.cav_debug_probe(h, buf.ctypes.data_as(C.c_void_p), C.byref(tg))
    tg = tg.value
    P = buf[:8 * tg * SLOTS].reshape(8, tg, SLOTS).astype(np.int64)

    out = {"workload": args.workload, "blocks": tg, "unit": "us from the first block's entry (min, median, max over blocks)"}
    prev_end = None
    for st in range(2, 8):
        g, c = P[st, :, :16], P[st, :, 16:]
        t0 = g[:, 0].min()

        def mmm(col):
            v = (g[:, col] - t0) / 1e3
            return [round(float(x), 2) for x in np.percentile(v, [0, 50, 100])]

        d = {MARKS[k]: mmm(k) for k in ((0, 15, 13, 9, 10, 1, 2, 6, 3, 5) if st >= 3 else (0, 15, 1, 2, 6, 3, 5))}
        d["main loop, median us"] = round(float(np.median(g[:, 3] - g[:, 2]) / 1e3), 2)
        d["main loop, slowest / median"] = round(float((g[:, 3] - g[:, 2]).max() / np.median(g[:, 3] - g[:, 2])), 3)
        if st == 7:
            last = int(np.argmax(g[:, 7]))
            d["stage_finish: block"] = last
            d["stage_finish: ticket -> entry, loads, arithmetic, write-back, graph condition (SM cycles)"] = [
                int(c[last, 8] - c[last, 4]), int(c[last, 9] - c[last, 8]), int(c[last, 10] - c[last, 9]),
                int(c[last, 11] - c[last, 10]), int(c[last, 12] - c[last, 11])]
            d["stage_finish: ticket -> exit, us"] = round(float((g[last, 5] - g[last, 4]) / 1e3), 2)
        d["kernel end -> next kernel's first entry, us"] = None if prev_end is None else round(float((t0 - prev_end) / 1e3), 2)
        prev_end = g[:, 5].max()
        out["stage %d" % st] = d
    txt = json.dumps(out, indent=1)
    print(txt)
    if args.json:
        with open(args.json, "w") as f:
            f.write(txt)


if __name__ == "__main__":
    main()
