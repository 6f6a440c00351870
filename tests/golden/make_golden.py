"""Writes tests/golden/oracle_cfg0_scan.txt from the CPU oracle alone (never the CUDA path): see README.md here."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "..", ".."))

import oracle                                           # noqa: E402
from paper_1908_01949_b200 import synth                 # noqa: E402  (seeded input generator only)

N_SAMPLE, KEY = 64, 2024


def compute():
    cfg = synth.CONFIGS[0]
    geom = synth.make_geometry(); field = synth.make_uniform_field()
    ev = synth.generate_events(cfg, geom, field, 1)[0]
    grid = synth.truth_anchored_grid(ev.seed, cfg.grid_n)[0]
    sel = synth.stratified_seed_sample(grid.n_seeds, N_SAMPLE, key=KEY)
    params = dict(h=cfg.h_mm, max_steps=cfg.max_steps, window=cfg.window_mm)
    bound = oracle.Bound(geom, field, params)
    out = oracle.scan(bound, ev.wire_id, ev.drift_mm, grid, index_list=sel)
    k, S = oracle.argmax(out["n_match"], out["chi2"], cfg.window_mm)
    best = int(sel[k])
    lab, _ = oracle.labels(bound, ev.wire_id, ev.drift_mm, oracle.seed_of_index(grid, best))
    lines = ["# configs[0], event 0, %d stratified seeds (key %d): index n_match chi2(hex double) n_steps" % (N_SAMPLE, KEY)]
    for i, s in enumerate(sel):
        lines.append("%d %d %s %d" % (int(s), int(out["n_match"][i]), float(out["chi2"][i]).hex(), int(out["n_steps"][i])))
    lines.append("best %d %s" % (best, float(S).hex()))
    lines.append("labels " + " ".join(str(int(v)) for v in lab))
    return "\n".join(lines) + "\n"


if __name__ == "__main__":
    with open(os.path.join(HERE, "oracle_cfg0_scan.txt"), "w") as f:
        f.write(compute())
    print("written")
