"""BASELINE.json configs[4]: per-GPU load sweep. Minkowski + seeded 1e-10 noise, periodic, block sizes 16^3 / 32^3 /
64^3, pack sizes from 8 blocks up to what fits the memory budget, 20 RK4 steps each; prints zone-cycles/s against
cells per GPU as a markdown table.

  python -m paper_2409_10383_b200.load_sweep [--budget-gb 120] [--steps 20]

The pack is filled on the device by tiling a 2x2x2-block (64^3: 1 block) seeded noise problem periodically, so host
memory never holds more than the small tile."""
from __future__ import annotations

import argparse
import ctypes as C
import json
from dataclasses import replace

import numpy as np

from . import build, inputs as I, z4c as Z

LATTICES = {16: [(2, 2, 2), (4, 4, 4), (8, 8, 8), (16, 16, 16), (24, 24, 24), (32, 32, 24)],
            32: [(2, 2, 2), (4, 4, 4), (8, 8, 8), (12, 12, 12), (16, 16, 12)],
            64: [(2, 2, 2), (4, 4, 4), (6, 6, 6), (8, 8, 8)]}


def bytes_needed(p) -> int:
    lib = Z.load_library()
    cp = Z.make_params(p)
    interior = I.NF * p.ncells * 8            # the tiled initial data, a temporary on the device
    return lib.z4c_state_bytes(C.byref(cp)) + lib.z4c_workspace_bytes(C.byref(cp)) + interior


def run_one(p, steps: int):
    import torch
    tile = (2, 2, 2)
    small = replace(p, nb=tile)
    base = torch.from_numpy(I.noise_data(small, 1000)).cuda()
    reps = (1, p.nb[2] // tile[2], p.nb[1] // tile[1], p.nb[0] // tile[0])
    u = base.repeat(*reps).contiguous()
    sim = Z.Z4c(p)
    sim.use_graph(True)
    sim.set_initial_data(u)
    del u
    sim.step(2)
    sim.sync()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(sim.stream)
    sim.step(steps)
    e1.record(sim.stream)
    sim.sync()
    ms = e0.elapsed_time(e1)
    dev = float(abs(sim.state[I.CHI, 0, 3:-3, 3:-3, 3:-3] - 1.0).max())
    sim.close()
    torch.cuda.empty_cache()
    return p.ncells * steps / (ms * 1e-3), ms / steps, dev


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--budget-gb", type=float, default=120.0)
    ap.add_argument("--steps", type=int, default=20)
    args = ap.parse_args()
    build.build()
    rows = []
    print("| n | blocks | cells per GPU | device GB | ms/step | zone-cycles/s | max |chi-1| |")
    print("|---|---|---|---|---|---|---|")
    for n, lats in LATTICES.items():
        for nb in lats:
            p = I.params_noise(n, nb, 0.1)
            gb = bytes_needed(p) / 1e9
            if gb > args.budget_gb:
                continue
            zcps, ms, dev = run_one(p, args.steps)
            rows.append({"n": n, "nb": nb, "cells": p.ncells, "gb": gb, "ms_per_step": ms, "zcps": zcps})
            print(f"| {n} | {nb[0]}x{nb[1]}x{nb[2]} = {p.nblocks} | {p.ncells:.3e} | {gb:.1f} | {ms:.3f} | {zcps:.3e} | {dev:.1e} |",
                  flush=True)
    print(json.dumps(rows))


if __name__ == "__main__":
    main()
