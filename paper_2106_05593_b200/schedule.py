"""Drive a workload's field / temperature schedule (BASELINE.json's configs 2, 3, 5 and the Fe film) through the library.

    python -m paper_2106_05593_b200.schedule --config 2 [--relax] [--shape nx,ny[,nz]]

Every schedule entry is (kind, value, n_sweeps) with kind "B" (applied field, tesla) or "T" (uniform temperature, kelvin).
With --relax a field step uses mmc_relax (the chunked convergence of PAPER.md:135, chunk = n_sweeps) instead of a fixed
number of iterations.  Prints one line per step: the value, the running means of the step and the acceptance rate.
Host-side orchestration only: every iteration runs in the CUDA library.
"""
from __future__ import annotations

import argparse
import sys


def run_schedule(sim, wl, relax=False, threshold=0.01, max_chunks=20, out=None):
    """Run wl.schedule on `sim` (an MMC context already configured with the workload).  Returns a list of dicts."""
    import numpy as np
    rows = []
    for kind, value, n in wl.schedule:
        if kind == "B":
            sim.set_field(*value)
        elif kind == "T":
            sim.set_temperature(float(value))
        else:
            raise ValueError(f"unknown schedule entry {kind!r}")
        sim.reset_counters()
        if relax and kind == "B" and any(value):
            r = sim.relax(value, chunk_sweeps=n, min_chunks=2, max_chunks=max_chunks, threshold=threshold)
            ob = sim.observables()
            row = dict(kind=kind, value=value, sweeps=int(r["sweeps"]), mean_m=r["mean_m"], mean_len=r["mean_len"],
                       chunks=r["chunks_done"], converged=r["converged"])
        else:
            sim.reset_averages()
            sim.sweep(n)
            ob = sim.observables()
            row = dict(kind=kind, value=value, sweeps=n, mean_m=ob["run_mean_m"], mean_len=ob["run_mean_len"], chunks=1, converged=True)
        row["acceptance"] = ob["accepted"] / max(1, ob["trials"])
        row["cone_deg"] = ob["cone_deg"]
        rows.append(row)
        if out is not None:
            v = value if kind == "T" else "(%.4g, %.4g, %.4g)" % tuple(value)
            print(f"{kind} {v}  sweeps {row['sweeps']:6d}  <m> = ({row['mean_m'][0]:+.5f}, {row['mean_m'][1]:+.5f}, {row['mean_m'][2]:+.5f})"
                  f"  <|m|> = {row['mean_len']:.5f}  acc = {row['acceptance']:.3f}  cone = {row['cone_deg']:.0f}", file=out)
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--relax", action="store_true")
    ap.add_argument("--shape", default=None)
    args = ap.parse_args()
    import paper_2106_05593_b200 as P
    import workloads as W
    kw = {}
    if args.shape:
        d = [int(x) for x in args.shape.split(",")]
        kw = dict(nx=d[0], ny=d[1])
        if len(d) > 2:
            kw["nz"] = d[2]
    wl = W.make(args.config, **kw)
    sim = P.MMC(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.pbc_mask)
    W.configure(sim, wl, P.Material)
    run_schedule(sim, wl, relax=args.relax, out=sys.stdout)
    sim.close()


if __name__ == "__main__":
    main()
