"""Run one of BASELINE.json's five configurations end to end through the C ABI and print one JSON line per
diagnostic output (xi, <v^2>, bound-state fraction, Gauss residual, ...), then a summary line with the timing.

    python -m paper_2208_01525_b200.run_config --config 5 [--size N] [--variant V] [--segments]

Schedules (readings R-3, R-11, R-19): tau0 = 1, dtau = 0.1, dx = 0.5, lambda = 2, e = 1,
sigma = 1, kappa = 0.9; the damping prephase is 200 steps with friction 0.5.  `--size` overrides the lattice size
(the step counts stay those of the config, capped at the half light-crossing time of the smaller box).
"""
from __future__ import annotations

import argparse
import json
import time

from . import Lattice, Params

DX, DTAU, TAU0 = 0.5, 0.1, 1.0
CONFIGS = {
    # N, era m, s, tau_norm (None: tau_end), prephase steps, main steps, init kind, diagnostics every
    1: dict(N=64, m=0.5, s=1.0, tau_norm=1.0, pre=0, steps=32, kind=0, every=32),
    2: dict(N=256, m=0.5, s=-1.0, tau_norm=1.0, pre=200, steps=1000, kind=0, every=20),
    3: dict(N=512, m=2.0 / 3.0, s=1.0, tau_norm=None, pre=0, steps=1270, kind=1, every=50),
    4: dict(N=768, m=0.5, s=0.0, tau_norm=1.0, pre=0, steps=1910, kind=0, every=100),
    5: dict(N=1024, m=0.5, s=1.0, tau_norm=None, pre=200, steps=2350, kind=0, every=100),
}
KEYS = ("tau", "a", "xi_W", "xi_p", "xi_q", "xi_pq", "xi_L", "v2_L", "v2_pq", "f_total", "f_p", "L_pq", "L_pq_tol",
        "sumW_p", "sumW_q", "cells_pq", "maxW", "energy")


def run(config: int, size: int | None = None, variant: int = 0, segments: bool = False, device: str = "cuda:0",
        emit=print, aux: bool = True):
    import torch
    c = dict(CONFIGS[config])
    N = size or c["N"]
    total = c["pre"] + c["steps"]
    if size and size < c["N"]:                       # stop at the half light-crossing time of the smaller box
        total = min(total, int((N * DX / 2 - TAU0) / DTAU))
    tau_end = TAU0 + total * DTAU
    tau_norm = c["tau_norm"] if c["tau_norm"] is not None else tau_end
    lat = Lattice(N, device=device)
    if aux:                                          # second momentum buffer: two steps per pass (same bits, faster)
        try:
            lat.set_aux(True)
        except Exception:
            pass
    prm = Params(init_kind=c["kind"], tau_norm=tau_norm, friction=0.5 if c["pre"] else 1.0, kernel_variant=variant)
    lat.init_fields(config, DX, prm)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    done, tau, t_diag = 0, TAU0, 0.0
    while done < total:
        if c["pre"] and done == c["pre"]:
            prm.friction = 1.0
            lat.set_params(prm)
        stop = c["pre"] if done < c["pre"] else total
        n = min(c["every"] - done % c["every"], stop - done)
        lat.step(n, tau, c["m"], c["s"])
        done += n
        tau = TAU0 + done * DTAU
        if done % c["every"] == 0 or done == total:
            torch.cuda.synchronize()
            td = time.perf_counter()
            d = lat.diagnostics()                 # one sweep: windings, cells, sums AND the Gauss-law norms
            row = {k: d[k] for k in KEYS}
            row.update(step=done, prephase=done <= c["pre"] and c["pre"] > 0, gauss_rel_p=d["gauss_rel_p"],
                       gauss_rel_q=d["gauss_rel_q"], gauss_max_p=d["gauss_max_p"], max_theta=d["max_theta"])
            if segments:
                row["segments"] = lat.pq_segments(8, True)
            t_diag += time.perf_counter() - td
            emit(json.dumps(row))
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    summary = {"config": config, "N": N, "steps": total, "tau_end": tau_end, "kernel_variant": variant,
               "wall_s": wall, "diagnostics_s": t_diag, "site_updates_per_s": N ** 3 * total / wall,
               "launches": lat.launch_count()}
    emit(json.dumps({"summary": summary}))
    return summary


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--config", type=int, default=1, choices=sorted(CONFIGS))
    ap.add_argument("--size", type=int, default=None)
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--no-aux", action="store_true", help="one step per pass (no second momentum buffer)")
    ap.add_argument("--segments", action="store_true", help="also label the pq segments (min 8 cells, one-cell tolerance)")
    a = ap.parse_args()
    run(a.config, a.size, a.variant, a.segments, aux=not a.no_aux)


if __name__ == "__main__":
    main()
