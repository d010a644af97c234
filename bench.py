#!/usr/bin/env python
"""bench.py -- site-updates/s of the fused U(1)xU(1) leapfrog step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--size 1024] [--impl ours|reference]

Workload (config.workload): BASELINE.json config 5 -- 1024^3 periodic lattice, dx=0.5, dtau=0.1,
radiation era, s=1, lambda=2, e=1, eta=1, kappa=0.9, seeded uniform random-phase init, damped
prephase (friction 0.5, 200 steps), full diagnostics every 100 steps.  A "step" is one fused kick+drift launch
(SURVEY.md 8(a) rows a1-a5); the diagnostics sweep (a6-a10: one fused read-only pass + the tolerant overlap count)
runs inside the timed region after every 100th timed step and, when fewer than 100 steps are timed, once after the
last one, so that every run's `value` contains at least one sweep; `value_steps_only` and
`value_at_config_cadence` (one sweep per 100 steps) are reported beside it.  Inputs (the 129 GB state) are far
larger than L2.

One JSON line on stdout (rank 0).  N > 1: replicas only (independent seeds per GPU, no collective on the
data path), launched by torchrun, timed as the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "lattice site-updates/sec (full 2-field step)"
UNIT = "site-updates/s"
BYTES_PER_SITE_UPDATE = 160          # read 20 + write 20 fp32 words
DX, DTAU, TAU0, ERA, S = 0.5, 0.1, 1.0, 0.5, 1.0
DIAG_EVERY = 100
PREPHASE_STEPS = 200                 # 20 tau units of friction 0.5 (config 5)


def workload_name(n, prephase=PREPHASE_STEPS):
    return (f"{n}^3 periodic, dx=0.5, dtau=0.1, fp32, radiation era, s=1, lambda=2, e=1, eta=1, kappa=0.9, "
            f"uniform random-phase init (seed 5+rank), {prephase}-step friction-0.5 prephase, diagnostics every "
            f"{DIAG_EVERY} steps (BASELINE.json config 5)")


# what the measured DRAM traffic depends on: the sources of the step kernels
TRAFFIC_SOURCES = ("step_tiled.cu", "step_tb.cu", "step_site.cuh", "f32x2.cuh", "stage.cuh", "common.cuh")


def csrc_sha():
    """sha256 (16 hex digits) of the sources of the step kernel: profiles/traffic.json carries the hash it was measured on."""
    import hashlib
    h = hashlib.sha256()
    for f in TRAFFIC_SOURCES:
        with open(os.path.join(ROOT, "paper_2208_01525_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def measured_traffic(N, two_step):
    """DRAM bytes per launch of the step kernel (one step, or two steps per pass) from profiles/traffic.json, or None if
    that file was measured on other sources than the ones being timed (the number would be stale)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            t = json.load(f)
        return t.get(f"step_tb_{N}" if two_step else f"step_{N}") if t.get("csrc_sha") == csrc_sha() else None
    except Exception:
        return None


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.path = tempfile.mktemp(prefix="u1u1_clocks_", suffix=".csv")
        self.proc = None
        self.gpu = gpu_index

    def start(self):
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            p = [t.strip() for t in line.split(",")]
            if len(p) < 9:
                continue
            try:
                sm.append(float(p[1])); mx.append(float(p[2]))
            except ValueError:
                continue
            for name, v in zip(names, p[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.path)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


def replica_seed(rank):
    """Replicas only: rank r evolves its own lattice from seed 5 + r."""
    return 5 + int(rank)


def max_over_ranks(values, dist, device):
    """Element-wise MAX of a list of floats over all ranks (identity when not distributed)."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_rate(world, steps, sites, ms):
    """Site-updates/s of the whole job: every rank advanced `sites` sites by `steps` steps in `ms` (max over ranks)."""
    return world * steps * sites / (ms * 1e-3)


def oracle_sample(n, steps, seed=5):
    """The oracle as it stands on an n^3 sample of the same workload; returns (site-updates/s, cores)."""
    from oracle import oracle as O
    s = O.init_random_phase(n, seed)
    K = O.Couplings()
    O.step(s, DX, K, TAU0, ERA, S, DTAU, tau_norm=256.0, friction=0.5, n=1)          # warm caches / page in
    t0 = time.perf_counter()
    O.step(s, DX, K, TAU0 + DTAU, ERA, S, DTAU, tau_norm=256.0, friction=0.5, n=steps)
    dt = time.perf_counter() - t0
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return n ** 3 * steps / dt, cores, dt


def run_reference(args):
    """--impl reference: the fp64 oracle on host cores (rank 0 only), bounded sample per step."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    n = 128
    from oracle import oracle as O
    s = O.init_random_phase(n, 5)
    K = O.Couplings()
    for k in range(args.warmup):
        O.step(s, DX, K, TAU0 + k * DTAU, ERA, S, DTAU, tau_norm=256.0, friction=0.5)
    t0 = time.perf_counter()
    for k in range(args.steps):
        O.step(s, DX, K, TAU0 + (args.warmup + k) * DTAU, ERA, S, DTAU, tau_norm=256.0, friction=0.5)
    dt = time.perf_counter() - t0
    value = n ** 3 * args.steps / dt
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    sample = f"{n}^3 sub-lattice of the workload per step (oracle fp64, gcc -O2, OpenMP over z-planes of the kick loops)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.size, args.prephase), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus > 1 and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs one rank per GPU: launch it as `python -m torch.distributed.run "
                         f"--nnodes=1 --nproc-per-node {args.gpus} --master-addr 127.0.0.1 --master-port P bench.py --gpus {args.gpus} ...` "
                         f"(WORLD_SIZE is {world})")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: CUDA device required (the library has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    from paper_2208_01525_b200 import Lattice, Params, build
    build.build()
    N = args.size
    V = N ** 3
    lat = Lattice(N, device=f"cuda:{local}")
    two_step = False
    if args.tb:
        # the second momentum buffer (43 GB at 1024^3, 172 + 11 GB in all): u1u1_step then takes two steps per pass
        try:
            lat.set_aux(True)
            two_step = True
        except Exception as e:          # not enough HBM: the one-step kernel
            print(f"bench.py: aux buffer not available ({e}); one step per pass", file=sys.stderr)
    prm = Params(tau_norm=256.0, friction=0.5, kernel_variant=args.variant)
    lat.init_fields(replica_seed(rank), DX, prm)
    lat.step(args.prephase, TAU0, ERA, S)                    # damped prephase (config 5: 200 steps)
    prm.friction = 1.0
    lat.set_params(prm)
    tau = TAU0 + args.prephase * DTAU
    lat.step(args.warmup, tau, ERA, S)                       # W >= 3 untimed warm-up steps
    tau += args.warmup * DTAU
    lat.diagnostics()                                        # warm the diagnostic kernels too

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    clocks = ClockSampler(local)
    launches0 = lat.launch_count()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    t_start, t_end, segs, dsegs = ev(), ev(), [], []
    barrier()
    clocks.start()
    t_start.record()
    done, diag = 0, None
    while done < args.steps:
        n = min(DIAG_EVERY - (done % DIAG_EVERY), args.steps - done)
        e0, e1 = ev(), ev()
        e0.record(); lat.step(n, tau, ERA, S); e1.record()
        segs.append((e0, e1))
        tau += n * DTAU
        done += n
        if done % DIAG_EVERY == 0 or (done == args.steps and not dsegs):
            d0, d1 = ev(), ev()
            d0.record(); diag = lat.diagnostics(); d1.record()      # one sweep: windings, cells, sums, Gauss norms
            dsegs.append((d0, d1))
    t_end.record()
    barrier()
    clk = clocks.stop()
    launches = lat.launch_count() - launches0
    ms_total = t_start.elapsed_time(t_end)
    ms_steps = sum(a.elapsed_time(b) for a, b in segs)
    ms_diag = sum(a.elapsed_time(b) for a, b in dsegs) / len(dsegs)
    ms_total, ms_steps, ms_diag = max_over_ranks([ms_total, ms_steps, ms_diag], dist, f"cuda:{local}")
    value = whole_job_rate(world, args.steps, V, ms_total)
    kernel_ms = ms_steps / args.steps
    step_launches = launches - 4 * len(dsegs)                # a diagnostics call is 4 launches (sweep, fold, overlap, fold)
    steps_per_launch = args.steps / step_launches
    # Roofline of the dominant kernel, per LAUNCH: a launch reads the 20 words of every site once and writes them once
    # (160 B x V) whether it advances one step or two, so that is the least it can move and `frac` stays <= 1.  The rate
    # on SURVEY.md 8(d)'s one-step basis (160 B per site-UPDATE, which two steps per pass can exceed) is reported beside
    # it as `one_step_equivalent_GBs`.
    launch_ms = kernel_ms * steps_per_launch
    achieved = BYTES_PER_SITE_UPDATE * V / (launch_ms * 1e-3) / 1e9
    one_step_equiv = BYTES_PER_SITE_UPDATE * V / (kernel_ms * 1e-3) / 1e9
    peak, peak_src = measured_peak_gbs()
    traffic = measured_traffic(N, two_step)

    e2e = run_e2e(args, lat, tau, world, dist, local)

    if rank != 0:
        return
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_s, steps_s = 192, 8
        v, cores, dt = oracle_sample(n_s, steps_s)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{n_s}^3 sub-lattice of the workload, {steps_s} steps ({dt:.1f} s), fp64 oracle as it stands"}
    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "value_steps_only": whole_job_rate(world, args.steps, V, ms_steps),
        "value_at_config_cadence": whole_job_rate(world, DIAG_EVERY, V, DIAG_EVERY * kernel_ms + ms_diag),
        "diagnostics_ms": ms_diag,
        "config": {"workload": workload_name(N, args.prephase), "N": N, "state_GB": (160 if two_step else 120) * V / 1e9,
                   "l2_policy": "inputs (129 GB state + 43 GB second momentum buffer) far larger than the 126 MB L2; no flush needed",
                   "prephase_steps_before_timing": args.prephase, "diag_calls_in_timed_region": len(dsegs),
                   "diag_every": DIAG_EVERY, "diag_every_effective": args.steps / len(dsegs),
                   "kernel_variant": args.variant, "two_steps_per_pass": two_step,
                   "parallelism": "replicas" if world > 1 else "single"},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "traffic_csrc_sha": csrc_sha(), "peak_source": peak_src,
                     "kernel": ("two fused kick+drift steps per pass (step_tb_kernel): a launch moves every site's 20 words "
                                "through HBM once for two site-updates (80 B per site-update)") if two_step
                               else "fused kick+drift step (step_tiled_kernel)",
                     "kernel_ms": kernel_ms, "launch_ms": launch_ms, "steps_per_launch": steps_per_launch,
                     "bytes_per_site_per_launch": BYTES_PER_SITE_UPDATE,
                     "algorithmic_bytes_per_launch": BYTES_PER_SITE_UPDATE * V,
                     "bytes_per_site_update": BYTES_PER_SITE_UPDATE / steps_per_launch,
                     "dram_GBs": (traffic / (launch_ms * 1e-3) / 1e9) if traffic else None,
                     "dram_frac_of_peak": (traffic / (launch_ms * 1e-3) / 1e9 / peak) if traffic else None,
                     "frac_of_8TBs_spec": achieved / 8000.0,
                     "one_step_equivalent_GBs": one_step_equiv, "one_step_equivalent_frac": one_step_equiv / peak,
                     "one_step_equivalent_note": "160 B per site-UPDATE (SURVEY.md 8(d)): what a one-step-per-pass kernel "
                                                 "would have to move for the same site-updates/s; exceeds 1 with two steps per pass",
                     "diagnostics": {"kernel": "fused diagnostics sweep + tolerant overlap", "ms": ms_diag,
                                     "algorithmic_bytes": 80 * V, "achieved": 80 * V / (ms_diag * 1e-3) / 1e9,
                                     "frac": 80 * V / (ms_diag * 1e-3) / 1e9 / peak}},
        "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clk,
        "diagnostics": {"tau": diag["tau"], "xi_W": diag["xi_W"], "xi_L": diag["xi_L"], "v2_L": diag["v2_L"],
                        "f_total": diag["f_total"], "maxW": diag["maxW"], "max_theta": diag["max_theta"],
                        "gauss_rel_p": diag["gauss_rel_p"], "gauss_rel_q": diag["gauss_rel_q"]},
    }))


def run_e2e(args, lat, tau, world, dist, local):
    """Same metric through the C ABI with HOST buffers: import_state_host (H2D of the 80 B/site state from
    pinned memory) -> K steps -> diagnostics (D2H scalars) -> export_state_host (D2H), all timed.  One host
    checkpoint per K steps: the copies are PCIe-bound, so the figure scales with `steps_per_checkpoint`."""
    import torch
    V = args.size ** 3
    nbytes = 80 * V
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 0
    if args.no_e2e or avail < 1.4 * nbytes * max(1, world):
        return {"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                "note": f"skipped: needs {nbytes / 1e9:.0f} GB pinned host memory per rank, {avail / 1e9:.0f} GB available"}
    host = torch.empty(20 * V, dtype=torch.float32, pin_memory=True)
    lat.export_state_host(host)                              # untimed: a valid checkpoint in host memory
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t0, t1, t2, t3 = (torch.cuda.Event(enable_timing=True) for _ in range(4))
    t0.record()
    lat.import_state_host(host)
    t1.record()
    lat.step(args.steps, tau, ERA, S)
    lat.diagnostics()
    t2.record()
    lat.export_state_host(host)
    t3.record()
    torch.cuda.synchronize()
    ms, ms_h2d, ms_d2h = max_over_ranks([t0.elapsed_time(t3), t0.elapsed_time(t1), t2.elapsed_time(t3)], dist, f"cuda:{local}")
    del host
    return {"value": whole_job_rate(world, args.steps, V, ms), "unit": UNIT,
            "h2d_bytes_per_step": nbytes / args.steps, "d2h_bytes_per_step": (nbytes + 8 * 48) / args.steps,
            "steps_per_checkpoint": args.steps, "ms_total": ms, "h2d_ms": ms_h2d, "d2h_ms": ms_d2h,
            "h2d_GBs": nbytes / ms_h2d / 1e6, "d2h_GBs": nbytes / ms_d2h / 1e6,
            "note": "checkpoint in pinned host memory -> H2D -> K steps -> diagnostics -> D2H; relayout kernels overlap the PCIe copies"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--size", type=int, default=1024)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--prephase", type=int, default=PREPHASE_STEPS)
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--tb", type=int, default=1, help="1: second momentum buffer -> two steps per pass (step_tb.cu); 0: one-step kernel")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
