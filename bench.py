#!/usr/bin/env python
"""bench.py -- whole-step throughput of the PM2D hot path on B200 (contract in the build brief).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c3] [--impl reference]

One "step" = one pass of the whole hot path (field update, 2 Poisson solves, 2 force grids, fused
gather-push-deposit stage A and B for every mobile species, periodic rebin) over the resident
particle set.  N = 1 workload: BASELINE.json configs[2], the 8192x4096 SRS-scale slab the
north_star target is quoted on (134 M electrons + 33.5 M deuterium ions, sine shape).  N > 1: the
path does not shard without the paper's domain decomposition (out of scope: "only one GPU is
used"), so every rank runs an independent replica -- weak scaling, no collective on the data path.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import pm2d_inputs as I  # noqa: E402

BYTES_STAGE_A = 28   # read x, y, ux, uy, w (20 B), write u^ (8 B)            -- DESIGN.md section 7
BYTES_STAGE_B = 44   # read x, y, ux, uy, w, u^ (28 B), write x, y, ux, uy (16 B)


def job_throughput(units_per_rank, steps, ms_local, world=1, device=None):
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's device time
    (max over ranks; the path does not shard, so ranks are independent replicas)."""
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    return units_per_rank * world * steps / (ms_max * 1e-3), ms_max


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def run(self):
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(self.rows))


def time_oracle(cfg, steps, warmup):
    """The CPU oracle as it stands (single thread, double precision) on a reduced copy of the workload."""
    import oracle
    oracle.build()
    orc, parts = oracle.from_config(cfg)
    nmob = sum(len(p["ix"]) for s, p in enumerate(parts) if p is not None and cfg["species"][s]["mobile"])
    orc.step(warmup)
    t0 = time.perf_counter()
    orc.step(steps)
    dt = time.perf_counter() - t0
    return nmob * steps / dt, dt / steps, nmob


def _oracle_worker(job):
    name, nx, ny, steps, warmup = job
    sys.path.insert(0, ROOT)
    return time_oracle(I.config(name, nx=nx, ny=ny), steps, warmup)


def time_oracle_all_cores(name, nx, ny, steps, warmup):
    """The same oracle, unchanged and single-threaded, as one independent copy of the sample per host core (the path has
    no shared state between independent problems): aggregate particle-steps/s over the slowest copy, and the copies run."""
    import multiprocessing as mp
    n = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    pool = mp.get_context("spawn").Pool(n)
    try:                                   # bounded: a worker that dies or stalls must not hold the bench line back
        res = pool.map_async(_oracle_worker, [(name, nx, ny, steps, warmup)] * n).get(timeout=300)
    finally:
        pool.terminate()
        pool.join()
    sec = max(r[1] for r in res)
    return sum(r[2] for r in res) / sec, n, sec


def sample_config(name, nx, ny):
    return I.config(name, nx=nx, ny=ny)


def workload_name(name, full_cfg, nmob=None):
    """config.workload of both arms: the full-size workload, whatever sample of it a CPU arm times."""
    g = full_cfg["grid"]
    if nmob is None:                      # the CPU arm: counted by the oracle's loader
        import oracle.loader as L
        nmob = sum(L.n_particles(full_cfg, s) for s, sp in enumerate(full_cfg["species"]) if sp["mobile"])
    src = (f"(BASELINE.json configs[{int(name[1]) - 1}])" if not name.startswith("cbet") else
           "(SURVEY 8f.1: the paper's CBET set-up P:L380, two beams at +-15 deg, particle step = 5 wave steps"
           + (", true vacuum margins P:L81)" if name == "cbet_vac" else ")"))
    return f"{name}: {g['nx']}x{g['ny']} cells, {nmob} mobile particles per GPU {src}"


def run_reference(args):
    """--impl reference: the oracle on host cores, same metric/config keys; each step is a bounded
    sample (a 512x256 copy of the workload: same dx, dt, particles per cell, profile, species, laser)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = sample_config(args.config, 512, 256)
    value, sec_per_step, nmob = time_oracle(cfg, args.steps, args.warmup)
    g = I.config(args.config)["grid"]
    line = dict(impl="reference", metric="particle-steps/s", value=value, unit="particle-steps/s", n_gpus=args.gpus,
                steps=args.steps, warmup=args.warmup, ms_per_step=sec_per_step * 1e3, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=workload_name(args.config, I.config(args.config)),
                            sample=f"{cfg['name']} reduced copy, {nmob} mobile particles"),
                cpu_baseline=dict(value=value, unit="particle-steps/s", cores=1, nproc=os.cpu_count(), kind="oracle",
                                  sample=f"{cfg['name']}: {nmob} mobile particles x {args.steps} steps"),
                e2e=dict(value=value, unit="particle-steps/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    if args.all_cores:      # opt-in here (the reference arm is one core by contract); the CUDA arm reports it by default
        va, nc, sa = time_oracle_all_cores(args.config, 512, 256, args.steps, args.warmup)
        line["cpu_baseline"]["all_cores"] = dict(value=va, unit="particle-steps/s", cores=nc,
                                                 how=f"{nc} independent copies of the sample, one per core, {sa * args.steps:.1f} s for the slowest")
    print(json.dumps(line))


def run_cuda(args):
    import torch
    import torch.distributed as dist

    import paper_2404_14293_b200 as pkg
    from paper_2404_14293_b200 import build
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if rank == 0:
        build.build()
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
        dist.barrier()
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    cfg = I.config(args.config)
    cfg["seed"] = int(cfg["seed"]) + 1000 * rank          # independent replicas
    g = cfg["grid"]
    order = {"auto": pkg.ORDER_AUTO, "cellmajor": pkg.ORDER_CELL_MAJOR, "layered": pkg.ORDER_LAYERED, "random": pkg.ORDER_RANDOM}[args.order]
    sim = pkg.PM2D(cfg, device=f"cuda:{local}", eager_moments=args.eager, rebin_every=args.rebin_every, particle_order=order)
    nmob = sum(sim.particle_count(s) for s, sp in enumerate(cfg["species"]) if sp["mobile"])
    nodes = (g["nx"] + 1) * g["ny"]

    # The loader's order holds exactly ppc particles in every cell; a run lives in the thermally mixed order that the
    # rebin leaves.  One rebin period is evolved before the warm-up so that the timed steps see that steady state.
    preroll = sim.grid.rebin_every if (sim.grid.rebin_every > 0 and args.order != "random") else 0
    sim.step(preroll)
    # ---- device-timed region: K steps, inputs resident in HBM ---------------------------------
    sim.step(args.warmup)
    sim.stray_count()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    sim.profile_enable(True)
    l0 = sim.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sim.step_async(args.steps)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = sim.launch_count() - l0
    prof = sim.profile_get()
    sim.profile_enable(False)
    clocks = sampler.stop() if sampler else None
    strays = sim.stray_count()
    value, ms_max = job_throughput(nmob, args.steps, ms, world, dev)

    # ---- end to end through the C ABI with host buffers: per step the host sends the laser table
    # (H2D, kernel arguments) and reads back the left-boundary probe column of a ----------
    probe = np.empty((1, g["ny"]), np.float32)
    lasers = cfg["lasers"]
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        sim.set_lasers(lasers)
        sim.step(1)
        sim.get_fields(pkg.FIELD_A, 0, 0, window=(0, 1, 0, g["ny"]), out=probe)
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    e2e_value, _ = job_throughput(nmob, args.steps, e2e_s * 1e3, world, dev)

    if rank == 0:
        peak, peak_src = hbm_peak()
        steps_p = max(prof["steps"], 1)
        stage_ms = (prof["ms"]["stage_a"] + prof["ms"]["stage_b"]) / steps_p
        per_particle = BYTES_STAGE_A + BYTES_STAGE_B + (8 if args.order == "random" else 0)   # random order: + the tile index, read at both stages
        # SURVEY 8(d)'s strict minimum: state read at both stages, written once = 56 B; 48 B where the weights are one
        # constant (c1: uniform profile without y taper is still tapered in x, so only the number-weighted c5 qualifies)
        uniform_w = all(sp["load"] == I.NUMBER_WEIGHTED for sp in cfg["species"] if sp["mobile"])
        min_bytes = 48 if uniform_w else 56
        alg_bytes = per_particle * nmob
        achieved = alg_bytes / (stage_ms * 1e-3) / 1e9 if stage_ms > 0 else 0.0
        achieved_min = min_bytes * nmob / (stage_ms * 1e-3) / 1e9 if stage_ms > 0 else 0.0
        # measured DRAM bytes of the stage launches of one step (ncu --set full), valid for the build that was profiled only
        traffic, traffic_src = None, None
        tp = os.path.join(ROOT, "profiles", "stage_traffic_bytes.txt")
        if os.path.exists(tp) and args.config == "c3" and world == 1 and args.order == "auto":
            try:
                # bytes, hash of the stage kernel's sources at the time of the capture, the profile that holds the capture
                from paper_2404_14293_b200.build import stage_id
                tok = open(tp).read().split()
                if tok[1] == stage_id():
                    traffic, traffic_src = float(tok[0]), f"{tok[2]} (ncu --set full, stage-kernel sources {tok[1]})"
                else:
                    traffic_src = f"stale: {tok[2]} was captured on stage-kernel sources {tok[1]}, these are {stage_id()}"
            except Exception:
                traffic = None
        line = dict(metric="particle-steps/s", value=value, unit="particle-steps/s", n_gpus=world, steps=args.steps,
                    warmup=args.warmup, ms_per_step=ms_max / args.steps, higher_is_better=True, scaling="weak",
                    vs_baseline=None, dtype="f32", data="synthetic",
                    config=dict(workload=workload_name(args.config, cfg, nmob),
                                shapes=[["cic", "tsc", "sine"][sp["shape"]] for sp in cfg["species"] if sp["mobile"]],
                                eager_moments=bool(args.eager), subcycle=int(g.get("subcycle", 1)), bc_y=("absorbing" if g.get("bc_y", 0) else "periodic"), rebin_every=sim.grid.rebin_every, particle_order=args.order, preroll_steps=preroll,
                                l2="inputs larger than L2 (particle state %.1f GB, grids %.1f GB)" % (nmob * 28 / 1e9, nodes * 60 / 1e9),
                                parallelism="replicas only" if world > 1 else "1 GPU",
                                **({"particles_note": "BASELINE.json asks for 1.0e9; the x edge taper (Q9) of the number-weighted loading leaves 9.44e8"} if args.config == "c5" else {})),
                    ns_per_particle_step=1e9 / value * world,
                    cell_updates_per_s=nodes * g["ncomp"] * max(int(g.get("subcycle", 1)), 1) * world * args.steps / (ms_max * 1e-3),
                    field_kernel_node_updates_per_s=(nodes * g["ncomp"] * max(int(g.get("subcycle", 1)), 1) / (prof["ms"]["field"] / steps_p * 1e-3)) if prof["ms"]["field"] > 0 else None,
                    phases_ms_per_step={k: v / steps_p for k, v in prof["ms"].items()},
                    stray_fraction=strays / max(2.0 * nmob * args.steps, 1.0),
                    clocks=clocks, gpu_launches=int(launches),
                    e2e=dict(value=e2e_value, unit="particle-steps/s",
                             h2d_bytes_per_step=int(len(lasers) * 48), d2h_bytes_per_step=int(g["ny"] * 4 + 16)),
                    rebin_share=(prof["ms"]["rebin"] / steps_p) / (ms_max / args.steps),
                    roofline=dict(bound="hbm", kernel="k_stage_lanes / k_stage (fused gather-push-deposit; per step: stage A + stage B launches of every mobile species)",
                                  achieved=achieved, peak=peak, unit="GB/s", frac=achieved / peak, peak_source=peak_src,
                                  frac_basis=f"{per_particle} B per particle-step (the layout: stage A 28 + stage B 44)",
                                  algorithmic_bytes_per_particle_step=per_particle,
                                  frac_min_bytes=achieved_min / peak, min_bytes_per_particle_step=min_bytes,
                                  ms_per_step=stage_ms, traffic=traffic, traffic_source=traffic_src))
        if world == 1 and not args.no_cpu_baseline:
            # about 10-30 s of CPU work: c5 holds ~56 particles per cell, so its sample is a smaller box
            snx, sny = (256, 256) if args.config == "c5" else (1024, 512)
            scfg = sample_config(args.config, snx, sny)
            v, sec, n = time_oracle(scfg, 8, 1)
            line["cpu_baseline"] = dict(value=v, unit="particle-steps/s", cores=1, nproc=os.cpu_count(), kind="oracle",
                                        sample=f"{scfg['name']} reduced copy of the workload: {n} mobile particles x 8 steps ({sec * 8:.1f} s)")
            if not args.no_all_cores:
                try:      # S§8d: the oracle on every host core (one independent copy of the sample each; the oracle itself stays single-threaded)
                    va, nc, sa = time_oracle_all_cores(args.config, snx, sny, 8, 1)
                    line["cpu_baseline"]["all_cores"] = dict(value=va, unit="particle-steps/s", cores=nc,
                                                             how=f"{nc} independent copies of the sample, one per core, {sa * 8:.1f} s for the slowest")
                except Exception as e:      # a reported baseline, never a reason to lose the line
                    line["cpu_baseline"]["all_cores"] = dict(value=None, error=str(e)[:200])
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=96,
                    help="timed steps; the default spans six rebin periods of c3 (0.7 s: several clock samples, the rebin at its long-run share)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--no-all-cores", action="store_true", help="skip the all-core leg of cpu_baseline")
    ap.add_argument("--all-cores", action="store_true", help="--impl reference: add cpu_baseline.all_cores")
    ap.add_argument("--config", default="c3", choices=["c1", "c2", "c3", "c4", "c5", "cbet", "cbet_vac"])
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--eager", type=int, default=1, help="1: deposit n, Px, Py at both stages (paper's flow); 0: n only")
    ap.add_argument("--rebin-every", type=int, default=None)
    ap.add_argument("--order", default="auto", choices=["auto", "cellmajor", "layered", "random"],
                    help="particle storage order; random = BASELINE config 5 run A (no tile staging, global atomics, no rebin)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--selftest-cpu", action="store_true", help=argparse.SUPPRESS)   # the rank plumbing alone, gloo, no GPU (tests)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    worker = run_reference if args.impl == "reference" else (run_selftest_cpu if args.selftest_cpu else run_cuda)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        spawn_ranks(args, worker)      # not under torchrun: start the N local ranks here
    else:
        worker(args)


def _rank_entry(rank, args, worker, port):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(args.gpus), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    worker(args)


def spawn_ranks(args, worker):
    """`python bench.py --gpus N` without torchrun: one process per GPU on this node, the same environment torchrun
    would set (replicas only: the ranks meet in the barrier and the MAX over their device times)."""
    import socket

    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    mp.spawn(_rank_entry, args=(args, worker, port), nprocs=args.gpus, join=True)


def run_selftest_cpu(args):
    """The multi-rank plumbing of run_cuda with the device work replaced by a fixed per-rank time (gloo, CPU): what the
    world_size-2 test drives through the spawn entry."""
    import torch.distributed as dist
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo", rank=rank, world_size=world)
    value, ms_max = job_throughput(1000, args.steps, 10.0 + rank, world, None)
    if rank == 0:
        print(json.dumps(dict(metric="particle-steps/s", value=value, unit="particle-steps/s", n_gpus=world, steps=args.steps,
                              warmup=args.warmup, ms_per_step=ms_max / args.steps, scaling="weak", selftest=True)))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
