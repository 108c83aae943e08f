"""N > 1 path of bench.py on CPU: the hot path does not shard (replicas only), so the
only multi-rank logic is the max-over-ranks timing and the whole-job aggregation.  world_size 2, gloo."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import oracle.loader as L
    import pm2d_inputs as I
    # rank r is slower by r ms: every rank must report the job value computed from the slowest one
    ms_local = 10.0 + rank
    value, ms_max = bench.job_throughput(1000, 5, ms_local, world, None)
    # replicas get distinct seeds (bench.run_cuda: seed + 1000 * rank) -> distinct particles
    cfg = I.config("c1", nx=32, ny=16)
    cfg["seed"] = int(cfg["seed"]) + 1000 * rank
    ux = torch.from_numpy(L.generate_particles(cfg, 0)["ux"][:64].copy())
    gathered = [torch.zeros_like(ux) for _ in range(world)]
    dist.all_gather(gathered, ux)
    out.put((rank, value, ms_max, bool(torch.equal(gathered[0], gathered[1]))))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_max_over_ranks_and_aggregate():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms_max, same in res:
        assert ms_max == 11.0                                  # max over ranks
        assert abs(value - 1000 * 2 * 5 / 11.0e-3) < 1e-6 * value  # units of ALL ranks / slowest time
        assert not same                                        # independent replicas


def test_bench_spawns_its_own_ranks():
    """`python bench.py --gpus 2` outside torchrun starts the two local ranks itself (bench.spawn_ranks) and rank 0
    prints one line for the whole job: n_gpus 2, the units of both ranks over the slower rank's time.  The device work
    is replaced by a fixed per-rank time (--selftest-cpu: gloo, no GPU); spawn, rendezvous, MAX and aggregation are
    the code `--gpus N` runs on a GPU node."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "5", "--selftest-cpu"],
                       capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                     # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["steps"] == 5 and d["scaling"] == "weak"
    assert abs(d["ms_per_step"] - 11.0 / 5) < 1e-9             # the slower rank (10 + rank ms)
    assert abs(d["value"] - 1000 * 2 * 5 / 11.0e-3) < 1e-6 * d["value"]
