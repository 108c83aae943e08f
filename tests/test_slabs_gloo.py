"""SURVEY 8(f).3 without a second GPU: the x-slab decomposition of the deposit, of the Poisson solve and of the particle
lists (oracle/slabs.py) against the single-domain oracle.  world_size 2 over gloo, and the same
arithmetic for three and five slabs in one process; the wave equation by slabs with a one-column halo of `a` (SlabField),
bit for bit.  CPU only."""
import os
import socket
import sys

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402


class _SerialComm:
    """all_gather for ranks that run one after the other in one process: two passes (publish, then compute)."""

    def __init__(self, world):
        self.world, self.box, self.replay = world, [], None

    def all_gather(self, obj):
        if self.replay is None:
            self.box.append(obj)
            raise _Publish
        return self.replay


class _Publish(Exception):
    pass


def _run_serial(world, fn):
    """fn(rank, comm) with exactly one all_gather inside: first pass collects, second pass computes."""
    comm = _SerialComm(world)
    for r in range(world):
        try:
            fn(r, comm)
        except _Publish:
            pass
    comm.replay = comm.box
    return [fn(r, comm) for r in range(world)]


class _DistComm:
    def all_gather(self, obj):
        out = [None] * dist.get_world_size()
        dist.all_gather_object(out, obj)
        return out


def _case(nx=72, ny=16):
    import oracle.loader as L
    import pm2d_inputs as I
    cfg = I.config("c3", nx=nx, ny=ny)
    parts = [L.generate_particles(cfg, s) for s in (0, 1)]
    return cfg, parts


def _slab_density_and_phi(cfg, parts, world, rank, comm_n, comm_p):
    from oracle import slabs
    g = cfg["grid"]
    nx, ny, dx, dy, dt = g["nx"], g["ny"], g["dx"], g["dy"], g["dt"]
    x_lo, x_hi = slabs.slab_cells(nx, world, rank)
    rho = 0.0
    dens = []
    for s, sp in enumerate(cfg["species"]):
        p = parts[s]
        X = p["ix"] + p["fx"].astype(np.float64)
        Y = p["iy"] + p["fy"].astype(np.float64)
        mine = (X >= x_lo) & (X < x_hi)
        n, px, py, g_lo = slabs.slab_deposit(nx, ny, dx, dy, dt, sp["shape"], sp["DD"], X[mine], Y[mine], p["ux"][mine], p["uy"][mine],
                                             p["w"][mine].astype(np.float64), x_lo, x_hi)
        own = slabs.add_ghosts(nx, ny, world, rank, n, g_lo, comm_n[s])
        dens.append(own)
        rho = rho + sp["sign"] * own
    phi = slabs.slab_poisson(nx, ny, dx, dy, world, rank, rho, comm_p)
    return dens, phi


def _reference(cfg, parts):
    import oracle
    g = cfg["grid"]
    grid = oracle.make_grid(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"])
    dens, rho = [], 0.0
    for s, sp in enumerate(cfg["species"]):
        p = parts[s]
        n, _, _ = oracle.deposit(grid, sp["shape"], sp["DD"], p["ix"] + p["fx"].astype(np.float64), p["iy"] + p["fy"].astype(np.float64),
                                 p["ux"], p["uy"], p["w"].astype(np.float64))
        dens.append(n)
        rho = rho + sp["sign"] * n
    return dens, oracle.poisson(grid, rho).reshape(g["nx"] + 1, g["ny"])


def _serial_check(world, nx):
    """Every all_gather of the slab routines in its own two-pass communicator."""
    cfg, parts = _case(nx=nx)
    from oracle import slabs
    g = cfg["grid"]
    nxx, ny = g["nx"], g["ny"]
    ref_dens, ref_phi = _reference(cfg, parts)
    # pass 1: deposits + ghost sums, per species
    owned = []
    for s, sp in enumerate(cfg["species"]):
        p = parts[s]
        X = p["ix"] + p["fx"].astype(np.float64)
        Y = p["iy"] + p["fy"].astype(np.float64)

        def dep(rank, comm, X=X, Y=Y, p=p, sp=sp):
            x_lo, x_hi = slabs.slab_cells(nxx, world, rank)
            mine = (X >= x_lo) & (X < x_hi)
            n, _, _, g_lo = slabs.slab_deposit(nxx, ny, g["dx"], g["dy"], g["dt"], sp["shape"], sp["DD"], X[mine], Y[mine], p["ux"][mine],
                                               p["uy"][mine], p["w"][mine].astype(np.float64), x_lo, x_hi)
            return slabs.add_ghosts(nxx, ny, world, rank, n, g_lo, comm)
        owned.append(_run_serial(world, dep))
        assert np.abs(np.concatenate(owned[s]) - ref_dens[s]).max() < 1e-13 * np.abs(ref_dens[s]).max()
    rho = [sum(sp["sign"] * owned[s][r] for s, sp in enumerate(cfg["species"])) for r in range(world)]
    phis = _run_serial(world, lambda rank, comm: slabs.slab_poisson(nxx, ny, g["dx"], g["dy"], world, rank, rho[rank], comm))
    phi = np.concatenate(phis)
    assert phi.shape == ref_phi.shape
    assert np.abs(phi - ref_phi).max() < 1e-11 * np.abs(ref_phi).max()


def test_three_and_five_slabs_equal_the_single_domain():
    """Ghost-column deposit sums and the interface system for 3 slabs (72 cells) and 5 slabs of unequal width (73 cells:
    15, 15, 15, 14, 14): densities to rounding, phi to 1e-11 of its maximum."""
    sys.path.insert(0, ROOT)
    _serial_check(3, 72)
    _serial_check(5, 73)


FIELD_STEPS = 120


def _field_case(nx=72, ny=16, ncomp=1):
    """A fixed electron density (the reduced c3 deposit) and an oblique Gaussian beam that crosses the cuts."""
    cfg, parts = _case(nx=nx, ny=ny)
    g = cfg["grid"]
    p = parts[0]
    grid = oracle.make_grid(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"])
    n_e, _, _ = oracle.deposit(grid, cfg["species"][0]["shape"], cfg["species"][0]["DD"], p["ix"] + p["fx"].astype(np.float64),
                               p["iy"] + p["fy"].astype(np.float64), p["ux"].astype(np.float64), p["uy"].astype(np.float64), p["w"].astype(np.float64))
    Ly = g["ny"] * g["dy"]
    lasers = [dict(a0=0.02, omega=1.0, y0=0.5 * Ly, w0=0.3 * Ly, t_rise=0.5, alpha=0.15, comp=0)]
    return g, n_e, lasers


def _field_reference(g, n_e, lasers, nsteps):
    fixed = dict(sign=-1, mass=1.0, T_keV=0.0, mobile=0, n_fixed=n_e)
    orc = oracle.Oracle(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"], [fixed], lasers, 1)
    orc.step(nsteps)
    return orc.a_now.copy()


def test_wave_equation_by_slabs_with_a_one_column_halo_is_the_single_domain_bit_for_bit():
    """SURVEY 8e (1) / P:L256: Eqs. 6-8 advanced slab by slab, one halo column of `a` exchanged per cut and step, give on
    every owned node exactly the bits of the single-domain run (the update of a node reads its four neighbours and n_e,
    nothing else) -- for 3 equal and 5 unequal slabs, through the turn-on of an oblique beam that crosses every cut.  A
    halo taken from the wrong time level, a wall condition applied at a cut, or an off-by-one in the owned range fails."""
    sys.path.insert(0, ROOT)
    from oracle import slabs
    for world, nx in ((3, 72), (5, 73)):
        g, n_e, lasers = _field_case(nx=nx)
        nsteps = 140
        ref = _field_reference(g, n_e, lasers, nsteps)
        assert np.abs(ref).max() > 0.005 and np.abs(ref[0, g["nx"] - 4:]).max() > 1e-4          # the beam has reached the right wall
        ranks = [slabs.SlabField(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"], 1, n_e, lasers, world, r) for r in range(world)]
        for _ in range(nsteps):
            for f in ranks:
                f.step()
            edges = [f.boundary() for f in ranks]
            for r, f in enumerate(ranks):
                f.set_halo(edges[r - 1][1] if r > 0 else None, edges[r + 1][0] if r < world - 1 else None)
        got = np.concatenate([f.owned() for f in ranks], axis=1)
        assert got.shape == ref.shape and np.array_equal(got, ref)


class _ThreadComm:
    """all_gather between ranks that run as threads of one process (any number of exchanges, in lockstep)."""

    def __init__(self, world):
        import threading
        self.world, self.slots, self.bar = world, [None] * world, threading.Barrier(world)

    def bind(self, rank):
        comm = self

        class _Bound:
            def all_gather(self, obj):
                comm.slots[rank] = obj
                comm.bar.wait()
                out = list(comm.slots)
                comm.bar.wait()
                return out
        return _Bound()


def _whole_step_by_slabs(cfg, parts, world, nsteps, comm_of_rank, ranks):
    from oracle import slabs
    out = {}
    for rank in ranks:
        r = slabs.SlabRank(cfg, parts, world, rank)
        comm = comm_of_rank(rank)
        r.initial_deposit(comm)
        for _ in range(nsteps):
            r.step(comm)
        out[rank] = (r.sp, r.field.owned(), r.n_own_s)
    return out


def _compare_with_single_domain(cfg, parts, res, world, nsteps, a_min=5e-3):
    orc, _ = oracle.from_config(cfg, parts)
    orc.step(nsteps)
    a = np.concatenate([res[r][1] for r in range(world)], axis=1)
    assert np.abs(a - orc.a_now).max() < 1e-12 * np.abs(orc.a_now).max() and np.abs(orc.a_now).max() > a_min, (
        np.abs(a - orc.a_now).max(), np.abs(orc.a_now).max())
    from oracle import slabs
    moved = 0
    for s in range(len(cfg["species"])):
        n = np.concatenate([res[r][2][s] for r in range(world)])
        assert np.abs(n - orc.moment(s, "n")).max() < 1e-11 * np.abs(orc.moment(s, "n")).max()
        ids = np.concatenate([res[r][0][s]["id"] for r in range(world)])
        order = np.argsort(ids)
        assert np.array_equal(ids[order], np.sort(parts[s]["id"]))               # every particle exactly once
        ref_order = np.argsort(parts[s]["id"])
        for key in ("X", "Y", "ux", "uy"):
            got = np.concatenate([res[r][0][s][key] for r in range(world)])[order]
            want = orc.sp[s][key][ref_order]
            assert np.abs(got - want).max() < 1e-10, (s, key, np.abs(got - want).max())
        for r in range(world):
            x_lo, x_hi = slabs.slab_cells(cfg["grid"]["nx"], world, r)
            X = res[r][0][s]["X"]
            assert ((X >= x_lo) & (X < x_hi)).all()
            X0 = parts[s]["ix"][np.isin(parts[s]["id"], res[r][0][s]["id"])]
            moved += int(((X0 < x_lo) | (X0 >= x_hi)).sum())
    return moved


def test_the_whole_time_step_by_slabs_equals_the_single_domain():
    """three ranks (threads of this process) carry the program flow of P:L229-238 on x-slabs
    for ten steps of the reduced c3 set-up (electrons and mobile ions, sine clouds, the laser turning on) -- deposit with
    ghost sums, wave equation with its halo, slab Poisson with the interface system, Eq. 16 on the rank's window, gather,
    predictor, corrector, walls, migration -- and end with the single-domain oracle's particles (1e-10 cell, by id), field
    and densities; particles have crossed the cuts."""
    import threading
    cfg, parts = _case(nx=72, ny=16)
    cfg["lasers"][0]["t_rise"] = 0.2               # the beam is at full amplitude within the run: the ponderomotive term of Eq. 16 acts
    world, nsteps = 3, 10
    comm = _ThreadComm(world)
    res, err = {}, []

    def run(rank):
        try:
            res.update(_whole_step_by_slabs(cfg, parts, world, nsteps, comm.bind, [rank]))
        except BaseException as e:          # a dead rank would leave the others at the barrier
            err.append(e)
            comm.bar.abort()

    th = [threading.Thread(target=run, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join(timeout=600)
    assert not err, err
    moved = _compare_with_single_domain(cfg, parts, res, world, nsteps)
    assert moved > 20


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import slabs
    cfg, parts = _case()
    comm = _DistComm()
    dens, phi = _slab_density_and_phi(cfg, parts, world, rank, [comm, comm], comm)
    # the particle lists after a displacement that sends some particles across the cut (both ways)
    g = cfg["grid"]
    x_lo, x_hi = slabs.slab_cells(g["nx"], world, rank)
    p = parts[0]
    X = p["ix"] + p["fx"].astype(np.float64)
    mine = (X >= x_lo) & (X < x_hi)
    rng = np.random.default_rng(7 + rank)
    mov = dict(X=np.clip(X[mine] + rng.normal(0.0, 1.5, mine.sum()), 0.0, g["nx"] - 1e-9), id=p["id"][mine].copy(),
               ux=p["ux"][mine].copy())
    got = slabs.migrate(mov, x_lo, x_hi, rank, world, comm)
    # the wave equation with its halo column sent over the process group, one exchange per step
    gg, n_e, lasers = _field_case()
    f = slabs.SlabField(gg["nx"], gg["ny"], gg["dx"], gg["dy"], gg["dt"], 1, n_e, lasers, world, rank)
    for _ in range(FIELD_STEPS):
        f.step()
        edges = comm.all_gather(f.boundary())
        f.set_halo(edges[rank - 1][1] if rank > 0 else None, edges[rank + 1][0] if rank < world - 1 else None)
    # and the whole time step (SlabRank), four steps
    whole = _whole_step_by_slabs(cfg, parts, world, 4, lambda r: comm, [rank])[rank]
    out.put((rank, dens, phi, mov, got, f.owned(), whole))
    dist.barrier()
    dist.destroy_process_group()


def test_two_slabs_over_gloo_equal_the_single_domain():
    sys.path.insert(0, ROOT)
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=300) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg, parts = _case()
    ref_dens, ref_phi = _reference(cfg, parts)
    for s in (0, 1):
        n = np.concatenate([r[1][s] for r in res])
        assert np.abs(n - ref_dens[s]).max() < 1e-13 * np.abs(ref_dens[s]).max()
    phi = np.concatenate([r[2] for r in res])
    assert np.abs(phi - ref_phi).max() < 1e-11 * np.abs(ref_phi).max()
    # migration: every rank ends with exactly the particles of its slab; nothing lost, nothing doubled; the fields of a
    # particle travel together
    from oracle import slabs
    g = cfg["grid"]
    before = {int(i): (x, u) for r in res for i, x, u in zip(r[3]["id"], r[3]["X"], r[3]["ux"])}
    after = {}
    crossed = 0
    gg, n_e, lasers = _field_case()
    assert np.array_equal(np.concatenate([r[5] for r in res], axis=1), _field_reference(gg, n_e, lasers, FIELD_STEPS))
    _compare_with_single_domain(cfg, parts, {r[0]: r[6] for r in res}, world, 4, a_min=0.0)
    for rank, _, _, mov, got, _, _ in res:
        x_lo, x_hi = slabs.slab_cells(g["nx"], world, rank)
        assert ((got["X"] >= x_lo) & (got["X"] < x_hi)).all()
        crossed += int(((mov["X"] < x_lo) | (mov["X"] >= x_hi)).sum())
        for i, x, u in zip(got["id"], got["X"], got["ux"]):
            assert int(i) not in after
            after[int(i)] = (x, u)
    assert crossed > 50 and after == before
