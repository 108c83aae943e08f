"""x-slab decomposition of the PM2D step, written out on the CPU -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

SURVEY 8(f).3 / DESIGN.md section 10: "the domain decomposition method to partition a 2D grid ... into m parts along the
x-coordinate direction", the per-slab tridiagonal solves joined by an interface system ("distributed arrowhead
decomposition") and the particle-list reconstruction (indicator vector I, scan A, filter a_{id+1} > a_{id},
MPI_SEND / MPI_RECV, "the received macroparticles are then inserted into the positions previously occupied by the sent
macro-particles ... any extra particles obtained are added at the end").  The library runs on one GPU
(BASELINE.json north_star); this module states what each rank of a multi-GPU version would compute and exchange, so that
the world_size-2 gloo test can check it against the single-domain oracle:

  * slab_cells            cells [x_lo, x_hi) of rank r; rank r owns the nodes x_lo .. x_hi - 1 (the last rank also nx)
  * slab_deposit          Eq. 14 of the rank's own particles on its nodes plus GHOST node columns on either side
  * ghost exchange        the ghost columns travel to the neighbour that owns those nodes and are added there
  * slab_poisson_local    FFT in y of the rank's rows (local: the cut is along x), then per k_y the chasing method on
                          the rank's interior nodes with its two interface values as unknowns g: phi = y + g_l V + g_r W
  * interface_solve       the (world - 1) x (world - 1) tridiagonal system for the interface values, per k_y
  * migrate               the paper's leaver / arrival bookkeeping
  * SlabField             Eqs. 6-8 on the rank's node columns plus one halo column of `a` per internal cut, exchanged
                          once per step: bit for bit the single-domain field
  * SlabRank              the whole program flow of P:L229-238 for one rank: the pieces above plus Eq. 16 / 18 on the
                          rank's window of nodes (HALO columns of n_s, phi, a from each neighbour), gather, predictor,
                          corrector and walls for the rank's own particles; equals the single-domain oracle step

`comm` is any object with all_gather(obj) -> list (torch.distributed in the test, a loop in the serial check).
"""
from __future__ import annotations

import numpy as np

from . import deposit as _deposit, make_grid as _make_grid

GHOST = 2          # ghost node columns per side: a footprint reaches one node beyond the nearest node, + the shared node


def slab_cells(nx: int, world: int, rank: int):
    """Cells [x_lo, x_hi) of a rank: as equal as possible ("as square-like as possible" is a statement about ny)."""
    base, rem = divmod(nx, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def slab_deposit(nx, ny, dx, dy, dt, shape, DD, X, Y, ux, uy, w, x_lo, x_hi):
    """Deposit (Eq. 14, oracle.deposit) of the particles with x_lo <= X < x_hi on the local node range
    [x_lo - GHOST, x_hi + GHOST] clipped to the box.  At the true x walls the local grid ends on the wall, so the
    wall treatment of the oracle (fold, half control volume) applies there and nowhere else: no particle of the slab
    comes within GHOST - 1/2 cells of an internal cut's local wall.  -> (n, Px, Py, g_lo) with g_lo = first node."""
    g_lo, g_hi = max(0, x_lo - GHOST), min(nx, x_hi + GHOST)
    sub = _make_grid(g_hi - g_lo, ny, dx, dy, dt)
    n, px, py = _deposit(sub, shape, DD, np.asarray(X) - g_lo, Y, ux, uy, w)
    return n, px, py, g_lo


def add_ghosts(nx, ny, world, rank, local, g_lo, comm):
    """Ghost exchange: every rank publishes its local array with its first node; each rank sums, over all ranks, the
    rows that fall on the nodes it owns.  (A real exchange sends GHOST + 1 columns to each neighbour; all_gather keeps
    the test small.)  -> owned rows [x_lo, x_hi) (+ row nx on the last rank)."""
    x_lo, x_hi = slab_cells(nx, world, rank)
    n_own = x_hi - x_lo + (1 if rank == world - 1 else 0)
    own = np.zeros((n_own, ny))
    for other, other_lo in comm.all_gather((local, g_lo)):
        lo = max(other_lo, x_lo)
        hi = min(other_lo + other.shape[0], x_lo + n_own)
        if hi > lo:
            own[lo - x_lo:hi - x_lo] += other[lo - other_lo:hi - other_lo]
    return own


def _thomas(b, rhs):
    """Chasing method for sub = super = 1, diag = b (scalar per system) on m unknowns; rhs (m, L) complex,
    b (L,).  Vectorised over the L systems, the recurrence in x is the plain one of orc_poisson."""
    m = rhs.shape[0]
    if m == 0:
        return rhs.copy()
    cp = np.empty((m, b.size))
    d = np.empty((m, b.size), complex)
    cp[0] = 1.0 / b
    d[0] = rhs[0] / b
    for i in range(1, m):
        den = b - cp[i - 1]
        cp[i] = 1.0 / den
        d[i] = (rhs[i] - d[i - 1]) / den
    x = np.empty_like(d)
    x[m - 1] = d[m - 1]
    for i in range(m - 2, -1, -1):
        x[i] = d[i] - cp[i] * x[i + 1]
    return x


def slab_poisson_local(nx, ny, dx, dy, world, rank, rho_own):
    """Local part of Eqs. 9-11 on a slab.  rho_own: the rank's owned rows of rho = n_i - n_e.  The rank's INTERFACE node
    is its first owned node x_lo (rank > 0); its interior unknowns are the nodes x_lo + 1 .. x_hi - 1 (rank 0: 1 .. x_hi
    - 1; the walls hold phi^ = 0, Q5).  Returns what the interface system needs and what the back-substitution needs."""
    x_lo, x_hi = slab_cells(nx, world, rank)
    rh = np.fft.fft(rho_own, axis=1) * dx * dx                     # dx^2 rho^ (Eq. 11 times dx^2), rows x_lo ..
    ls = np.fft.fftfreq(ny, 1.0 / ny)                                # l = -N/2 .. N/2 (Eq. 10)
    ky = 2.0 * np.pi * ls / (ny * dy)
    b = -2.0 - (ky * dx) ** 2
    first = 1 if rank == 0 else x_lo + 1                             # interior unknowns first .. last
    last = x_hi - 1
    m = last - first + 1
    rhs = rh[first - x_lo:first - x_lo + m]
    y = _thomas(b, rhs)                                              # both ends 0
    eL = np.zeros((m, ny), complex)
    eR = np.zeros((m, ny), complex)
    if m > 0:
        eL[0] = -1.0                                                 # unit value on the left end moves to the right-hand side
        eR[m - 1] = -1.0
    V = _thomas(b, eL)                                               # response to phi(left end) = 1
    W = _thomas(b, eR)                                               # response to phi(right end) = 1
    return dict(b=b, first=first, m=m, y=y, V=V, W=W, rho_if=rh[0] if rank > 0 else None)


def interface_solve(world, parts):
    """The interface system.  Unknowns g_k = phi^(first node of rank k), k = 1 .. world - 1.  Equation at that node:
    phi^(node + 1) + b g_k + phi^(node - 1) = dx^2 rho^(node), with phi^(node + 1) = y_k[0] + g_k V_k[0] + g_{k+1} W_k[0]
    (first interior node of rank k) and phi^(node - 1) = y_{k-1}[-1] + g_{k-1} V_{k-1}[-1] + g_k W_{k-1}[-1] (last
    interior node of rank k - 1).  A (world - 1)-tridiagonal system per k_y; g_0 = g_world = 0 are the walls.
    parts[k] = dict(b, m, y_first, y_last, V_first, V_last, W_first, W_last, rho_if) of every rank."""
    L = parts[0]["b"].size
    n = world - 1
    if n == 0:
        return np.zeros((world + 1, L), complex)
    A = np.zeros((L, n, n), complex)
    r = np.zeros((L, n), complex)
    for k in range(1, world):
        right, left = parts[k], parts[k - 1]
        row = k - 1
        diag = right["b"].astype(complex)
        rhs = right["rho_if"].copy()
        if right["m"] > 0:
            diag = diag + right["V_first"]
            rhs -= right["y_first"]
            if k + 1 < world:
                A[:, row, row + 1] += right["W_first"]
        else:                                                        # no interior node: the neighbour node is the next interface
            if k + 1 < world:
                A[:, row, row + 1] += 1.0
        if left["m"] > 0:
            diag = diag + left["W_last"]
            rhs -= left["y_last"]
            if k - 1 >= 1:
                A[:, row, row - 1] += left["V_last"]
        else:
            if k - 1 >= 1:
                A[:, row, row - 1] += 1.0
        A[:, row, row] = diag
        r[:, row] = rhs
    g = np.linalg.solve(A, r[..., None])[..., 0]                     # (L, n)
    out = np.zeros((world + 1, L), complex)
    out[1:world] = g.T
    return out


def slab_poisson(nx, ny, dx, dy, world, rank, rho_own, comm):
    """phi on the rank's owned nodes: local solve, all_gather of six numbers per k_y and rank, interface solve (done
    redundantly by every rank), back-substitution, inverse FFT."""
    loc = slab_poisson_local(nx, ny, dx, dy, world, rank, rho_own)
    m = loc["m"]
    z = np.zeros(ny, complex)
    mine = dict(b=loc["b"], m=m, rho_if=loc["rho_if"],
                y_first=loc["y"][0] if m else z, y_last=loc["y"][-1] if m else z,
                V_first=loc["V"][0] if m else z, V_last=loc["V"][-1] if m else z,
                W_first=loc["W"][0] if m else z, W_last=loc["W"][-1] if m else z)
    g = interface_solve(world, comm.all_gather(mine))
    gl, gr = g[rank], g[rank + 1]
    x_lo, x_hi = slab_cells(nx, world, rank)
    n_own = x_hi - x_lo + (1 if rank == world - 1 else 0)
    ph = np.zeros((n_own, ny), complex)
    ph[0] = gl                                                       # the interface node (rank 0: the wall, 0)
    if m:
        f0 = loc["first"] - x_lo
        ph[f0:f0 + m] = loc["y"] + gl * loc["V"] + gr * loc["W"]
    return np.fft.ifft(ph, axis=1).real                              # last rank: row nx stays 0 (wall)


def migrate(parts, x_lo, x_hi, rank, world, comm):
    """Particle-list reconstruction after the push, for the particles dict of one rank (arrays of equal
    length, key "X" in cells).  Indicator I (1 = crossed the slab boundary), scan A = inclusive_scan(I), leavers =
    the ids with a_{id+1} > a_{id} (A with a leading 0), packets to the left / right neighbour, arrivals fill the holes
    the leavers left, extras go to the end, remaining holes are closed from the end."""
    X = parts["X"]
    n = X.size
    I = ((X < x_lo) | (X >= x_hi)).astype(np.int64)
    A = np.concatenate([[0], np.cumsum(I)])
    leavers = np.flatnonzero(A[1:] > A[:-1])
    to_left = leavers[X[leavers] < x_lo]
    to_right = leavers[X[leavers] >= x_hi]
    if (rank == 0 and to_left.size) or (rank == world - 1 and to_right.size):
        raise ValueError("a particle left the box: the walls reflect before the migration")
    packets = comm.all_gather({rank - 1: {k: v[to_left] for k, v in parts.items()}, rank + 1: {k: v[to_right] for k, v in parts.items()}})
    arrivals = [p[rank] for p in packets if rank in p and p[rank]["X"].size]
    arr = {k: np.concatenate([a[k] for a in arrivals]) if arrivals else v[:0] for k, v in parts.items()}
    na, holes = arr["X"].size, leavers
    out = {k: v.copy() for k, v in parts.items()}
    nfill = min(na, holes.size)
    for k in out:
        out[k][holes[:nfill]] = arr[k][:nfill]
    if na > holes.size:                                              # extras at the end of the list
        out = {k: np.concatenate([out[k], arr[k][nfill:]]) for k in out}
    elif holes.size > na:                                            # close the remaining holes with particles from the end
        keep = np.ones(n, bool)
        keep[holes[nfill:]] = False
        out = {k: v[keep] for k, v in out.items()}
    return out


# ---- the stencil halo of the wave equation --------------------------------------------------------------------------------
class SlabField:
    """Eqs. 6-8 on one x-slab: the rank's owned node columns plus ONE halo column of `a` per internal cut
    ("a stencil halo for a"; Eq. 6 reaches one node in x).  The local grid is an ordinary oracle grid whose
    end columns are either a true wall of the box (rank 0: the left wall with the injected beams, last rank: the right
    wall; Eq. 8 applies there and only there) or a halo column, whose value after a step is whatever the local wall
    condition made of it and is overwritten by the neighbour's owned column before the next step.  n_e is held fixed (the
    deposit exchange is slab_deposit / add_ghosts).  One exchange per step and cut: ncomp x ny values each way.

    step()            one wave step of the local grid
    boundary()        -> (first owned column, last owned column) of the newest level, each [ncomp][ny]
    set_halo(l, r)    the neighbours' columns into the halo (None at a true wall)
    owned()           the owned columns of the newest level, [ncomp][n_own][ny]"""

    def __init__(self, nx, ny, dx, dy, dt, ncomp, n_e, lasers, world, rank, bc_y=0):
        from . import Oracle
        x_lo, x_hi = slab_cells(nx, world, rank)
        self.left_halo, self.right_halo = rank > 0, rank < world - 1
        self.first = x_lo - (1 if self.left_halo else 0)                 # first local node (global index)
        self.last = x_hi if self.right_halo else nx                      # last local node
        self.n_own = x_hi - x_lo + (0 if self.right_halo else 1)
        fixed = dict(sign=-1, mass=1.0, T_keV=0.0, mobile=0, n_fixed=np.ascontiguousarray(n_e[self.first:self.last + 1]))
        self.orc = Oracle(self.last - self.first, ny, dx, dy, dt, [fixed], lasers if rank == 0 else [], ncomp, bc_y=bc_y)

    def step(self):
        self.orc.step(1)

    def _cols(self):
        a = self.orc.a_now                                               # [ncomp][local nodes][ny]
        lo = 1 if self.left_halo else 0
        return a, lo, lo + self.n_own

    def boundary(self):
        a, lo, hi = self._cols()
        return a[:, lo].copy(), a[:, hi - 1].copy()

    def set_halo(self, from_left, from_right):
        a, lo, hi = self._cols()
        if self.left_halo:
            a[:, 0] = from_left
        if self.right_halo:
            a[:, hi] = from_right

    def owned(self):
        a, lo, hi = self._cols()
        return a[:, lo:hi].copy()


# ---- the whole time step, slab by slab ------------------------------------------------------------------------------------
HALO = 4       # node columns of n_s, phi and a that a rank reads beyond its owned nodes when it builds the force grid its own
#                particles gather from: a footprint reaches 2 nodes beyond the slab at the predicted position, Eq. 16 one more
#                (central differences, E on cell centres), and the last column of a window that ends on a cut is not used


class SlabRank:
    """One rank of the program flow of P:L229-238 on x-slabs: everything a rank computes is on its own nodes and
    its own particles; what it reads from its neighbours is named at each exchange.  `comm.all_gather` stands in for
    the neighbour exchanges (a device version sends HALO / GHOST columns to two neighbours instead of gathering
    everything; the values used are the same).  All species mobile, no sub-cycling, periodic y.

    per step:   halo of n_s^n  ->  a^{n+1} (SlabField, 1-column halo of a)  ->  halo of a^{n+1}
                rho -> slab Poisson (interface system) -> halo of phi  ->  E, F_s^n on the rank's window (Eq. 16)
                gather + predictor (Eqs. 15, 17) for the rank's particles  ->  deposit (x^, u^) + ghost sums
                slab Poisson again -> F_s^ (Eq. 18)  ->  gather at x^ + corrector (Eq. 19) + walls
                migrate  ->  deposit (x^{n+1}, u^{n+1}) + ghost sums = item (1) of the next step"""

    def __init__(self, cfg, parts, world, rank):
        from . import Oracle
        g = cfg["grid"]
        assert all(sp["mobile"] for sp in cfg["species"]) and g.get("subcycle", 1) <= 1 and not g.get("bc_y", 0)
        self.cfg, self.world, self.rank = cfg, world, rank
        self.nx, self.ny, self.dx, self.dy, self.dt, self.ncomp = g["nx"], g["ny"], g["dx"], g["dy"], g["dt"], g["ncomp"]
        self.x_lo, self.x_hi = slab_cells(self.nx, world, rank)
        self.n_own = self.x_hi - self.x_lo + (1 if rank == world - 1 else 0)
        self.w_lo, self.w_hi = max(0, self.x_lo - HALO), min(self.nx, self.x_hi + HALO)         # the rank's window of nodes
        self.wgrid = _make_grid(self.w_hi - self.w_lo, self.ny, self.dx, self.dy, self.dt, self.ncomp)
        self.sp = []
        for s, q in enumerate(cfg["species"]):
            p = parts[s]
            X = p["ix"] + p["fx"].astype(np.float64)
            m = (X >= self.x_lo) & (X < self.x_hi)
            self.sp.append(dict(X=X[m], Y=(p["iy"] + p["fy"].astype(np.float64))[m], ux=p["ux"][m].astype(np.float64),
                                uy=p["uy"][m].astype(np.float64), w=p["w"][m].astype(np.float64), id=p["id"][m].copy()))
        lasers = [dict(a0=l["a0"], omega=l["omega"], y0=l["y0"], w0=l["w0"], t_rise=l["t_rise"], comp=l["comp"], alpha=l.get("alpha", 0.0))
                  for l in cfg["lasers"]]
        self.field = SlabField(self.nx, self.ny, self.dx, self.dy, self.dt, self.ncomp, np.zeros((self.nx + 1, self.ny)), lasers, world, rank)
        nw = self.w_hi - self.w_lo + 1
        fixed = [dict(sign=q["sign"], mass=q["mass"], T_keV=q["T_keV"], C=q["pressure_coeff"], shape=q["shape"], DD=q["DD"], mobile=0,
                      n_fixed=np.zeros((nw, self.ny))) for q in cfg["species"]]
        self.loc = Oracle(self.w_hi - self.w_lo, self.ny, self.dx, self.dy, self.dt, fixed, [], self.ncomp)      # Eq. 16 on the window
        self.a_win = np.zeros((self.ncomp, nw, self.ny))                                                 # a^n
        self.n_own_s = None

    # -- exchanges ----------------------------------------------------------------------------------------------------
    def _window(self, comm, own):
        """Owned node columns [.., n_own, ny] of every rank -> this rank's window (its own columns + HALO columns of each
        neighbour's)."""
        full = np.concatenate(comm.all_gather(own), axis=-2)
        return np.ascontiguousarray(full[..., self.w_lo:self.w_hi + 1, :])

    def _deposit(self, comm, s, X, Y, ux, uy):
        """Eq. 14 of the rank's particles on its window, ghost columns summed at their owners -> owned n, Px, Py."""
        q = self.cfg["species"][s]
        loc = _deposit(self.wgrid, q["shape"], q["DD"], X - self.w_lo, Y, ux, uy, self.sp[s]["w"])
        return [add_ghosts(self.nx, self.ny, self.world, self.rank, a, self.w_lo, comm) for a in loc]

    def initial_deposit(self, comm):
        self.n_own_s = [self._deposit(comm, s, d["X"], d["Y"], d["ux"], d["uy"])[0] for s, d in enumerate(self.sp)]

    # -- Eq. 16 / 18 on the window --------------------------------------------------------------------------------------
    def _forces(self, comm, n_own_s, a_win):
        import ctypes as C
        from . import efield, lib, _p
        signs = [q["sign"] for q in self.cfg["species"]]
        rho_own = sum(sg * n for sg, n in zip(signs, n_own_s))
        phi_win = self._window(comm, slab_poisson(self.nx, self.ny, self.dx, self.dy, self.world, self.rank, rho_own, comm))
        Ex, Ey = efield(self.loc.g, phi_win)
        Ex, Ey = np.ascontiguousarray(Ex), np.ascontiguousarray(Ey)
        F = []
        for s in range(len(self.sp)):
            self.loc.sp[s]["n"][:] = self._window(comm, n_own_s[s]).ravel()
            Fx, Fy = np.zeros(self.loc.nn), np.zeros(self.loc.nn)
            lib().orc_force(C.byref(self.loc.g), C.byref(self.loc._sp[s]), _p(np.ascontiguousarray(a_win)), _p(Ex), _p(Ey), _p(Fx), _p(Fy))
            F.append((Fx, Fy))
        return F

    # -- one step -------------------------------------------------------------------------------------------------------
    def step(self, comm):
        from . import gather, predictor, corrector
        nx, ny, dt = self.nx, self.ny, self.dt
        hx, hy = dt / (2.0 * self.dx), dt / (2.0 * self.dy)
        cfgs = self.cfg["species"]
        # (2) the wave equation with n_e^n on the field's local nodes (1-column halo of a^n is in place), then the halos
        n_e = sum(self._window(comm, n) for n, q in zip(self.n_own_s, cfgs) if q["sign"] < 0)
        f = self.field
        f.orc.sp[0]["n"][:] = n_e[f.first - self.w_lo:f.last - self.w_lo + 1].ravel()
        f.step()
        edges = comm.all_gather(f.boundary())
        f.set_halo(edges[self.rank - 1][1] if self.rank > 0 else None, edges[self.rank + 1][0] if self.rank < self.world - 1 else None)
        a_new_win = self._window(comm, f.owned())
        # (2)(3) E^n, F^n with a^n;  (3)(4) gather at x^n, predictor
        F = self._forces(comm, self.n_own_s, self.a_win)
        hat = []
        for s, d in enumerate(self.sp):
            q = cfgs[s]
            npart = d["X"].size
            uhx, uhy, Xh, Yh = (np.zeros(npart) for _ in range(4))
            for p in range(npart):
                fx, fy = gather(self.wgrid, q["shape"], q["DD"], d["X"][p] - self.w_lo, d["Y"][p], F[s][0], F[s][1])
                uhx[p], Xh[p] = predictor(dt, hx, d["X"][p], d["ux"][p], fx)
                uhy[p], Yh[p] = predictor(dt, hy, d["Y"][p], d["uy"][p], fy)
            d["uhx"], d["uhy"] = uhx, uhy
            hat.append(self._deposit(comm, s, Xh, Yh, uhx, uhy)[0])                                   # (5)
        # (6)(7) E^, F^ with a^{n+1} and n^;  (8) gather at x^, corrector, walls
        F = self._forces(comm, hat, a_new_win)
        for s, d in enumerate(self.sp):
            q = cfgs[s]
            for p in range(d["X"].size):
                xh = d["X"][p] + hx * (d["uhx"][p] + d["ux"][p])
                yh = d["Y"][p] + hy * (d["uhy"][p] + d["uy"][p])
                fx, fy = gather(self.wgrid, q["shape"], q["DD"], xh - self.w_lo, yh, F[s][0], F[s][1])
                unx, xn = corrector(dt, hx, d["X"][p], d["ux"][p], d["uhx"][p], fx)
                uny, yn = corrector(dt, hy, d["Y"][p], d["uy"][p], d["uhy"][p], fy)
                if xn < 0.0:
                    xn, unx = -xn, -unx
                if xn > nx:
                    xn, unx = 2.0 * nx - xn, -unx
                yn -= np.floor(yn / ny) * ny
                if yn >= ny:
                    yn -= ny
                d["X"][p], d["Y"][p], d["ux"][p], d["uy"][p] = xn, yn, unx, uny
            # the list reconstruction of P:L274-276, then item (1) of the next step
            moved = migrate({k: d[k] for k in ("X", "Y", "ux", "uy", "w", "id")}, self.x_lo, self.x_hi, self.rank, self.world, comm)
            self.sp[s] = moved
        self.n_own_s = [self._deposit(comm, s, d["X"], d["Y"], d["ux"], d["uy"])[0] for s, d in enumerate(self.sp)]
        self.a_win = a_new_win
