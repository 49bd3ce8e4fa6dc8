"""Slab decomposition of the lattice along y (SURVEY.md section 8e, row f4 of section 8f).

The paper's runs are single-GPU; this is the way the same step shards over several GPUs.
Host logic only: which halo rows are still valid, when they must be refreshed, and who sends what to whom.
Every arithmetic step still runs in the kernels behind the C ABI (nh_step, nh_update_force); the halo rows
move with nh_get_rows / nh_set_rows and, between processes, with torch.distributed point-to-point calls
(NCCL over NVLink on GPUs; gloo, staged through host memory, in the tests).

Geometry.  Slab s owns rows [y0_s, y0_s + rows_s) of the global lattice and stores them as rows
[H, H + rows_s) of a local lattice of rows_s + 2H rows; local rows [0, H) mirror the last H rows of slab
s - 1, local rows [H + rows_s, 2H + rows_s) the first H rows of slab s + 1 (periodic in s).  The local
lattice is periodic in y like any other, so after one operator of stencil radius R the outermost R halo
rows hold values computed from the wrong neighbour: each operator "eats" R rows of valid halo, and an
exchange restores all H.  `HaloSchedule` keeps that count per field and emits the cheapest sequence of
(exchange, step, force) actions; results are bit-identical to the undivided lattice because every cell is
computed by the same kernels from the same neighbour values (tests/test_gpu_slabs.py).

Reach of the operators in rows (DESIGN.md section 8 derives them from the stencils):
  LB step               populations 1, force 0                        (pull streaming, Eq. 18)
  velocity store        populations 1, force 0                        (Eqs. 20-21 on gathered populations)
  director update       director 2, velocity 2   one-constant energy  (two Heun stages of radius 1, Eqs. 13-15)
                        director 4, velocity 3   three-constant energy (h = -df/dn + d_b pi_b. has radius 2)
  force                 director 2               elastic stress       (sigma from grad n, then its divergence)
                        director 2, velocity 2   + Leslie stress, one-constant (N needs h and grad u)
                        director 3, velocity 2   + Leslie stress, three-constant
"""
from __future__ import annotations

from dataclasses import dataclass


def partition(ny: int, parts: int):
    """Rows of each slab: [(y0, rows)], sizes differing by at most one, larger slabs first."""
    if parts < 1 or ny < parts:
        raise ValueError("cannot cut %d rows into %d slabs" % (ny, parts))
    base, extra = divmod(ny, parts)
    out, y0 = [], 0
    for s in range(parts):
        rows = base + (1 if s < extra else 0)
        out.append((y0, rows))
        y0 += rows
    return out


@dataclass(frozen=True)
class Reach:
    """Stencil radii in rows of the operators of one lattice (see the module docstring)."""
    fd_director: int
    fd_velocity: int      # 0: the director update does not read u (coupling bit1 off)
    force_director: int
    force_velocity: int   # 0: no Leslie viscosities
    stores_velocity: bool

    @staticmethod
    def of(coupling=3, alpha=(0.0,) * 6, K3=(0.0,) * 3, **_):
        three = any(float(k) != 0.0 for k in K3)
        visc = any(float(a) != 0.0 for a in alpha)
        flow = bool(coupling & 2)
        return Reach(fd_director=4 if three else 2,
                     fd_velocity=(3 if three else 2) if flow else 0,
                     force_director=3 if (three and visc) else 2,
                     force_velocity=2 if visc else 0,
                     stores_velocity=flow or visc)

    def populations_before_update(self) -> int:
        """Valid halo rows of the populations needed BEFORE the LB step that a director update follows:
        that step eats one row, the velocity store another, the update needs fd_velocity of u."""
        need = 1
        if self.fd_velocity:
            need = max(need, self.fd_velocity + 2)
        if self.stores_velocity:
            need = max(need, 2)                     # u must at least be right on the slab's own rows
        return need

    def min_halo(self) -> int:
        return max(self.populations_before_update(), self.fd_director, self.force_director, self.force_velocity, 1)


class HaloSchedule:
    """How many halo rows of the populations are still valid, and the actions that advance n_lb steps.

    The director, the force (and the stored velocity, where the force reads it) are refreshed to the full
    halo after every director update, so only the populations' count varies between updates."""

    def __init__(self, halo: int, reach: Reach, fd_ratio: int, t: int = 0):
        if halo < reach.min_halo():
            raise ValueError("halo of %d rows is too narrow: these operators need %d" % (halo, reach.min_halo()))
        self.H, self.reach, self.r, self.t = int(halo), reach, int(fd_ratio), int(t)
        self.valid_f = self.H

    def refresh(self, actions):
        """Only the outermost H - valid_f halo rows have gone stale: those are the rows that travel."""
        if self.valid_f < self.H:
            actions.append(("exchange", "populations", self.H - max(self.valid_f, 0)))
            self.valid_f = self.H

    def after_director(self, actions):
        """Halo traffic and force recomputation that follow a director update (or nh_set_director)."""
        actions.append(("exchange", "director"))
        if self.reach.force_velocity:
            actions.append(("exchange", "velocity"))
        actions.append(("force",))
        actions.append(("exchange", "force"))

    def plan(self, n_lb: int, n_fd: int = -1):
        """Actions that advance n_lb LB steps.  A ("step", m, n_fd) action is one nh_step call per slab; a director
        update can only be the LAST thing such a call does (the halos must be refreshed right after it).  Calls of
        an even number of steps are preferred: the two-step LB kernel takes the steps of a call in pairs."""
        r = self.r if n_fd < 0 else int(n_fd)
        need = self.reach.populations_before_update()

        def even(m):
            return m - 1 if m > 2 and m % 2 else m

        actions, left = [], int(n_lb)
        while left > 0:
            T = r - (self.t % r) if r > 0 else left + 1          # the T-th step from now is followed by an update
            if T <= left and self.valid_f - (T - 1) >= need:     # the halo lasts up to and including that step
                actions.append(("step", T, n_fd))
                self.valid_f -= T
                self.t += T
                left -= T
                self.after_director(actions)
                continue
            if left < T:
                cap = left                                       # this call ends before the update
            else:
                last = even(min(T, self.H - need + 1))           # steps of the call that ends with the update, after a refresh
                cap = T - last
                if cap == 0:
                    self.refresh(actions)
                    continue
            if self.valid_f < min(2, cap):
                self.refresh(actions)
            m = even(min(cap, self.valid_f))
            actions.append(("step", m, n_fd))
            self.valid_f -= m
            self.t += m
            left -= m
        return actions


class SlabLattice:
    """The lattice of `nx x ny x nz` cells cut into y-slabs.

    group=None: this process holds all `slabs` slabs (one device; how the decomposition is tested on one GPU:
    the slabs are advanced one after the other by the host, none waits for another on the device).
    group=a torch.distributed group: one slab per rank, slabs = world size, neighbours exchange halo rows with
    batched isend/irecv.  `factory(nx, ny_local, nz, **params)` makes the per-slab lattice
    (default: paper_2503_06610_b200.Lattice)."""

    def __init__(self, nx, ny, nz, *, slabs=None, group=None, halo=None, factory=None, **params):
        self.group = group
        if group is not None:
            import torch.distributed as dist
            self.rank, self.size = dist.get_rank(group), dist.get_world_size(group)
            if slabs not in (None, self.size):
                raise ValueError("one slab per rank: slabs must equal the group's size")
        else:
            self.rank, self.size = 0, int(slabs or 1)
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.reach = Reach.of(**params)
        # two rows more than the minimum: the step before a director update can then share a two-step LB launch
        self.H = int(halo) if halo is not None else self.reach.min_halo() + 2
        self.parts = partition(self.ny, self.size)
        if min(rows for _, rows in self.parts) < self.H:
            raise ValueError("slabs of fewer than halo = %d rows" % self.H)
        if factory is None:
            from .binding import Lattice as factory
        mine = [self.rank] if group is not None else list(range(self.size))
        self.local = {}
        for s in mine:
            y0, rows = self.parts[s]
            self.local[s] = factory(self.nx, rows + 2 * self.H, self.nz, **params)
            self.local[s].defer_force(True)      # the force follows the director's halo refresh (after_director)
        self.fd_ratio = int(params.get("fd_ratio", 1))
        self.schedule = HaloSchedule(self.H, self.reach, self.fd_ratio)
        self._buf = {}
        self.exchanges = 0
        self.bytes_sent = 0

    # ---- halo exchange -------------------------------------------------------------------------------
    def _buffers(self, s, field):
        """Per slab and field: `send` = [rows for the slab below | rows for the slab above], `recv` = [rows from the
        slab below | rows from the slab above]; each half holds up to H packed rows."""
        key = (s, field)
        if key not in self._buf:
            lat = self.local[s]
            half = lat.rows_bytes(field, self.H)
            self._buf[key] = {k: lat.new_rows_buffer(field, 2 * self.H) for k in ("send", "recv")}
            self._buf[key]["half"] = half
        return self._buf[key]

    def _on_stream(self, lat):
        """Everything an exchange enqueues must be ordered with the lattice's own launches: make the lattice's stream
        torch's current stream for the duration (torch copies and NCCL then wait on it, whatever the ambient stream)."""
        import contextlib
        st = getattr(lat, "_stream", None)
        if st is None:
            return contextlib.nullcontext()
        import torch
        return torch.cuda.stream(st)

    def exchange(self, field, m=None):
        """Refresh the outermost `m` (default: all H) rows of both halos of `field` on every slab from its two
        neighbours.  One pack launch and one unpack launch per slab (both faces at once)."""
        H = self.H
        m = H if m is None else int(m)
        assert 1 <= m <= H
        for s, lat in self.local.items():
            rows = self.parts[s][1]
            b = self._buffers(s, field)
            with self._on_stream(lat):
                # first half: my first owned rows that the slab below lacks at the far end of its upper halo;
                # second half: my last owned rows that the slab above lacks at the far end of its lower halo
                lat.get_rows_pair(field, 2 * H - m, rows, m, b["send"])
        if self.group is None or self.size == 1:
            for s, lat in self.local.items():
                rows = self.parts[s][1]
                lo, hi = (s - 1) % self.size, (s + 1) % self.size
                nb = lat.rows_bytes(field, m)
                with self._on_stream(lat):
                    if lo == s and hi == s:      # one slab, its own neighbour on both sides: its two halves, swapped
                        lat.set_rows_pair(field, 2 * H + rows - m, 0, m, self._buffers(s, field)["send"])
                    else:
                        lat.set_rows(field, 0, m, self._buffers(lo, field)["send"][nb:2 * nb])
                        lat.set_rows(field, 2 * H + rows - m, m, self._buffers(hi, field)["send"][:nb])
        else:
            import torch.distributed as dist
            s = self.rank
            lat, rows, b = self.local[s], self.parts[s][1], self._buffers(s, field)
            nb = lat.rows_bytes(field, m)
            lo = dist.get_global_rank(self.group, (s - 1) % self.size)
            hi = dist.get_global_rank(self.group, (s + 1) % self.size)
            with self._on_stream(lat):
                # Same order on every rank.  With two ranks both neighbours are the same peer and messages between a
                # pair match in posting order: my first send (to below) meets the peer's first receive (from above).
                staged = b["send"].is_cuda and dist.get_backend(self.group) == "gloo"
                send = b["send"][:2 * nb].cpu() if staged else b["send"]      # gloo moves host memory only
                recv = send.new_empty(2 * nb) if staged else b["recv"]
                ops = [dist.P2POp(dist.isend, send[:nb], lo, self.group),
                       dist.P2POp(dist.isend, send[nb:2 * nb], hi, self.group),
                       dist.P2POp(dist.irecv, recv[nb:2 * nb], hi, self.group),
                       dist.P2POp(dist.irecv, recv[:nb], lo, self.group)]
                for req in dist.batch_isend_irecv(ops):
                    req.wait()
                if staged:
                    b["recv"][:2 * nb].copy_(recv)
                lat.set_rows_pair(field, 0, 2 * H + rows - m, m, b["recv"])
        self.exchanges += 1
        self.bytes_sent += sum(2 * lat.rows_bytes(field, m) for lat in self.local.values())

    def _run(self, actions):
        for a in actions:
            if a[0] == "exchange":
                self.exchange(*a[1:])
            elif a[0] == "step":
                for lat in self.local.values():
                    lat.step(a[1], a[2])
            else:
                for lat in self.local.values():
                    lat.update_force()

    # ---- the C ABI's calls, on the cut lattice -----------------------------------------------------
    def set_director(self, n_global):
        """`n_global`: host FP64 [3][nz][ny][nx], the whole lattice (every rank passes the same array)."""
        import numpy as np
        n_global = np.asarray(n_global, dtype=np.float64)
        assert n_global.shape == (3, self.nz, self.ny, self.nx)
        acts = []
        self.schedule.refresh(acts)      # the velocity the force may read gathers the populations
        self._run(acts)
        for s, lat in self.local.items():
            y0, rows = self.parts[s]
            idx = np.arange(y0 - self.H, y0 + rows + self.H) % self.ny
            lat.set_director(np.ascontiguousarray(n_global[:, :, idx, :]))
        # F is right on the slab's own rows (director halo H, u from the refreshed populations H - 1): fill its halo
        self._run([("exchange", "force")])

    def step(self, n_lb, n_fd=-1):
        self._run(self.schedule.plan(n_lb, n_fd))

    def get_fields(self, which=("rho", "u", "n", "F")):
        """The rows this process holds: {slab index: (y0, rows, {name: array [..][nz][rows][nx]})}."""
        acts = []
        if self.schedule.valid_f < 1:
            self.schedule.refresh(acts)      # rho and u gather the populations
        self._run(acts)
        out = {}
        for s, lat in self.local.items():
            y0, rows = self.parts[s]
            f = lat.get_fields(which=which)
            out[s] = (y0, rows, {k: v[..., self.H:self.H + rows, :].copy() for k, v in f.items()})
        return out

    def gather_fields(self, which=("rho", "u", "n", "F")):
        """Whole-lattice arrays (group=None only; across ranks use get_fields and the caller's own gather)."""
        import numpy as np
        assert self.group is None
        parts = self.get_fields(which)
        out = {}
        for k in which:
            out[k] = np.concatenate([parts[s][2][k] for s in range(self.size)], axis=-2)
        return out

    @property
    def time(self):
        return self.schedule.t

    def synchronize(self):
        for lat in self.local.values():
            lat.synchronize()

    def close(self):
        for lat in self.local.values():
            lat.close()
        self.local = {}
        self._buf = {}
