"""A stand-in for paper_2503_06610_b200.Lattice with NO physics: integer stencils on numpy uint64 arrays whose
reach in y equals the reach of the real operators (slabs.Reach), so that the halo bookkeeping of
paper_2503_06610_b200.slabs can be tested on the CPU, exactly (wrap-around integer arithmetic), without a GPU.
`extra` widens every stencil by that many rows: the negative control (a schedule that is too optimistic
must then give a different answer)."""
import numpy as np
import torch

from paper_2503_06610_b200.slabs import Reach

COMPS = {"populations": 2, "director": 1, "velocity": 1, "force": 1}


def _sum(field, radius, salt):
    out = np.zeros_like(field)
    for d in range(-radius, radius + 1):
        out += np.uint64(d + salt) * np.roll(field, d, axis=-2)
    return out


class MockLattice:
    def __init__(self, nx, ny, nz, fd_ratio=1, extra=0, **params):
        self.shape = (nz, ny, nx)
        self.reach = Reach.of(**params)
        self.r, self.t, self.extra = int(fd_ratio), 0, int(extra)
        z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
        self.fld = {k: np.zeros((c, nz, ny, nx), dtype=np.uint64) for k, c in COMPS.items()}
        self.fld["populations"][:] = 1          # uniform, like the lattice at rest
        self.device = "cpu"
        self.deferred = False

    def defer_force(self, on=True):
        self.deferred = bool(on)

    # --- the operators: same reach as the real ones, arbitrary integer content ---
    def _lb(self):
        f, F = self.fld["populations"], self.fld["force"]
        e = 1 + self.extra
        self.fld["populations"] = _sum(f, e, 5) + f[::-1] * np.uint64(3) + F

    def _velocity(self):
        f, F = self.fld["populations"], self.fld["force"]
        self.fld["velocity"] = (_sum(f[:1], 1 + self.extra, 9) ^ f[1:]) + F

    def _director(self):
        R, e = self.reach, self.extra
        n = _sum(self.fld["director"], R.fd_director + e, 7)
        if R.fd_velocity:
            n += _sum(self.fld["velocity"], R.fd_velocity + e, 11)
        self.fld["director"] = n

    def update_force(self):
        R, e = self.reach, self.extra
        F = _sum(self.fld["director"], R.force_director + e, 13)
        if R.force_velocity:
            F += _sum(self.fld["velocity"], R.force_velocity + e, 17)
        self.fld["force"] = F

    # --- the Lattice interface SlabLattice uses ---
    def set_director(self, n):
        assert n.shape == (3,) + self.shape
        self.fld["director"] = np.ascontiguousarray((n[:1] * 1e6).astype(np.int64).astype(np.uint64))
        if self.reach.force_velocity:
            self._velocity()
        self.update_force()

    def step(self, n_lb, n_fd=-1):
        r = self.r if n_fd < 0 else n_fd
        for _ in range(n_lb):
            self._lb()
            self.t += 1
            if r > 0 and self.t % r == 0:
                if self.reach.stores_velocity:
                    self._velocity()
                self._director()
                if not self.deferred:
                    self.update_force()

    def get_fields(self, which=("rho", "u", "n", "F")):
        f = self.fld["populations"]
        full = {"rho": _sum(f[0], 1 + self.extra, 3), "u": _sum(f[1:], 1 + self.extra, 4) + self.fld["force"],
                "n": self.fld["director"], "F": self.fld["force"]}
        return {k: full[k] for k in which}

    def rows_bytes(self, field, nrows):
        return COMPS[field] * self.shape[0] * nrows * self.shape[2] * 8

    def new_rows_buffer(self, field, nrows):
        return torch.zeros(self.rows_bytes(field, nrows), dtype=torch.uint8)

    def get_rows(self, field, y0, nrows, buf):
        a = np.ascontiguousarray(self.fld[field][:, :, y0:y0 + nrows, :])
        buf[:a.nbytes].copy_(torch.from_numpy(a.view(np.uint8).reshape(-1)))

    def set_rows(self, field, y0, nrows, buf):
        a = buf[:self.rows_bytes(field, nrows)].numpy().view(np.uint64).reshape(COMPS[field], self.shape[0], nrows, self.shape[2])
        self.fld[field][:, :, y0:y0 + nrows, :] = a

    def get_rows_pair(self, field, y0_a, y0_b, nrows, buf):
        nb = self.rows_bytes(field, nrows)
        self.get_rows(field, y0_a, nrows, buf[:nb])
        self.get_rows(field, y0_b, nrows, buf[nb:2 * nb])

    def set_rows_pair(self, field, y0_a, y0_b, nrows, buf):
        nb = self.rows_bytes(field, nrows)
        self.set_rows(field, y0_a, nrows, buf[:nb])
        self.set_rows(field, y0_b, nrows, buf[nb:2 * nb])

    def synchronize(self):
        pass

    def close(self):
        pass
