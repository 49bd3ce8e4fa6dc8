"""Host logic of the slab decomposition (paper_2503_06610_b200/slabs.py) on
the CPU: the partition, the halo schedule, and the neighbour exchange -- in one process over several slabs
and over a world_size-2 gloo group -- driven through a mock lattice whose integer stencils have the reach of
the real operators (tests/slab_mock.py).  The cut lattice must reproduce the undivided one EXACTLY."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "tests"))

from paper_2503_06610_b200.slabs import HaloSchedule, Reach, SlabLattice, partition  # noqa: E402
from slab_mock import MockLattice  # noqa: E402

MODELS = {
    "one-constant": dict(),
    "no flow coupling": dict(coupling=1),
    "leslie": dict(alpha=(0.1, -0.4, -0.02, 0.9, 0.3, -0.16)),
    "three-constant": dict(K3=(1.0, 0.5, 1.5)),
    "three-constant + leslie": dict(K3=(1.0, 0.5, 1.5), alpha=(0.1, -0.4, -0.02, 0.9, 0.3, -0.16)),
}


def test_partition_covers_the_rows_once():
    for ny, parts in ((256, 8), (10, 3), (7, 7), (320, 6)):
        p = partition(ny, parts)
        assert p[0][0] == 0 and sum(r for _, r in p) == ny
        assert all(p[i][0] + p[i][1] == p[i + 1][0] for i in range(parts - 1))
        assert max(r for _, r in p) - min(r for _, r in p) <= 1
    with pytest.raises(ValueError):
        partition(3, 4)


def test_reach_and_minimum_halo():
    assert Reach.of().min_halo() == 4                                   # Heun on a radius-1 stencil, u two rows out
    assert Reach.of(coupling=1).min_halo() == 2
    assert Reach.of(K3=(1, 1, 1)).min_halo() == 5                       # u three rows out + velocity store + LB step
    assert Reach.of(K3=(1, 1, 1), alpha=(1,) * 6).force_director == 3
    with pytest.raises(ValueError):
        HaloSchedule(3, Reach.of(), 10)


@pytest.mark.parametrize("r", [1, 2, 5, 10, 0])
def test_schedule_never_uses_an_invalid_row(r):
    """Replay the plan with the validity rules written out independently of HaloSchedule's own counter."""
    for name, params in MODELS.items():
        reach = Reach.of(**params)
        H = max(4, reach.min_halo())
        sch = HaloSchedule(H, reach, r)
        vf, vn, vu, vF, t, steps = H, H, H, H, 0, 0
        for chunk in (1, 3, 7, 10, 2, 25):
            for a in sch.plan(chunk):
                if a[0] == "exchange":
                    if a[1] == "populations":
                        assert vf >= 0
                        vf = H
                    elif a[1] == "director":
                        assert vn >= 0
                        vn = H
                    elif a[1] == "velocity":
                        assert vu >= 0
                        vu = H
                    else:
                        assert vF >= 0
                        vF = H
                elif a[0] == "force":
                    vF = vn - reach.force_director
                    if reach.force_velocity:
                        vF = min(vF, vu - reach.force_velocity)
                else:
                    for _ in range(a[1]):
                        vf = min(vf - 1, vF)
                        assert vf >= 0, (name, r, t)
                        t += 1
                        steps += 1
                        if r > 0 and t % r == 0:
                            if reach.stores_velocity:
                                vu = min(vf - 1, vF)
                            vn = vn - reach.fd_director
                            if reach.fd_velocity:
                                vn = min(vn, vu - reach.fd_velocity)
                            assert vn >= 0, (name, r, t)
                            vF = -1                      # the force nh_step computed from the stale halo is unusable
            assert vf >= 0 and vn == H and vF == H, (name, r, vf, vn, vF)
        assert steps == 48 and sch.t == 48


def _director(nx, ny, nz):
    rng = np.random.default_rng(3)
    return rng.normal(size=(3, nz, ny, nx))


def _run_global(nx, ny, nz, r, chunks, params, extra=0):
    g = MockLattice(nx, ny, nz, fd_ratio=r, extra=extra, **params)
    g.set_director(_director(nx, ny, nz))
    for c in chunks:
        g.step(c)
    return g.get_fields()


@pytest.mark.parametrize("model", sorted(MODELS))
@pytest.mark.parametrize("slabs", [1, 2, 3])
def test_cut_lattice_equals_the_whole_one(model, slabs):
    params = MODELS[model]
    nx, ny, nz, chunks = 3, 29, 2, (1, 4, 10, 6)
    for r in (1, 3, 10):
        ref = _run_global(nx, ny, nz, r, chunks, params)
        s = SlabLattice(nx, ny, nz, slabs=slabs, factory=MockLattice, fd_ratio=r, **params)
        s.set_director(_director(nx, ny, nz))
        for c in chunks:
            s.step(c)
        got = s.gather_fields()
        for k in ref:
            assert np.array_equal(got[k], ref[k]), (model, slabs, r, k)
        assert s.exchanges > 0 and s.time == sum(chunks)


def test_a_too_narrow_halo_is_caught_by_this_test():
    """Negative control: stencils one row wider than the schedule assumes must change the answer."""
    nx, ny, nz, chunks, r = 3, 23, 2, (5, 10), 5   # not 16: two slabs of 8 + 2 x 4 rows would be the whole ring
    ref = _run_global(nx, ny, nz, r, chunks, {}, extra=1)
    s = SlabLattice(nx, ny, nz, slabs=2, factory=lambda *a, **k: MockLattice(*a, extra=1, **k), fd_ratio=r)
    s.set_director(_director(nx, ny, nz))
    for c in chunks:
        s.step(c)
    got = s.gather_fields()
    assert any(not np.array_equal(got[k], ref[k]) for k in ref)


WORKER = r"""
import os, sys
sys.path.insert(0, %r); sys.path.insert(0, os.path.join(%r, "tests"))
import numpy as np
import torch.distributed as dist
from paper_2503_06610_b200.slabs import SlabLattice
from slab_mock import MockLattice
import test_slabs_host as T
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", rank=rank, world_size=2)
for model in ("one-constant", "three-constant + leslie"):
    params = T.MODELS[model]
    nx, ny, nz, chunks, r = 3, 29, 2, (1, 4, 10, 6), 5
    ref = T._run_global(nx, ny, nz, r, chunks, params)
    s = SlabLattice(nx, ny, nz, group=dist.group.WORLD, factory=MockLattice, fd_ratio=r, **params)
    s.set_director(T._director(nx, ny, nz))
    for c in chunks:
        s.step(c)
    (idx, (y0, rows, f)), = s.get_fields().items()
    assert idx == rank and rows in (14, 15)
    for k in ref:
        assert np.array_equal(f[k], ref[k][..., y0:y0 + rows, :]), (model, k)
dist.barrier()
print("rank", rank, "slabs ok", s.exchanges)
dist.destroy_process_group()
"""


def test_two_ranks_exchange_halos_over_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % (ROOT, ROOT))
    port = 31500 + os.getpid() % 2000
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=300)[0] for p in procs]
    for rank, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert "rank %d slabs ok" % rank in o
