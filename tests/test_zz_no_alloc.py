"""nh_lb_two_steps_noalloc (include/nh_noalloc.h) against the handle path, on a B200.

Why the entry point exists: nh_init_lattice creates host objects, a pinned host word and, on demand, events and graphs,
and its scratch (plane ring, flags) comes out of a workspace the caller must allocate.  A host that handed the whole
device to its own pool at start-up, or that sits in a time-critical loop where cudaMalloc's device-wide wait is not
acceptable, cannot use that.  The no-alloc call keeps the kernel's scratch in a 16 MiB array inside the library and
allocates nothing; all it asks for is the input and output arrays.

What is checked here: the call produces the very same bits as two LB steps of nh_step (the tolerance the two-step tests
of test_gpu_parity.py use: none), on calls made back to back -- the second and third call find the previous call's ring,
flags and ticket in the shared array and must not be confused by them, also when the grid changes in between -- that
device memory in use does not move across a call, and that a lattice beyond the limit is refused with a message.

This file is named so that pytest collects it last: under `pytest -x` a failure here hides nothing that comes after.
It passes on its own in a fresh process (the first call then does the per-device set-up) and after the other tests.
"""
import numpy as np
import pytest

import nh_inputs as I

pytestmark = pytest.mark.gpu


def nh():
    import paper_2503_06610_b200 as m
    from paper_2503_06610_b200 import build
    build.build()
    return m


def reference_lattice(m, nx, ny, nz, precision, tau, g):
    """A lattice of the handle path with a non-trivial state: noisy director (so F^LC != 0), a few steps done."""
    lat = m.Lattice(nx=nx, ny=ny, nz=nz, tau=tau, K=0.015, pitch=9.0, xi=0.8, gamma1=1.3, g=g, fd_ratio=3, precision=precision)
    lat.set_options(m.OPT_LB_TWOSTEP)
    lat.set_director(I.noisy_homeotropic(nx, ny, nz, 0.1))
    lat.step(7)
    return lat


def field(lat, name, dtype):
    """All rows of one field as a device tensor [comps][nz][ny][nx] (the layout the no-alloc call takes)."""
    import torch
    nz, ny, nx = lat.shape
    buf = lat.new_rows_buffer(name, ny)
    lat.get_rows(name, 0, ny, buf)
    lat.synchronize()
    return buf.view(dtype).view(-1, nz, ny, nx)


@pytest.mark.parametrize("shape,precision", [((64, 48, 12), 1), ((128, 15, 5), 1), ((256, 24, 9), 2),
                                             ((64, 30, 11), 0), ((512, 6, 7), 3)])
def test_no_alloc_two_steps_match_the_handle_path_call_after_call(shape, precision):
    import torch
    m = nh()
    nx, ny, nz = shape
    tau, g = 0.7, (2e-6, -1e-6, 1.5e-6)
    dtype = torch.float32 if precision in (1, 2) else torch.float64
    lat = reference_lattice(m, nx, ny, nz, precision, tau, g)
    f_in = field(lat, "populations", dtype).clone()
    F = field(lat, "force", dtype).clone()
    assert float(F.abs().max()) > 0.0
    outs = [torch.zeros_like(f_in), torch.zeros_like(f_in)]
    torch.cuda.synchronize()
    src = f_in
    for call in range(3):
        # the handle path: two more LB steps with director and force frozen (r = 0)
        lat.step(2, 0)
        want = field(lat, "populations", dtype)
        dst = outs[call % 2]
        free_before = torch.cuda.mem_get_info()[0]
        m.lb_two_steps_noalloc(nx, ny, nz, precision, tau, g, src, F, dst)
        if call > 0:      # (the first call on a device may load the kernels)
            assert torch.cuda.mem_get_info()[0] == free_before, "device memory in use moved across the call"
        got = dst[:, 1:nz - 1]
        assert torch.equal(got, want[:, 1:nz - 1]), (shape, precision, call, float((got - want[:, 1:nz - 1]).abs().max()))
        assert torch.all(dst[:, 0] == 0) and torch.all(dst[:, nz - 1] == 0)      # plate layers are not written
        src = dst
    lat.close()


def test_no_alloc_without_force_and_on_a_side_stream():
    """F_lc = NULL is 'no LC force' (coupling bit0 off on the handle path); the work goes to the stream it is given."""
    import torch
    m = nh()
    nx, ny, nz, tau, g = 64, 20, 8, 0.9, (1e-6, 0.0, 0.0)
    lat = m.Lattice(nx=nx, ny=ny, nz=nz, tau=tau, K=0.015, g=g, fd_ratio=0, precision=1, coupling=2)
    lat.set_options(m.OPT_LB_ONESTEP)
    lat.set_director(I.noisy_homeotropic(nx, ny, nz, 0.1))
    lat.step(5)
    f_in = field(lat, "populations", torch.float32).clone()
    lat.step(2)
    want = field(lat, "populations", torch.float32)
    out = torch.empty_like(f_in)
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    m.lb_two_steps_noalloc(nx, ny, nz, 1, tau, g, f_in, None, out, stream=side)
    assert torch.equal(out[:, 1:nz - 1], want[:, 1:nz - 1])
    lat.close()


def test_no_alloc_refuses_what_does_not_fit():
    import torch
    m = nh()
    tiny = torch.zeros(256, dtype=torch.uint8, device="cuda")
    g = (0.0, 0.0, 0.0)
    # beyond the scratch: three ring planes of 19 * 512 * 514 floats are 60 MB
    with pytest.raises(m.NhError) as ei:
        m.lb_two_steps_noalloc(512, 512, 64, 1, 0.8, g, tiny, None, tiny[128:])
    assert ei.value.code == -1 and "beyond the static scratch" in str(ei.value) and "16777216" in str(ei.value)
    # FP64 doubles the plane: 256 x 256 fits in FP32 only
    with pytest.raises(m.NhError) as ei:
        m.lb_two_steps_noalloc(256, 256, 16, 0, 0.8, g, tiny, None, tiny[128:])
    assert ei.value.code == -1 and "beyond the static scratch" in str(ei.value)
    for bad, word in ((dict(nx=96), "nx must be"), (dict(nz=4), "nz >= 5"), (dict(tau=0.5), "tau"), (dict(precision=4), "precision")):
        kw = dict(nx=64, ny=8, nz=6, precision=1, tau=0.8)
        kw.update(bad)
        with pytest.raises(m.NhError) as ei:
            m.lb_two_steps_noalloc(kw["nx"], kw["ny"], kw["nz"], kw["precision"], kw["tau"], g, tiny, None, tiny[128:])
        assert ei.value.code == -1 and word in str(ei.value), str(ei.value)
    # in place is not possible: the second phase writes while the first still reads
    buf = torch.zeros(19 * 64 * 8 * 6, dtype=torch.float32, device="cuda")
    with pytest.raises(m.NhError) as ei:
        m.lb_two_steps_noalloc(64, 8, 6, 1, 0.8, g, buf, None, buf)
    assert "overlap" in str(ei.value)
