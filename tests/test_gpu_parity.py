"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances are BASELINE.json's: FP64 relative L_inf <= 1e-10 on u and n after 100 steps; shifted
FP32 max|du|/max|u| <= 1e-3 and max|dn| <= 1e-4 after 1000 steps; the unshifted FP32 error is
reported (printed), not gated.
"""
import numpy as np
import pytest

import nh_inputs as I
from oracle import Oracle

pytestmark = pytest.mark.gpu

FP64_TOL = 1e-10
FP32_TOL_U = 1e-3
FP32_TOL_N = 1e-4


def nh():
    import paper_2503_06610_b200 as m
    from paper_2503_06610_b200 import build
    build.build()
    return m


def pair(p, precision, options=0):
    """(oracle, gpu lattice) for a config dict from nh_inputs.config()."""
    p = dict(p)
    d = p.pop("director")
    p.pop("steps", None)
    o = Oracle(**dict(p, precision=precision))
    o.set_director(d)
    g = nh().Lattice(**dict(p, precision=precision))
    if options:
        g.set_options(options)
    g.set_director(d)
    return o, g


def rel_linf(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


def compare(o, g, tol_u, tol_n, tol_f=None, label=""):
    fo, fg = o.get_fields(), g.get_fields()
    eu = rel_linf(fg["u"], fo["u"])
    en = np.abs(fg["n"] - fo["n"]).max()
    er = np.abs(fg["rho"] - fo["rho"]).max()
    ef = rel_linf(fg["F"], fo["F"]) if np.abs(fo["F"]).max() > 0 else np.abs(fg["F"]).max()
    print("%s t=%d  rel|du|=%.3e  max|dn|=%.3e  max|drho|=%.3e  rel|dF|=%.3e" % (label, o.time, eu, en, er, ef))
    assert g.time == o.time
    assert eu <= tol_u, (label, eu)
    assert en <= tol_n, (label, en)
    assert ef <= (tol_f if tol_f is not None else 100 * tol_u), (label, ef)
    return eu, en


@pytest.mark.parametrize("precision", [0, 3])
def test_config0_fp64(precision):
    """configs[0]: 16x16x8 noisy homeotropic channel, 200 steps, r = 1, FP64."""
    o, g = pair(I.config(0), precision)
    compare(o, g, 1e-300 + FP64_TOL, FP64_TOL, label="init")
    for _ in range(2):
        o.step(100)
        g.step(100)
        compare(o, g, FP64_TOL, FP64_TOL, label="cfg0 fp64 p%d" % precision)
    f = g.get_fields()
    for zz in (0, -1):  # plates: rho = 1, u = 0, F = 0, n = z_hat
        assert np.all(f["rho"][zz] == 1.0) and np.all(f["u"][:, zz] == 0.0) and np.all(f["F"][:, zz] == 0.0)
        assert np.all(f["n"][2, zz] == 1.0) and np.all(f["n"][:2, zz] == 0.0)


def test_config0_fp32_shifted_and_unshifted():
    """configs[0] in FP32: shifted within tolerance at 200 and 1000 steps; unshifted reported."""
    o, g = pair(I.config(0), 1)
    _, gu = pair(I.config(0), 2)
    for n in (200, 800):
        o.step(n)
        g.step(n)
        gu.step(n)
        compare(o, g, FP32_TOL_U, FP32_TOL_N, tol_f=2e-3, label="cfg0 fp32 shifted")
        fo, fu = o.get_fields(), gu.get_fields()
        print("cfg0 fp32 UNSHIFTED t=%d rel|du|=%.3e max|dn|=%.3e (reported, not gated)"
              % (o.time, rel_linf(fu["u"], fo["u"]), np.abs(fu["n"] - fo["n"]).max()))


def test_config1_skyrmion_tube():
    """configs[1]: 64x64x32 single skyrmion tube in Poiseuille flow, chiral (p = 16), r = 1, run as
    SURVEY.md section 8(d) prescribes: the oracle over the full 5000 LB steps (6.1e8 fluid-cell updates,
    about two minutes of host time, one run serving both precisions); FP64 gated at 1e-10 at step 100,
    shifted FP32 gated at (1e-3, 1e-4) at steps 100 and 1000 (north_star's bar); both reported at step
    5000 and gated there at 1e-8 (FP64: round-off growth only) and at the FP32 bars for u, 10x for n (five
    times the length north_star quotes its director bar at)."""
    p = I.config(1)
    assert p["steps"] == 5000 and p["fd_ratio"] == 1
    o, g64 = pair(p, 0)
    _, g32 = pair(p, 1)
    compare(o, g64, 1e-300 + FP64_TOL, FP64_TOL, label="init")
    for n in (100, 900, 4000):
        o.step(n)
        g64.step(n)
        g32.step(n)
        if o.time == 100:
            compare(o, g64, FP64_TOL, FP64_TOL, label="cfg1 fp64")
            compare(o, g32, FP32_TOL_U, FP32_TOL_N, label="cfg1 fp32 shifted")
        elif o.time == 1000:
            compare(o, g64, 1e-9, 1e-9, label="cfg1 fp64")
            compare(o, g32, FP32_TOL_U, FP32_TOL_N, label="cfg1 fp32 shifted")
        else:
            assert o.time == 5000
            compare(o, g64, 1e-8, 1e-8, label="cfg1 fp64 (full length)")
            compare(o, g32, FP32_TOL_U, 10 * FP32_TOL_N, tol_f=0.2, label="cfg1 fp32 shifted (full length)")


def test_config4_lattice_of_tubes_128():
    """configs[4] ("Oracle parity on the 128x128x64 case for 100 steps only"): the jittered
    lattice of tubes (nh_inputs.lattice_centres), r = 10, element by element: FP64 within 1e-10, shifted FP32
    within north_star's bars, at step 100."""
    p = I.config(4, size=(128, 128, 64))
    assert p["fd_ratio"] == 10
    o, g64 = pair(p, 0)
    _, g32 = pair(p, 1)
    o.step(100)
    g64.step(100)
    g32.step(100)
    compare(o, g64, FP64_TOL, FP64_TOL, label="cfg4 128x128x64 fp64")
    compare(o, g32, FP32_TOL_U, FP32_TOL_N, tol_f=5e-3, label="cfg4 128x128x64 fp32 shifted")


@pytest.mark.parametrize("r", [2, 5, 10])
@pytest.mark.parametrize("precision", [0, 1])
def test_fd_ratio_schedule(r, precision):
    """Sub-cycling: FD fires every r steps with Delta t_FD = r; step() called in
    uneven chunks must give the same result as the oracle's single call."""
    p = I.config(0, fd_ratio=r)
    o, g = pair(p, precision)
    o.step(60)
    for chunk in (1, 7, r, 60 - 8 - r):
        g.step(chunk)
    tol = (FP64_TOL, FP64_TOL) if precision == 0 else (FP32_TOL_U, FP32_TOL_N)
    compare(o, g, *tol, label="r=%d p%d" % (r, precision))
    # explicit n_fd overrides the default, 0 freezes the director
    n_before = g.get_fields(which=("n",))["n"].copy()
    o.step(9, 0)
    g.step(9, 0)
    assert np.array_equal(g.get_fields(which=("n",))["n"], n_before)
    o.step(6, 3)
    g.step(6, 3)
    compare(o, g, *tol, label="r=3 override p%d" % precision)


@pytest.mark.parametrize("gz", [0.0, 3e-6])
@pytest.mark.parametrize("shape", [(17, 5, 6), (1, 1, 3), (3, 2, 9), (130, 3, 4), (33, 31, 5)])
def test_ragged_and_degenerate_grids(shape, gz):
    """Sizes that are not multiples of the block / tile / vector width, down to a single fluid cell;
    with and without a wall-normal body acceleration (bounce-back under g_z, pin P14)."""
    nx, ny, nz = shape
    d = I.noisy_homeotropic(nx, ny, nz, 0.1)
    p = dict(nx=nx, ny=ny, nz=nz, tau=0.7, K=0.015, pitch=9.0, xi=0.8, gamma1=1.3,
             g=(2e-6, -1e-6, gz), fd_ratio=2, director=d)
    for precision, tol in ((0, (FP64_TOL, FP64_TOL)), (1, (FP32_TOL_U, FP32_TOL_N))):
        o, g = pair(p, precision)
        o.step(40)
        g.step(40)
        compare(o, g, *tol, tol_f=None if precision == 0 else 5e-3, label="ragged %s p%d" % (shape, precision))


@pytest.mark.parametrize("shape,anchoring,W0", [((64, 8, 5), 0, 0.0), ((128, 21, 9), 0, 0.0), ((192, 7, 12), 1, 2e-3),
                                                ((64, 40, 23), 1, -1e-3)])
def test_director_kernel_forms_agree(shape, anchoring, W0):
    """Rows that are a multiple of 64 cells take the four-cells-per-thread director kernels in FP32 (nh_fd_vec.cuh):
    against the oracle, and against the one-cell-per-thread tiled (NH_OPT_FD_NOVEC) and plain (NH_OPT_FD_DIRECT)
    forms of the same update, with ny not a multiple of the tile height, z-chunks of one plane, free plates and W0."""
    m = nh()
    nx, ny, nz = shape
    d = I.noisy_homeotropic(nx, ny, nz, 0.1)
    p = dict(nx=nx, ny=ny, nz=nz, tau=0.7, K=0.015, pitch=9.0, xi=0.8, gamma1=1.3, g=(2e-6, -1e-6, 1e-6), fd_ratio=2,
             anchoring=anchoring, W0=W0, director=d)
    o, g = pair(p, 1)
    o.step(40)
    g.step(40)
    compare(o, g, FP32_TOL_U, FP32_TOL_N, tol_f=5e-3, label="vec %s" % (shape,))
    ref = g.get_fields()
    for opt, knobs in ((m.OPT_FD_NOVEC, {}), (m.OPT_FD_DIRECT, {}), (0, dict(fd_planes=1)), (0, dict(fd_planes=3))):
        _, h = pair(p, 1, options=opt)
        h.debug_tune(**knobs)
        h.step(40)
        f = h.get_fields()
        assert rel_linf(f["u"], ref["u"]) < 1e-4 and np.abs(f["n"] - ref["n"]).max() < 2e-5, (shape, opt, knobs)
        if not opt:                      # the same kernels in other z-chunks: the same arithmetic per cell
            for k in ref:
                assert np.array_equal(f[k], ref[k]), (shape, knobs, k)


@pytest.mark.parametrize("coupling", [0, 1, 2])
def test_coupling_switches(coupling):
    p = I.config(0, coupling=coupling, fd_ratio=2)
    o, g = pair(p, 0)
    o.step(50)
    g.step(50)
    compare(o, g, FP64_TOL, FP64_TOL, label="coupling=%d" % coupling)


def test_poiseuille_closed_form_on_gpu():
    """The GPU itself reproduces the exact discrete Poiseuille profile (pin P1) in FP64."""
    nz, tau, gx = 8, 0.8, 1e-6
    nu = (tau - 0.5) / 3.0
    g = nh().Lattice(4, 3, nz, tau, g=(gx, 0, 0), fd_ratio=0, precision=0, coupling=0)
    g.step(4000, 0)
    ux = g.get_fields(which=("u",))["u"][0]
    z = np.arange(nz, dtype=np.float64)
    exact = gx / (2 * nu) * (z - 0.5) * (nz - 1.5 - z) + gx * (16 * (tau - 0.5) ** 2 - 3) / (24 * nu)
    assert np.abs(ux[1:-1] - exact[1:-1, None, None]).max() / exact.max() < 1e-10


@pytest.mark.parametrize("precision", [0, 1])
def test_hydrostatic_column_on_gpu(precision):
    """The GPU itself reproduces pin P14: under g = (0, 0, g_z) the fluid comes to rest with
    ln rho rising by 3 g_z per layer toward +z (PAPER.md:43 with u = 0, c_s^2 = 1/3 PAPER.md:127), element by
    element equal to the oracle; a non-uniform state under a wall-normal force."""
    nz, gz = 14, 1e-4
    p = dict(nx=5, ny=3, nz=nz, tau=0.8, K=0.0, g=(0.0, 0.0, gz), fd_ratio=0, coupling=0)
    o = Oracle(**dict(p, precision=precision))
    g = nh().Lattice(**dict(p, precision=precision))
    o.step(20000, 0)
    g.step(20000, 0)
    fo, fg = o.get_fields(), g.get_fields()
    rho = fg["rho"][1:-1, 0, 0]
    dln = np.diff(np.log(rho))
    tol = 2 * gz * gz if precision == 0 else 2e-3
    assert np.all(dln > 0.0) and np.abs(dln / (3 * gz) - 1.0).max() < tol
    assert np.abs(fg["u"]).max() <= (gz * gz if precision == 0 else 1e-6)
    assert np.abs(fg["rho"] - fo["rho"]).max() < (1e-12 if precision == 0 else 2e-6)


def test_invariants_long_run_fp32():
    """Properties that hold at any size: mass conserved, |n| = 1, plates fixed (FP32 shifted)."""
    p = I.config(1, fd_ratio=5)
    d = p.pop("director")
    p.pop("steps")
    g = nh().Lattice(**dict(p, precision=1))
    g.set_director(d)
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    g.step(2000)
    f = g.get_fields()
    assert abs((f["rho"][1:-1] - 1.0).sum()) / nf < 1e-7
    assert np.abs(np.sqrt((f["n"] ** 2).sum(0)) - 1.0).max() < 5e-7
    assert np.isfinite(f["u"]).all() and np.abs(f["u"]).max() < 0.01


def test_set_director_rejects_bad_input_and_keeps_state():
    m = nh()
    g = m.Lattice(8, 8, 6, 0.8, K=0.01, precision=0)
    d = I.noisy_homeotropic(8, 8, 6, 0.05)
    g.set_director(d)
    before = g.get_fields()
    bad = d.copy()
    bad[:, 2, 3, 4] = 0.0
    with pytest.raises(m.NhError) as ei:
        g.set_director(bad)
    assert ei.value.code == -1
    bad[0, 2, 3, 4] = np.nan
    with pytest.raises(m.NhError):
        g.set_director(bad)
    after = g.get_fields()
    for k in before:
        assert np.array_equal(before[k], after[k])
    with pytest.raises(m.NhError):
        g.step(-1)


def test_options_do_not_change_results():
    """Scheduling / kernel-variant switches are bit-neutral or within round-off of each other."""
    m = nh()
    ref = None
    for opt in (0, m.OPT_TIMING, m.OPT_GRAPH, m.OPT_FD_DIRECT, m.OPT_FD_NOVEC, m.OPT_FD_DIRECT | m.OPT_NO_SERPENTINE):
        p = I.config(0, fd_ratio=3)
        d = p.pop("director")
        p.pop("steps")
        import torch
        # graph replay needs a capturable stream (not the legacy default stream)
        stream = torch.cuda.Stream() if opt & m.OPT_GRAPH else None
        g = m.Lattice(stream=stream, **dict(p, precision=0))
        g.set_options(opt)
        g.set_director(d)
        g.step(50)
        g.step(31)
        if opt & m.OPT_GRAPH:          # replays of cached graphs, and a schedule that cycles through keys
            for _ in range(4):
                g.step(3)
            g.step(7)
            h = m.Lattice(**dict(p, precision=0))
            h.set_director(d)
            h.step(100)
            fg, fh = g.get_fields(), h.get_fields()
            for k in fg:
                assert np.array_equal(fg[k], fh[k]), k
            assert g.launch_count == h.launch_count and g.time == h.time == 100
            continue
        f = g.get_fields()
        if ref is None:
            ref = f
        else:
            assert rel_linf(f["u"], ref["u"]) < 1e-12 and np.abs(f["n"] - ref["n"]).max() < 1e-13, opt
        if opt & m.OPT_TIMING:
            ms, cnt = g.kernel_time("lb")
            assert cnt == 81 and ms > 0.0
            assert g.kernel_time("predictor")[1] == 27
        assert g.launch_count > 81


def test_check_finite_option_reports_a_nan_on_the_next_call():
    """NH_OPT_CHECK_FINITE: a NaN in the populations (planted through nh_set_rows) is found by the check that follows
    the steps of nh_step and makes every later call return NH_ENUMERIC; without the option nothing is reported, and a
    healthy run with the option on is bit-identical to one without."""
    import torch
    m = nh()
    p = I.config(0, fd_ratio=3)
    d = p.pop("director")
    p.pop("steps")
    for precision, dtype in ((1, torch.float32), (0, torch.float64)):
        ref = m.Lattice(**dict(p, precision=precision))
        ref.set_director(d)
        ref.step(12)
        g = m.Lattice(**dict(p, precision=precision))
        g.set_options(m.OPT_CHECK_FINITE)
        g.set_director(d)
        for _ in range(4):
            g.step(3)
        fr, fg = ref.get_fields(), g.get_fields()               # no error, same bits
        for k in fr:
            assert np.array_equal(fr[k], fg[k]), k
        for lat, checked in ((ref, False), (g, True)):
            rows = lat.new_rows_buffer("populations", 1)
            lat.get_rows("populations", 5, 1, rows)
            rows.view(dtype)[p["nx"] * 1 + 7] = float("nan")       # rest population of the cell (7, 5, 1): a fluid cell
            lat.set_rows("populations", 5, 1, rows)
            lat.step(2)                                          # asynchronous: this call cannot know yet
            lat.synchronize()
            if checked:
                for call in (lambda: lat.step(1), lambda: lat.get_fields(), lambda: lat.update_force()):
                    with pytest.raises(m.NhError) as ei:
                        call()
                    assert ei.value.code == -4 and "not finite" in str(ei.value)
            else:
                lat.step(1)
                assert not np.isfinite(lat.get_fields(which=("u",))["u"]).all()
            lat.close()


def test_unknown_option_bits_are_refused_and_option_changes_drop_graphs():
    """nh_set_options: bits that are not in include/nh.h (the launch-shape bits of earlier builds, now nh_debug_tune
    keys) are NH_EINVAL and leave the options as they were; switching a kernel-selecting bit while graphs are held
    drops them, and the steps that follow are those of a lattice that ran with plain launches throughout."""
    import torch
    m = nh()
    p = I.config(0, fd_ratio=3)
    d = p.pop("director")
    p.pop("steps")
    g = m.Lattice(stream=torch.cuda.Stream(), **dict(p, precision=0))
    g.set_options(m.OPT_GRAPH)
    for bad in (8, 1 << 26, 1 << 9, m.OPT_GRAPH | (1 << 30)):
        with pytest.raises(m.NhError) as ei:
            g.set_options(bad)
        assert ei.value.code == -1 and "unknown option bit" in str(ei.value)
    g.set_director(d)
    for _ in range(4):
        g.step(6)                                   # captured once, replayed three times
    g.set_options(m.OPT_GRAPH | m.OPT_FD_DIRECT)    # other FD kernels: the held graphs go
    for _ in range(4):
        g.step(6)
    g.set_options(m.OPT_GRAPH)
    g.step(6)
    h = m.Lattice(**dict(p, precision=0))
    h.set_director(d)
    h.step(24)
    h.set_options(m.OPT_FD_DIRECT)
    h.step(24)
    h.set_options(0)
    h.step(6)
    fg, fh = g.get_fields(), h.get_fields()
    for k in fg:
        assert np.array_equal(fg[k], fh[k]), k
    assert g.time == h.time == 54



@pytest.mark.parametrize("shape,r", [((64, 64, 32), 10), ((128, 5, 20), 7), ((32, 7, 9), 3), ((512, 4, 6), 2),
                                     ((1024, 3, 5), 2), ((64, 3, 3), 2), ((256, 9, 8), 4), ((16, 16, 8), 1),
                                     ((128, 24, 12), 3), ((512, 16, 9), 4), ((64, 40, 7), 2),
                                     # rows that do not tile into 512-cell pieces: CTAs of 160, 96, 224, 96 x 3, 160 x 2 threads
                                     ((320, 6, 9), 3), ((192, 10, 8), 2), ((448, 4, 7), 4), ((576, 3, 6), 2), ((640, 4, 6), 3)])
def test_two_step_kernel_is_bit_identical(shape, r):
    """The two-steps-per-sweep LB kernel (L2-resident plane ring, wavefront along z) does the same
    arithmetic per cell as the one-step kernel, so every field must agree bit for bit, whatever
    the lead / ring size / CTA shape, for uneven step() chunks and odd FD ratios; grids that do
    not tile into pieces (16 wide) silently take the one-step kernel."""
    m = nh()
    nx, ny, nz = shape
    d = I.noisy_homeotropic(nx, ny, nz, 0.1)
    p = dict(nx=nx, ny=ny, nz=nz, tau=0.7, K=0.015, pitch=9.0, xi=0.8, gamma1=1.3, g=(2e-6, -1e-6, 1.5e-6), fd_ratio=r)

    def run(precision, opt, chunks, **knobs):
        g = m.Lattice(**dict(p, precision=precision))
        g.set_options(opt)
        g.debug_tune(**knobs)
        g.set_director(d)
        for c in chunks:
            g.step(c)
        f = g.get_fields()
        g.close()
        return f

    T = m.OPT_LB_TWOSTEP
    variants = [(T, {}), (T | m.OPT_NO_SERPENTINE, {}), (T, dict(lb2_cells=1)), (T, dict(lb2_threads=256)), (T, dict(lb2_threads=64)),
                (T, dict(lb2_lead=1, lb2_ring=3)), (T, dict(lb2_lead=3, lb2_ring=12, lb2_blockorder=1)),
                (T, dict(lb2_blockorder=1, lb2_cells=1)), (T, dict(lb2_strips=2)),
                (T, dict(lb2_strips=4, lb2_lead=2, lb2_ring=5)), (T, dict(lb2_strips=8, lb2_blockorder=1)),
                # four consecutive cells per thread, 16-byte loads and stores (rows a multiple of 128 cells, FP32)
                (T, dict(lb2_cells=4)), (T, dict(lb2_cells=4, lb2_threads=128, lb2_strips=2))]
    for precision in (0, 1):
        ref = run(precision, m.OPT_LB_ONESTEP, [43])
        for opt, knobs in variants:
            if ny % knobs.get("lb2_strips", 1):
                continue                      # (the number of strips must divide ny)
            f = run(precision, opt, [1, 7, 20, 15], **knobs)
            for k in ref:
                assert np.array_equal(ref[k], f[k]), (shape, precision, hex(opt), knobs, k)


def test_wavefront_timeout_is_reported_by_the_next_calls():
    """A dependency wait of the two-step LB kernel that is not met within its bound ends the launch and makes
    every later call on the lattice fail with NH_ECUDA -- nh_step included, not only nh_get_fields.  Forced with
    the test hook that makes the waits ask for an epoch that never comes (include/nh_debug.h)."""
    m = nh()
    p = I.config(1, nx=64, ny=32, nz=14, fd_ratio=4)
    d = p.pop("director")
    p.pop("steps")
    g = m.Lattice(**dict(p, precision=1))
    g.set_options(m.OPT_LB_TWOSTEP)
    g.set_director(d)
    g.step(8)
    g.get_fields()                                      # fine so far
    g.debug_tune(lb2_fault=1, lb2_timeout_ms=20)
    g.step(2)                                           # asynchronous: this call cannot know yet
    g.synchronize()
    for call in (lambda: g.step(2), lambda: g.get_fields(), lambda: g.update_force(), lambda: g.set_director(d)):
        with pytest.raises(m.NhError) as ei:
            call()
        assert ei.value.code == -3 and "wavefront" in str(ei.value)
    g.close()
    # another lattice is unaffected
    h = m.Lattice(**dict(p, precision=1))
    h.set_options(m.OPT_LB_TWOSTEP)
    h.set_director(d)
    h.step(8)
    h.get_fields()


def test_config3_full_size_bench_configuration():
    """BASELINE.json configs[3] at FULL size (256x256x64, two tubes, r = 10), in the launch
    configurations bench.py times (default options: the two-step LB kernel in FP32; and one step
    per launch): FP64 within 1e-10 at 100 steps, shifted FP32 within (1e-3, 1e-4) at 100 and at 1000
    steps (north_star's bar), every output element compared with the oracle; the one-step run must
    equal the default FP32 run bit for bit.  One oracle run (about 90 s of host time) serves all of them."""
    m = nh()
    p = I.config(3)
    d = p.pop("director")
    p.pop("steps")
    o = Oracle(**dict(p, precision=0))
    o.set_director(d)
    g64 = m.Lattice(**dict(p, precision=0))
    g32 = m.Lattice(**dict(p, precision=1))
    g32w = m.Lattice(**dict(p, precision=1))
    g32w.set_options(m.OPT_LB_ONESTEP)
    for g in (g64, g32, g32w):
        g.set_director(d)
    for n in (100, 900):
        o.step(n)
        for g in (g64, g32, g32w):
            g.step(n)
        if o.time == 100:
            compare(o, g64, FP64_TOL, FP64_TOL, label="cfg3 full fp64")
        compare(o, g32, FP32_TOL_U, FP32_TOL_N, tol_f=5e-3, label="cfg3 full fp32 shifted")
        a, b = g32.get_fields(), g32w.get_fields()
        for k in a:
            assert np.array_equal(a[k], b[k]), k
    # the default picks the two-step kernel on this grid in FP32 and the one-step kernel in FP64
    assert g32.kernel_time("lb2")[1] > 0 and g32w.kernel_time("lb2")[1] == 0 and g64.kernel_time("lb2")[1] == 0
    f = g64.get_fields()
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    assert abs((f["rho"][1:-1] - 1.0).sum()) / nf < 1e-12          # mass (pin P2) on the GPU at full size
    assert np.abs(np.sqrt((f["n"] ** 2).sum(0)) - 1.0).max() < 1e-14


def test_config4_largest_grid_properties():
    """configs[4] at its largest size (512x512x128, 33.5 M cells, about 7 GB in FP32), far beyond what the oracle is
    run for: what holds at any size.  The default FP32 path there is the two-step LB kernel over FOUR y-strips; it must
    equal one LB step per launch bit for bit; mass is conserved, |n| = 1, the plates keep their values, and FP32
    stays close to the FP64 run of the same GPU path."""
    m = nh()
    p = I.config(4, size=(512, 512, 128))
    d = p.pop("director")
    p.pop("steps")
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    out = {}
    for name, precision, opt in (("two", 1, 0), ("one", 1, m.OPT_LB_ONESTEP), ("f64", 0, 0)):
        g = m.Lattice(**dict(p, precision=precision))
        g.set_options(opt)
        g.set_director(d)
        g.step(23)                                   # two director updates and an odd tail
        if name == "two":
            assert g.kernel_time("lb2")[1] > 0       # the two-step kernel is what ran
        out[name] = g.get_fields(which=("rho", "u", "n"))
        g.close()
    for k in out["two"]:
        assert np.array_equal(out["two"][k], out["one"][k]), k
    for name, tol_m, tol_n in (("two", 2e-7, 5e-7), ("f64", 1e-12, 1e-14)):
        f = out[name]
        assert abs((f["rho"][1:-1] - 1.0).sum()) / nf < tol_m
        assert np.abs(np.sqrt((f["n"] ** 2).sum(0)) - 1.0).max() < tol_n
        assert np.all(f["n"][2, 0] == 1.0) and np.all(f["u"][:, -1] == 0.0)
    assert rel_linf(out["two"]["u"], out["f64"]["u"]) < FP32_TOL_U
    assert np.abs(out["two"]["n"] - out["f64"]["n"]).max() < FP32_TOL_N


def test_config3_full_length_invariants():
    """configs[3] over its full 20 000 LB steps (far beyond what the oracle is run for): properties
    that hold at any length -- mass conserved, |n| = 1, plates fixed, no wavefront error -- and the
    shifted-FP32 run stays close to the FP64 run of the same GPU path."""
    m = nh()
    p = I.config(3)
    d = p.pop("director")
    steps = p.pop("steps")
    assert steps == 20000
    out = {}
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    for precision in (0, 1):
        g = m.Lattice(**dict(p, precision=precision))
        g.set_director(d)
        m0 = (g.get_fields(which=("rho",))["rho"][1:-1] - 1.0).sum()
        g.step(steps)
        f = g.get_fields()
        assert g.time == steps
        assert np.isfinite(f["u"]).all() and np.isfinite(f["n"]).all()
        assert abs((f["rho"][1:-1] - 1.0).sum() - m0) / nf < (1e-12 if precision == 0 else 2e-7)
        assert np.abs(np.sqrt((f["n"] ** 2).sum(0)) - 1.0).max() < (1e-14 if precision == 0 else 5e-7)
        assert np.all(f["n"][2, 0] == 1.0) and np.all(f["u"][:, 0] == 0.0) and np.all(f["F"][:, -1] == 0.0)
        out[precision] = f
        g.close()
    eu = rel_linf(out[1]["u"], out[0]["u"])
    en = np.abs(out[1]["n"] - out[0]["n"]).max()
    print("cfg3 20000 steps: FP32 vs FP64 on the GPU rel|du|=%.3e max|dn|=%.3e umax=%.3e" % (eu, en, np.abs(out[0]["u"]).max()))
    # 20x the length north_star gates at 1e-3 / 1e-4; measured 1.9e-3 / 3.9e-3 (deterministic arithmetic: 2x margin)
    assert eu < 5e-3 and en < 8e-3


def test_two_lattices_interleaved_on_two_streams():
    """The two-step kernel keeps its tickets, flags and launch numbers per lattice: two lattices stepped
    in alternation, each on its own stream, give what each gives alone."""
    import torch
    m = nh()
    p = I.config(1, fd_ratio=4, nx=64, ny=32, nz=14)
    d = p.pop("director")
    p.pop("steps")
    q = dict(p, g=(-3e-7, 2e-7, 0.0), tau=0.9)

    def alone(par):
        g = m.Lattice(**dict(par, precision=1))
        g.set_options(m.OPT_LB_TWOSTEP)
        g.set_director(d)
        g.step(37)
        f = g.get_fields()
        g.close()
        return f

    ra, rb = alone(p), alone(q)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ga = m.Lattice(stream=sa, **dict(p, precision=1))
    gb = m.Lattice(stream=sb, **dict(q, precision=1))
    for g in (ga, gb):
        g.set_options(m.OPT_LB_TWOSTEP)
        g.set_director(d)
    for chunk in (5, 9, 2, 13, 8):
        ga.step(chunk)
        gb.step(chunk)
    fa, fb = ga.get_fields(), gb.get_fields()
    for k in ra:
        assert np.array_equal(fa[k], ra[k]) and np.array_equal(fb[k], rb[k]), k


def test_chained_lb_launches_with_two_lattices_on_one_stream():
    """Consecutive one-step LB launches are chained by programmatic dependent launch.  Two
    lattices of different sizes stepped one LB step at a time in alternation on the SAME stream put the other
    lattice's launch between every two of a lattice's own: each must still give exactly what it gives alone,
    in plain launches and under graph replay."""
    import torch
    m = nh()
    p = I.config(1, fd_ratio=7, nx=96, ny=40, nz=12)
    d = p.pop("director")
    p.pop("steps")
    q = I.config(1, fd_ratio=3, nx=32, ny=24, nz=30, g=(-3e-7, 2e-7, 0.0), tau=0.9)
    e = q.pop("director")
    q.pop("steps")

    def alone(par, n0):
        g = m.Lattice(**dict(par, precision=1))
        g.set_options(m.OPT_LB_ONESTEP)
        g.set_director(n0)
        g.step(60)
        f = g.get_fields()
        g.close()
        return f

    ra, rb = alone(p, d), alone(q, e)
    for opt in (m.OPT_LB_ONESTEP, m.OPT_LB_ONESTEP | m.OPT_GRAPH):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            ga = m.Lattice(stream=st, **dict(p, precision=1))
            gb = m.Lattice(stream=st, **dict(q, precision=1))
            for g, n0 in ((ga, d), (gb, e)):
                g.set_options(opt)
                g.set_director(n0)
            for chunk in (1,) * 20 + (3, 2, 5, 10, 20):
                ga.step(chunk)
                gb.step(chunk)
            fa, fb = ga.get_fields(), gb.get_fields()
            ga.close()
            gb.close()
        for k in ra:
            assert np.array_equal(fa[k], ra[k]) and np.array_equal(fb[k], rb[k]), (opt, k)


@pytest.mark.parametrize("shape,r", [((64, 64, 16), 20), ((16, 16, 8), 50), ((33, 7, 5), 16), ((64, 64, 32), 0)])
def test_resident_multi_step_kernel_is_bit_identical(shape, r):
    """Small lattices take all the LB steps between two director updates in ONE cooperative launch
    (lb_resident_kernel, 16 steps or more): same arithmetic per cell as one launch per step, so bit for bit
    the same fields, for uneven step() chunks; and far fewer launches."""
    m = nh()
    nx, ny, nz = shape
    d = I.noisy_homeotropic(nx, ny, nz, 0.1)
    p = dict(nx=nx, ny=ny, nz=nz, tau=0.7, K=0.004, pitch=9.0, xi=0.8, gamma1=1.3, g=(2e-6, -1e-6, 0.0), fd_ratio=r)
    for precision in (0, 1, 2):
        out = []
        for opt, chunks in ((m.OPT_LB_ONESTEP, [137]), (0, [137]), (0, [1, 40, 17, 60, 19])):
            g = m.Lattice(**dict(p, precision=precision))
            g.set_options(opt)
            g.set_director(d)
            for c in chunks:
                g.step(c)
            out.append((g.get_fields(), g.launch_count))
            assert g.time == 137
            g.close()
        for f, _ in out[1:]:
            for k in out[0][0]:
                assert np.array_equal(out[0][0][k], f[k]), (shape, precision, k)
        # FP64 keeps 2 CTAs of 256 threads per SM resident (296 on 148 SMs): larger lattices stay on one launch per step
        if precision != 0 or nx * ny * (nz - 2) <= 296 * 256:
            assert out[1][1] < out[0][1] // 2
