"""One small run of every kernel family of libnh_b200.so, for use under compute-sanitizer.

    compute-sanitizer --tool memcheck  --error-exitcode 1 python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck --error-exitcode 1 python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck --error-exitcode 1 python tests/sanitizer_cases.py
    compute-sanitizer --tool initcheck --error-exitcode 1 python tests/sanitizer_cases.py

(compute-sanitizer is closed on the pool this repository is built on -- profiles/r03_sanitizers.md -- so there the same
cases run in tests/test_gpu_poisoned_workspace.py on a workspace filled with NaN bit patterns between guard bands.)

Not a pytest file (pytest does not collect it): the parity tests say whether the numbers are right, this only drives
each kernel once on grids small enough for the tools -- two-step wavefront (one and several strips, FP32 and FP64, 64 ...
256 threads), the cooperative small-lattice launch, one LB step per launch, velocity store, the director kernels in their
tiled, four-cells-per-thread, element-wise-staged and one-thread-per-cell forms on aligned and ragged grids, force with and
without the Leslie stress, the three-constant energy, free plates, row pack / unpack, graph replay, the conversions of
nh_set_director / nh_get_fields, and the no-alloc entry point -- and checks that what comes back is finite.
It never touches the oracle.  Results of the last run: profiles/r03_sanitizers.md.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import nh_inputs as I  # noqa: E402

ALPHA = tuple(0.1 * a for a in I.MBBA_ALPHA)


def finite(lat, label):
    f = lat.get_fields()
    for k, v in f.items():
        assert np.isfinite(v).all(), (label, k)
    n2 = (f["n"] ** 2).sum(0)
    assert abs(n2 - 1.0).max() < 1e-4, label
    print("ok  %-58s launches=%d" % (label, lat.launch_count), flush=True)


def run(nh, label, shape, precision, steps, options=0, knobs=None, make=None, **params):
    nx, ny, nz = shape
    base = dict(nx=nx, ny=ny, nz=nz, tau=0.8, K=0.012, pitch=9.0, xi=0.7, gamma1=1.2, g=(2e-6, -1e-6, 1e-6), fd_ratio=3)
    base.update(params)
    lat = (make or nh.Lattice)(**dict(base, precision=precision))
    lat.set_options(options)
    if knobs:
        lat.debug_tune(**knobs)
    lat.set_director(I.noisy_homeotropic(nx, ny, nz, 0.1))
    for c in steps:
        lat.step(c)
    finite(lat, label)
    return lat


def lattice_cases(nh):
    """(label, shape, precision, step chunks, options, tuning knobs, extra parameters) of one small run per kernel family."""
    T, ONE = nh.OPT_LB_TWOSTEP, nh.OPT_LB_ONESTEP
    F32, F64, F32U, F64U = nh.FP32_SHIFTED, nh.FP64_SHIFTED, nh.FP32_UNSHIFTED, nh.FP64_UNSHIFTED
    k3 = (0.012, 0.006, 0.018)

    def case(label, shape, precision, steps, options=0, knobs=None, **params):
        return (label, shape, precision, steps, options, knobs, params)

    return [
        case("two-step wavefront FP32, 128 threads", (64, 16, 9), F32, [1, 6, 5], T),
        case("two-step wavefront FP32 unshifted, 4 strips, D=2 R=5", (64, 16, 9), F32U, [8], T, dict(lb2_strips=4, lb2_lead=2, lb2_ring=5)),
        case("two-step wavefront FP64, 256 threads", (128, 8, 7), F64, [7], T, dict(lb2_threads=256)),
        case("two-step wavefront FP32, 64 threads, block order", (64, 8, 7), F32, [6], T, dict(lb2_threads=64, lb2_blockorder=1)),
        case("two-step wavefront FP32, four cells per thread", (128, 8, 7), F32, [6], T, dict(lb2_cells=4)),
        case("two-step wavefront FP64 unshifted, one cell per thread", (64, 8, 6), F64U, [4], T, dict(lb2_cells=1)),
        case("cooperative small-lattice launch (20 steps per launch)", (16, 16, 8), F32, [40], 0, fd_ratio=20),
        case("one LB step per launch, ragged grid", (20, 12, 7), F64, [7], ONE),
        case("director four cells per thread + tiled force (FP32, nx=64)", (64, 20, 9), F32, [6], ONE),
        case("director and force tiled, 16-byte staging (FP64, nx=32)", (32, 20, 9), F64, [6], ONE),
        case("director and force tiled, element-wise staging (ragged)", (20, 12, 7), F32, [6], ONE),
        case("director and force tiled, NOVEC on an aligned grid", (64, 12, 7), F32, [6], ONE | nh.OPT_FD_NOVEC),
        case("director and force one thread per cell", (20, 12, 7), F64, [6], ONE | nh.OPT_FD_DIRECT),
        case("Leslie viscous stress, tiled", (32, 12, 7), F64, [6], ONE, alpha=ALPHA),
        case("Leslie viscous stress, one thread per cell", (20, 12, 7), F32, [6], ONE | nh.OPT_FD_DIRECT, alpha=ALPHA),
        case("three-constant energy, tiled", (32, 12, 7), F64, [6], ONE, K3=k3),
        case("three-constant energy + Leslie stress, tiled, ragged", (20, 12, 7), F32, [6], ONE, K3=k3, alpha=ALPHA),
        case("three-constant energy + Leslie stress, one thread per cell", (20, 12, 7), F64, [6], ONE | nh.OPT_FD_DIRECT, K3=k3, alpha=ALPHA),
        case("free plates + bulk anchoring W0", (32, 12, 7), F32, [6], ONE, anchoring=1, W0=1e-3),
        case("graph replay", (16, 16, 8), F64, [6, 6, 6], nh.OPT_GRAPH),
        case("per-launch timing events", (16, 16, 8), F32, [6], nh.OPT_TIMING),
    ]


def main():
    import torch
    import paper_2503_06610_b200 as nh
    from paper_2503_06610_b200 import build
    build.build()
    assert torch.cuda.is_available()
    torch.cuda.set_stream(torch.cuda.Stream())      # graph replay cannot capture the legacy default stream
    ONE, F32, F64 = nh.OPT_LB_ONESTEP, nh.FP32_SHIFTED, nh.FP64_SHIFTED
    for label, shape, precision, steps, options, knobs, params in lattice_cases(nh):
        run(nh, label, shape, precision, steps, options, knobs, **params).close()

    # ---- rows of a slab: pack, unpack, pairs; deferred force ----
    lat = run(nh, "rows: lattice", (32, 20, 7), F32, [4], ONE)
    for field in ("populations", "director", "velocity", "force"):
        one, two = lat.new_rows_buffer(field, 3), torch.empty(2 * lat.rows_bytes(field, 3), dtype=torch.uint8, device="cuda")
        lat.get_rows(field, 2, 3, one)
        lat.set_rows(field, 9, 3, one)
        lat.get_rows_pair(field, 0, 17, 3, two)
        lat.set_rows_pair(field, 17, 0, 3, two)
    lat.defer_force(True)
    lat.step(3)
    lat.update_force()
    finite(lat, "rows pack / unpack / pairs, deferred force")
    lat.close()

    # ---- the no-alloc entry point, twice, on two grids ----
    for shape, precision, dtype in (((64, 12, 7), F32, torch.float32), ((128, 6, 6), F64, torch.float64)):
        nx, ny, nz = shape
        f_in = torch.zeros((19, nz, ny, nx), dtype=dtype, device="cuda")
        F = torch.full((3, nz, ny, nx), 1e-7, dtype=dtype, device="cuda")
        f_out = torch.zeros_like(f_in)
        nh.lb_two_steps_noalloc(nx, ny, nz, precision, 0.8, (1e-6, 0.0, 0.0), f_in, F, f_out)
        nh.lb_two_steps_noalloc(nx, ny, nz, precision, 0.8, (1e-6, 0.0, 0.0), f_out, None, f_in)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(f_in).all()) and float(f_in.abs().max()) > 0.0
        print("ok  no-alloc entry point %dx%dx%d precision %d, two calls" % (nx, ny, nz, precision), flush=True)
    print("sanitizer cases done")


if __name__ == "__main__":
    main()
