"""The paper's accuracy experiment (Figs. 2, 4) re-measured on its own test-case
parameters as far as the container allows (see test_gpu_frank3.test_paper_test_case_parameters):
56x56x16, MBBA's three Frank constants, P = 14, g = 2e-9, free plates, W0 = 1.5e-8, |u| ~ 1e-7, elastic
stress only (the explicit viscous force is unstable for Delta t_FD >= 10 in this scheme).

For Delta t_FD in {1, 10, 50, 250, 1000} at the matched time T = 2000 LB steps, for unshifted FP32, shifted
FP32 and FP64 on the GPU:
  eps   = sum |u - u_ref| / sum |u_ref| (Eq. 24, vector norms) against the ORACLE at Delta t_FD = 1, the
          paper's reference choice
  eps_r = the same against the ORACLE AT THE SAME Delta t_FD (isolates the arithmetic precision)
  dn    = max |n - n_ref(same Delta t_FD)|
Printed and written to gpurun_out/paper_case_sweep.md.  Gated: FP64 eps_r <= 1e-9; shifted FP32 eps_r <= 1e-3;
shifted FP32 beats unshifted FP32 at every ratio (the paper's claim).

test_paper_case_full_model: the same with the FULL model -- Leslie viscous stress included -- under reading G25 of
DESIGN.md ("We choose the same viscosity both in LBM and in FD": alpha4' = rho c_s^2 (tau - 1/2) = alpha4 / 2,
which fixes tau = 1/2 + 3 alpha4 / 2 = 1.898 for Table 1): with it the frozen alpha4' term stays below the limit that
pin V7 locates at every Delta t_FD, and the full model runs at Delta t_FD = 1, 5, 250, 1000, 5000 over T = 5000 steps
(the anisotropic alphas still leave an unstable window around Delta t_FD = 10 ... 50, profiles/r02_paper_case_sweep.md)."""
import os

import numpy as np
import pytest

import nh_inputs as I
from oracle import Oracle

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
MBBA = (0.0373, -0.4496, -0.0203, 0.9318, 0.3084, -0.1617)
RATIOS = (1, 10, 50, 250, 1000)
T_END = 2000


def eps24(u, ref):
    return float(np.sqrt(((u - ref) ** 2).sum(0)).sum() / np.sqrt((ref ** 2).sum(0)).sum())


def test_paper_case_precision_vs_fd_ratio():
    import paper_2503_06610_b200 as nh
    from paper_2503_06610_b200 import build
    build.build()
    nx, ny, nz, tau = 56, 56, 16, 1.0
    gamma1 = MBBA[2] - MBBA[1]
    xi = -(MBBA[2] + MBBA[1]) / gamma1
    d = I.skyrmion_tubes(nx, ny, nz, [((nx - 1) / 2.0, (ny - 1) / 2.0)], 7.0)
    base = dict(nx=nx, ny=ny, nz=nz, tau=tau, K3=(1.67e-7, 7.88e-8, 2.62e-7), pitch=14.0, xi=xi, gamma1=gamma1,
                g=(2e-9, 0.0, 0.0), anchoring=1, W0=1.5e-8)
    rows, ref1 = [], None
    for r in RATIOS:
        o = Oracle(**dict(base, fd_ratio=r, precision=0))
        o.set_director(d)
        o.step(T_END)
        fo = o.get_fields()
        if r == 1:
            ref1 = fo["u"].copy()
        for name, prec in (("fp32u", 2), ("fp32s", 1), ("fp64", 0)):
            g = nh.Lattice(**dict(base, fd_ratio=r, precision=prec))
            g.set_director(d)
            g.step(T_END)
            fg = g.get_fields()
            g.close()
            rows.append(dict(r=r, prec=name, eps=eps24(fg["u"], ref1), eps_r=eps24(fg["u"], fo["u"]),
                             dn=float(np.abs(fg["n"] - fo["n"]).max()), umax=float(np.abs(fo["u"]).max())))
    lines = ["", "### paper's test-case parameters: error vs Delta t_FD at T = %d LB steps (max|u| = %.2e)" % (T_END, rows[0]["umax"]), "",
             "| Delta t_FD | precision | eps (Eq. 24) vs oracle(Delta t_FD = 1) | eps vs oracle(same Delta t_FD) | max|dn| vs oracle(same) |",
             "|---|---|---|---|---|"]
    for q in rows:
        lines.append("| %d | %s | %.3e | %.3e | %.3e |" % (q["r"], q["prec"], q["eps"], q["eps_r"], q["dn"]))
    text = "\n".join(lines)
    print(text)
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "paper_case_sweep.md"), "w") as fh:
            fh.write(text + "\n")
    by = {(q["r"], q["prec"]): q for q in rows}
    for r in RATIOS:
        assert by[(r, "fp64")]["eps_r"] <= 1e-9
        assert by[(r, "fp32s")]["eps_r"] <= 1e-3
        assert by[(r, "fp32s")]["eps_r"] < by[(r, "fp32u")]["eps_r"]


RATIOS_FULL = (1, 5, 250, 1000, 5000)
T_FULL = 5000


def test_paper_case_full_model():
    import paper_2503_06610_b200 as nh
    from paper_2503_06610_b200 import build
    build.build()
    nx, ny, nz = 56, 56, 16
    tau = 0.5 + 1.5 * MBBA[3]                      # reading G25: rho c_s^2 (tau - 1/2) = alpha4' = alpha4 / 2
    alpha = list(MBBA)
    alpha[3] = MBBA[3] / 2.0
    gamma1 = MBBA[2] - MBBA[1]
    xi = -(MBBA[2] + MBBA[1]) / gamma1
    d = I.skyrmion_tubes(nx, ny, nz, [((nx - 1) / 2.0, (ny - 1) / 2.0)], 7.0)
    base = dict(nx=nx, ny=ny, nz=nz, tau=tau, K3=(1.67e-7, 7.88e-8, 2.62e-7), pitch=14.0, xi=xi, gamma1=gamma1,
                g=(2e-9, 0.0, 0.0), anchoring=1, W0=1.5e-8, alpha=tuple(alpha))
    rows, ref1 = [], None
    for r in RATIOS_FULL:
        o = Oracle(**dict(base, fd_ratio=r, precision=0))
        o.set_director(d)
        o.step(T_FULL)
        fo = o.get_fields()
        assert np.isfinite(fo["u"]).all() and np.abs(fo["u"]).max() < 1e-6, r      # stable under G25 at this ratio
        if r == 1:
            ref1 = fo["u"].copy()
        for name, prec in (("fp32u", 2), ("fp32s", 1), ("fp64", 0)):
            g = nh.Lattice(**dict(base, fd_ratio=r, precision=prec))
            g.set_director(d)
            g.step(T_FULL)
            fg = g.get_fields()
            g.close()
            rows.append(dict(r=r, prec=name, eps=eps24(fg["u"], ref1), eps_r=eps24(fg["u"], fo["u"]),
                             dn=float(np.abs(fg["n"] - fo["n"]).max()), umax=float(np.abs(fo["u"]).max())))
    lines = ["", "### paper's test case, FULL model (Leslie stress, reading G25: tau = %.4f, alpha4' = alpha4/2): error vs Delta t_FD "
             "at T = %d LB steps (max|u| = %.2e)" % (tau, T_FULL, rows[0]["umax"]), "",
             "| Delta t_FD | precision | eps (Eq. 24) vs oracle(Delta t_FD = 1) | eps vs oracle(same Delta t_FD) | max|dn| vs oracle(same) |",
             "|---|---|---|---|---|"]
    for q in rows:
        lines.append("| %d | %s | %.3e | %.3e | %.3e |" % (q["r"], q["prec"], q["eps"], q["eps_r"], q["dn"]))
    text = "\n".join(lines)
    print(text)
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "paper_case_full_model.md"), "w") as fh:
            fh.write(text + "\n")
    by = {(q["r"], q["prec"]): q for q in rows}
    for r in RATIOS_FULL:
        assert by[(r, "fp64")]["eps_r"] <= 1e-9
        assert by[(r, "fp32s")]["eps_r"] <= 1e-3          # measured 5e-7 ... 2e-5 (profiles/r02_paper_case_sweep.md)
        assert by[(r, "fp32s")]["eps_r"] < by[(r, "fp32u")]["eps_r"]


LONG = os.environ.get("NH_LONG_SWEEP", "")
RATIOS_LONG = (1, 5, 50, 250, 1000, 5000, 50000)


@pytest.mark.skipif(LONG in ("", "0"), reason="slow (minutes): set NH_LONG_SWEEP=1 (T = 5e4 vs the oracle and 2e5 vs GPU FP64) or 2 (adds T = 1e6)")
def test_paper_case_long_horizon():
    """The far end of the paper's sweep (Delta t_FD up to 50 000; the FP32 minimum at 250),
    elastic stress only, on the horizons this container can afford.  Table 1: T = 50 000 LB steps, reference = the ORACLE at
    Delta t_FD = 1 (2.2e9 cell updates).  Tables 2 (and 3): T = 2e5 (1e6), reference = the GPU's FP64 path at Delta t_FD = 1 --
    legitimate as a reference because its parity with the oracle is gated at 1e-10 (test_gpu_parity.py) and re-checked here at
    T = 50 000.  Reports eps of Eq. 24 per (Delta t_FD, precision); gates only what must hold at any horizon."""
    import paper_2503_06610_b200 as nh
    from paper_2503_06610_b200 import build
    build.build()
    nx, ny, nz, tau = 56, 56, 16, 1.0
    gamma1 = MBBA[2] - MBBA[1]
    xi = -(MBBA[2] + MBBA[1]) / gamma1
    d = I.skyrmion_tubes(nx, ny, nz, [((nx - 1) / 2.0, (ny - 1) / 2.0)], 7.0)
    base = dict(nx=nx, ny=ny, nz=nz, tau=tau, K3=(1.67e-7, 7.88e-8, 2.62e-7), pitch=14.0, xi=xi, gamma1=gamma1,
                g=(2e-9, 0.0, 0.0), anchoring=1, W0=1.5e-8)

    def gpu(r, prec, T):
        g = nh.Lattice(**dict(base, fd_ratio=r, precision=prec))
        g.set_director(d)
        g.step(T)
        f = g.get_fields(which=("u", "n"))
        g.close()
        return f

    text = []
    horizons = [(50000, "oracle")] + [(200000, "gpu")] + ([(1000000, "gpu")] if LONG == "2" else [])
    for T, ref_kind in horizons:
        if ref_kind == "oracle":
            o = Oracle(**dict(base, fd_ratio=1, precision=0))
            o.set_director(d)
            o.step(T)
            ref = o.get_fields()
            g64 = gpu(1, 0, T)
            parity = eps24(g64["u"], ref["u"])
            assert parity <= 1e-9, parity          # the GPU's FP64 path is a fair stand-in for the oracle further out
            ref_name = "the ORACLE at Delta t_FD = 1 (GPU FP64 at Delta t_FD = 1 differs from it by eps = %.2e)" % parity
        else:
            ref = gpu(1, 0, T)
            ref_name = "the GPU's FP64 path at Delta t_FD = 1"
        rows = []
        for r in RATIOS_LONG:
            if r > T:
                continue
            for name, prec in (("fp32u", 2), ("fp32s", 1), ("fp64", 0)):
                f = gpu(r, prec, T)
                assert np.isfinite(f["u"]).all() and np.isfinite(f["n"]).all(), (T, r, name)
                rows.append(dict(r=r, prec=name, eps=eps24(f["u"], ref["u"]), dn=float(np.abs(f["n"] - ref["n"]).max())))
        text += ["", "### elastic model, T = %d LB steps, reference = %s (max|u_ref| = %.2e)" % (T, ref_name, np.abs(ref["u"]).max()), "",
                 "| Delta t_FD | precision | eps (Eq. 24) vs reference | max|dn| vs reference |", "|---|---|---|---|"]
        text += ["| %d | %s | %.3e | %.3e |" % (q["r"], q["prec"], q["eps"], q["dn"]) for q in rows]
        by = {(q["r"], q["prec"]): q for q in rows}
        best = min((q for q in rows if q["prec"] == "fp32s"), key=lambda q: q["eps"])
        text += ["", "shifted FP32: smallest eps %.3e at Delta t_FD = %d" % (best["eps"], best["r"])]
        for r in RATIOS_LONG:
            if r <= T:
                assert by[(r, "fp32s")]["eps"] < by[(r, "fp32u")]["eps"] or by[(r, "fp64")]["eps"] > 0.1 * by[(r, "fp32u")]["eps"], (T, r)
                assert by[(r, "fp32s")]["eps"] <= max(1e-3, 2.0 * by[(r, "fp64")]["eps"]), (T, r)   # FP32 adds at most 1e-3 to the scheme's own error
    out = "\n".join(text)
    print(out)
    dest = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(dest):
        with open(os.path.join(dest, "paper_case_long.md"), "w") as fh:
            fh.write(out + "\n")
