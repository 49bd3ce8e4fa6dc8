"""GPU parity of the Leslie viscous stress in the force (row f1: Eqs. 3, 12):
the CUDA path through the C ABI against the oracle, element by element, same seeded inputs.
alpha = Table 1 (tests/golden/table1_mbba.txt) scaled by 0.1 in the stress (the explicit viscous
force must stay stable at FD ratios up to 5), gamma1 = alpha3 - alpha2 and xi = -(alpha3 + alpha2)/gamma1
from the unscaled numbers."""
import numpy as np
import pytest

import nh_inputs as I
from conftest import read_golden
from oracle import Oracle

pytestmark = pytest.mark.gpu

FP64_TOL, FP32_TOL_U, FP32_TOL_N = 1e-10, 1e-3, 1e-4


def nh():
    import paper_2503_06610_b200 as m
    from paper_2503_06610_b200 import build
    build.build()
    return m


def mbba(scale=0.1):
    t = {r[0]: float(r[1]) for r in read_golden("table1_mbba.txt")}
    a = np.array([t["alpha%d" % i] for i in range(1, 7)])
    gamma1 = a[2] - a[1]                 # unscaled: K r / gamma1 stays inside the explicit stability limit
    xi = -(a[2] + a[1]) / gamma1
    return tuple(a * scale), gamma1, xi


def rel_linf(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


def run_pair(p, d, precision, steps, options=0):
    o = Oracle(**dict(p, precision=precision))
    o.set_director(d)
    g = nh().Lattice(**dict(p, precision=precision))
    g.set_options(options)
    g.set_director(d)
    f0o, f0g = o.get_fields(), g.get_fields()
    o.step(steps)
    g.step(steps)
    return o.get_fields(), g.get_fields(), f0o, f0g


@pytest.mark.parametrize("r", [1, 5])
@pytest.mark.parametrize("precision", [0, 1])
def test_config0_with_viscous_stress(r, precision):
    al, gamma1, xi = mbba()
    p = I.config(0, fd_ratio=r, alpha=al, gamma1=gamma1, xi=xi)
    d = p.pop("director")
    p.pop("steps")
    m = nh()
    tol_u, tol_n = (FP64_TOL, FP64_TOL) if precision == 0 else (FP32_TOL_U, FP32_TOL_N)
    for opt in (0, m.OPT_FD_DIRECT):
        fo, fg, f0o, f0g = run_pair(p, d, precision, 100, opt)
        assert rel_linf(f0g["F"], f0o["F"]) <= (1e-12 if precision == 0 else 2e-4)   # force at set_director (u = 0)
        eu, en, ef = rel_linf(fg["u"], fo["u"]), np.abs(fg["n"] - fo["n"]).max(), rel_linf(fg["F"], fo["F"])
        print("visc cfg0 r=%d p%d opt=%d rel|du|=%.3e max|dn|=%.3e rel|dF|=%.3e" % (r, precision, opt, eu, en, ef))
        assert np.isfinite(fo["u"]).all()
        assert eu <= tol_u and en <= tol_n and ef <= 100 * tol_u
    # the viscous stress really is in there: the same run without it differs
    q = dict(p, alpha=(0.0,) * 6)
    fo0, _, _, _ = run_pair(q, d, precision, 100)
    assert rel_linf(fo0["u"], fo["u"]) > 1e-3


@pytest.mark.parametrize("coupling", [1, 2, 3])
def test_viscous_stress_with_coupling_switches(coupling):
    """coupling bit1 off: the director ignores the flow, but the viscous stress still needs u(t)."""
    al, gamma1, xi = mbba()
    p = I.config(0, fd_ratio=2, alpha=al, gamma1=gamma1, xi=xi, coupling=coupling)
    d = p.pop("director")
    p.pop("steps")
    fo, fg, _, _ = run_pair(p, d, 0, 60)
    assert rel_linf(fg["u"], fo["u"]) <= FP64_TOL and np.abs(fg["n"] - fo["n"]).max() <= FP64_TOL
    assert rel_linf(fg["F"], fo["F"]) <= 1e-8


@pytest.mark.parametrize("shape", [(17, 5, 6), (1, 1, 3), (33, 31, 5), (64, 64, 12)])
def test_viscous_stress_on_ragged_grids(shape):
    nx, ny, nz = shape
    al, gamma1, xi = mbba()
    d = I.noisy_homeotropic(nx, ny, nz, 0.1)
    p = dict(nx=nx, ny=ny, nz=nz, tau=0.7, K=0.015, pitch=9.0, xi=xi, gamma1=gamma1, g=(2e-6, -1e-6, 0.0),
             fd_ratio=2, alpha=al)
    for precision, tu, tn in ((0, FP64_TOL, FP64_TOL), (1, FP32_TOL_U, FP32_TOL_N)):
        fo, fg, _, _ = run_pair(p, d, precision, 40)
        assert rel_linf(fg["u"], fo["u"]) <= tu and np.abs(fg["n"] - fo["n"]).max() <= tn, (shape, precision)


def test_skyrmion_tube_with_viscous_stress():
    """configs[1] domain (64x64x32 tube, chiral) with the full force of Eq. 12, r = 2, 60 steps."""
    al, gamma1, xi = mbba()
    p = I.config(1, fd_ratio=2, alpha=al, gamma1=gamma1, xi=xi)
    d = p.pop("director")
    p.pop("steps")
    for precision, tu, tn in ((0, FP64_TOL, FP64_TOL), (1, FP32_TOL_U, FP32_TOL_N)):
        fo, fg, _, _ = run_pair(p, d, precision, 60)
        eu, en = rel_linf(fg["u"], fo["u"]), np.abs(fg["n"] - fo["n"]).max()
        print("visc cfg1 p%d rel|du|=%.3e max|dn|=%.3e" % (precision, eu, en))
        assert eu <= tu and en <= tn
