"""GPU parity of the anchoring options (row f3 ingredients, readings G14,
G23): free plates (anchoring = 1) and the bulk anchoring W0, through the C ABI against the oracle."""
import numpy as np
import pytest

import nh_inputs as I
from oracle import Oracle

pytestmark = pytest.mark.gpu

FP64_TOL, FP32_TOL_U, FP32_TOL_N = 1e-10, 1e-3, 1e-4


def nh():
    import paper_2503_06610_b200 as m
    from paper_2503_06610_b200 import build
    build.build()
    return m


def rel_linf(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


@pytest.mark.parametrize("anchoring,W0", [(1, 0.0), (0, 2e-3), (1, 2e-3), (1, -1e-3)])
@pytest.mark.parametrize("precision", [0, 1])
def test_anchoring_options_match_the_oracle(anchoring, W0, precision):
    m = nh()
    tol_u, tol_n = (FP64_TOL, FP64_TOL) if precision == 0 else (FP32_TOL_U, FP32_TOL_N)
    for cfg, r, steps in ((0, 2, 100), (1, 1, 60)):
        p = I.config(cfg, fd_ratio=r, anchoring=anchoring, W0=W0)
        d = p.pop("director")
        p.pop("steps")
        for opt in ((0, m.OPT_FD_DIRECT) if cfg == 0 else (0,)):
            o = Oracle(**dict(p, precision=precision))
            g = m.Lattice(**dict(p, precision=precision))
            g.set_options(opt)
            o.set_director(d)
            g.set_director(d)
            assert np.abs(g.get_fields()["n"] - o.get_fields()["n"]).max() <= (1e-15 if precision == 0 else 1e-7)
            o.step(steps)
            g.step(steps)
            fo, fg = o.get_fields(), g.get_fields()
            eu, en = rel_linf(fg["u"], fo["u"]), np.abs(fg["n"] - fo["n"]).max()
            print("anchoring=%d W0=%g cfg%d p%d opt=%d rel|du|=%.3e max|dn|=%.3e" % (anchoring, W0, cfg, precision, opt, eu, en))
            assert eu <= tol_u and en <= tol_n
            if anchoring == 1:       # the plate layers follow the fluid
                assert np.array_equal(fg["n"][:, 0], fg["n"][:, 1]) and np.array_equal(fg["n"][:, -1], fg["n"][:, -2])
            else:
                assert np.all(fg["n"][2, 0] == 1.0) and np.all(fg["n"][2, -1] == 1.0)
            g.close()


def test_free_plates_with_viscous_stress_and_ragged_grid():
    nx, ny, nz = 33, 7, 6
    d = I.noisy_homeotropic(nx, ny, nz, 0.2)
    al = tuple(0.1 * a for a in (0.0373, -0.4496, -0.0203, 0.9318, 0.3084, -0.1617))
    p = dict(nx=nx, ny=ny, nz=nz, tau=0.7, K=0.015, pitch=9.0, xi=1.0946, gamma1=0.4293, g=(2e-6, -1e-6, 0.0),
             fd_ratio=2, alpha=al, anchoring=1, W0=1e-3)
    for precision, tu, tn in ((0, FP64_TOL, FP64_TOL), (1, FP32_TOL_U, FP32_TOL_N)):
        o = Oracle(**dict(p, precision=precision))
        g = nh().Lattice(**dict(p, precision=precision))
        o.set_director(d)
        g.set_director(d)
        o.step(40)
        g.step(40)
        fo, fg = o.get_fields(), g.get_fields()
        assert rel_linf(fg["u"], fo["u"]) <= tu and np.abs(fg["n"] - fo["n"]).max() <= tn
