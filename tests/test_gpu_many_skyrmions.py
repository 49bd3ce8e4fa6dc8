"""Second workload (single-GPU half): the paper's closing demonstration, a
320x320x16 cell with 20 randomly placed skyrmions at Delta t_FD = 250 in single precision (PAPER.md:284,
Fig. 6), on the test case's material (three Frank constants, free plates, W0).  The tubes
are nh_inputs' ansatz standing in for the ref.-[18] toron.  Through the C ABI against the oracle, element by
element, after 500 LB steps (two director updates)."""
import numpy as np
import pytest

import nh_inputs as I
from oracle import Oracle

pytestmark = pytest.mark.gpu


def test_many_skyrmion_demonstration_against_the_oracle():
    import paper_2503_06610_b200 as nh
    from paper_2503_06610_b200 import build
    build.build()
    p = I.many_skyrmions()
    d = p.pop("director")
    p.pop("steps")
    assert (p["nx"], p["ny"], p["nz"], p["fd_ratio"]) == (320, 320, 16, 250)
    o = Oracle(**dict(p, precision=0))
    o.set_director(d)
    o.step(500)
    fo = o.get_fields()
    assert np.abs(fo["n"] - d).max() > 1e-3                       # the director did move
    for prec, tol_u, tol_n in ((nh.FP64_SHIFTED, 1e-10, 1e-10), (nh.FP32_SHIFTED, 1e-3, 1e-4)):
        g = nh.Lattice(**dict(p, precision=prec))
        g.set_director(d)
        g.step(500)
        fg = g.get_fields()
        g.close()
        eu = np.abs(fg["u"] - fo["u"]).max() / np.abs(fo["u"]).max()
        en = np.abs(fg["n"] - fo["n"]).max()
        print("many skyrmions precision %d: max|du|/max|u| = %.3e  max|dn| = %.3e  max|u| = %.3e" % (prec, eu, en, np.abs(fo["u"]).max()))
        assert eu <= tol_u and en <= tol_n
        assert np.abs(np.sqrt((fg["n"] ** 2).sum(0)) - 1.0).max() <= (1e-12 if prec == nh.FP64_SHIFTED else 1e-6)
