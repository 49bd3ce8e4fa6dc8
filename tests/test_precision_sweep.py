"""BASELINE.json configs[2]: the precision sweep (row a15 of SURVEY.md section 8a).

Unshifted FP32 vs shifted FP32 vs FP64 on the config-0 domain (16x16x8 noisy homeotropic channel),
FD/LB ratios r in {1, 2, 5, 10, 20, 50}, body forces g_x in {1e-7, 1e-6}, run to the common time
T = 1000 LB steps.  Reported per case (printed, and written to gpurun_out/precision_sweep.md when
that folder exists):
  (i)  L_inf of u (relative to max|u|) and of n against the ORACLE AT THE SAME r  -> isolates precision
  (ii) the paper's eps (Eq. 24: sum|u - u_ref| / sum|u_ref|) against the ORACLE AT r = 1,
       the paper's reference choice                             -> adds the sub-cycling error
K = 0.01 is beyond the explicit stability limit of the Heun step for r = 20, 50 (K r / gamma1 > 1/6,
DESIGN.md reading G20): those rows are reported as such, not gated; the supplementary sweep with
K = 1e-3 is stable at every ratio.

Gated: FP64 rel L_inf <= 1e-9 and shifted FP32 within north_star's (1e-3, 1e-4) on every stable
case; shifted FP32 is more accurate in u than unshifted FP32 at the low body force (the paper's
claim) on every stable case.
"""
import os

import numpy as np
import pytest

import nh_inputs as I
from oracle import Oracle

pytestmark = pytest.mark.gpu

RATIOS = (1, 2, 5, 10, 20, 50)
FORCES = (1e-7, 1e-6)
T_END = 1000
PREC = (("fp32u", 2), ("fp32s", 1), ("fp64", 0))
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _fields(obj):
    f = obj.get_fields()
    return f["u"], f["n"]


def _sweep(K):
    import paper_2503_06610_b200 as nh
    from paper_2503_06610_b200 import build
    build.build()
    rows = []
    for gx in FORCES:
        ref1 = None
        for r in RATIOS:
            p = I.config(2, K=K, g=(gx, 0.0, 0.0), fd_ratio=r)
            d = p.pop("director")
            p.pop("steps")
            o = Oracle(**dict(p, precision=0))
            o.set_director(d)
            o.step(T_END)
            uo, no = _fields(o)
            if r == 1:
                ref1 = uo.copy()
            stable = bool(np.isfinite(uo).all() and np.isfinite(no).all()) and K * r / p["gamma1"] <= 1.0 / 6.0
            for name, prec in PREC:
                g = nh.Lattice(**dict(p, precision=prec))
                g.set_director(d)
                g.step(T_END)
                ug, ng = _fields(g)
                g.close()
                with np.errstate(all="ignore"):
                    eu = float(np.abs(ug - uo).max() / np.abs(uo).max())
                    en = float(np.abs(ng - no).max())
                    eps = float(np.abs(ug - ref1).sum() / np.abs(ref1).sum())
                rows.append(dict(K=K, gx=gx, r=r, prec=name, eu=eu, en=en, eps=eps, stable=stable,
                                 umax=float(np.abs(uo).max())))
    return rows


def _report(rows, title):
    lines = ["", "### " + title, "",
             "| g_x | r | precision | max|du|/max|u| vs oracle(r) | max|dn| vs oracle(r) | eps (Eq. 24) vs oracle(r=1) | note |",
             "|---|---|---|---|---|---|---|"]
    for q in rows:
        note = "" if q["stable"] else "beyond the explicit stability limit (K r/gamma1 > 1/6)"
        lines.append("| %g | %d | %s | %.3e | %.3e | %.3e | %s |" % (q["gx"], q["r"], q["prec"], q["eu"], q["en"], q["eps"], note))
    text = "\n".join(lines)
    print(text)
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "precision_sweep.md"), "a") as fh:
            fh.write(text + "\n")
    return text


@pytest.mark.parametrize("K", [0.01, 1e-3])
def test_precision_sweep(K):
    rows = _sweep(K)
    _report(rows, "configs[2] precision sweep, K = %g, T = %d LB steps, 16x16x8" % (K, T_END))
    by = {(q["gx"], q["r"], q["prec"]): q for q in rows}
    for gx in FORCES:
        for r in RATIOS:
            q64, q32s, q32u = by[(gx, r, "fp64")], by[(gx, r, "fp32s")], by[(gx, r, "fp32u")]
            if not q64["stable"]:
                continue
            assert q64["eu"] <= 1e-9 and q64["en"] <= 1e-9, q64
            assert q32s["eu"] <= 1e-3 and q32s["en"] <= 1e-4, q32s
            if gx == FORCES[0]:
                assert q32s["eu"] < q32u["eu"], (q32s, q32u)
    if K == 1e-3:
        assert all(q["stable"] for q in rows)
