"""Pins of the CPU oracle against what the paper and the mathematics fix (SURVEY.md 8(c) P1-P11,
plus P12 moment identities and P13 advected shear wave).  CPU only: -m "not gpu".

None of these retypes an oracle formula: each compares the oracle with a closed form, an
invariant, a brute-force definition or a printed constant.
"""
import math

import numpy as np
import pytest

import nh_inputs as I
from conftest import read_golden
from oracle import Oracle, director_rhs, elastic_force, elastic_stress, molecular_field

# D3Q19 table written out independently of the oracle's (order documented in oracle/nh_oracle.h)
E = np.array([(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1),
              (1, 1, 0), (-1, -1, 0), (1, -1, 0), (-1, 1, 0), (1, 0, 1), (-1, 0, -1), (1, 0, -1),
              (-1, 0, 1), (0, 1, 1), (0, -1, -1), (0, 1, -1), (0, -1, 1)], dtype=np.float64)


def weights_from_golden():
    w_of = {int(r[0]): float(r[2]) / float(r[3]) for r in read_golden("d3q19.txt")}
    mult = {int(r[0]): int(r[1]) for r in read_golden("d3q19.txt")}
    w = np.array([w_of[int(e @ e)] for e in E])
    for k, m in mult.items():
        assert int(sum(int(e @ e) == k for e in E)) == m
    return w


# ------------------------------------------------------------------------------------------
# LB side
# ------------------------------------------------------------------------------------------
def test_d3q19_constants_and_rest_state():
    """PAPER.md:127 weights; rest state f_i = w_i (Eq. 15 at rho = 1, u = 0); shifted rest = 0 (Eq. 19)."""
    w = weights_from_golden()
    assert abs(w.sum() - 1.0) < 1e-15
    assert np.allclose(np.einsum("i,ia,ib->ab", w, E, E), np.eye(3) / 3.0, atol=1e-15)  # c_s^2 = 1/3
    o = Oracle(4, 3, 5, tau=0.8, precision=2)
    f = o.get_populations()
    assert np.array_equal(f[:, 1:-1], np.broadcast_to(w[:, None, None, None], f[:, 1:-1].shape))
    o = Oracle(4, 3, 5, tau=0.8, precision=0)
    assert np.all(o.get_populations() == 0.0)


@pytest.mark.parametrize("nz,tau", [(8, 0.8), (8, 1.0), (12, 0.6), (10, 0.5 + math.sqrt(3.0) / 4.0)])
@pytest.mark.parametrize("precision", [0, 2])
def test_P1_poiseuille_closed_form(nz, tau, precision):
    """P1: LC coupling off, uniform g_x: the steady D3Q19-SRT-Guo-halfway-bounce-back profile is
    exactly u_x(z) = g/(2 nu) (z - 1/2)(nz - 3/2 - z) + g (16 (tau-1/2)^2 - 3)/(24 nu), rho = 1."""
    g = 1e-6
    nu = (tau - 0.5) / 3.0
    H = nz - 2
    o = Oracle(3, 2, nz, tau=tau, K=0.0, g=(g, 0, 0), fd_ratio=0, precision=precision, coupling=0)
    o.step(int(45 * H * H / nu / 9.87) + 200, 0)
    fld = o.get_fields()
    z = np.arange(nz, dtype=np.float64)
    exact = g / (2 * nu) * (z - 0.5) * (nz - 1.5 - z) + g * (16 * (tau - 0.5) ** 2 - 3) / (24 * nu)
    ux = fld["u"][0]
    scale = exact[1:-1].max()
    assert np.abs(ux[1:-1] - exact[1:-1, None, None]).max() / scale < 1e-10
    assert np.abs(fld["u"][1:]).max() < 1e-14 * scale / 1e-5
    assert np.abs(fld["rho"] - 1.0).max() < 1e-12
    assert np.all(ux[0] == 0.0) and np.all(ux[-1] == 0.0)
    # the wall sits half-way: the parabola part vanishes at z = 1/2 and z = nz - 3/2; the slip
    # vanishes at tau = 1/2 + sqrt(3)/4
    if abs(tau - (0.5 + math.sqrt(3.0) / 4.0)) < 1e-12:
        assert abs(ux[1, 0, 0] - g / (2 * nu) * 0.5 * (nz - 2.5)) / scale < 1e-10


def test_P2_mass_conservation_coupled_run():
    """P2: sum of delta rho is constant to round-off over a coupled LC + flow run."""
    p = I.config(0)
    d = p.pop("director")
    p.pop("steps")
    o = Oracle(**p)
    o.set_director(d)
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    m0 = (o.get_fields()["rho"][1:-1] - 1.0).sum()
    for _ in range(4):
        o.step(50)
        m = (o.get_fields()["rho"][1:-1] - 1.0).sum()
        assert abs(m - m0) <= 1e-12 * nf


def test_P3_shifted_equals_unshifted_in_fp64():
    """P3: in FP64 the shifted and unshifted schemes agree (paper: eps = 2.68e-9)."""
    p = I.config(0)
    d = p.pop("director")
    p.pop("steps")
    out = []
    for prec in (0, 2):
        o = Oracle(**dict(p, precision=prec))
        o.set_director(d)
        o.step(200)
        out.append(o.get_fields())
    du = np.sqrt(((out[0]["u"] - out[1]["u"]) ** 2).sum(0)).sum()
    eps = du / np.sqrt((out[0]["u"] ** 2).sum(0)).sum()  # Eq. 24
    assert eps < 1e-8
    assert np.abs(out[0]["n"] - out[1]["n"]).max() < 1e-10


def test_P12_one_step_moment_identities():
    """P12: after one step from a uniform equilibrium state the moments obey the textbook
    constraints of Guo forcing (sum S = 0, sum e S = F, sum e e S = uF + Fu) and of Eq. 15:
      rho' = 1,  j' = u0 + F,  Pi' = Pi0 - (Pi0 - Pi_eq(u))/tau + (1 - 1/(2 tau)) (uF + Fu),
    u = u0 + F/2.  Interior cell, uniform state, so streaming does not change it."""
    tau = 0.77
    g = np.array([3e-4, -2e-4, 1.5e-4])
    u0 = np.array([0.011, -0.007, 0.004])
    for prec in (0, 2):
        o = Oracle(4, 4, 9, tau=tau, g=tuple(g), fd_ratio=0, precision=prec, coupling=0)
        uf = np.zeros((3, 9, 4, 4))
        uf[:, 1:-1] = u0[:, None, None, None]
        o.set_velocity(uf)
        w = weights_from_golden()
        o.step(1, 0)
        f = o.get_populations()[:, 4, 2, 1] + (w if prec == 0 else 0.0)
        u = u0 + 0.5 * g
        assert abs(f.sum() - 1.0) < 1e-14
        assert np.abs(E.T @ f - (u0 + g)).max() < 1e-15
        Pi = np.einsum("i,ia,ib->ab", f, E, E)
        Pi0 = np.eye(3) / 3 + np.outer(u0, u0)
        Pieq = np.eye(3) / 3 + np.outer(u, u)
        expect = Pi0 - (Pi0 - Pieq) / tau + (1 - 0.5 / tau) * (np.outer(u, g) + np.outer(g, u))
        assert np.abs(Pi - expect).max() < 1e-15


@pytest.mark.parametrize("axis", [0, 1])
def test_P13_advected_shear_wave(axis):
    """P13: a transverse shear wave on a uniform drift U decays with nu k^2 and travels WITH the
    drift: u_t(s, t) = A sin(k (s - U t)) exp(-nu k^2 t) up to O(k^2) lattice corrections.
    Pins the direction of streaming along x and y and the viscosity nu = (tau - 1/2)/3
    (PAPER.md:137).  The plates are 20 cells from the mid-plane that is read, further than the
    momentum diffusion length sqrt(nu T) = 4.6, so they do not matter."""
    L, nz, tau, U, A, T = 32, 42, 0.9, 0.05, 1e-4, 160
    nu = (tau - 0.5) / 3.0
    k = 2 * math.pi / L
    nx, ny = (L, 4) if axis == 0 else (4, L)
    sv = np.arange(L, dtype=np.float64)
    s = sv[None, None, :] if axis == 0 else sv[None, :, None]
    u = np.zeros((3, nz, ny, nx))
    u[axis] = U
    u[1 - axis] = A * np.sin(k * s)  # polarised along the other in-plane axis
    u[:, 0] = 0.0
    u[:, -1] = 0.0
    o = Oracle(nx, ny, nz, tau=tau, fd_ratio=0, coupling=0)
    o.set_velocity(u)
    o.step(T, 0)
    fld = o.get_fields()["u"]
    got = fld[1 - axis, nz // 2]
    got = got[0, :] if axis == 0 else got[:, 0]
    assert abs(fld[axis, nz // 2].mean() - U) < 0.01 * U  # drift (almost) intact at the mid-plane
    a_s = 2.0 / L * (got * np.sin(k * sv)).sum()
    a_c = 2.0 / L * (got * np.cos(k * sv)).sum()
    phase = math.atan2(-a_c, a_s)  # got = amp * sin(k s - phase)
    assert abs(phase - k * U * T) < 0.01 * k * U * T  # moved downstream by U T
    amp = math.hypot(a_s, a_c)
    assert abs(amp / (A * math.exp(-nu * k * k * T)) - 1.0) < 0.01


@pytest.mark.parametrize("gz", [1e-4, -1e-4])
@pytest.mark.parametrize("tau", [0.8, 1.0])
def test_P14_hydrostatic_column_pins_the_z_orientation_of_streaming(gz, tau):
    """P14: LC coupling off, body acceleration along z only.  With u = 0 Eq. 1 reduces
    to c_s^2 d(rho)/dz = rho g_z with c_s^2 = 1/3: ln rho rises by 3 g_z per layer
    TOWARD +z for g_z > 0.  Populations move to x + e_i (Eq. 14 / Eq. 23 LHS)
    and are reflected at the plate between two nodes; a stream mirrored in z stacks
    the fluid on the other plate.  None of P1, P2, P3 (mirror-symmetric in z), P12 (uniform state)
    or P13 (x and y) would notice that.  Expected values are from the hydrostatic balance, with the
    O(g_z^2) lattice correction as the tolerance."""
    nz = 14
    o = Oracle(3, 2, nz, tau=tau, K=0.0, g=(0.0, 0.0, gz), fd_ratio=0, precision=0, coupling=0)
    # transient: after a few steps mass has moved along the acceleration, away from one plate, onto the other
    o.step(3, 0)
    rho = o.get_fields()["rho"][:, 0, 0]
    far, near = (nz - 2, 1) if gz > 0 else (1, nz - 2)
    assert rho[far] > 1.0 + abs(gz) and rho[near] < 1.0 - abs(gz)
    # steady state (acoustic modes damp with nu k^2; (nz-2)^2/nu ~ 1.4e3 steps, run 30x that)
    o.step(40000, 0)
    f = o.get_fields()
    rho = f["rho"][1:-1]
    assert np.abs(f["u"]).max() <= gz * gz  # at rest up to the O(g^2) lattice term (measured 0.25 g^2)
    dln = np.diff(np.log(rho[:, 0, 0]))
    assert np.all(dln * np.sign(gz) > 0.0)  # denser toward +z for g_z > 0, toward -z for g_z < 0
    assert np.abs(dln / (3.0 * gz) - 1.0).max() < 2.0 * gz * gz  # measured 0.75 g^2
    assert np.abs(rho - rho[:, :1, :1]).max() == 0.0  # uniform in x and y
    assert abs((rho - 1.0).sum()) < 1e-12 * rho.size  # mass (P2) under a wall-normal force


# ------------------------------------------------------------------------------------------
# FD side
# ------------------------------------------------------------------------------------------
def cdiff(a, axis):
    """Central difference along a periodic array axis (independent numpy restatement of Eq. 13)."""
    return 0.5 * (np.roll(a, -1, axis) - np.roll(a, 1, axis))


def curl_c(n):
    """n: [3][nz][ny][nx]; array axes (1, 2, 3) are (z, y, x)."""
    dx = lambda a: cdiff(a, 2)  # noqa: E731  (component arrays are [nz][ny][nx])
    dy = lambda a: cdiff(a, 1)  # noqa: E731
    dz = lambda a: cdiff(a, 0)  # noqa: E731
    return np.stack([dy(n[2]) - dz(n[1]), dz(n[0]) - dx(n[2]), dx(n[1]) - dy(n[0])])


def discrete_energy_periodic(n, K, q0):
    """E_d = sum_x [ K/2 sum_b |n(x+e_b) - n(x)|^2 + K q0 n.(curl_c n) ]  (reading G1/G2)."""
    e = 0.0
    for ax in (1, 2, 3):
        d = np.roll(n, -1, ax) - n
        e += 0.5 * K * (d * d).sum()
    e += K * q0 * (n * curl_c(n)).sum()
    return e


@pytest.mark.parametrize("case", ["no_flow", "flow_does_not_act_on_n"])
def test_P4_uniform_director_is_a_fixed_point(case):
    """P4: n = z_hat everywhere and no flow acting on n: R = 0, F^LC = 0, n stays exactly z_hat,
    |n| = 1 (a uniform director in shear is NOT a fixed point: flow alignment turns it, see P7)."""
    p = I.config(0)
    p.pop("director")
    p.pop("steps")
    over = dict(g=(0.0, 0.0, 0.0)) if case == "no_flow" else dict(coupling=1)
    o = Oracle(**dict(p, pitch=7.0, **over))
    o.set_director(I.uniform_director(p["nx"], p["ny"], p["nz"]))
    o.step(60)
    f = o.get_fields()
    assert np.all(f["n"][2] == 1.0) and np.all(f["n"][:2] == 0.0)
    assert np.all(f["F"] == 0.0)
    if case == "no_flow":
        assert np.all(f["u"] == 0.0) and np.all(f["rho"] == 1.0)
    else:
        assert f["u"][0].max() > 1e-6  # the flow did develop


@pytest.mark.parametrize("q0", [0.0, 0.37])
def test_P5_molecular_field_is_minus_energy_gradient(q0):
    """P5: h(x) = -dE_d/dn(x) by centred numerical differentiation on a 4^3 fully periodic grid."""
    K = 0.013
    n = I.random_unit_field(4, 4, 4)
    h = molecular_field(n, K, q0, periodic_z=True)
    eps = 1e-6
    worst = 0.0
    for c in range(3):
        for z in range(4):
            for y in range(4):
                for x in range(4):
                    npl = n.copy()
                    nmi = n.copy()
                    npl[c, z, y, x] += eps
                    nmi[c, z, y, x] -= eps
                    g = (discrete_energy_periodic(npl, K, q0) - discrete_energy_periodic(nmi, K, q0)) / (2 * eps)
                    worst = max(worst, abs(h[c, z, y, x] + g))
    assert worst < 5e-9 * K / 0.013


def test_P8_discrete_helix_closed_forms():
    """P8: n = (0, cos qx, sin qx): lap_7pt n = (2 cos q - 2) n, curl_c n = -sin q n, so
    h = K [(2 cos q - 2) + 2 q0 sin q] n exactly, R = 0 for any q0; with a uniform drift u_x the
    advection term alone remains: R = -u_x d_x n = -u_x sin q (0, -sin qx, cos qx)."""
    nx, K, q0 = 16, 0.02, 0.41
    q = 2 * math.pi / nx
    x = np.arange(nx, dtype=np.float64)[None, None, :] + np.zeros((4, 4, 1))
    n = np.stack([np.zeros_like(x), np.cos(q * x), np.sin(q * x)])
    h = molecular_field(n, K, q0, periodic_z=True)
    assert np.abs(h - K * ((2 * math.cos(q) - 2) + 2 * q0 * math.sin(q)) * n).max() < 1e-16
    u = np.zeros_like(n)
    R = director_rhs(n, u, K, q0, 0.7, 1.3, periodic_z=True)
    assert np.abs(R).max() < 1e-16
    u[0] = 0.03
    R = director_rhs(n, u, K, q0, 0.7, 1.3, periodic_z=True)
    expect = -0.03 * math.sin(q) * np.stack([np.zeros_like(x), -np.sin(q * x), np.cos(q * x)])
    assert np.abs(R - expect).max() < 1e-16
    # uniform stress => no force (P9, second half)
    assert np.abs(elastic_force(n, K, q0, periodic_z=True)).max() < 1e-16


def test_P7_flow_alignment_signs_and_leslie_angle():
    """P7: homogeneous shear u_x = gd z, K = 0, n = (cos th, 0, sin th):
    R.theta_hat = (gd/2)(xi cos 2th - 1), zero and stable at the Leslie angle.  With the MBBA values
    the paper prints (Table 1) the textbook angle tan^2 th_L = alpha3/alpha2 is 12.0 degrees."""
    a = {r[0]: float(r[1]) for r in read_golden("table1_mbba.txt")}
    gamma1 = a["alpha3"] - a["alpha2"]
    gamma2 = a["alpha3"] + a["alpha2"]
    xi = -gamma2 / gamma1                # reading G4
    thL = math.atan(math.sqrt(a["alpha3"] / a["alpha2"]))
    assert abs(math.degrees(thL) - 12.0) < 0.05
    gd = 2e-3
    nz = 7
    z = np.arange(nz, dtype=np.float64)[:, None, None] + np.zeros((1, 3, 3))
    u = np.stack([gd * z, np.zeros_like(z), np.zeros_like(z)])

    def rate(th, xi_):
        n = np.stack([np.full_like(z, math.cos(th)), np.zeros_like(z), np.full_like(z, math.sin(th))])
        R = director_rhs(n, u, 0.0, 0.0, xi_, 1.0, periodic_z=False)[:, 3, 1, 1]
        assert abs(R @ np.array([math.cos(th), 0.0, math.sin(th)])) < 1e-18  # R perpendicular to n
        assert R[1] == 0.0
        return R @ np.array([-math.sin(th), 0.0, math.cos(th)])

    for th in (0.0, 0.3, 1.1, -0.8, math.pi / 2):
        assert abs(rate(th, xi) - 0.5 * gd * (xi * math.cos(2 * th) - 1.0)) < 1e-17
    assert abs(rate(thL, xi)) < 1e-9 * gd            # stationary at the Leslie angle ...
    assert rate(thL + 0.05, xi) < 0 < rate(thL - 0.05, xi)   # ... and stable there
    assert rate(-thL + 0.05, xi) < 0 < rate(-thL - 0.05, xi) or abs(rate(-thL, xi)) < 1e-9 * gd
    # xi = 0: pure co-rotation with half the vorticity, clockwise for gd > 0 (tumbling)
    assert abs(rate(0.4, 0.0) + 0.5 * gd) < 1e-17


def test_P9_net_elastic_force_vanishes_on_a_periodic_grid():
    """P9: F = div sigma telescopes: sum_x F = 0 to round-off for any unit field."""
    n = I.random_unit_field(6, 5, 4)
    F = elastic_force(n, 0.02, 0.3, periodic_z=True)
    assert np.abs(F).max() > 1e-3
    assert np.abs(F.sum(axis=(1, 2, 3))).max() < 1e-15


def smooth_unit_field(L):
    s = 2 * math.pi * np.arange(L, dtype=np.float64) / L
    z, y, x = np.meshgrid(s, s, s, indexing="ij")
    v = np.stack([0.6 * np.sin(x) + 0.3 * np.cos(y + z), 0.5 * np.cos(x - y) + 0.4 * np.sin(z),
                  1.0 + 0.3 * np.sin(y) * np.cos(z) + 0.2 * np.cos(x)])
    return v / np.sqrt((v * v).sum(0))


def test_P10_stress_divergence_identity():
    """P10: d_b sigma_ab = -d_a f - h_c d_a n_c (Eq. 6 with the energy of G1) holds to O(dx^2) on a
    smooth field; pins sign and index order of sigma (the chiral part is not symmetric)."""
    K, q0l = 0.02, 0.35
    errs = []
    for L in (32, 64):
        n = smooth_unit_field(L)
        dxl = 2 * math.pi / L            # grid spacing in the field's own length unit
        q0 = q0l * dxl                   # keeps q0 * (length unit) fixed under refinement
        F = elastic_force(n, K, q0, periodic_z=True)
        h = molecular_field(n, K, q0, periodic_z=True)
        grad = [np.stack([cdiff(n[c], ax) for c in range(3)]) for ax in (2, 1, 0)]  # grad[a][c] = d_a n_c
        fdens = 0.5 * K * sum((g * g).sum(0) for g in grad) + K * q0 * (n * curl_c(n)).sum(0)
        rhs = np.stack([-cdiff(fdens, ax) - (h * grad[a]).sum(0) for a, ax in enumerate((2, 1, 0))])
        errs.append(np.abs(F - rhs).max() / np.abs(F).max())
    assert errs[0] < 0.2 and errs[1] < errs[0] / 3.4  # second order; a wrong sign gives ~2
    # the chiral part: -K q0 eps_{mu b c} n_mu d_a n_c = +K q0 (n x d_a n)_b, not symmetric in (a, b)
    n = smooth_unit_field(16)
    s = elastic_stress(n, K, 0.3, periodic_z=True)
    s0 = elastic_stress(n, K, 0.0, periodic_z=True)
    assert np.abs(s0 - s0.transpose(1, 0, 2, 3, 4)).max() < 1e-17          # one-constant part symmetric
    grad = [np.stack([cdiff(n[c], ax) for c in range(3)]) for ax in (2, 1, 0)]
    chir = np.stack([np.cross(n, g, axis=0) for g in grad])                 # chir[a][b] = (n x d_a n)_b
    assert np.abs((s - s0) - K * 0.3 * chir).max() < 1e-16


# ------------------------------------------------------------------------------------------
# time stepping, schedule, error behaviour
# ------------------------------------------------------------------------------------------
def plate_energy(n, K, q0):
    """Discrete Frank energy between fixed plates: bonds (K/2)|n(x+e_b) - n(x)|^2 over every pair of
    neighbours with at least one fluid cell (x, y periodic; z bonds include those to the plate
    layers) plus K q0 n.curl_c n summed over the fluid cells."""
    e = 0.0
    fl = n[:, 1:-1]
    for ax in (2, 3):
        d = np.roll(fl, -1, ax) - fl
        e += 0.5 * K * (d * d).sum()
    d = n[:, 1:] - n[:, :-1]
    e += 0.5 * K * (d * d).sum()
    if q0 != 0.0:
        dz = lambda a: 0.5 * (a[2:] - a[:-2])                                   # noqa: E731
        dy = lambda a: 0.5 * (np.roll(a, -1, 1) - np.roll(a, 1, 1))[1:-1]       # noqa: E731
        dx = lambda a: 0.5 * (np.roll(a, -1, 2) - np.roll(a, 1, 2))[1:-1]       # noqa: E731
        curl = np.stack([dy(n[2]) - dz(n[1]), dz(n[0]) - dx(n[2]), dx(n[1]) - dy(n[0])])
        e += K * q0 * (fl * curl).sum()
    return e


@pytest.mark.parametrize("K,r,pitch", [(0.01, 1, 0.0), (0.01, 10, 0.0), (0.01, 16, 0.0), (0.02, 2, 16.0)])
def test_P6_energy_descends_in_flow_free_relaxation(K, r, pitch):
    """P6: with the flow switched off the update is a projected gradient flow of the discrete Frank
    energy: it decreases monotonically while |n| = 1 (explicit-stability range K r / gamma1 <= 1/6)."""
    nx, ny, nz = 12, 10, 8
    if pitch > 0:
        d = I.skyrmion_tubes(nx, ny, nz, [((nx - 1) / 2, (ny - 1) / 2)], 4.5)
    else:
        d = I.noisy_homeotropic(nx, ny, nz, 0.05)
    o = Oracle(nx, ny, nz, tau=0.8, K=K, pitch=pitch, xi=0.5, gamma1=1.0, fd_ratio=r, coupling=0)
    o.set_director(d)
    q0 = 2 * math.pi / pitch if pitch > 0 else 0.0
    e_prev = plate_energy(o.get_fields()["n"], K, q0)
    e0 = e_prev
    for _ in range(30):
        o.step(r)
        n = o.get_fields()["n"]
        e = plate_energy(n, K, q0)
        assert e < e_prev
        assert np.abs((n * n).sum(0) - 1.0).max() < 1e-15
        e_prev = e
    assert e_prev < 0.9 * e0


def test_P11_heun_is_second_order():
    """P11 (PAPER.md:251 'typically second-order'): flow-free relaxation to a fixed physical time with
    Delta t_FD = 4, 2, 1: the differences shrink by a factor 4."""
    nx, ny, nz = 10, 8, 8
    d = I.skyrmion_tubes(nx, ny, nz, [((nx - 1) / 2, (ny - 1) / 2)], 4.0)
    res = {}
    for r in (4, 2, 1):
        o = Oracle(nx, ny, nz, tau=0.8, K=0.02, pitch=12.0, xi=0.5, gamma1=1.0, fd_ratio=r, coupling=0)
        o.set_director(d)
        o.step(16)
        res[r] = o.get_fields()["n"]
    ratio = np.abs(res[4] - res[2]).max() / np.abs(res[2] - res[1]).max()
    assert 3.4 < ratio < 5.0  # first order would give 2, third order 8


def test_schedule_and_heun_composition():
    """Fig. 1 / PAPER.md:204 (reading G10): the FD update fires after the LB step that makes t a
    multiple of r, with Delta t_FD = r; and one update is the predictor-corrector of PAPER.md:105-112
    composed from the RHS routine: n_P = nrm(n + r k1), n' = nrm(n + r (k1 + k2)/2)."""
    nx, ny, nz, r = 8, 6, 7, 5
    K, xi, gamma1, pitch = 0.015, 0.6, 1.2, 9.0
    q0 = 2 * math.pi / pitch
    d = I.skyrmion_tubes(nx, ny, nz, [((nx - 1) / 2, (ny - 1) / 2)], 3.0)
    o = Oracle(nx, ny, nz, tau=0.9, K=K, pitch=pitch, xi=xi, gamma1=gamma1, g=(1e-5, 0, 0), fd_ratio=r)
    o.set_director(d)
    n0 = o.get_fields()["n"]
    F0 = o.get_fields()["F"]
    assert np.array_equal(F0, elastic_force(n0, K, q0))           # G9: force from the initial director
    o.step(r - 1)
    assert o.time == r - 1
    assert np.array_equal(o.get_fields()["n"], n0) and np.array_equal(o.get_fields()["F"], F0)
    o.step(1)
    f = o.get_fields()
    assert not np.array_equal(f["n"], n0)
    # recompute the update from the velocity the oracle itself saw: u(t = r) with the OLD force.
    o2 = Oracle(nx, ny, nz, tau=0.9, K=K, pitch=pitch, xi=xi, gamma1=gamma1, g=(1e-5, 0, 0), fd_ratio=0)
    o2.set_director(d)
    o2.step(r, 0)
    u = o2.get_fields()["u"]

    def nrm(v):
        out = v / np.sqrt((v * v).sum(0))
        out[:, 0] = n0[:, 0]
        out[:, -1] = n0[:, -1]
        return out

    k1 = director_rhs(n0, u, K, q0, xi, gamma1)
    nP = nrm(n0 + r * k1)
    k2 = director_rhs(nP, u, K, q0, xi, gamma1)
    n1 = nrm(n0 + 0.5 * r * (k1 + k2))
    assert np.abs(f["n"] - n1).max() < 1e-15
    assert np.abs(f["F"] - elastic_force(n1, K, q0)).max() < 1e-17
    # explicit n_fd overrides params.fd_ratio; n_fd = 0 freezes the director
    o.step(7, 0)
    assert np.array_equal(o.get_fields()["n"], f["n"])


def test_plates_stay_fixed_and_set_director_normalises():
    """solid node values fixed (n = z_hat, u = 0); set_director normalises its input."""
    p = I.config(0)
    d = p.pop("director") * 1.7
    p.pop("steps")
    o = Oracle(**p)
    o.set_director(d)
    n = o.get_fields()["n"]
    assert np.abs((n * n).sum(0) - 1.0).max() < 1e-15
    o.step(20)
    f = o.get_fields()
    for zz in (0, -1):
        assert np.all(f["n"][2, zz] == 1.0) and np.all(f["n"][:2, zz] == 0.0)
        assert np.all(f["u"][:, zz] == 0.0) and np.all(f["F"][:, zz] == 0.0) and np.all(f["rho"][zz] == 1.0)


def test_invalid_arguments_are_rejected():
    from oracle import OracleError
    for bad in (dict(tau=0.5), dict(nz=2), dict(gamma1=0.0), dict(K=-1.0), dict(fd_ratio=-1), dict(W0=float("nan")),
                dict(anchoring=2)):
        kw = dict(nx=4, ny=4, nz=5, tau=0.8)
        kw.update(bad)
        with pytest.raises(OracleError):
            Oracle(**kw)
    o = Oracle(4, 4, 5, tau=0.8)
    with pytest.raises(OracleError):
        o.set_director(np.zeros((3, 5, 4, 4)))
    with pytest.raises(OracleError):
        o.step(-1)
