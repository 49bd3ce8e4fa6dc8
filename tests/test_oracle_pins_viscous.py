"""Pins of the oracle's Leslie viscous stress (row f1 of SURVEY.md section 8f; Eqs. 3, 4, 12 of the
paper).  CPU only: -m "not gpu".

alpha values are the paper's Table 1 (tests/golden/table1_mbba.txt).

V1  homogeneous shear u_x = s z, K = 0, uniform director: every component of sigma^v worked out by
    hand from Eq. 3 with N = (xi n.D) projected (reading G22) -- for n along x, y, z and in the
    shear plane at 30 degrees; catches a swapped alpha2/alpha3 or alpha5/alpha6 and a wrong alpha1 contraction
V2  torque identity on random fields: eps_abc sigma^v_bc = (alpha3 - alpha2)/gamma1 (n x h)_a
    + [(alpha3 - alpha2) xi + (alpha6 - alpha5)] (n x (n.D))_a, exact algebra whatever the fields; with
    gamma1 = alpha3 - alpha2 and xi = -gamma2/gamma1 = -(alpha6 - alpha5)/gamma1 (Parodi) the viscous torque
    is exactly n x h: the balance of angular momentum the Ericksen-Leslie stress is built on
V3  the viscous force sums to zero on a fully periodic grid (divergence form telescopes)
V4  alpha4' alone on a sinusoidal shear wave u_x = a sin(k z): F_x = -(alpha4'/2) sin^2(k) u_x, the
    central difference applied twice; F_y = F_z = 0
V5  alpha all zero: the force is the elastic force bit for bit (the default path is untouched)
V6  Poiseuille flow with alpha4' only: the plateau velocity drops as the total viscosity rises,
    u_max(alpha4') / u_max(0) close to nu / (nu + alpha4'/2)  (Newtonian stress 2 mu D = alpha4 D)
V7  WHERE the explicit viscous force stops being stable when it is frozen for r LB steps:
    alpha4' alone on a transverse shear wave; amplification per FD period and its |G| = 1 crossing
    against the closed form that the scheme's own statements give (below)
"""
import math

import numpy as np
import pytest

import nh_inputs as I
from conftest import read_golden
from oracle import Oracle, elastic_force, lc_force, molecular_field, viscous_stress


def mbba():
    t = {r[0]: float(r[1]) for r in read_golden("table1_mbba.txt")}
    return np.array([t["alpha1"], t["alpha2"], t["alpha3"], t["alpha4"], t["alpha5"], t["alpha6"]])


def shear_field(nx, ny, nz, s):
    u = np.zeros((3, nz, ny, nx))
    u[0] = s * np.arange(nz, dtype=np.float64)[:, None, None]
    return u


def uniform(nx, ny, nz, v):
    v = np.asarray(v, dtype=np.float64)
    v = v / np.linalg.norm(v)
    n = np.empty((3, nz, ny, nx))
    n[:] = v[:, None, None, None]
    return n


@pytest.mark.parametrize("direction", ["x", "y", "z", "tilt"])
def test_V1_shear_stress_of_a_uniform_director_by_hand(direction):
    a1, a2, a3, a4, a5, a6 = mbba()
    xi, s = 1.0946, 3e-4
    nx, ny, nz = 4, 3, 7
    th = math.radians(30.0)
    nvec = {"x": (1, 0, 0), "y": (0, 1, 0), "z": (0, 0, 1), "tilt": (math.cos(th), 0, math.sin(th))}[direction]
    n = uniform(nx, ny, nz, nvec)
    sig = viscous_stress(n, shear_field(nx, ny, nz, s), K=0.0, q0=0.0, xi=xi, gamma1=0.4293, alpha=mbba())
    got = sig[:, :, 3, 1, 2]                       # an interior cell; the field is uniform there
    d = s / 2.0                                     # D_xz = D_zx
    exp = np.zeros((3, 3))
    if direction == "y":                            # n.D = 0, N = 0: only alpha4' D
        exp[0, 2] = exp[2, 0] = a4 * d
    elif direction == "x":                          # n.D = (0,0,d), N = xi (0,0,d)
        exp[0, 2] = (a3 * xi + a4 + a6) * d
        exp[2, 0] = (a2 * xi + a4 + a5) * d
    elif direction == "z":                          # n.D = (d,0,0), N = xi (d,0,0)
        exp[0, 2] = (a2 * xi + a4 + a5) * d
        exp[2, 0] = (a3 * xi + a4 + a6) * d
    else:
        c, w = math.cos(th), math.sin(th)
        nD = np.array([w * d, 0.0, c * d])          # n_m D_mb
        nnD = 2 * c * w * d
        A = xi * nD
        nv = np.array([c, 0.0, w])
        N = A - nv * (nv @ A)
        for a in range(3):
            for b in range(3):
                Dab = d if {a, b} == {0, 2} else 0.0
                exp[a, b] = (a1 * nv[a] * nv[b] * nnD + a2 * nv[b] * N[a] + a3 * nv[a] * N[b] + a4 * Dab
                             + a5 * nv[b] * nD[a] + a6 * nv[a] * nD[b])
    assert np.abs(got - exp).max() <= 1e-15 * max(1.0, np.abs(exp).max() / 1e-4)
    assert np.abs(exp).max() > 1e-5                 # the case is not trivially zero


def _cross(a, b):
    return np.stack([a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]])


def _central(f, axis):
    return 0.5 * (np.roll(f, -1, axis=axis) - np.roll(f, 1, axis=axis))


def test_V2_viscous_torque_identity_on_random_fields():
    rng = np.random.default_rng(5)
    nx = ny = nz = 5
    n = rng.normal(size=(3, nz, ny, nx))
    n /= np.sqrt((n ** 2).sum(0))
    u = 1e-3 * rng.normal(size=(3, nz, ny, nx))
    K, q0 = 0.013, 0.31
    al = mbba()
    gamma1 = al[2] - al[1]
    for xi in (0.7, -(al[5] - al[4]) / gamma1):
        sig = viscous_stress(n, u, K, q0, xi, gamma1, al, periodic_z=True)
        h = molecular_field(n, K, q0, periodic_z=True)
        # D from numpy's own central differences (axes: z = 1, y = 2, x = 3 of [c][z][y][x])
        du = np.stack([_central(u, 3), _central(u, 2), _central(u, 1)])    # du[b][c] = d_b u_c
        D = 0.5 * (du + du.transpose(1, 0, 2, 3, 4))
        nD = np.einsum("m...,mb...->b...", n, D)
        torque = np.stack([sig[1, 2] - sig[2, 1], sig[2, 0] - sig[0, 2], sig[0, 1] - sig[1, 0]])
        expect = (al[2] - al[1]) / gamma1 * _cross(n, h) + ((al[2] - al[1]) * xi + (al[5] - al[4])) * _cross(n, nD)
        assert np.abs(torque - expect).max() <= 1e-15 + 1e-12 * np.abs(expect).max()
    # with Parodi's xi the viscous torque is n x h alone
    assert np.abs(torque - _cross(n, h)).max() <= 1e-12 * np.abs(_cross(n, h)).max() + 1e-18


def test_V3_net_viscous_force_vanishes_on_a_periodic_grid():
    rng = np.random.default_rng(11)
    n = rng.normal(size=(3, 4, 5, 6))
    n /= np.sqrt((n ** 2).sum(0))
    u = 1e-3 * rng.normal(size=n.shape)
    F = lc_force(n, u, K=0.0, q0=0.0, xi=0.9, gamma1=0.43, alpha=mbba(), periodic_z=True)
    assert np.abs(F).max() > 1e-6
    assert np.abs(F.sum(axis=(1, 2, 3))).max() <= 1e-13 * np.abs(F).sum()


def test_V4_newtonian_part_on_a_shear_wave():
    nx, ny, nz = 3, 2, 12
    k = 2 * math.pi / nz
    z = np.arange(nz, dtype=np.float64)
    u = np.zeros((3, nz, ny, nx))
    u[0] = 2e-4 * np.sin(k * z)[:, None, None]
    n = uniform(nx, ny, nz, (0.3, -0.5, 0.8))
    a4 = 0.37
    F = lc_force(n, u, K=0.0, q0=0.0, xi=0.5, gamma1=1.0, alpha=(0, 0, 0, a4, 0, 0), periodic_z=True)
    assert np.abs(F[0] - (-(a4 / 2.0) * math.sin(k) ** 2 * u[0])).max() <= 1e-18
    assert np.abs(F[1:]).max() <= 1e-20


def test_V5_zero_alphas_leave_the_elastic_force_untouched():
    n = I.skyrmion_tubes(12, 12, 8, [(5.5, 5.5)], 4.0)
    u = 1e-3 * np.random.default_rng(2).normal(size=n.shape)
    a = lc_force(n, u, K=0.02, q0=0.4, xi=0.6, gamma1=1.0, alpha=(0.0,) * 6)
    b = elastic_force(n, K=0.02, q0=0.4)
    assert np.array_equal(a, b)
    p = I.config(0)
    d = p.pop("director")
    p.pop("steps")
    o0, o1 = Oracle(**p), Oracle(**dict(p, alpha=(0.0,) * 6))
    for o in (o0, o1):
        o.set_director(d)
        o.step(20)
    f0, f1 = o0.get_fields(), o1.get_fields()
    assert all(np.array_equal(f0[k], f1[k]) for k in f0)


def test_V6_extra_newtonian_viscosity_slows_poiseuille_flow():
    nz, tau, g = 18, 0.8, 1e-6
    nu = (tau - 0.5) / 3.0
    res = []
    for a4 in (0.0, 0.1):
        o = Oracle(3, 2, nz, tau=tau, K=0.0, g=(g, 0, 0), fd_ratio=1, coupling=1, alpha=(0, 0, 0, a4, 0, 0))
        o.step(12000)
        res.append(o.get_fields()["u"][0, :, 0, 0].max())
    ratio = res[1] / res[0]
    expect = nu / (nu + 0.1 / 2.0)
    # the FD viscous term sees u = 0 on the plate NODES (one spacing away), the LB wall is half-way:
    # the two agree to a few per cent on 16 fluid layers
    assert abs(ratio / expect - 1.0) < 0.05, (ratio, expect)


def frozen_force_model(L, tau, r, a4):
    """Amplification per FD period of the transverse shear wave u_y = a sin(k x), k = 2 pi / L, under the alpha4'
    force frozen for r LB steps, from the scheme as the paper states it, and the alpha4' at which it reaches -1:
      - the force is F = -(alpha4'/2) sin^2(k) u                      (Eq. 12's alpha4' D term with Eq. 13 twice: pin V4)
        evaluated from the velocity of Eq. 21, u = j + F_old/2        (rho = 1), and then frozen
      - a shear wave of the LB fluid decays by lam = exp(-nu k^2) per step, nu = (tau - 1/2)/3  (pin P13),
        and every step adds F to the momentum, half before and half after the step's decay (Guo forcing, Eq. 18)
    so with c = alpha4' sin^2(k)/2 and B = (1 + lam)/2 (1 - lam^r)/(1 - lam):
        F_n = -c (j_n + F_{n-1}/2),   j_{n+1} = lam^r j_n + B F_n
    a 2x2 linear map whose dominant eigenvalue is G; G = -1 at c = (1 + lam^r) / (B + (1 + lam^r)/2).
    Long waves only (lam is the hydrodynamic decay, right to O(k^2))."""
    nu, k = (tau - 0.5) / 3.0, 2.0 * math.pi / L
    lam = math.exp(-nu * k * k)
    lr = lam ** r
    B = 0.5 * (1.0 + lam) * (1.0 - lr) / (1.0 - lam)
    c = a4 * math.sin(k) ** 2 / 2.0
    tr, det = lr - c * B - c / 2.0, -(c / 2.0) * lr
    disc = math.sqrt(tr * tr - 4.0 * det)
    G = max(((tr - disc) / 2.0, (tr + disc) / 2.0), key=abs)
    a4_crit = 2.0 * (1.0 + lr) / (math.sin(k) ** 2 * (B + (1.0 + lr) / 2.0))
    return G, a4_crit


def oracle_amplification(L, tau, r, a4, periods=6, nz=82):
    """Ratio of the wave's amplitude at the mid-plane between the last two of `periods` FD updates.  The plates are 40
    cells from the plane that is read: what they seed (a z-structure with a larger discrete k^2, which goes unstable
    earlier) spreads by viscous diffusion, sqrt(nu T) < 4 cells here, and does not reach it."""
    k = 2.0 * math.pi / L
    x = np.arange(L, dtype=np.float64)
    u = np.zeros((3, nz, 2, L))
    u[1] = 1e-6 * np.sin(k * x)[None, None, :]
    u[:, 0] = 0.0
    u[:, -1] = 0.0
    o = Oracle(L, 2, nz, tau=tau, K=0.0, fd_ratio=r, coupling=1, alpha=(0, 0, 0, a4, 0, 0))
    o.set_velocity(u)
    amps = []
    for _ in range(periods):
        o.step(r)
        uy = o.get_fields()["u"][1, nz // 2, 0, :]
        amps.append(2.0 / L * (uy * np.sin(k * x)).sum())
    return amps[-1] / amps[-2]


@pytest.mark.parametrize("L,tau,r", [(16, 0.9, 10), (16, 0.9, 4), (32, 1.0, 20)])
def test_V7_stability_limit_of_the_frozen_viscous_force(L, tau, r):
    """With the force frozen over r steps the explicit alpha4' term over-corrects: the wave flips sign every FD update
    and grows once alpha4' exceeds a limit that FALLS with r (for r -> infinity: alpha4'/2 sin^2 k < nu k^2, the
    explicit viscosity must stay below the lattice's own).  The oracle crosses |G| = 1 where the closed form says."""
    _, a4c = frozen_force_model(L, tau, r, 0.0)
    # no extra viscosity: plain decay of the LB shear wave
    assert abs(oracle_amplification(L, tau, r, 0.0) / math.exp(-(tau - 0.5) / 3.0 * (2 * math.pi / L) ** 2 * r) - 1.0) < 0.01
    below, above = oracle_amplification(L, tau, r, 0.92 * a4c), oracle_amplification(L, tau, r, 1.08 * a4c)
    assert -1.0 < below < 0.0 and above < -1.0, (below, above, a4c)
    for f, got in ((0.92, below), (1.08, above)):
        G, _ = frozen_force_model(L, tau, r, f * a4c)
        assert abs(got / G - 1.0) < 0.04, (f, got, G)
    # the limit falls with r, towards 2 nu k^2 / sin^2 k
    assert frozen_force_model(L, tau, 8 * r, 0.0)[1] < a4c
    k = 2 * math.pi / L
    lam = math.exp(-(tau - 0.5) / 3.0 * k * k)
    assert frozen_force_model(L, tau, 10 ** 6, 0.0)[1] == pytest.approx(2.0 * (1.0 - lam) / math.sin(k) ** 2, rel=1e-9)
