"""Pins of the oracle's three-constant Frank energy (row f2 of SURVEY.md section 8f; Eqs. 6-8, 10 of the
paper; discrete form: DESIGN.md reading G24).  CPU only: -m "not gpu".

K11, K22, K33 are the paper's Table-1 values scaled to order 1e-2 (their ratios 1.67 : 0.788 : 2.62).

F1  h = -dE_d/dn by brute-force differentiation of the oracle's own total energy on a fully periodic
    grid (random unit field, chiral): the variational structure h = -df/dn + d_b pi_b. is exact
F2  the energy itself against closed forms (central differences of sines are sines):
    twist only   n = (cos qz, sin qz, 0):      f = K22/2 (q0 - sin q)^2, and h is parallel to n
    splay + bend n = (cos kx, sin kx, 0):      f = K11/2 sin^2k sin^2(kx) + K33/2 sin^2k cos^2(kx) + K22/2 q0^2
    so a swapped K11/K33 or a wrong sign of the twist term fails
F3  the stress against the energy: d_b sigma_ab = -d_a f - h_c d_a n_c to O(dx^2) on a smooth field, and
    sigma_ab = -d_a n_c pi_bc rebuilt in numpy from the closed-form pi of the helix
F4  flow-free relaxation between homeotropic plates: the discrete energy descends, |n| = 1
F5  K3 = 0 leaves the one-constant path bit for bit; K11 = K22 = K33 = K agrees with the one-constant
    molecular field to O(dx^2) on a smooth unit field (they differ by a null Lagrangian and by the
    compact vs wide Laplacian only)
"""
import math

import numpy as np
import pytest

import nh_inputs as I
from oracle import Oracle, frank3, molecular_field
from test_oracle_pins import cdiff, curl_c, smooth_unit_field

K3 = (0.0167, 0.00788, 0.0262)


def test_F1_h_is_minus_the_energy_gradient():
    rng = np.random.default_rng(17)
    n = rng.normal(size=(3, 6, 4, 5))
    n /= np.sqrt((n ** 2).sum(0))
    q0 = 0.37
    h, _, _ = frank3(n, K3, q0, periodic_z=True)
    eps = 1e-6
    for idx in [(0, 1, 2, 3), (1, 0, 0, 0), (2, 5, 3, 4), (2, 3, 1, 2), (0, 4, 0, 1), (1, 2, 3, 0)]:
        a, b = n.copy(), n.copy()
        a[idx] += eps
        b[idx] -= eps
        dE = (frank3(a, K3, q0, periodic_z=True)[2] - frank3(b, K3, q0, periodic_z=True)[2]) / (2 * eps)
        assert abs(h[idx] + dE) < 2e-9, (idx, h[idx], -dE)


def test_F2_energy_closed_forms():
    q0 = 0.21
    # twist: helix along z
    nz = 12
    q = 2 * math.pi / nz
    z = np.arange(nz, dtype=np.float64)
    n = np.zeros((3, nz, 3, 4))
    n[0] = np.cos(q * z)[:, None, None]
    n[1] = np.sin(q * z)[:, None, None]
    h, _, E = frank3(n, K3, q0, periodic_z=True)
    assert abs(E - n[0].size * 0.5 * K3[1] * (q0 - math.sin(q)) ** 2) < 1e-15
    hperp = h - n * (h * n).sum(0)
    assert np.abs(hperp).max() < 1e-16
    # splay and bend: planar director turning along x
    nx = 16
    k = 2 * math.pi / nx
    x = np.arange(nx, dtype=np.float64)
    n = np.zeros((3, 3, 2, nx))
    n[0] = np.cos(k * x)[None, None, :]
    n[1] = np.sin(k * x)[None, None, :]
    _, _, E = frank3(n, K3, q0, periodic_z=True)
    f = (0.5 * K3[0] * math.sin(k) ** 2 * np.sin(k * x) ** 2 + 0.5 * K3[2] * math.sin(k) ** 2 * np.cos(k * x) ** 2
         + 0.5 * K3[1] * q0 ** 2)
    assert abs(E - 6 * f.sum()) < 1e-15
    # a pure splay and a pure bend configuration separate K11 from K33: radial-like vs circular at x = 0
    assert abs(frank3(n, (1.0, 0, 0), 0.0, periodic_z=True)[2] - 6 * (0.5 * math.sin(k) ** 2 * np.sin(k * x) ** 2).sum()) < 1e-13
    assert abs(frank3(n, (0, 0, 1.0), 0.0, periodic_z=True)[2] - 6 * (0.5 * math.sin(k) ** 2 * np.cos(k * x) ** 2).sum()) < 1e-13


def _grad(n):
    return [np.stack([cdiff(n[c], ax) for c in range(3)]) for ax in (2, 1, 0)]   # grad[a][c] = d_a n_c


def _fdens(n, K3, q0):
    g = _grad(n)
    div = g[0][0] + g[1][1] + g[2][2]
    T = (n * curl_c(n)).sum(0) + q0
    b = n[0] * g[0] + n[1] * g[1] + n[2] * g[2]
    return 0.5 * K3[0] * div ** 2 + 0.5 * K3[1] * T ** 2 + 0.5 * K3[2] * (b * b).sum(0)


def test_F3_stress_divergence_identity_and_helix_stress():
    q0l = 0.35
    errs = []
    for L in (32, 64):
        n = smooth_unit_field(L)
        dxl = 2 * math.pi / L
        q0 = q0l * dxl
        h, sig, _ = frank3(n, K3, q0, periodic_z=True)
        F = np.stack([sum(cdiff(sig[a, b], ax) for b, ax in enumerate((2, 1, 0))) for a in range(3)])
        g = _grad(n)
        fd = _fdens(n, K3, q0)
        rhs = np.stack([-cdiff(fd, ax) - (h * g[a]).sum(0) for a, ax in enumerate((2, 1, 0))])
        errs.append(np.abs(F - rhs).max() / np.abs(F).max())
    assert errs[0] < 0.25 and errs[1] < errs[0] / 3.3, errs
    # helix along z: only d_z n is non-zero, pi_bc = K22 T eps_{abc} n_a: sigma_zb = -d_z n_c pi_bc
    nz = 10
    q = 2 * math.pi / nz
    z = np.arange(nz, dtype=np.float64)
    n = np.zeros((3, nz, 2, 2))
    n[0] = np.cos(q * z)[:, None, None]
    n[1] = np.sin(q * z)[:, None, None]
    q0 = 0.4
    _, sig, _ = frank3(n, K3, q0, periodic_z=True)
    T = q0 - math.sin(q)
    dzn = math.sin(q) * np.stack([-np.sin(q * z), np.cos(q * z), 0 * z])
    nn = np.stack([np.cos(q * z), np.sin(q * z), 0 * z])
    eps = np.zeros((3, 3, 3))
    eps[0, 1, 2] = eps[1, 2, 0] = eps[2, 0, 1] = 1
    eps[0, 2, 1] = eps[2, 1, 0] = eps[1, 0, 2] = -1
    pi = K3[1] * T * np.einsum("abc,az->bcz", eps, nn)
    expect_zb = -np.einsum("cz,bcz->bz", dzn, pi)
    assert np.abs(sig[2, :, :, 0, 0] - expect_zb).max() < 1e-17
    assert np.abs(sig[:2]).max() < 1e-18 and np.abs(expect_zb[2]).max() > 1e-4    # sigma_zz = K22 T sin q


def test_F4_energy_descends_between_plates():
    d = I.skyrmion_tubes(12, 12, 10, [(5.5, 5.5)], 4.0)
    o = Oracle(12, 12, 10, tau=0.8, K3=K3, pitch=8.0, gamma1=1.0, fd_ratio=2, coupling=0)
    o.set_director(d)
    q0 = 2 * math.pi / 8.0
    last = None
    for _ in range(25):
        n = o.get_fields()["n"]
        e = frank3(n, K3, q0)[2]
        if last is not None:
            assert e <= last + 1e-12 * abs(last)
        last = e
        assert np.abs(np.sqrt((n ** 2).sum(0)) - 1.0).max() < 1e-14
        o.step(4)


def test_F5_defaults_and_one_constant_limit():
    p = I.config(0)
    d = p.pop("director")
    p.pop("steps")
    a, b = Oracle(**p), Oracle(**dict(p, K3=(0.0, 0.0, 0.0)))
    for o in (a, b):
        o.set_director(d)
        o.step(15)
    fa, fb = a.get_fields(), b.get_fields()
    assert all(np.array_equal(fa[k], fb[k]) for k in fa)
    K, errs = 0.02, []
    for L in (32, 64):
        n = smooth_unit_field(L)
        q0 = 0.3 * 2 * math.pi / L
        h3 = frank3(n, (K, K, K), q0, periodic_z=True)[0]
        h1 = molecular_field(n, K, q0, periodic_z=True)
        p3 = h3 - n * (h3 * n).sum(0)          # only the part perpendicular to n moves the director
        p1 = h1 - n * (h1 * n).sum(0)
        errs.append(np.abs(p3 - p1).max() / np.abs(p1).max())
    assert errs[0] < 0.3 and errs[1] < errs[0] / 3.0, errs
