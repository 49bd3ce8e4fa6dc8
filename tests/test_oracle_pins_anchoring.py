"""Pins of the oracle's plate and bulk anchoring options (row f3 of SURVEY.md section 8f; the paper's
own test case has "no anchoring at the plates" and "a weak effective bulk anchoring" of strength W0,
PAPER.md:229; their discrete form is readings G14 and G23 of DESIGN.md).  CPU only: -m "not gpu".

A1  W0 term = minus the gradient of the energy -(W0/2) sum (n_z)^2, by brute-force differentiation
A2  uniform tilted director, no flow, K irrelevant, periodic x, y and FREE plates: the polar angle obeys
    d(theta)/dt = -(W0/gamma1) sin(theta) cos(theta), i.e. tan(theta(t)) = tan(theta0) exp(-W0 t/gamma1);
    the Heun steps follow it to second order and the field stays uniform (no torque from the plates)
A3  free plates, W0 = 0: ANY uniform director is a fixed point (with homeotropic plates only z_hat is:
    the same tilted field relaxes there) -- the plates exert no torque
A4  free plates: the discrete energy with mirrored plate layers still descends monotonically
A5  W0 = 0 and anchoring = 0 reproduce the default path bit for bit
"""
import math

import numpy as np
import pytest

import nh_inputs as I
from oracle import Oracle, molecular_field


def uniform(nx, ny, nz, theta, phi=0.3):
    v = np.array([math.sin(theta) * math.cos(phi), math.sin(theta) * math.sin(phi), math.cos(theta)])
    n = np.empty((3, nz, ny, nx))
    n[:] = v[:, None, None, None]
    return n


def test_A1_bulk_anchoring_is_minus_the_energy_gradient():
    rng = np.random.default_rng(3)
    n = rng.normal(size=(3, 4, 4, 4))
    n /= np.sqrt((n ** 2).sum(0))
    W0, K, q0 = 0.037, 0.01, 0.2
    dh = molecular_field(n, K, q0, periodic_z=True, W0=W0) - molecular_field(n, K, q0, periodic_z=True)
    E = lambda m: -(W0 / 2.0) * (m[2] ** 2).sum()
    eps = 1e-6
    for idx in [(0, 1, 2, 3), (1, 0, 0, 0), (2, 3, 1, 2), (2, 0, 0, 1)]:
        a, b = n.copy(), n.copy()
        a[idx] += eps
        b[idx] -= eps
        assert abs(dh[idx] - (-(E(a) - E(b)) / (2 * eps))) < 1e-9
    assert np.abs(dh[:2]).max() == 0.0 and np.abs(dh[2] - W0 * n[2]).max() < 1e-16


@pytest.mark.parametrize("r", [1, 4])
def test_A2_uniform_tilt_relaxes_under_W0_by_the_closed_form(r):
    W0, gamma1, th0 = 2e-3, 0.8, math.radians(55.0)
    o = Oracle(4, 3, 7, tau=0.8, K=0.02, gamma1=gamma1, W0=W0, anchoring=1, fd_ratio=r, coupling=0)
    o.set_director(uniform(4, 3, 7, th0))
    T = 400
    o.step(T)
    n = o.get_fields()["n"]
    assert np.abs(n - n[:, 3:4, 1:2, 2:3]).max() < 1e-14            # still uniform, plates included
    th = math.atan2(math.hypot(n[0, 3, 1, 2], n[1, 3, 1, 2]), n[2, 3, 1, 2])
    exact = math.atan(math.tan(th0) * math.exp(-W0 * T / gamma1))
    assert abs(th - exact) < 2e-6 * r * r                             # Heun: second order in r
    assert abs(math.atan2(n[1, 3, 1, 2], n[0, 3, 1, 2]) - 0.3) < 1e-12  # the azimuth does not move


def test_A3_free_plates_exert_no_torque():
    n0 = uniform(5, 4, 8, math.radians(40.0))
    free = Oracle(5, 4, 8, tau=0.8, K=0.02, anchoring=1, fd_ratio=2, coupling=0)
    free.set_director(n0)
    free.step(50)
    f = free.get_fields()
    assert np.abs(f["n"] - n0).max() < 1e-15 and np.abs(f["F"]).max() == 0.0
    fixed = Oracle(5, 4, 8, tau=0.8, K=0.02, anchoring=0, fd_ratio=2, coupling=0)
    fixed.set_director(n0)
    fixed.step(50)
    assert np.abs(fixed.get_fields()["n"][:, 1:-1] - n0[:, 1:-1]).max() > 1e-2


def _energy_free(n, K):
    """(K/2) sum over bonds |n(x+e) - n(x)|^2, periodic x, y; z bonds between fluid layers only
    (a mirrored plate layer adds a zero bond)."""
    e = 0.0
    m = n[:, 1:-1]
    e += ((np.roll(m, -1, 3) - m) ** 2).sum() + ((np.roll(m, -1, 2) - m) ** 2).sum()
    e += ((m[:, 1:] - m[:, :-1]) ** 2).sum()
    return 0.5 * K * e


def test_A4_energy_descends_with_free_plates():
    K = 0.02
    d = I.noisy_homeotropic(8, 8, 8, 0.3)
    o = Oracle(8, 8, 8, tau=0.8, K=K, anchoring=1, fd_ratio=2, coupling=0)
    o.set_director(d)
    last = _energy_free(o.get_fields()["n"], K)
    for _ in range(30):
        o.step(4)
        n = o.get_fields()["n"]
        e = _energy_free(n, K)
        assert e <= last * (1 + 1e-12)
        last = e
        assert np.array_equal(n[:, 0], n[:, 1]) and np.array_equal(n[:, -1], n[:, -2])
        assert np.abs(np.sqrt((n ** 2).sum(0)) - 1.0).max() < 1e-14


def test_A5_defaults_are_untouched():
    p = I.config(0)
    d = p.pop("director")
    p.pop("steps")
    a, b = Oracle(**p), Oracle(**dict(p, W0=0.0, anchoring=0))
    for o in (a, b):
        o.set_director(d)
        o.step(15)
    fa, fb = a.get_fields(), b.get_fields()
    assert all(np.array_equal(fa[k], fb[k]) for k in fa)
