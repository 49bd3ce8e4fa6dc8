"""Seeded synthetic inputs for the nematohydrodynamics hot path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2503_06610_b200/``).  It holds none of the method's arithmetic: it only
builds initial director fields and parameter sets (plain numpy, FP64) that are
then handed to either side through ``set_director`` / the params struct.

Recipe source: BASELINE.json ``configs`` and SURVEY.md §8(d) "Synthetic inputs";
the workloads stand in for the paper's skyrmion-tube-in-Poiseuille-flow runs
(§III.A) and its many-skyrmion domain (Fig. 6).

Random numbers are counter based: ``splitmix64(seed, cell, component)`` gives two
uniforms, Box-Muller turns them into one normal deviate, so the values do not
depend on traversal order or on the language that asks for them.
"""
from __future__ import annotations

import math
import numpy as np

SEED = 20250311  # the paper's date; SURVEY.md §8(d)

_U64 = np.uint64
_MASK = _U64(0xFFFFFFFFFFFFFFFF)


def splitmix64(x: np.ndarray) -> np.ndarray:
    """One round of the splitmix64 finaliser on uint64 counters (wraps mod 2^64)."""
    with np.errstate(over="ignore"):
        z = (np.asarray(x, dtype=np.uint64) + _U64(0x9E3779B97F4A7C15)) & _MASK
        z = ((z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)) & _MASK
        z = ((z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)) & _MASK
        return z ^ (z >> _U64(31))


def _counter(seed: int, cell: np.ndarray, comp: int, draw: int) -> np.ndarray:
    with np.errstate(over="ignore"):
        c = np.asarray(cell, dtype=np.uint64) * _U64(8) + _U64(2 * comp + draw)
        return splitmix64(splitmix64(np.full_like(c, _U64(seed))) ^ c)


def uniform01(seed: int, cell: np.ndarray, comp: int, draw: int = 0) -> np.ndarray:
    """Uniform in (0, 1): top 53 bits of the counter hash, offset by half an ulp."""
    bits = _counter(seed, cell, comp, draw) >> _U64(11)
    return (bits.astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed: int, cell: np.ndarray, comp: int) -> np.ndarray:
    """Standard normal by Box-Muller from two counter-based uniforms."""
    u1 = uniform01(seed, cell, comp, 0)
    u2 = uniform01(seed, cell, comp, 1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


def _normalise(n: np.ndarray) -> np.ndarray:
    return n / np.sqrt((n * n).sum(axis=0, keepdims=True))


def _plates_homeotropic(n: np.ndarray) -> np.ndarray:
    n[:, 0] = 0.0
    n[:, -1] = 0.0
    n[2, 0] = 1.0
    n[2, -1] = 1.0
    return n


def uniform_director(nx: int, ny: int, nz: int, direction=(0.0, 0.0, 1.0)) -> np.ndarray:
    """n = const everywhere; layout [3][nz][ny][nx], x fastest."""
    d = np.asarray(direction, dtype=np.float64)
    d = d / np.linalg.norm(d)
    return np.ascontiguousarray(np.broadcast_to(d[:, None, None, None], (3, nz, ny, nx)))


def noisy_homeotropic(nx: int, ny: int, nz: int, sigma: float = 0.05, seed: int = SEED) -> np.ndarray:
    """Config 1/3: normalise(z_hat + sigma N(0,1)^3) on fluid cells, z_hat on the plates."""
    cell = np.arange(nx * ny * nz, dtype=np.uint64).reshape(nz, ny, nx)
    n = np.zeros((3, nz, ny, nx))
    n[2] = 1.0
    for c in range(3):
        n[c] += sigma * normal(seed, cell, c)
    return np.ascontiguousarray(_plates_homeotropic(_normalise(n)))


def random_unit_field(nx: int, ny: int, nz: int, seed: int = SEED) -> np.ndarray:
    """Isotropic random unit vectors on every cell (used by fully periodic oracle pins)."""
    cell = np.arange(nx * ny * nz, dtype=np.uint64).reshape(nz, ny, nx)
    n = np.stack([normal(seed + 1, cell, c) for c in range(3)])
    return np.ascontiguousarray(_normalise(n))


def skyrmion_tubes(nx: int, ny: int, nz: int, centres, R: float, envelope: bool = True) -> np.ndarray:
    """Configs 2/4/5: skyrmion tubes with axes along z in a homeotropic background.

    theta(r) = pi (1 - r/R) s(z) for r < R, 0 outside; azimuth phi + pi/2, i.e.
    n = (-sin(theta) sin(phi), sin(theta) cos(phi), cos(theta)); s(z) = sin(pi z / nz)
    with z the layer index (BASELINE.json config 1, literal reading); plates z_hat.
    Distances use the periodic minimum image in x and y.
    """
    z = np.arange(nz, dtype=np.float64)[:, None, None]
    s = np.sin(math.pi * z / nz) if envelope else np.ones_like(z)
    n = np.zeros((3, nz, ny, nx))
    n[2] = 1.0
    w = int(math.ceil(R)) + 1                      # a tube only touches the window |x - xc|, |y - yc| <= R
    for (xc, yc) in centres:
        if 2 * w + 1 >= nx or 2 * w + 1 >= ny:     # the window would wrap onto itself: whole plane
            ix, iy = np.arange(nx), np.arange(ny)
        else:
            ix = np.arange(int(math.floor(xc)) - w, int(math.floor(xc)) + w + 2) % nx
            iy = np.arange(int(math.floor(yc)) - w, int(math.floor(yc)) + w + 2) % ny
        y = iy.astype(np.float64)[None, :, None]
        x = ix.astype(np.float64)[None, None, :]
        dx = x - xc
        dy = y - yc
        dx = dx - nx * np.round(dx / nx)
        dy = dy - ny * np.round(dy / ny)
        r = np.sqrt(dx * dx + dy * dy) + 0.0 * z
        inside = r < R
        theta = math.pi * (1.0 - r / R) * s
        phi = np.arctan2(dy, dx) + 0.0 * z
        tube = np.stack([-np.sin(theta) * np.sin(phi), np.sin(theta) * np.cos(phi), np.cos(theta)])
        sel = np.ix_(np.arange(3), np.arange(nz), iy, ix)
        n[sel] = np.where(inside[None], tube, n[sel])
    return np.ascontiguousarray(_plates_homeotropic(_normalise(n)))


def lattice_centres(nx: int, ny: int, spacing: float = 48.0, jitter: float = 6.0, seed: int = SEED):
    """Config 5: m = floor(L/spacing) tubes per axis, spacing L/m, centre jitter U[-jitter, jitter]^2."""
    mx, my = max(1, int(nx // spacing)), max(1, int(ny // spacing))
    out = []
    for j in range(my):
        for i in range(mx):
            k = np.array([j * mx + i], dtype=np.uint64)
            jx = (2.0 * uniform01(seed + 2, k, 0)[0] - 1.0) * jitter
            jy = (2.0 * uniform01(seed + 2, k, 1)[0] - 1.0) * jitter
            out.append(((i + 0.5) * nx / mx - 0.5 + jx, (j + 0.5) * ny / my - 0.5 + jy))
    return out


def random_centres(nx: int, ny: int, count: int, min_dist: float, seed: int = SEED):
    """`count` tube centres drawn uniformly on the periodic nx x ny plane, a draw being rejected when it
    falls within `min_dist` (periodic minimum image) of an accepted one: "randomly placed skyrmions"
     that do not overlap.  Counter-based draws, so the list depends on the seed only."""
    out, k = [], 0
    while len(out) < count:
        if k > 10000 * count:
            raise ValueError("cannot place %d centres %g apart on %dx%d" % (count, min_dist, nx, ny))
        c = np.array([k], dtype=np.uint64)
        x = uniform01(seed + 3, c, 0)[0] * nx
        y = uniform01(seed + 3, c, 1)[0] * ny
        k += 1
        ok = True
        for (xa, ya) in out:
            dx, dy = x - xa, y - ya
            dx -= nx * round(dx / nx)
            dy -= ny * round(dy / ny)
            if dx * dx + dy * dy < min_dist * min_dist:
                ok = False
                break
        if ok:
            out.append((float(x), float(y)))
    return out


# alpha1..alpha6 of MBBA in simulation units as the paper's Table 1 prints them (
# tests/golden/table1_mbba.txt holds the same numbers with the citation)
MBBA_ALPHA = (0.0373, -0.4496, -0.0203, 0.9318, 0.3084, -0.1617)
MBBA_K3 = (1.67e-7, 7.88e-8, 2.62e-7)


def many_skyrmions(nx: int = 320, ny: int = 320, nz: int = 16, count: int = 20, **over) -> dict:
    """The paper's closing demonstration (Fig. 6): a 320x320x16 cell with 20 randomly placed
    skyrmions, single precision, Delta t_FD = 250, on the test case's material (MBBA's
    three Frank constants, pitch 14, free plates, W0 = 1.5e-8, g = 2e-9; gamma1, xi from Table 1 with
    Parodi's relation).  Stand-in: the tubes are this module's ansatz, not the ref.-[18] toron
    (out of scope); elastic stress only unless ``alpha`` is given (the explicit viscous force is
    unstable at this Delta t_FD)."""
    gamma1 = MBBA_ALPHA[2] - MBBA_ALPHA[1]
    xi = -(MBBA_ALPHA[2] + MBBA_ALPHA[1]) / gamma1
    p = dict(nx=nx, ny=ny, nz=nz, tau=1.0, K3=MBBA_K3, pitch=14.0, xi=xi, gamma1=gamma1,
             g=(2e-9, 0.0, 0.0), anchoring=1, W0=1.5e-8, fd_ratio=250, steps=1000)
    p.update(over)
    seed = p.pop("seed", SEED)
    p["director"] = skyrmion_tubes(nx, ny, nz, random_centres(nx, ny, count, 2.0 * 7.0 + 4.0, seed), 7.0)
    return p


def config(k: int, **over) -> dict:
    """Parameter set + director for BASELINE.json ``configs[k]`` (k = 0..4).

    Returns a dict with the nh_params fields, ``steps`` and ``director`` ([3][nz][ny][nx] FP64).
    k = 2 (the precision sweep) returns the config-0 domain; the sweep itself lives in the tests.
    k = 4 takes ``size=(nx, ny, nz)`` (default 128x128x64).
    """
    if k in (0, 2):
        p = dict(nx=16, ny=16, nz=8, tau=0.8, K=0.01, pitch=0.0, xi=0.5, gamma1=1.0,
                 g=(1e-6, 0.0, 0.0), fd_ratio=1, steps=200 if k == 0 else 1000)
        p.update(over)
        p["director"] = noisy_homeotropic(p["nx"], p["ny"], p["nz"], 0.05, over.get("seed", SEED))
    elif k == 1:
        p = dict(nx=64, ny=64, nz=32, tau=1.0, K=0.02, pitch=16.0, xi=0.6, gamma1=1.0,
                 g=(5e-7, 0.0, 0.0), fd_ratio=1, steps=5000)
        p.update(over)
        c = [((p["nx"] - 1) / 2.0, (p["ny"] - 1) / 2.0)]
        p["director"] = skyrmion_tubes(p["nx"], p["ny"], p["nz"], c, 12.0)
    elif k == 3:
        p = dict(nx=256, ny=256, nz=64, tau=0.8, K=0.01, pitch=32.0, xi=0.5, gamma1=1.0,
                 g=(1e-6, 0.0, 0.0), fd_ratio=10, steps=20000)
        p.update(over)
        xc, yc = (p["nx"] - 1) / 2.0, (p["ny"] - 1) / 2.0
        p["director"] = skyrmion_tubes(p["nx"], p["ny"], p["nz"], [(xc - 40.0, yc), (xc + 40.0, yc)], 16.0)
    elif k == 4:
        nx, ny, nz = over.pop("size", (128, 128, 64))
        p = dict(nx=nx, ny=ny, nz=nz, tau=0.8, K=0.01, pitch=32.0, xi=0.5, gamma1=1.0,
                 g=(1e-6, 0.0, 0.0), fd_ratio=10, steps=200)
        p.update(over)
        p["director"] = skyrmion_tubes(nx, ny, nz, lattice_centres(nx, ny), 16.0)
    else:
        raise ValueError("config index must be 0..4")
    p.pop("seed", None)
    return p
