"""Seeded synthetic particle sets shaped like the paper's workloads.

This module only *draws inputs*: it contains none of the method's arithmetic (no keys, no
tree, no forces) and imports neither the CUDA library nor the oracle.  Tests, ``bench.py``
and ``__graft_entry__.smoke()`` hand the same arrays to both sides.

The paper's production inputs are cosmological particle sets made with CLASS + 2LPTIC
 which are not available here; BASELINE.json's five ``configs``
prescribe seeded stand-ins of the same shape and they are what this file builds (recipe in
DESIGN.md "Input recipe").

All sets: ``numpy.random.Generator(PCG64(seed))``, double precision internally, returned as
C-contiguous float32 ``pos[n,3]`` and ``mass[n]`` plus the box ``(lo[3], size)``.
Seeds are ``SEED0 + config index``.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED0 = 1310450200


@dataclass
class Workload:
    name: str
    pos: np.ndarray  # float32 [n,3]
    mass: np.ndarray  # float32 [n]
    lo: tuple  # (x,y,z) of the root cube corner
    size: float  # side of the root cube / period
    periodic: bool
    eps: float
    theta: float
    order: int
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.pos.shape[0])


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def _inside_f32(x: np.ndarray, lo: float, size: float) -> np.ndarray:
    """Round to float32 and keep every coordinate a few float32 ulps inside [lo, lo+size).

    The library rejects particles whose scaled coordinate rounds to >= 1, so
    the generators never emit the last few representable values below the upper face.
    """
    hi = np.float32(lo + size)
    top = hi
    for _ in range(4):
        top = np.nextafter(top, np.float32(-np.inf), dtype=np.float32)
    xf = x.astype(np.float32)
    np.minimum(xf, top, out=xf)
    np.maximum(xf, np.float32(lo), out=xf)
    return xf


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    cz = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * np.pi, n)
    s = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
    return np.stack([s * np.cos(ph), s * np.sin(ph), cz], axis=1)


def _plummer_radii(rng: np.random.Generator, n: int, a: float, rcut: float) -> np.ndarray:
    """Radii of a Plummer sphere of scale a, truncated at rcut, by inverse CDF + rejection."""
    out = np.empty(n)
    filled = 0
    while filled < n:
        m = max(1024, int((n - filled) * 1.05))
        u = rng.uniform(0.0, 1.0, m)
        u = u[u > 0.0]
        r = a / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
        r = r[r <= rcut]
        k = min(n - filled, r.size)
        out[filled:filled + k] = r[:k]
        filled += k
    return out


def uniform_cube(n: int, seed: int = SEED0, eps: float = 1e-3, theta: float = 0.5,
                 order: int = 2) -> Workload:
    """C0: n equal-mass particles, iid uniform in the unit cube, open boundary."""
    rng = _rng(seed)
    x = rng.uniform(0.0, 1.0, (n, 3))
    pos = _inside_f32(x, 0.0, 1.0)
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return Workload(f"uniform_{n}", np.ascontiguousarray(pos), mass, (0.0, 0.0, 0.0), 1.0,
                    False, eps, theta, order)


def plummer_sphere(n: int, seed: int = SEED0 + 1, a: float = 0.05, eps: float = 1e-4,
                   theta: float = 0.5, order: int = 2) -> Workload:
    """C1: Plummer sphere, scale a, truncated at 20a, centred at the origin, box [-1,1)^3."""
    rng = _rng(seed)
    r = _plummer_radii(rng, n, a, 20.0 * a)
    x = r[:, None] * _isotropic(rng, n)
    pos = _inside_f32(x, -1.0, 2.0)
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return Workload(f"plummer_{n}", np.ascontiguousarray(pos), mass, (-1.0, -1.0, -1.0), 2.0,
                    False, eps, theta, order, {"a": a})


def clustered_mix(n: int, seed: int = SEED0 + 2, n_halos: int = 4096, halo_frac: float = 0.7,
                  eps: float = 5e-5, theta: float = 0.6, order: int = 2) -> Workload:
    """C2: 70% of the particles in Plummer halos with dN/dM ~ M^-1.9 over 3 decades,
    a_h = 0.02 (M/Mmax)^(1/3), truncated at 10 a_h, centres uniform; 30% uniform background;
    everything wrapped into the unit box."""
    rng = _rng(seed)
    n_halos = max(1, min(n_halos, n // 64 if n >= 64 else 1))
    n_in = int(round(halo_frac * n))
    m1, m2 = 1.0, 1.0e3
    u = rng.uniform(0.0, 1.0, n_halos)
    mh = (m1 ** -0.9 + u * (m2 ** -0.9 - m1 ** -0.9)) ** (-1.0 / 0.9)
    # particles per halo proportional to mass, largest-remainder rounding to hit n_in exactly
    share = mh / mh.sum() * n_in
    cnt = np.floor(share).astype(np.int64)
    rem = n_in - int(cnt.sum())
    if rem > 0:
        idx = np.argsort(-(share - cnt), kind="stable")[:rem]
        cnt[idx] += 1
    centres = rng.uniform(0.0, 1.0, (n_halos, 3))
    ah = 0.02 * (mh / m2) ** (1.0 / 3.0)
    x = np.empty((n, 3))
    # one vectorised draw for all halo particles
    hid = np.repeat(np.arange(n_halos), cnt)
    a_p = ah[hid]
    # unit-scale Plummer radii truncated at 10 (scale applied per particle)
    r = _plummer_radii(rng, n_in, 1.0, 10.0) * a_p
    x[:n_in] = centres[hid] + r[:, None] * _isotropic(rng, n_in)
    x[n_in:] = rng.uniform(0.0, 1.0, (n - n_in, 3))
    x -= np.floor(x)
    # a fixed shuffle so the caller's order carries no spatial structure
    p = rng.permutation(n)
    pos = _inside_f32(x[p], 0.0, 1.0)
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return Workload(f"clustered_{n}", np.ascontiguousarray(pos), mass, (0.0, 0.0, 0.0), 1.0,
                    False, eps, theta, order, {"n_halos": n_halos})


def zeldovich_lattice(ng: int, rms_cells: float, seed: int = SEED0 + 3, eps: float | None = None,
                      theta: float = 0.5, order: int = 4) -> Workload:
    """C3/C4: ng^3 lattice q=(i+1/2)/ng displaced by a Gaussian field with P(k) ~ k^-2,
    spherical cut at the Nyquist frequency, 3-D rms displacement = rms_cells/ng, periodic."""
    rng = _rng(seed)
    white = rng.standard_normal((ng, ng, ng))
    wk = np.fft.rfftn(white)
    del white
    kx = np.fft.fftfreq(ng, d=1.0 / ng) * 2.0 * np.pi
    kz = np.fft.rfftfreq(ng, d=1.0 / ng) * 2.0 * np.pi
    k2 = (kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2)
    knyq = np.pi * ng
    with np.errstate(divide="ignore", invalid="ignore"):
        amp = np.where((k2 > 0) & (k2 <= knyq * knyq), k2 ** -0.5, 0.0)  # delta_k ~ |k|^-1
        dk = wk * amp
        del wk
        ik2 = np.where(k2 > 0, 1.0 / k2, 0.0)
    comps = []
    for ax, kvec in enumerate((kx[:, None, None], kx[None, :, None], kz[None, None, :])):
        comps.append(np.fft.irfftn(1j * kvec * ik2 * dk, s=(ng, ng, ng), axes=(0, 1, 2)))
    del dk, ik2, k2
    rms = np.sqrt(np.mean(comps[0] ** 2 + comps[1] ** 2 + comps[2] ** 2))
    scale = (rms_cells / ng) / rms
    q1 = (np.arange(ng) + 0.5) / ng
    n = ng ** 3
    x = np.empty((n, 3))
    x[:, 0] = (q1[:, None, None] + scale * comps[0]).ravel()
    x[:, 1] = (q1[None, :, None] + scale * comps[1]).ravel()
    x[:, 2] = (q1[None, None, :] + scale * comps[2]).ravel()
    del comps
    x -= np.floor(x)
    pos = _inside_f32(x, 0.0, 1.0)
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    if eps is None:
        eps = 1.0 / (40.0 * ng)
    return Workload(f"zeldovich_{ng}^3", np.ascontiguousarray(pos), mass, (0.0, 0.0, 0.0), 1.0,
                    True, eps, theta, order, {"ng": ng, "rms_cells": rms_cells})


def config(idx: int, scale: int | None = None) -> Workload:
    """BASELINE.json ``configs[idx]`` (0-based).  ``scale`` (log2 n, or lattice side for the
    periodic configs) builds a smaller replica by the same code for tests."""
    if idx == 0:
        return uniform_cube(1 << (14 if scale is None else scale), SEED0 + 0)
    if idx == 1:
        return plummer_sphere(1 << (20 if scale is None else scale), SEED0 + 1)
    if idx == 2:
        return clustered_mix(1 << (24 if scale is None else scale), SEED0 + 2)
    if idx == 3:
        return zeldovich_lattice(256 if scale is None else scale, 0.3, SEED0 + 3, order=4)
    if idx == 4:
        ng = 512 if scale is None else scale
        return zeldovich_lattice(ng, 2.0, SEED0 + 4, eps=1.0 / (40.0 * ng), order=2)
    raise ValueError(f"no config {idx}")
