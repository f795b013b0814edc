"""Pins of the periodic part of the oracle (pins O-P1..O-P4)."""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_1310_4502_b200 import workloads as W

GOLD = {}
for _l in open(os.path.join(os.path.dirname(__file__), "golden", "ewald_constants.txt")):
    if _l.strip() and not _l.startswith("#"):
        _k, _v, _t = _l.split()
        GOLD[_k] = (float(_v), float(_t))


def _close(got, name):
    v, t = GOLD[name]
    assert abs(got - v) <= t, (name, got, v)


def test_ewald_constants_golden():
    _close(O.ewald_xi(), "xi")
    _close(O.ewald_psi([0.5, 0, 0])[0], "psi_half_0_0")
    _close(O.ewald_psi([0.5, 0.5, 0])[0], "psi_half_half_0")
    _close(O.ewald_psi([0.5, 0.5, 0.5])[0], "psi_half_half_half")
    _close(O.ewald_psi([0.25, 0, 0])[0], "psi_quarter_0_0")
    _close(O.psi_smooth([0, 0, 0]), "psi_sm_0")


def test_ewald_gradient_is_derivative_and_vanishes_by_symmetry():
    r = np.array([0.21, -0.13, 0.37]); h = 1e-4
    psi, g = O.ewald_psi(r)
    for k in range(3):
        e = np.zeros(3); e[k] = h
        fd = (8 * (O.ewald_psi(r + e)[0] - O.ewald_psi(r - e)[0]) - (O.ewald_psi(r + 2 * e)[0] - O.ewald_psi(r - 2 * e)[0])) / (12 * h)
        assert math.isclose(g[k], fd, rel_tol=1e-8)
    assert np.abs(O.ewald_psi([0.5, 0, 0])[1]).max() < 1e-12
    assert np.abs(O.ewald_psi([0.5, 0.5, 0.5])[1]).max() < 1e-12
    # psi is periodic and has zero box mean (midpoint rule on a grid that avoids r = 0)
    assert math.isclose(O.ewald_psi([0.3, 0.2, 0.1])[0], O.ewald_psi([1.3, -0.8, 0.1])[0], rel_tol=1e-10)
    k = 12
    q = (np.arange(k) + 0.5) / k
    mean = np.mean([O.ewald_psi([x, y, z])[0] for x in q for y in q for z in q])
    assert abs(mean) < 2e-2  # 1/r singularity limits the midpoint rule; the exact mean is 0


def test_far_table_is_the_taylor_series_of_psi_smooth():
    w = W.config(3, 4)
    T = O.Tree(w.pos, w.mass, w.lo, w.size, periodic=True)
    co = T.far_table()
    idx = {}
    q = 0
    for deg in range(9):
        for a in range(deg, -1, -1):
            for b in range(deg - a, -1, -1):
                idx[(a, b, deg - a - b)] = q; q += 1
    _close(co[idx[(0, 0, 0)]], "psi_sm_0")
    # the r^2 term is the uniform background: Laplacian of psi_sm = 4 pi  =>  c200 = 2 pi / 3
    assert math.isclose(co[idx[(2, 0, 0)]], 2 * math.pi / 3, rel_tol=1e-10)
    assert abs(co[idx[(2, 0, 0)]] - co[idx[(0, 2, 0)]]) < 1e-13 and abs(co[idx[(2, 0, 0)]] - co[idx[(0, 0, 2)]]) < 1e-13
    # every higher degree is harmonic: e.g. degree 4, 12 c400 + 2 c220 + 2 c202 = 0
    assert abs(12 * co[idx[(4, 0, 0)]] + 2 * co[idx[(2, 2, 0)]] + 2 * co[idx[(2, 0, 2)]]) < 1e-9
    # polynomial reproduces psi_sm near the centre to the size of the first neglected term
    rng = np.random.default_rng(1)
    for r in rng.uniform(-0.3, 0.3, (20, 3)):
        poly = sum(c * r[0]**a * r[1]**b * r[2]**cc for (a, b, cc), i in idx.items() for c in [co[i]])
        assert abs(poly - O.psi_smooth(r)) < 2e-7


def test_single_particle_and_perfect_lattices():
    # O-P1: one particle: a = 0, phi = -m xi / L
    pos = np.array([[0.3, 0.7, 0.2]], np.float32); mass = np.array([2.0], np.float32)
    T = O.Tree(pos, mass, (0, 0, 0), 1.0, periodic=True)
    a, p, _, _ = T.forces(0.5, 1e-6, 4)
    assert np.abs(a).max() < 1e-6 and abs(p[0] - (-2.0 * GOLD["xi"][0])) < 2e-5
    ad, pd = O.ewald_direct(pos, mass, 1.0, 1e-6)
    assert np.abs(ad).max() == 0 and abs(pd[0] + 2.0 * GOLD["xi"][0]) < 1e-10
    for K, name in ((2, "lattice_K2_phi"), (3, "lattice_K3_phi")):
        q = (np.arange(K) + 0.5) / K
        pos = np.array([[x, y, z] for x in q for y in q for z in q], np.float32)
        mass = np.full(K**3, 1.0 / K**3, np.float32)
        ad, pd = O.ewald_direct(pos, mass, 1.0, 1e-7)
        assert np.abs(ad).max() < (1e-10 if K == 2 else 1e-6)  # (i+1/2)/3 is not exact in float32
        assert np.abs(pd - GOLD[name][0]).max() < GOLD[name][1] * 10


def test_tree_images_farfield_vs_direct_ewald():
    """O-P2: algorithm (125 explicit cubes + degree-8 far field) against the direct Ewald sum."""
    w = W.config(3, 8)  # 512 particles
    T = O.Tree(w.pos, w.mass, w.lo, w.size, periodic=True, nleaf=8, ncrit=32)
    # the definition softens the nearest image only, the algorithm all 125 explicit ones: the two
    # differ by O(eps^2 ln) in the potential, so the comparison uses a small softening length
    eps = 2e-4
    ad, pd = O.ewald_direct(w.pos, w.mass, w.size, eps)
    rms = lambda a: math.sqrt(((a - ad) ** 2).sum() / (ad ** 2).sum())
    a0, p0, lpc, lpp = T.forces(0.0, eps, 4)
    assert (lpp == 125 * w.n).all() and (lpc == 0).all()
    e0 = rms(a0)
    assert e0 < 2e-5, e0
    assert np.abs(p0 - pd).max() < 2e-5 * np.abs(pd).max()
    e = [rms(T.forces(th, eps, 4)[0]) for th in (0.3, 0.5, 0.8)]
    assert e[0] < e[1] < e[2] and e[0] < 1e-3
    # O-P4: momentum
    m = w.mass.astype(np.float64)
    assert np.abs((m[:, None] * a0).sum(0)).max() < 1e-6 * (m[:, None] * np.abs(a0)).sum()


def test_translation_invariance():
    """O-P3: shifting every particle by the same vector modulo L changes a by round-off only."""
    w = W.config(3, 4)
    sh = np.array([0.25, 0.5, 0.125])  # exactly representable shift keeps float32 positions exact
    pos1 = np.floor(w.pos.astype(np.float64) * 2**20) / 2**20  # on a grid, so the shift is exact
    pos2 = (pos1 + sh) % 1.0
    assert (pos2.astype(np.float32) == pos2).all() and (pos1.astype(np.float32) == pos1).all()
    a1, p1 = O.ewald_direct(pos1.astype(np.float32), w.mass, 1.0, w.eps)
    a2, p2 = O.ewald_direct(pos2.astype(np.float32), w.mass, 1.0, w.eps)
    assert np.abs(a1 - a2).max() < 1e-9 * np.abs(a1).max() and np.abs(p1 - p2).max() < 1e-9
