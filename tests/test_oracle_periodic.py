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


# ---------------------------------------------------------------- f-1: per-cell background subtraction (R-18)
def test_cube_moments_and_closed_form_field():
    """PAPER.md:76-84.  Moments of the uniform cube (rho s^3, rho s^5/12, rho s^7/80, rho s^7/144), by the
    closed 1-D integrals and by quadrature; the closed-form potential and force of the homogeneous cube (refs [59, 46])
    against numerical integration, outside, inside, on a face and on the plane of a face."""
    s = 0.37
    mom = O.cube_moments(s)
    mi = O.multi_indices()
    want = {(0, 0, 0): s ** 3, (2, 0, 0): s ** 5 / 12, (0, 2, 0): s ** 5 / 12, (4, 0, 0): s ** 7 / 80, (2, 2, 0): s ** 7 / 144, (0, 2, 2): s ** 7 / 144}
    for k, ab in enumerate(mi):
        if ab in want:
            assert math.isclose(mom[k], want[ab], rel_tol=1e-14), ab
        elif any(e % 2 for e in ab):
            assert mom[k] == 0.0, ab
    n = 200
    q = ((np.arange(n) + 0.5) / n - 0.5) * s
    X, Y, Z = np.meshgrid(q, q, q, indexing="ij")
    wq = (s / n) ** 3
    assert math.isclose(mom[mi.index((2, 2, 0))], (X ** 2 * Y ** 2).sum() * wq, rel_tol=1e-4)
    assert math.isclose(mom[mi.index((4, 0, 0))], (X ** 4).sum() * wq, rel_tol=1e-4)
    lo = np.array([0.1, -0.2, 0.3]); side = 0.8
    n = 96
    q = (np.arange(n) + 0.5) / n * side
    X, Y, Z = np.meshgrid(lo[0] + q, lo[1] + q, lo[2] + q, indexing="ij")
    for x, tol in (([2.0, 1.0, -1.5], 1e-6), ([0.5, 0.1, 0.6], 3e-4), ([0.95, 0.3, 0.7], 1e-4), ([0.9, 0.2, 0.7], 3e-4), ([0.3, 0.6, 0.9], 3e-4)):
        x = np.array(x)
        d = np.stack([X - x[0], Y - x[1], Z - x[2]], -1)
        r = np.sqrt((d * d).sum(-1))
        pq = -((side / n) ** 3 / r).sum()
        aq = ((side / n) ** 3 * d / r[..., None] ** 3).sum((0, 1, 2))
        p, a = O.cube_field(x, lo, side)
        assert abs(p - pq) <= tol * abs(pq) * 10, (x, p, pq)
        assert np.abs(a - aq).max() <= max(tol * 200 * np.abs(aq).max(), 2e-3), (x, a, aq)
    # far away the cube is a point mass; inside, the Laplacian of the potential is 4 pi (finite differences)
    p, a = O.cube_field([30.0, -20.0, 10.0], lo, side)
    R = np.array([30.0, -20.0, 10.0]) - (lo + side / 2)
    assert math.isclose(p, -side ** 3 / np.linalg.norm(R), rel_tol=1e-4)
    x0 = lo + np.array([0.31, 0.42, 0.55]) * side
    hh = 1e-3
    lap = sum(O.cube_field(x0 + hh * e, lo, side)[0] + O.cube_field(x0 - hh * e, lo, side)[0] for e in np.eye(3)) - 6 * O.cube_field(x0, lo, side)[0]
    assert math.isclose(lap / hh ** 2, 4 * math.pi, rel_tol=1e-4)
    for k, e in enumerate(np.eye(3)):  # acceleration = -grad phi
        fd = -(O.cube_field(x0 + hh * e, lo, side)[0] - O.cube_field(x0 - hh * e, lo, side)[0]) / (2 * hh)
        assert math.isclose(O.cube_field(x0, lo, side)[1][k], fd, rel_tol=1e-5, abs_tol=1e-8)


@pytest.mark.parametrize("cfg,side,order,theta", [(3, 10, 2, 0.5), (4, 12, 4, 0.5), (4, 10, 0, 0.6)])
def test_background_subtraction_is_consistent_with_the_plain_periodic_tree(cfg, side, order, theta):
    """The background-subtracted walk computes the same periodic field as the plain one and as the direct Ewald sum
    (the subtracted cubes are added back in closed form): differences at the level of the truncation error; the
    subtracted cubes tile exactly (5 L)^3 minus the near cube; on a perfect lattice every subtracted monopole is 0."""
    w = W.config(cfg, side)
    T = O.Tree(w.pos, w.mass, w.lo, w.size, periodic=True, nleaf=8, ncrit=32)
    sel = np.arange(0, T.ngroups, max(1, T.ngroups // 12))
    a0, p0, lpc0, lpp0 = T.forces(theta, w.eps, order, groups=sel)
    a1, p1, lpc1, lbg, lv, lpp1 = T.forces_bg(theta, w.eps, order, groups=sel)
    m = ~np.isnan(p0)
    sinks = np.nonzero(m)[0]
    ae, pe = O.ewald_direct(w.pos, w.mass, w.size, w.eps, sinks=sinks)
    arms = np.sqrt((ae ** 2).sum(1).mean())
    e0 = np.sqrt(((a0[m] - ae) ** 2).sum(1).mean()) / arms
    e1 = np.sqrt(((a1[m] - ae) ** 2).sum(1).mean()) / arms
    assert e1 < max(3 * e0, 2e-3) and e1 < 0.05, (e0, e1)
    prms = np.sqrt(((pe - pe.mean()) ** 2).mean())
    assert np.abs(p1[m] - pe).max() < max(3 * np.abs(p0[m] - pe).max(), 1e-3 * prms), (np.abs(p1[m] - pe).max(), np.abs(p0[m] - pe).max())
    assert (lbg > 0).all() and (lbg <= lpc1).all() and (lpp1 <= lpp0).all()
    c = T.cells()
    gs = w.size * np.ldexp(1.0, -c["level"][T.groups()[sel]].astype(np.int64))
    assert np.allclose(T.bg_volume, 125.0 - (5 * gs / w.size) ** 3, rtol=1e-12)
    # a lazy tree (moments of the accepted cells only, as the 2^27-body test uses) does the same arithmetic
    T2 = O.Tree(w.pos, w.mass, w.lo, w.size, periodic=True, nleaf=8, ncrit=32, moments=2)
    a3, p3, *_ = T2.forces_bg(theta, w.eps, order, groups=sel)
    assert np.array_equal(a3, a1, equal_nan=True) and np.array_equal(p3, p1, equal_nan=True)
    # smaller theta: both converge to the Ewald sum
    a2, p2, *_ = T.forces_bg(0.3, w.eps, order, groups=sel)
    e2 = np.sqrt(((a2[m] - ae) ** 2).sum(1).mean()) / arms
    assert e2 < e1 or e2 < 1e-5


def test_background_subtracted_moments_vanish_on_a_perfect_lattice():
    K = 8
    q = (np.arange(K) + 0.5) / K
    pos = np.stack(np.meshgrid(q, q, q, indexing="ij"), -1).reshape(-1, 3).astype(np.float32)
    mass = np.full(K ** 3, 1.0 / K ** 3, np.float32)
    T = O.Tree(pos, mass, (0, 0, 0), 1.0, periodic=True, nleaf=1, ncrit=8)
    a, p, lpc, lbg, lv, lpp = T.forces_bg(0.5, 1e-3, 4, groups=np.array([0, T.ngroups // 2, T.ngroups - 1]))
    m = ~np.isnan(p)
    a0, p0, *_ = T.forces(0.5, 1e-3, 4, groups=np.array([0, T.ngroups // 2, T.ngroups - 1]))
    # zero force on a lattice: what is left is the truncation error of the near region, no worse than without subtraction
    assert np.abs(a[m]).max() < 5e-6 and np.abs(a[m]).max() <= 1.5 * np.abs(a0[m]).max()
    assert np.allclose(p[m], 2.8372974794806 / K ** 2, rtol=1e-3)
    assert (lv == 0).all()   # a full lattice has no empty octants outside the near cube
