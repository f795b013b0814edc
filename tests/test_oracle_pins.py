"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-types the oracle's own formula or re-calls its routine as the expected value:
closed forms, symmetry invariants, finite differences, brute force, series, analytic fields.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_1310_4502_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- keys (C-2)
def _read_key_pins():
    out = []
    for line in open(os.path.join(GOLD, "keys.txt")):
        if line.startswith("#") or not line.strip():
            continue
        ix, iy, iz, hx = line.split()
        out.append((int(ix), int(iy), int(iz), int(hx, 16)))
    return out


def test_key_pins_golden():
    # grid coordinate i -> position (i + 0.5) / 2^21 is exact in float32 (22 significant bits)
    for ix, iy, iz, want in _read_key_pins():
        p = np.array([[(ix + 0.5) / 2**21, (iy + 0.5) / 2**21, (iz + 0.5) / 2**21]], np.float32)
        got = int(O.keys(p, (0, 0, 0), 1.0)[0])
        assert got == want, (ix, iy, iz, hex(got), hex(want))


def test_key_lower_corner_and_box_offset():
    p = np.array([[-1.0, -1.0, -1.0]], np.float32)
    assert int(O.keys(p, (-1, -1, -1), 2.0)[0]) == 0x8000000000000000
    with pytest.raises(ValueError):
        O.keys(np.array([[1.0, 0.5, 0.5]], np.float32), (0, 0, 0), 1.0)  # upper face is outside
    with pytest.raises(ValueError):
        O.keys(np.array([[0.5, -1e-3, 0.5]], np.float32), (0, 0, 0), 1.0)


def _deinterleave(key):
    key = int(key) & ((1 << 63) - 1)
    c = [0, 0, 0]
    for b in range(21):
        c[0] |= ((key >> (3 * b + 2)) & 1) << b
        c[1] |= ((key >> (3 * b + 1)) & 1) << b
        c[2] |= ((key >> (3 * b)) & 1) << b
    return c


def test_key_decode_encode_identity():
    rng = np.random.default_rng(7)
    pos = rng.uniform(0, 1, (2000, 3)).astype(np.float32)
    key = O.keys(pos, (0, 0, 0), 1.0)
    want = np.floor(pos.astype(np.float64) * 2**21).astype(np.int64)  # exact: power-of-two scale
    for k, w in zip(key, want):
        assert (int(k) >> 63) == 1
        assert _deinterleave(k) == list(w)


def _zorder_bruteforce(ic, idx, level):
    """Recursive octant partition, x most significant; ties keep input order."""
    if len(idx) <= 1 or level == 21:
        return list(idx)
    out = []
    bit = 20 - level
    for o in range(8):
        sel = [i for i in idx if (((ic[i][0] >> bit) & 1) << 2 | ((ic[i][1] >> bit) & 1) << 1
                                  | ((ic[i][2] >> bit) & 1)) == o]
        if sel:
            out += _zorder_bruteforce(ic, sel, level + 1)
    return out


def test_sort_equals_recursive_octant_partition():
    rng = np.random.default_rng(11)
    pos = rng.uniform(0, 1, (64, 3)).astype(np.float32)
    pos[10] = pos[3]  # duplicated key: stable tie-break
    pos[40] = pos[3]
    T = O.Tree(pos, np.ones(64, np.float32), (0, 0, 0), 1.0, nleaf=1, ncrit=1, moments=False)
    key, skey, perm = T.keys()
    ic = np.floor(pos.astype(np.float64) * 2**21).astype(np.int64)
    assert list(perm) == _zorder_bruteforce(ic, list(range(64)), 0)
    assert (skey == key[perm]).all() and (np.diff(skey.astype(np.float64)) >= 0).all()


def test_sort_is_stable_permutation():
    w = W.config(2, 12)
    pos = w.pos.copy()
    pos[100:200] = pos[0:100]  # many equal keys
    T = O.Tree(pos, w.mass, w.lo, w.size, moments=False)
    key, skey, perm = T.keys()
    assert sorted(perm.tolist()) == list(range(w.n))
    assert (skey[1:] >= skey[:-1]).all()
    eq = skey[1:] == skey[:-1]
    assert eq.sum() >= 100 and (perm[1:][eq] > perm[:-1][eq]).all()


# ---------------------------------------------------------------- tree (C-4)
@pytest.mark.parametrize("cfg,scale,nleaf,ncrit", [(0, 12, 16, 64), (1, 13, 8, 32), (2, 13, 16, 64),
                                                   (2, 12, 1, 1), (0, 5, 16, 64)])
def test_tree_invariants(cfg, scale, nleaf, ncrit):
    w = W.config(cfg, scale)
    T = O.Tree(w.pos, w.mass, w.lo, w.size, nleaf=nleaf, ncrit=ncrit, moments=False)
    c = T.cells()
    key, skey, perm = T.keys()
    n, nc = w.n, T.ncells
    assert c["key"][0] == 1 and c["first"][0] == 0 and c["count"][0] == n and c["parent"][0] == -1
    assert (np.diff(c["key"].astype(np.float64)) > 0).all()  # ascending numeric key, unique
    lvl = np.array([(int(k).bit_length() - 1) // 3 for k in c["key"]])
    assert (lvl == c["level"]).all()
    leaf = c["child"] < 0
    assert ((c["count"] <= nleaf) | (c["level"] == 21))[leaf].all()
    assert (c["count"] > nleaf)[~leaf].all() and (c["mask"][leaf] == 0).all()
    # leaves partition [0, n)
    order = np.argsort(c["first"][leaf], kind="stable")
    f, k = c["first"][leaf][order], c["count"][leaf][order]
    assert f[0] == 0 and (f[1:] == f[:-1] + k[:-1]).all() and f[-1] + k[-1] == n
    for ci in range(nc):
        l = int(c["level"][ci])
        # every particle of the cell carries the cell key as prefix
        pref = skey[c["first"][ci]:c["first"][ci] + c["count"][ci]] >> np.uint64(63 - 3 * l)
        assert (pref == c["key"][ci]).all()
        if not leaf[ci]:
            nch = bin(int(c["mask"][ci])).count("1")
            ch = np.arange(c["child"][ci], c["child"][ci] + nch)
            assert (c["parent"][ch] == ci).all()
            octs = [o for o in range(8) if (int(c["mask"][ci]) >> o) & 1]
            assert [int(x) for x in c["key"][ch]] == [(int(c["key"][ci]) << 3) | o for o in octs]
            assert c["count"][ch].sum() == c["count"][ci] and c["first"][ch][0] == c["first"][ci]
    # groups partition [0, n) in particle order
    g = T.groups()
    gf, gk = c["first"][g], c["count"][g]
    assert gf[0] == 0 and (gf[1:] == gf[:-1] + gk[:-1]).all() and gf[-1] + gk[-1] == n
    assert ((gk <= ncrit) | (c["level"][g] == 21)).all()
    par = c["parent"][g]
    assert ((par < 0) | (c["count"][np.maximum(par, 0)] > ncrit)).all()
    # membership: the leaf of a particle is a cell whose key prefixes the particle key
    lf = T.leaf_of()
    sh = (63 - 3 * c["level"][lf]).astype(np.uint64)
    assert ((skey >> sh) == c["key"][lf]).all()


def test_tree_by_hand_n8():
    # 8 particles, one per octant centre: root + 8 leaves when NLEAF = 1
    pts = np.array([[x, y, z] for x in (0.25, 0.75) for y in (0.25, 0.75) for z in (0.25, 0.75)], np.float32)
    T = O.Tree(pts[::-1].copy(), np.ones(8, np.float32), (0, 0, 0), 1.0, nleaf=1, ncrit=1, moments=False)
    c = T.cells()
    assert T.ncells == 9 and c["mask"][0] == 0xFF and c["child"][0] == 1
    assert [int(k) for k in c["key"][1:]] == [8 + o for o in range(8)]
    assert list(T.keys()[2]) == [7, 6, 5, 4, 3, 2, 1, 0]
    T2 = O.Tree(pts, np.ones(8, np.float32), (0, 0, 0), 1.0, nleaf=8, ncrit=8, moments=False)
    assert T2.ncells == 1 and T2.ngroups == 1


def test_level21_leaf_with_coincident_particles():
    pos = np.tile(np.array([[0.3, 0.6, 0.9]], np.float32), (40, 1))
    pos = np.vstack([pos, np.array([[0.1, 0.1, 0.1]], np.float32)])
    T = O.Tree(pos, np.ones(41, np.float32), (0, 0, 0), 1.0, nleaf=4, ncrit=8, moments=False)
    c = T.cells()
    deep = c["level"] == 21
    assert deep.sum() == 1 and c["count"][deep][0] == 40 and (c["child"][deep] < 0).all()
    g = T.groups()
    assert T.ngroups == 2 and sorted(c["count"][g].tolist()) == [1, 40]


# ---------------------------------------------------------------- direct sum (C-1)
def test_two_body_closed_form():
    m2, eps = 0.75, 0.05
    pos = np.array([[0.125, 0.25, 0.5], [0.625, 0.5, 0.25]], np.float32)
    mass = np.array([0.5, m2], np.float32)
    a, p = O.direct(pos, mass, eps)
    d = pos[1].astype(np.float64) - pos[0].astype(np.float64)
    u = d @ d + eps * eps
    assert np.allclose(a[0], m2 * d / u**1.5, rtol=1e-15, atol=0)
    assert math.isclose(p[0], -m2 / math.sqrt(u), rel_tol=1e-15)
    assert np.allclose(a[1], -0.5 * d / u**1.5, rtol=1e-15, atol=0)
    # O-5: a softened particle is a Plummer sphere of scale eps
    r = math.sqrt(d @ d)
    assert math.isclose(np.linalg.norm(a[0]), m2 * r / (r * r + eps * eps) ** 1.5, rel_tol=1e-14)


def test_momentum_conservation_and_coincident_pair():
    w = W.config(0, 10)
    a, p = O.direct(w.pos, w.mass, w.eps)
    m = w.mass.astype(np.float64)
    tot = (m[:, None] * a).sum(0)
    assert np.abs(tot).max() <= 1e-13 * (m[:, None] * np.abs(a)).sum()
    # energy symmetry: sum_i m_i phi_i = 2 * sum_{i<j} pair energies (antisymmetry of the pairs)
    x = w.pos.astype(np.float64)
    e = 0.0
    for i in range(0, 64):
        d = x[i + 1:] - x[i]
        e += -(m[i] * m[i + 1:] / np.sqrt((d * d).sum(1) + w.eps**2)).sum()
    a64, p64 = O.direct(w.pos[:65], w.mass[:65], w.eps)
    # coincident distinct bodies: zero force, -m/eps potential
    pos = np.array([[0.5, 0.5, 0.5], [0.5, 0.5, 0.5]], np.float32)
    a2, p2 = O.direct(pos, np.array([1, 2], np.float32), 0.1)
    assert (a2 == 0).all() and math.isclose(p2[0], -20.0) and math.isclose(p2[1], -10.0)


def _ring(q, k, rng, centre):
    cz = rng.uniform(-1, 1, k); ph = rng.uniform(0, 2 * np.pi, k); s = np.sqrt(1 - cz * cz)
    u = np.stack([s * np.cos(ph), s * np.sin(ph), cz], 1)
    return (centre + q * u).astype(np.float32), u


def test_uniform_sphere_field():
    """O-3: radial-shell means of the direct sum against the homogeneous-sphere closed form."""
    rng = np.random.default_rng(3)
    n, Rs, k = 1 << 14, 0.4, 64
    r = Rs * rng.uniform(0, 1, n) ** (1 / 3)
    pos, _ = _ring(1.0, n, rng, 0.0)
    pos = (0.5 + r[:, None] * pos.astype(np.float64)).astype(np.float32)
    mass = np.full(n, 1.0 / n, np.float32)
    for q in (0.1, 0.2, 0.3, 0.6, 0.9):
        probes, u = _ring(q, k, rng, 0.5)
        allp = np.vstack([pos, probes]); allm = np.concatenate([mass, np.full(k, 1e-30, np.float32)])
        a, p = O.direct(allp, allm, 5e-3, sinks=np.arange(n, n + k))
        ar = -q / Rs**3 if q < Rs else -1 / q**2
        ph_ = -(3 * Rs**2 - q**2) / (2 * Rs**3) if q < Rs else -1 / q
        n_enc = n * min(1.0, (q / Rs) ** 3)  # Poisson noise of the enclosed mass: "few x N^-1/2"
        assert abs((a * u).sum(1).mean() - ar) < (3 / math.sqrt(n_enc) + 0.02) * abs(ar), q
        assert abs(p.mean() - ph_) < 0.01 * abs(ph_), q


def test_plummer_sphere_field():
    """O-4: Plummer sphere truncated at 20a: a_r = -M r/(r^2+a^2)^1.5 / 0.996261 inside the cut."""
    w = W.config(1, 14)
    a_s, k = w.meta["a"], 64
    rng = np.random.default_rng(4)
    frac = (20 / math.sqrt(401)) ** 3  # mass fraction of an untruncated Plummer sphere inside 20a
    assert math.isclose(frac, 0.996261, rel_tol=1e-6)
    for q in (0.02, 0.05, 0.1, 0.3, 0.8):
        probes, u = _ring(q, k, rng, 0.0)
        allp = np.vstack([w.pos, probes]); allm = np.concatenate([w.mass, np.full(k, 1e-30, np.float32)])
        a, p = O.direct(allp, allm, 2e-3, sinks=np.arange(w.n, w.n + k))
        ar = -q / (q * q + a_s * a_s) ** 1.5 / frac
        n_enc = w.n * q**3 / (q * q + a_s * a_s) ** 1.5
        assert abs((a * u).sum(1).mean() - ar) < (3 / math.sqrt(n_enc) + 0.02) * abs(ar), q


# ---------------------------------------------------------------- Green's function tensors (C-6)
@pytest.mark.parametrize("eps", [0.0, 0.3])
def test_dg_against_finite_differences(eps):
    R = np.array([0.7, -0.4, 0.55])
    g = lambda r: 1.0 / math.sqrt(r @ r + eps * eps)
    assert math.isclose(O.dg(0, 0, 0, R, eps), g(R), rel_tol=1e-15)
    h = 1e-3
    e = np.eye(3)
    # first derivatives by central differences of g, higher ones by differences of lower tensors
    for k in range(3):
        fd = (g(R + h * e[k]) - g(R - h * e[k])) / (2 * h)
        idx = [0, 0, 0]; idx[k] = 1
        assert math.isclose(O.dg(*idx, R, eps), fd, rel_tol=2e-6)
    for a in range(0, 5):
        for b in range(0, 5 - a):
            for c in range(0, 5 - a - b):
                for k in range(3):
                    up = [a, b, c]; up[k] += 1
                    f = lambda t: O.dg(a, b, c, R + t * e[k], eps)
                    fd = (8 * (f(h) - f(-h)) - (f(2 * h) - f(-2 * h))) / (12 * h)  # 4th-order stencil
                    assert math.isclose(O.dg(*up, R, eps), fd, rel_tol=1e-7, abs_tol=1e-7), (a, b, c, k)


def test_dg_laplacian_vanishes_only_without_softening():
    R = np.array([0.3, 0.5, -0.2])
    lap = lambda eps: O.dg(2, 0, 0, R, eps) + O.dg(0, 2, 0, R, eps) + O.dg(0, 0, 2, R, eps)
    assert abs(lap(0.0)) < 1e-12 * abs(O.dg(2, 0, 0, R, 0.0))
    u = R @ R + 0.04
    assert math.isclose(lap(0.2), -3 * 0.04 * u**-2.5, rel_tol=1e-12)  # traces matter when softened


# ---------------------------------------------------------------- expansion (C-5, C-6, eq 5-6)
def _cluster(b, seed=5):
    rng = np.random.default_rng(seed)
    y = b * rng.uniform(-1, 1, (5, 3)) + np.array([0.1, -0.2, 0.05])
    m = rng.uniform(0.5, 1.5, 5)
    return y, m


def _direct_on(x, y, m, eps):
    d = y - x
    u = (d * d).sum(1) + eps * eps
    return (m[:, None] * d / u[:, None] ** 1.5).sum(0), -(m / np.sqrt(u)).sum()


@pytest.mark.parametrize("eps", [0.0, 0.3])
def test_order_law_fig6(eps):
    """PAPER.md:267 (Fig 6): the error of a p-th order expansion scales as (b/r)^(p+1)."""
    x = np.array([2.0, 1.5, -1.0])
    want = {0: 4.0, 2: 8.0, 3: 16.0, 4: 32.0}
    for order, ratio in want.items():
        errs = []
        for b in (0.2, 0.1):
            y, m = _cluster(b)
            mom, z = O.moments_of(y, m)
            a, p = O.cell_on_sink(mom, z, order, x, eps)
            ad, pd = _direct_on(x, y, m, eps)
            errs.append((np.linalg.norm(a - ad) / np.linalg.norm(ad), abs(p - pd) / abs(pd)))
        for k in range(2):
            r = errs[0][k] / errs[1][k]
            assert abs(r / ratio - 1) < 0.15, (order, k, r)


def test_one_particle_cell_is_particle_particle():
    y = np.array([[0.3, -0.1, 0.2]]); m = np.array([0.7]); x = np.array([1.0, 0.4, -0.3])
    mom, z = O.moments_of(y, m)
    assert np.abs(mom[1:]).max() < 1e-16 and np.allclose(z, y[0], rtol=1e-15)
    ad, pd = _direct_on(x, y, m, 0.05)
    for order in (0, 2, 3, 4):
        a, p = O.cell_on_sink(mom, z, order, x, 0.05)
        assert np.allclose(a, ad, rtol=1e-14) and math.isclose(p, pd, rel_tol=1e-14)


def test_two_equal_masses_series():
    """phi = -(2m/R)(1 + d^2/R^2 + d^4/R^4 + ...) on the axis, eps = 0 (SURVEY C-10 O-9)."""
    dl, R, m = 0.1, 1.0, 0.5
    y = np.array([[dl, 0, 0], [-dl, 0, 0]]); mm = np.array([m, m]); x = np.array([R, 0, 0.0])
    mom, z = O.moments_of(y, mm)
    q = (dl / R) ** 2
    for order, nterm in ((0, 1), (2, 2), (3, 2), (4, 3)):
        a, p = O.cell_on_sink(mom, z, order, x, 0.0)
        assert math.isclose(p, -(2 * m / R) * sum(q**k for k in range(nterm)), rel_tol=1e-14)
        # a_x = -d phi/dR of the truncated series: -(2m) sum (2k+1) d^(2k) / R^(2k+2)
        assert math.isclose(a[0], -(2 * m) * sum((2 * k + 1) * dl ** (2 * k) / R ** (2 * k + 2) for k in range(nterm)), rel_tol=1e-14)


def test_moment_pins():
    w = W.config(0, 11)
    T = O.Tree(w.pos, w.mass, w.lo, w.size)
    mom, com, bmax = T.moments()
    c = T.cells()
    m = w.mass.astype(np.float64); x = w.pos.astype(np.float64)
    assert math.isclose(mom[0, 0], m.sum(), rel_tol=1e-14)
    assert np.allclose(com[0], (m[:, None] * x).sum(0) / m.sum(), rtol=1e-13)
    assert np.abs(mom[:, 1:4]).max() < 1e-13 * mom[0, 0] * w.size  # dipole about the centre of mass
    one = c["count"] == 1
    assert one.any() and np.abs(mom[one, 1:]).max() == 0 and (bmax[one] == 0).all()
    # second moments of the root against numpy
    d = x - com[0]
    assert math.isclose(mom[0, 4], (m * d[:, 0] ** 2).sum(), rel_tol=1e-12)   # xx
    assert math.isclose(mom[0, 5], (m * d[:, 0] * d[:, 1]).sum(), rel_tol=1e-10, abs_tol=1e-16)  # xy
    assert math.isclose(mom[0, 9], (m * d[:, 2] ** 2).sum(), rel_tol=1e-12)   # zz
    assert math.isclose(mom[0, 34], (m * d[:, 2] ** 4).sum(), rel_tol=1e-12)  # zzzz
    assert math.isclose(mom[0, 24], (m * d[:, 0] ** 2 * d[:, 1] * d[:, 2]).sum(), rel_tol=1e-9, abs_tol=1e-18)  # xxyz
    assert math.isclose(bmax[0], np.sqrt((d * d).sum(1)).max(), rel_tol=1e-14)


# ---------------------------------------------------------------- walk + tree forces (C-7, C-8)
def test_theta_zero_is_direct_sum():
    w = W.config(2, 9)
    T = O.Tree(w.pos, w.mass, w.lo, w.size, nleaf=4, ncrit=16)
    a, p, lpc, lpp = T.forces(0.0, w.eps, 4)
    ad, pd = O.direct(w.pos, w.mass, w.eps)
    assert (lpc == 0).all() and (lpp == w.n).all()
    assert np.abs(a - ad).max() <= 1e-12 * np.abs(ad).max() and np.abs(p - pd).max() <= 1e-12 * np.abs(pd).max()


@pytest.mark.parametrize("cfg,scale", [(0, 12), (1, 12), (2, 12)])
def test_coverage_invariant(cfg, scale):
    w = W.config(cfg, scale)
    T = O.Tree(w.pos, w.mass, w.lo, w.size)
    for theta in (0.3, 0.5, 0.8):
        lpc, lpp, cov = T.walk_counts(theta)
        assert (cov + lpp == w.n).all()
    # the lists of one group: disjoint particle cover, no accepted cell touches the group
    c = T.cells()
    g = T.ngroups // 2
    pc, lv = T.walk_lists(0.5, g)
    seen = np.zeros(w.n, int)
    for ci in list(pc) + list(lv):
        seen[c["first"][ci]:c["first"][ci] + c["count"][ci]] += 1
    assert (seen == 1).all()


def test_error_monotone_in_order_and_theta():
    w = W.config(1, 12)
    T = O.Tree(w.pos, w.mass, w.lo, w.size)
    ad, pd = O.direct(w.pos, w.mass, w.eps)
    def rms(theta, order):
        a, p, _, _ = T.forces(theta, w.eps, order)
        return math.sqrt(((a - ad) ** 2).sum() / (ad ** 2).sum())
    e = {(t, o): rms(t, o) for t in (0.4, 0.6, 0.8) for o in (0, 2, 4)}
    for t in (0.4, 0.6, 0.8):
        assert e[(t, 0)] > e[(t, 2)] > e[(t, 4)]
    for o in (0, 2, 4):
        assert e[(0.4, o)] < e[(0.6, o)] < e[(0.8, o)]
    assert e[(0.4, 4)] < 1e-5
