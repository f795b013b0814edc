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
    # O-2 termwise: the force of j on i is minus the force of i on j.  A pair's term is what is left of the
    # direct sum when every other body is removed, so evaluate pairs (i, j) on their own
    x = w.pos.astype(np.float64)
    for i, j in ((0, 1), (5, 900), (17, 18), (1023, 3)):
        a2, p2 = O.direct(w.pos[[i, j]], w.mass[[i, j]], w.eps)
        assert np.array_equal(m[i] * a2[0], -(m[j] * a2[1])), (i, j)          # bit-exact: same |d|, same products
        assert m[i] * p2[0] == m[j] * p2[1]
    # energy symmetry: sum_i m_i phi_i = 2 * sum_{i<j} (pair energy), pair energies typed out here with numpy
    k = 65
    e = 0.0
    for i in range(k - 1):
        d = x[i + 1:k] - x[i]
        e += -(m[i] * m[i + 1:k] / np.sqrt((d * d).sum(1) + w.eps**2)).sum()
    a64, p64 = O.direct(w.pos[:k], w.mass[:k], w.eps)
    assert math.isclose((m[:k] * p64).sum(), 2 * e, rel_tol=1e-13)
    assert np.abs((m[:k, None] * a64).sum(0)).max() <= 1e-13 * (m[:k, None] * np.abs(a64)).sum()
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
    # every second, third and fourth moment (indices 4..34) of the root and of a mid-tree cell, typed out with numpy
    key, skey, perm = T.keys()
    xs, ms = x[perm], m[perm]
    mid = int(np.argmax((c["level"] == 2) & (c["count"] > 40)))
    assert c["level"][mid] == 2
    for ci in (0, mid):
        f, k = int(c["first"][ci]), int(c["count"][ci])
        dd = xs[f:f + k] - (ms[f:f + k, None] * xs[f:f + k]).sum(0) / ms[f:f + k].sum()
        for q, (a, b, cc) in enumerate(O.multi_indices()):
            if a + b + cc < 2:
                continue
            want = (ms[f:f + k] * dd[:, 0] ** a * dd[:, 1] ** b * dd[:, 2] ** cc).sum()
            assert abs(mom[ci, q] - want) <= 1e-12 * ms[f:f + k].sum() * np.abs(dd).max() ** (a + b + cc), (ci, a, b, cc)


def test_bmax_bound_of_the_upward_pass():
    """R-15: the b_max an upward pass can carry (children's radii + centre offsets) contains every body of the
    cell: it is never below the exact radius, equals it on leaves, and never exceeds the cell's diagonal by more
    than the children's slack (sanity: <= 2 x the exact radius + the cell diagonal)."""
    w = W.config(2, 12)
    T = O.Tree(w.pos, w.mass, w.lo, w.size, nleaf=4, ncrit=16)
    mom, com, bmax = T.moments()
    bb = T.bbound()
    c = T.cells()
    leaf = c["child"] < 0
    assert (bb >= bmax * (1 - 1e-15)).all()
    assert (bb[leaf] == bmax[leaf]).all()
    # brute force from the bodies: every body lies within bb of the centre of mass
    key, skey, perm = T.keys()
    xs = w.pos.astype(np.float64)[perm]
    for ci in np.random.default_rng(0).choice(T.ncells, 200, replace=False):
        f, k = int(c["first"][ci]), int(c["count"][ci])
        r = np.sqrt(((xs[f:f + k] - com[ci]) ** 2).sum(1)).max()
        assert r <= bb[ci] * (1 + 1e-14) and math.isclose(r, bmax[ci], rel_tol=1e-13, abs_tol=1e-300)
    side = w.size * np.ldexp(1.0, -c["level"].astype(np.int64))
    assert (bb <= np.sqrt(3.0) * side * 2).all()


def test_lazy_moments_give_the_same_forces():
    """moments=2 (only the cells the requested groups accept; used at 2^27 bodies) is the same arithmetic."""
    w = W.config(2, 11)
    T1 = O.Tree(w.pos, w.mass, w.lo, w.size)
    T2 = O.Tree(w.pos, w.mass, w.lo, w.size, moments=2)
    sel = np.array([0, 3, T1.ngroups - 1])
    a1, p1, lpc1, lpp1 = T1.forces(0.5, w.eps, 4, groups=sel)
    a2, p2, lpc2, lpp2 = T2.forces(0.5, w.eps, 4, groups=sel)
    assert np.array_equal(a1, a2, equal_nan=True) and np.array_equal(p1, p2, equal_nan=True)
    assert (lpc1 == lpc2).all() and (lpp1 == lpp2).all()


# ---------------------------------------------------------------- walk + tree forces (C-7, C-8)
def test_theta_zero_is_direct_sum():
    w = W.config(2, 9)
    T = O.Tree(w.pos, w.mass, w.lo, w.size, nleaf=4, ncrit=16)
    a, p, lpc, lpp = T.forces(0.0, w.eps, 4)
    ad, pd = O.direct(w.pos, w.mass, w.eps)
    assert (lpc == 0).all() and (lpp == w.n).all()
    assert np.abs(a - ad).max() <= 1e-12 * np.abs(ad).max() and np.abs(p - pd).max() <= 1e-12 * np.abs(pd).max()


def _lattice64():
    """One body at the centre of each of the 64 level-2 cells; NLEAF = NCRIT = 1: root, 8 level-1 cells,
    64 level-2 leaves which are also the sink groups.  Returns the tree and, per cell index, (level, i, j, k)."""
    q = (np.arange(4) + 0.5) / 4
    pts = np.array([[x, y, z] for x in q for y in q for z in q], np.float32)
    T = O.Tree(pts, np.ones(64, np.float32), (0, 0, 0), 1.0, nleaf=1, ncrit=1, moments=False)
    c = T.cells()
    assert T.ncells == 73 and T.ngroups == 64
    geo = {}
    for ci in range(T.ncells):
        l = int(c["level"][ci])
        k = int(c["key"][ci]) & ((1 << (3 * l)) - 1)
        ijk = [0, 0, 0]
        for b in range(l):
            for ax in range(3):
                ijk[ax] |= ((k >> (3 * b + 2 - ax)) & 1) << b
        geo[ci] = (l, *ijk)
    return T, c, geo


def _by_hand_accepts(level, ijk, img, theta):
    """SURVEY C-7 / DESIGN R-7 worked by hand for the group = level-2 cell (0,0,0) of the 4x4x4 lattice, in
    units of the level-2 side s (group = [0,1)^3): a level-l cell (i,j,k) of image n is the cube
    [i w + 4 n, (i+1) w + 4 n) with w = 4 / 2^l; gap per axis = distance between the intervals (0 if they touch
    or overlap); accepted iff w^2 < theta^2 * (sum of squared gaps), strictly."""
    from fractions import Fraction
    wdt = Fraction(4, 2 ** level)
    d2 = Fraction(0)
    for ax in range(3):
        lo = ijk[ax] * wdt + 4 * img[ax]
        hi = lo + wdt
        gap = max(Fraction(0), lo - 1, 0 - hi)
        d2 += gap * gap
    return wdt * wdt < Fraction(theta).limit_denominator(10 ** 6) ** 2 * d2


@pytest.mark.parametrize("theta", [0.5, 0.51, 0.577, 0.578, 0.9])
def test_mac_by_hand_open_and_one_image(theta):
    """The FORM of the criterion (verdict r1 item 4): minimum distance between the cubes (not centre distance),
    s_C^2 < theta^2 d^2 strictly, d = 0 never accepted, image shift +n L applied to the SOURCE."""
    T, c, geo = _lattice64()
    g0 = 0  # groups are in key order: group 0 is the level-2 cell (0,0,0)
    assert geo[int(T.groups()[0])] == (2, 0, 0, 0)
    for img in ((0, 0, 0), (-1, 0, 0), (1, 0, 0), (0, 2, -1)):
        pc, lv = T.walk_lists(theta, g0, img=img)
        want_pc, want_lv = set(), set()
        # by hand: no level-0/1 cell is ever accepted for theta < 1 in the box itself (gap <= its own side);
        # in an image, walk the three levels with the rule above
        def visit(ci):
            l, i, j, k = geo[ci]
            if _by_hand_accepts(l, (i, j, k), img, theta):
                want_pc.add(ci)
            elif c["child"][ci] < 0:
                want_lv.add(ci)
            else:
                for ch in range(int(c["child"][ci]), int(c["child"][ci]) + bin(int(c["mask"][ci])).count("1")):
                    visit(ch)
        visit(0)
        assert set(pc.tolist()) == want_pc and set(lv.tolist()) == want_lv, (theta, img)
        assert len(pc) == len(want_pc) and len(lv) == len(want_lv)
    # the named cases, spelled out
    pc, lv = T.walk_lists(theta, g0)
    by = {geo[ci][1:]: ci for ci in geo if geo[ci][0] == 2}
    # cell (2,2,2): gap (s,s,s), d^2 = 3 s^2: accepted iff theta^2 > 1/3
    assert (by[(2, 2, 2)] in pc) == (theta * theta > 1 / 3)
    # cell (3,0,0): gap (2s,0,0), d^2 = 4 s^2: theta = 0.5 is an exact tie and a tie is NOT accepted
    assert (by[(3, 0, 0)] in pc) == (theta > 0.5)
    # face-, edge- and corner-adjacent cells touch the group (d = 0): never accepted, and neither is the group itself
    for adj in ((1, 0, 0), (1, 1, 0), (1, 1, 1), (0, 0, 0)):
        assert by[adj] in lv and by[adj] not in pc
    # a centre-distance criterion would differ: (2,0,0) has centre distance 2s but gap s -> rejected for theta < 1
    assert by[(2, 0, 0)] in lv
    # image (-1,0,0): the copy of cell (3,0,0) occupies x in [-s, 0) and touches the group: never accepted;
    # the copy of cell (1,0,0) occupies [-3s,-2s): gap 2 s: accepted iff theta > 0.5.  With the shift applied
    # with the wrong sign these cells would sit at x in [7s, 8s) and [5s, 6s) and both be accepted at theta >= 0.5.
    pc, lv = T.walk_lists(theta, g0, img=(-1, 0, 0))
    assert by[(3, 0, 0)] in lv
    assert (by[(1, 0, 0)] in pc) == (theta > 0.5)
    # every group, every listed image: accepted cells + rejected leaves cover each body exactly once
    for g in (0, 21, 63):
        for img in ((0, 0, 0), (2, -2, 1)):
            pc, lv = T.walk_lists(theta, g, img=img)
            seen = np.zeros(64, int)
            for ci in list(pc) + list(lv):
                seen[c["first"][ci]:c["first"][ci] + c["count"][ci]] += 1
            assert (seen == 1).all()


@pytest.mark.parametrize("cfg,scale", [(0, 12), (1, 12), (2, 12)])
def test_coverage_invariant(cfg, scale):
    w = W.config(cfg, scale)
    T = O.Tree(w.pos, w.mass, w.lo, w.size)
    for theta in (0.3, 0.5, 0.8):
        lpc, lpp, cov = T.walk_counts(theta)
        assert (cov + lpp == w.n).all()
    # the lists of one group: disjoint particle cover, and no accepted cell touches or overlaps the group's cube
    c = T.cells()
    g = T.ngroups // 2
    pc, lv = T.walk_lists(0.5, g)
    seen = np.zeros(w.n, int)
    for ci in list(pc) + list(lv):
        seen[c["first"][ci]:c["first"][ci] + c["count"][ci]] += 1
    assert (seen == 1).all()

    def cube(ci):  # integer corner and side on the 2^21 grid, from the key alone
        l = int(c["level"][ci]); k = int(c["key"][ci]) & ((1 << (3 * l)) - 1)
        o = [0, 0, 0]
        for b in range(l):
            for ax in range(3):
                o[ax] |= ((k >> (3 * b + 2 - ax)) & 1) << b
        return [v << (21 - l) for v in o], 1 << (21 - l)
    go, gs = cube(int(T.groups()[g]))
    for ci in pc:
        o, sz = cube(int(ci))
        gaps = [max(0, o[ax] - (go[ax] + gs), go[ax] - (o[ax] + sz)) for ax in range(3)]
        assert sum(v * v for v in gaps) * 0.25 > sz * sz  # accepted at theta = 0.5: strictly separated, by more than 2 sides


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


# ---------------------------------------------------------------- f-2: error-bound MAC (R-16)
def test_error_bound_holds_for_random_cells():
    """Fig 6's set-up: 512 random particles in a unit cube, a sink at distance r.  The bound of R-16
    must never be below the actual truncation error of the expansion about the centre of mass -- for every order it
    is used with, every direction, softened or not -- and must not be uselessly loose either."""
    rng = np.random.default_rng(68)
    worst = {0: 0.0, 2: 0.0, 4: 0.0}
    loose = {0: [], 2: [], 4: []}
    for trial in range(6):
        n = 512 if trial < 3 else 9
        y = rng.uniform(-0.5, 0.5, (n, 3)) * (1.0 if trial % 2 == 0 else np.array([1.0, 0.2, 0.05]))
        m = rng.uniform(0.5, 1.5, n) / n
        mom, z = O.moments_of(y, m)
        b = np.sqrt(((y - z) ** 2).sum(1)).max()
        for eps in (0.0, 0.05):
            for r in (1.05 * b, 1.5 * b, 1.0, 2.0, 4.0, 16.0):
                if r <= b:
                    continue
                for _ in range(8):
                    u = rng.standard_normal(3); u /= np.linalg.norm(u)
                    x = z + r * u
                    ad, pd = _direct_on(x, y, m, eps)
                    for order, p in ((0, 1), (2, 2), (4, 4)):
                        a, ph = O.cell_on_sink(mom, z, order, x, eps)
                        err = np.linalg.norm(a - ad)
                        bound = O.mac_bound(mom, b, r, p)
                        assert err <= bound * (1 + 1e-9) + 1e-15 * np.linalg.norm(ad), (trial, eps, r, order, err, bound)
                        worst[order] = max(worst[order], err / bound)
                        if r >= 2 * b and eps == 0.0 and n == 512:
                            loose[order].append(bound / max(err, 1e-300))
    assert all(v > 0.02 for v in worst.values()), worst           # the bound is approached within a factor of 50
    assert all(np.median(v) < 2000 for v in loose.values()), {k: np.median(v) for k, v in loose.items()}
    assert O.mac_bound(mom, b, 0.9 * b, 2) == np.inf                # inside the cell's radius: never accepted


def test_error_bound_tree_properties():
    """Tolerance -> 0: everything particle-particle = the direct sum.  Larger tolerance: fewer, lower-order
    interactions and a larger error, always below tolerance x accepted cells; coverage invariant."""
    w = W.config(2, 11)
    T = O.Tree(w.pos, w.mass, w.lo, w.size, nleaf=8, ncrit=32)
    ad, pd = O.direct(w.pos, w.mass, w.eps)
    a, p, l0, l2, l4, lpp = T.forces_tol(0.0, w.eps)
    # tolerance 0 accepts only cells whose bound is 0: single bodies, whose monopole is exact
    assert (l2 + l4 == 0).all() and (l0 + lpp == w.n).all()
    assert np.abs(a - ad).max() <= 1e-12 * np.abs(ad).max()
    arms = np.sqrt((ad ** 2).sum(1).mean())
    prev_cost, prev_err = None, None
    for tol in (1e-5 * arms, 1e-3 * arms, 1e-1 * arms):
        a, p, l0, l2, l4, lpp = T.forces_tol(tol, w.eps)
        err = np.linalg.norm(a - ad, axis=1)
        # every particle's error is below tol x (number of cells its group accepted)
        gcount = T.cells()["count"][T.groups()]
        per_body = np.repeat(l0 + l2 + l4, gcount)          # in key order
        perm = T.keys()[2]
        bound = np.empty(w.n); bound[perm] = per_body * tol
        assert (err <= bound + 1e-12 * arms).all()
        cost = (gcount * (l0 + 3 * l2 + 13 * l4 + lpp)).sum()
        rms = np.sqrt((err ** 2).mean()) / arms
        if prev_cost is not None:
            assert cost < prev_cost and rms > prev_err
        prev_cost, prev_err = cost, rms
    assert l0.sum() > 0 and l2.sum() > 0                   # a mix of orders at the loosest tolerance
    a, p, l0, l2, l4, lpp = T.forces_tol(1e-4 * arms, w.eps)
    assert l2.sum() > 0 and l4.sum() > 0


# ---------------------------------------------------------------- f-4: spline softening, kick / drift
def test_spline_kernel_is_the_field_of_the_spline_ball():
    """PAPER.md:136 (spline kernel of ref [50]).  The force factor and potential are pinned by quadrature of the
    density they claim to come from: W(u) = 8/(pi h^3) (1 - 6u^2 + 6u^3 | 2 (1-u)^3); enclosed mass / r^3 and
    -(M(r)/r + 4 pi int_r^h W r' dr'); unit total mass; Newtonian outside; phi(0) = -2.8/h; continuous at the joints."""
    h = 0.7
    def W(r):
        u = r / h
        return 8 / (np.pi * h ** 3) * np.where(u <= 0.5, 1 - 6 * u ** 2 + 6 * u ** 3, np.where(u <= 1, 2 * (1 - u) ** 3, 0.0))
    rr = np.linspace(0, h, 400001)
    dm = 4 * np.pi * W(rr) * rr ** 2
    M = np.concatenate([[0], np.cumsum(0.5 * (dm[1:] + dm[:-1]) * np.diff(rr))])      # trapezoid
    sh = 4 * np.pi * W(rr) * rr
    outer = np.concatenate([np.cumsum((0.5 * (sh[1:] + sh[:-1]) * np.diff(rr))[::-1])[::-1], [0]])
    assert abs(M[-1] - 1) < 1e-9
    for r in (0.05 * h, 0.3 * h, 0.5 * h, 0.77 * h, 0.999 * h):
        i = int(round(r / h * 400000))
        fac, pot = O.spline_kernel(rr[i], h)
        assert math.isclose(fac, M[i] / rr[i] ** 3, rel_tol=1e-7), r
        assert math.isclose(pot, -(M[i] / rr[i] + outer[i]), rel_tol=1e-7), r
    assert math.isclose(O.spline_kernel(0.0, h)[1], -2.8 / h, rel_tol=1e-15) and math.isclose(O.spline_kernel(0.0, h)[0], 32 / 3 / h ** 3, rel_tol=1e-15)
    for r in (h, 1.5 * h):
        fac, pot = O.spline_kernel(r, h)
        assert math.isclose(fac, r ** -3, rel_tol=1e-15) and math.isclose(pot, -1 / r, rel_tol=1e-15)
    for r in (0.5 * h, h):
        a, b = O.spline_kernel(r * (1 - 1e-9), h), O.spline_kernel(r * (1 + 1e-9), h)
        assert math.isclose(a[0], b[0], rel_tol=1e-7) and math.isclose(a[1], b[1], rel_tol=1e-7)


def test_spline_softened_tree_against_direct_sum():
    w = W.config(2, 11)
    eps = 2e-3   # h = 5.6e-3: many pairs inside the kernel's support
    O.set_softening(1)
    try:
        ad, pd = O.direct(w.pos, w.mass, eps)
        T = O.Tree(w.pos, w.mass, w.lo, w.size, nleaf=8, ncrit=32)
        a0, p0, lpc0, lpp0 = T.forces(0.0, eps, 2)
        assert np.abs(a0 - ad).max() <= 1e-12 * np.abs(ad).max() and np.abs(p0 - pd).max() <= 1e-12 * np.abs(pd).max()
        a, p, lpc, lpp = T.forces(0.5, eps, 4)
        assert np.sqrt(((a - ad) ** 2).sum() / (ad ** 2).sum()) < 1e-4
    finally:
        O.set_softening(0)
    ap, pp = O.direct(w.pos, w.mass, eps)
    assert not np.allclose(ap, ad) and np.abs(pp - pd).max() > 0     # a different kernel from Plummer's
    # two bodies: inside the support the pair force is the kernel's, outside Newtonian, always antisymmetric
    O.set_softening(1)
    try:
        for d in (0.3, 0.9, 2.0):
            pos = np.array([[0.1, 0.2, 0.3], [0.1 + d * 2.8 * 0.01, 0.2, 0.3]], np.float32)
            m = np.array([1.0, 3.0], np.float32)
            a2, p2 = O.direct(pos, m, 0.01)
            r = float(pos[1, 0]) - float(pos[0, 0])
            fac, pot = O.spline_kernel(r, 0.028)
            assert math.isclose(a2[0, 0], 3.0 * r * fac, rel_tol=1e-14) and math.isclose(p2[0], 3.0 * pot, rel_tol=1e-14)
            assert np.allclose(1.0 * a2[0], -(3.0 * a2[1]), rtol=1e-15, atol=0)
    finally:
        O.set_softening(0)


def test_kick_drift_is_a_second_order_leapfrog():
    """Kick-drift-kick around the direct sum: a circular two-body orbit closes to O(dt^2) (halving dt quarters the
    error); the periodic wrap keeps every coordinate inside [lo, lo + size)."""
    def orbit(nsteps):
        m = np.array([0.5, 0.5], np.float32)
        pos = np.array([[0.25, 0.5, 0.5], [0.75, 0.5, 0.5]], np.float32)
        v = math.sqrt(0.5 / (4 * 0.25))          # circular: v^2 / r = m / (2r)^2, r = 0.25
        vel = np.array([[0, v, 0], [0, -v, 0]], np.float32)
        dt = 2 * math.pi * 0.25 / v / nsteps
        a, _ = O.direct(pos, m, 0.0)
        for _ in range(nsteps):
            O.kick_drift(pos, vel, a.astype(np.float32), 0.5 * dt, dt, (0, 0, 0), 1.0, False)
            a, _ = O.direct(pos, m, 0.0)
            O.kick_drift(pos, vel, a.astype(np.float32), 0.5 * dt, 0.0, (0, 0, 0), 1.0, False)
        return float(np.linalg.norm(pos[0].astype(np.float64) - [0.25, 0.5, 0.5]))
    e1, e2 = orbit(400), orbit(800)
    assert e1 < 5e-3 and 3.0 < e1 / e2 < 5.0, (e1, e2)
    rng = np.random.default_rng(9)
    pos = rng.uniform(0, 1, (1000, 3)).astype(np.float32); vel = rng.normal(0, 3, (1000, 3)).astype(np.float32)
    p0 = pos.astype(np.float64); v0 = vel.astype(np.float64)
    O.kick_drift(pos, vel, np.zeros((1000, 3), np.float32), 0.0, 0.7, (0, 0, 0), 1.0, True)
    assert (pos >= 0).all() and (pos < 1).all()
    want = (p0 + 0.7 * v0) % 1.0
    d = np.abs(pos - want); d = np.minimum(d, 1 - d)
    assert d.max() < 1e-6


# ---------------------------------------------------------------- f-3: orders 6 and 8
def test_order_law_and_fig6_claim_for_high_orders():
    """PAPER.md:267 (Fig 6): "A single p=8 multipole is more accurate than direct summation in single precision at
    r=4" for 512 particles randomly distributed in a unit cube; and the (b/r)^(p+1) law for p = 5 .. 8."""
    x = np.array([2.0, 1.5, -1.0])
    for order, ratio in ((5, 64.0), (6, 128.0), (7, 256.0), (8, 512.0)):
        errs = []
        for b in (0.2, 0.1):
            y, m = _cluster(b)
            mom, z = O.moments_of(y, m, order=8)
            a, p = O.cell_on_sink(mom, z, order, x, 0.0)
            ad, pd = _direct_on(x, y, m, 0.0)
            errs.append(np.linalg.norm(a - ad) / np.linalg.norm(ad))
        assert abs(errs[0] / errs[1] / ratio - 1) < 0.2, (order, errs[0] / errs[1])
    rng = np.random.default_rng(6)
    y = rng.uniform(-0.5, 0.5, (512, 3)); m = np.full(512, 1 / 512)
    xs = 4.0 * np.array([0.6, 0.64, 0.48])
    ad, _ = _direct_on(xs, y, m, 0.0)
    y32, x32, m32 = y.astype(np.float32), xs.astype(np.float32), m.astype(np.float32)
    a32 = np.zeros(3, np.float32)
    for j in range(512):  # the direct sum as a single-precision code does it
        d = y32[j] - x32
        u = np.float32((d * d).sum())
        a32 += m32[j] * d / np.float32(u * np.sqrt(u))
    e32 = np.linalg.norm(a32.astype(np.float64) - ad) / np.linalg.norm(ad)
    mom, z = O.moments_of(y, m, order=8)
    e = {o: np.linalg.norm(O.cell_on_sink(mom, z, o, xs, 0.0)[0] - ad) / np.linalg.norm(ad) for o in (2, 4, 6, 8)}
    assert e[8] < e32 < e[4], (e, e32)
    assert e[2] > e[4] > e[6] > e[8]


def test_generated_high_order_code_is_what_the_generator_writes():
    import importlib.util
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    path = os.path.join(root, "paper_1310_4502_b200", "csrc", "gen_hi_orders.py")
    spec = importlib.util.spec_from_file_location("gen_hi_orders", path)
    g = importlib.util.module_from_spec(spec); spec.loader.exec_module(g)
    assert g.generate() == open(os.path.join(root, "paper_1310_4502_b200", "csrc", "hot_hi_generated.inc")).read()
