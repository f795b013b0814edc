"""ctypes front end of oracle/hot_oracle.c (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import this module.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hot_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
NMOM = 35


def build(force: bool = False) -> str:
    """Compile hot_oracle.c with gcc (double precision, OpenMP over sink groups only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
               _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_create.restype = C.c_void_p
        _lib.orc_n.restype = C.c_int64
        _lib.orc_ncells.restype = C.c_int64
        _lib.orc_ngroups.restype = C.c_int64
        _lib.orc_dg.restype = C.c_double
        _lib.orc_psi_smooth.restype = C.c_double
        _lib.orc_ewald_xi.restype = C.c_double
        _lib.orc_mac_bound.restype = C.c_double
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int64)


def set_moment_order(order):
    """Trees created from now on keep moments through this degree (4 by default; 6 or 8 for the high orders of f-3)."""
    global NMOM
    lib().orc_set_moment_order(int(order))
    NMOM = (order + 1) * (order + 2) * (order + 3) // 6


def multi_indices(order=4):
    """(a,b,c) of the moments, degree-major then x>y>z, as hot_oracle.c orders them."""
    out = []
    for d in range(order + 1):
        for a in range(d, -1, -1):
            for b in range(d - a, -1, -1):
                out.append((a, b, d - a - b))
    return out


def keys(pos, lo, size):
    pos = _f32(pos)
    n = pos.shape[0]
    key = np.empty(n, dtype=np.uint64)
    lo = _f32(lo)
    st = lib().orc_keys(_p(pos), C.c_int64(n), _p(lo), C.c_float(size), _p(key))
    if st:
        raise ValueError("particle outside the box")
    return key


def direct(pos, mass, eps, sinks=None):
    pos, mass = _f32(pos), _f32(mass)
    n = pos.shape[0]
    sinks = _i64(sinks)
    ns = n if sinks is None else sinks.shape[0]
    acc = np.empty((ns, 3))
    pot = np.empty(ns)
    lib().orc_direct(_p(pos), _p(mass), C.c_int64(n), C.c_double(eps), _p(sinks), C.c_int64(ns),
                     _p(acc), _p(pot))
    return acc, pot


def ewald_direct(pos, mass, size, eps, sinks=None):
    pos, mass = _f32(pos), _f32(mass)
    n = pos.shape[0]
    sinks = _i64(sinks)
    ns = n if sinks is None else sinks.shape[0]
    acc = np.empty((ns, 3))
    pot = np.empty(ns)
    lib().orc_ewald_direct(_p(pos), _p(mass), C.c_int64(n), C.c_double(size), C.c_double(eps),
                           _p(sinks), C.c_int64(ns), _p(acc), _p(pot))
    return acc, pot


def ewald_psi(r):
    r = np.ascontiguousarray(r, dtype=np.float64)
    psi = C.c_double()
    g = np.empty(3)
    lib().orc_ewald_psi(_p(r), C.byref(psi), _p(g))
    return psi.value, g


def psi_smooth(r):
    r = np.ascontiguousarray(r, dtype=np.float64)
    return lib().orc_psi_smooth(_p(r))


def ewald_xi():
    return lib().orc_ewald_xi()


def dg(a, b, c, R, eps):
    R = np.ascontiguousarray(R, dtype=np.float64)
    return lib().orc_dg(a, b, c, _p(R), C.c_double(eps))


def moments_of(y, m, order=4):
    y = np.ascontiguousarray(y, dtype=np.float64)
    m = np.ascontiguousarray(m, dtype=np.float64)
    mom = np.empty((order + 1) * (order + 2) * (order + 3) // 6)
    z = np.empty(3)
    lib().orc_moments_of_order(_p(y), _p(m), C.c_int64(y.shape[0]), int(order), _p(mom), _p(z))
    return mom, z


def cell_on_sink(mom, z, order, x, eps):
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    z = np.ascontiguousarray(z, dtype=np.float64)
    x = np.ascontiguousarray(x, dtype=np.float64)
    acc = np.empty(3)
    pot = C.c_double()
    lib().orc_cell_on_sink(_p(mom), _p(z), order, _p(x), C.c_double(eps), _p(acc), C.byref(pot))
    return acc, pot.value


def mac_bound(mom35, b, R, p):
    """Error bound of DESIGN.md R-16 for a cell with moments mom35 (about its centre of mass), radius b, at distance R."""
    mom35 = np.ascontiguousarray(mom35, dtype=np.float64)
    return lib().orc_mac_bound(_p(mom35), C.c_double(b), C.c_double(R), int(p))


def set_softening(kind):
    """0: Plummer (default); 1: cubic spline with h = 2.8 eps.  Global to the oracle library."""
    lib().orc_set_softening(int(kind))


def spline_kernel(r, h):
    fac, pot = C.c_double(), C.c_double()
    lib().orc_spline_kernel(C.c_double(r), C.c_double(h), C.byref(fac), C.byref(pot))
    return fac.value, pot.value


def kick_drift(pos, vel, acc, dtk, dtd, lo, size, periodic):
    """In place on float32 arrays: v += a dtk; x += v dtd (one fmaf each), periodic wrap."""
    assert pos.dtype == np.float32 and vel.dtype == np.float32 and pos.flags["C_CONTIGUOUS"] and vel.flags["C_CONTIGUOUS"]
    acc = _f32(acc); lo = _f32(lo)
    lib().orc_kick_drift(_p(pos), _p(vel), _p(acc), C.c_int64(pos.shape[0]), C.c_float(dtk), C.c_float(dtd), _p(lo), C.c_float(size), int(bool(periodic)))


def set_num_threads(n):
    lib().orc_set_num_threads(int(n))


def cube_field(x, lo, side):
    """Potential and acceleration at x of the homogeneous unit-density cube [lo, lo+side)^3 (closed form)."""
    x = np.ascontiguousarray(x, dtype=np.float64); lo = np.ascontiguousarray(lo, dtype=np.float64)
    phi = C.c_double(); a = np.empty(3)
    lib().orc_cube_field(_p(x), _p(lo), C.c_double(side), C.byref(phi), _p(a))
    return phi.value, a


def cube_moments(side):
    mom = np.empty(35)
    lib().orc_cube_moments(C.c_double(side), _p(mom))
    return mom


def num_threads():
    return lib().orc_num_threads()


class Tree:
    """Keys, stable sort, bucket oct-tree, groups and moments of one particle set."""

    def __init__(self, pos, mass, lo, size, periodic=False, nleaf=16, ncrit=64, moments=True):
        self.pos, self.mass = _f32(pos), _f32(mass)
        self.n = self.pos.shape[0]
        self.lo = _f32(lo)
        self.size = float(size)
        self.periodic = bool(periodic)
        st = C.c_int()
        self._h = lib().orc_create(_p(self.pos), _p(self.mass), C.c_int64(self.n), _p(self.lo),
                                   C.c_float(size), int(periodic), nleaf, ncrit, int(moments),
                                   C.byref(st))
        if not self._h:
            raise ValueError(f"orc_create failed: {st.value}")
        self._h = C.c_void_p(self._h)
        self.ncells = lib().orc_ncells(self._h)
        self.ngroups = lib().orc_ngroups(self._h)
        self.nmom = NMOM  # moments per cell of this tree (set_moment_order at creation time)
        self.has_moments = bool(moments)  # moments = 2 ("lazy"): only the cells that forces() needs, on demand

    def __del__(self):
        if getattr(self, "_h", None):
            try:
                lib().orc_destroy(self._h)
            except TypeError:  # interpreter shutdown: the module globals are already gone
                pass
            self._h = None

    def keys(self):
        key = np.empty(self.n, dtype=np.uint64)
        skey = np.empty(self.n, dtype=np.uint64)
        perm = np.empty(self.n, dtype=np.uint32)
        lib().orc_get_keys(self._h, _p(key), _p(skey), _p(perm))
        return key, skey, perm

    def cells(self):
        nc = self.ncells
        out = dict(key=np.empty(nc, np.uint64), level=np.empty(nc, np.int32),
                   first=np.empty(nc, np.int64), count=np.empty(nc, np.int64),
                   mask=np.empty(nc, np.uint8), child=np.empty(nc, np.int64),
                   parent=np.empty(nc, np.int64))
        lib().orc_get_cells(self._h, _p(out["key"]), _p(out["level"]), _p(out["first"]),
                            _p(out["count"]), _p(out["mask"]), _p(out["child"]), _p(out["parent"]))
        return out

    def groups(self):
        g = np.empty(self.ngroups, dtype=np.int64)
        lib().orc_get_groups(self._h, _p(g))
        return g

    def leaf_of(self):
        leaf = np.empty(self.n, dtype=np.int64)
        lib().orc_get_leaf_of(self._h, _p(leaf))
        return leaf

    def moments(self):
        nc = self.ncells
        mom = np.empty((nc, self.nmom))
        com = np.empty((nc, 3))
        bmax = np.empty(nc)
        lib().orc_get_moments(self._h, _p(mom), _p(com), _p(bmax))
        return mom, com, bmax

    def bbound(self):
        """b_max as an upward pass carries it (children's radii + centre offsets); >= moments()[2]."""
        bb = np.empty(self.ncells)
        lib().orc_get_bbound(self._h, _p(bb))
        return bb

    def walk_counts(self, theta, groups=None):
        groups = _i64(groups)
        ng = self.ngroups if groups is None else groups.shape[0]
        lpc = np.empty(ng, np.int64)
        lpp = np.empty(ng, np.int64)
        cov = np.empty(ng, np.int64)
        lib().orc_walk_counts(self._h, C.c_double(theta), _p(groups), C.c_int64(ng), _p(lpc),
                              _p(lpp), _p(cov))
        return lpc, lpp, cov

    def walk_lists(self, theta, group, img=(0, 0, 0)):
        cap = self.ncells
        pc = np.empty(cap, np.int64)
        lv = np.empty(cap, np.int64)
        npc = C.c_int64()
        nlv = C.c_int64()
        im = np.ascontiguousarray(img, dtype=np.int32)
        lib().orc_walk_lists(self._h, C.c_double(theta), C.c_int64(group), _p(im), C.c_int64(cap),
                             _p(pc), C.byref(npc), _p(lv), C.byref(nlv))
        return pc[:npc.value].copy(), lv[:nlv.value].copy()

    def forces(self, theta, eps, order, groups=None):
        """acc[n,3], pot[n] (caller's order; NaN where not evaluated), Lpc, Lpp per listed group."""
        groups = _i64(groups)
        ng = self.ngroups if groups is None else groups.shape[0]
        acc = np.full((self.n, 3), np.nan)
        pot = np.full(self.n, np.nan)
        lpc = np.empty(ng, np.int64)
        lpp = np.empty(ng, np.int64)
        lib().orc_tree_forces(self._h, C.c_double(theta), C.c_double(eps), int(order), _p(groups),
                              C.c_int64(ng), _p(acc), _p(pot), _p(lpc), _p(lpp))
        return acc, pot, lpc, lpp

    def forces_tol(self, tol, eps, groups=None, evaluate=True):
        """Error-bound MAC with per-interaction order (R-16): acc, pot, and per listed group the accepted cells by
        order (monopole, quadrupole, hexadecapole) and L_pp."""
        groups = _i64(groups)
        ng = self.ngroups if groups is None else groups.shape[0]
        acc = np.full((self.n, 3), np.nan) if evaluate else None
        pot = np.full(self.n, np.nan) if evaluate else None
        l0, l2, l4, lpp = (np.empty(ng, np.int64) for _ in range(4))
        lib().orc_tree_forces_tol(self._h, C.c_double(tol), C.c_double(eps), _p(groups), C.c_int64(ng),
                                  _p(acc), _p(pot), _p(l0), _p(l2), _p(l4), _p(lpp))
        return acc, pot, l0, l2, l4, lpp

    def forces_bg(self, theta, eps, order, groups=None):
        """Periodic boxes with per-cell background subtraction (R-18): acc, pot, and per listed group the accepted
        cells (all), the background-subtracted ones among them, the accepted virtual cubes, and L_pp."""
        groups = _i64(groups)
        ng = self.ngroups if groups is None else groups.shape[0]
        acc = np.full((self.n, 3), np.nan); pot = np.full(self.n, np.nan)
        lpc, lbg, lv, lpp = (np.empty(ng, np.int64) for _ in range(4))
        vol = np.empty(ng)
        lib().orc_tree_forces_bg(self._h, C.c_double(theta), C.c_double(eps), int(order), _p(groups), C.c_int64(ng),
                                 _p(acc), _p(pot), _p(lpc), _p(lbg), _p(lv), _p(lpp), _p(vol))
        self.bg_volume = vol  # subtracted volume per group in units of the box: 125 - (5 s_G / size)^3 exactly
        return acc, pot, lpc, lbg, lv, lpp

    def far_table(self):
        co = np.empty(165)
        lib().orc_far_table(self._h, _p(co))
        return co
