"""ctypes marshalling for include/hot.h.  Same names as the C entry points."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libhot.so")
_lib = None

STATUS = {0: "HOT_OK", -1: "HOT_EINVAL", -2: "HOT_ERANGE", -3: "HOT_ENOMEM", -4: "HOT_ECUDA",
          -5: "HOT_EORDER", -6: "HOT_EINTERNAL"}


class HotError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class hot_box(C.Structure):
    _fields_ = [("lo", C.c_float * 3), ("size", C.c_float)]


class hot_stats_t(C.Structure):
    _fields_ = [("n", C.c_int64), ("n_cells", C.c_int64), ("n_leaves", C.c_int64), ("n_groups", C.c_int64),
                ("max_level", C.c_int32), ("nleaf", C.c_int32), ("ncrit", C.c_int32), ("periodic", C.c_int32),
                ("hash_capacity", C.c_int64), ("hash_max_probe", C.c_int32), ("order", C.c_int32),
                ("pp_interactions", C.c_uint64), ("pc_interactions", C.c_uint64),
                ("cells_visited", C.c_uint64), ("walk_spills", C.c_uint64),
                ("ms_keygen", C.c_float), ("ms_sort", C.c_float), ("ms_gather", C.c_float), ("ms_tree", C.c_float),
                ("ms_moments", C.c_float), ("ms_walk", C.c_float), ("ms_eval", C.c_float), ("ms_farfield", C.c_float),
                ("ms_build_total", C.c_float), ("ms_forces_total", C.c_float),
                ("list_chunks", C.c_int32), ("ms_coarse", C.c_float), ("list_entries", C.c_uint64),
                ("bytes_allocated", C.c_int64),
                ("launches_build", C.c_int64), ("launches_forces", C.c_int64),
                ("pc_monopole", C.c_uint64), ("pc_quadrupole", C.c_uint64), ("pc_hexadecapole", C.c_uint64)]


def library_path() -> str:
    return _LIBPATH


def _load():
    """Load libhot.so; fail loudly if it was not built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise ImportError(f"{_LIBPATH} is missing: run `python -m paper_1310_4502_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        lib = C.CDLL(_LIBPATH)
        lib.hot_last_error.restype = C.c_char_p
        lib.hot_build.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, hot_box, C.c_int]
        lib.hot_forces.argtypes = [C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_void_p]
        lib.hot_stats.argtypes = [C.POINTER(hot_stats_t)]
        lib.hot_forces_tol.argtypes = [C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        lib.hot_export_group_orders.argtypes = [C.c_void_p] * 3 + [C.c_int64, C.POINTER(C.c_int64)]
        lib.hot_step_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, hot_box, C.c_int, C.c_double,
                                      C.c_double, C.c_int, C.c_void_p, C.c_void_p]
        lib.hot_set_stream.argtypes = [C.c_void_p]
        lib.hot_set_params.argtypes = [C.c_int, C.c_int]
        lib.hot_set_list_arena.argtypes = [C.c_int64]
        lib.hot_set_softening.argtypes = [C.c_int]
        lib.hot_sort_keys_noalloc.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        lib.hot_noalloc_last_error.restype = C.c_char_p
        lib.hot_set_background.argtypes = [C.c_int]
        lib.hot_kick_drift.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_float, C.c_float, hot_box, C.c_int]
        lib.hot_far_coefficients.argtypes = [C.c_void_p]
        lib.hot_measure_fp32.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        lib.hot_measure_fp32_operands.argtypes = [C.POINTER(C.c_double)]
        lib.hot_free.restype = None
        lib.hot_export_keys.argtypes = [C.c_void_p, C.c_void_p]
        lib.hot_export_cells.argtypes = [C.c_void_p] * 6 + [C.c_int64, C.POINTER(C.c_int64)]
        lib.hot_export_groups.argtypes = [C.c_void_p] * 6 + [C.c_int64, C.POINTER(C.c_int64)]
        lib.hot_export_lists.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64),
                                         C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
        lib.hot_export_moments.argtypes = [C.c_void_p] * 6 + [C.c_int64]
        lib.hot_lookup_keys.argtypes = [C.c_void_p, C.c_int64, C.c_void_p]
        _lib = lib
    return _lib


def _check(rc: int):
    if rc != 0:
        raise HotError(rc, _load().hot_last_error().decode())


def _box(lo, size) -> hot_box:
    b = hot_box()
    b.lo[0], b.lo[1], b.lo[2] = float(lo[0]), float(lo[1]), float(lo[2])
    b.size = float(size)
    return b


def hot_last_error() -> str:
    return _load().hot_last_error().decode()


def hot_set_stream(stream=None):
    """Pass a torch.cuda.Stream (or None for the legacy default stream)."""
    ptr = None if stream is None else C.c_void_p(stream.cuda_stream)
    _check(_load().hot_set_stream(ptr))


def hot_measure_fp32():
    """(scalar FFMA, packed FFMA2) TFLOP/s of a register-only FMA chain on the current device."""
    a, b = C.c_double(), C.c_double()
    _check(_load().hot_measure_fp32(C.byref(a), C.byref(b)))
    return a.value, b.value


def hot_measure_fp32_operands():
    """TFLOP/s of FMAs reading (packed, 2 registers), (packed, 3 registers), (scalar, 3 registers) per instruction."""
    out = (C.c_double * 3)()
    _check(_load().hot_measure_fp32_operands(out))
    return tuple(out)


def hot_far_coefficients() -> np.ndarray:
    """The 165 far-field Taylor coefficients (host computation, no GPU needed)."""
    out = np.empty(165, dtype=np.float64)
    _check(_load().hot_far_coefficients(out.ctypes.data_as(C.c_void_p)))
    return out


def hot_set_list_arena(max_bytes: int = 0):
    """Cap the interaction-list arena (0 = default); smaller caps make hot_forces work in chunks of groups."""
    _check(_load().hot_set_list_arena(int(max_bytes)))


def hot_set_params(nleaf: int = 16, ncrit: int = 256):
    _check(_load().hot_set_params(int(nleaf), int(ncrit)))


def hot_set_softening(kind: int = 0):
    """0: Plummer (default); 1: cubic spline with h = 2.8 eps."""
    _check(_load().hot_set_softening(int(kind)))


def hot_set_background(on: bool = False):
    """Per-cell background subtraction in periodic boxes for the following hot_forces calls."""
    _check(_load().hot_set_background(int(bool(on))))


def hot_kick_drift(pos, vel, acc, dt_kick, dt_drift, lo, size, periodic=False):
    """In place on contiguous CUDA float32 [n,3] tensors: vel += acc * dt_kick; pos += vel * dt_drift (periodic wrap)."""
    import torch

    for t_, name in ((pos, "pos"), (vel, "vel"), (acc, "acc")):
        if not (t_.is_cuda and t_.dtype == torch.float32 and t_.is_contiguous() and t_.dim() == 2 and t_.shape[1] == 3
                and t_.shape[0] == pos.shape[0] and t_.device.index == torch.cuda.current_device()):
            raise TypeError(f"hot_kick_drift wants {name} as a contiguous CUDA float32 [n,3] tensor on the current device")
    _check(_load().hot_kick_drift(pos.data_ptr(), vel.data_ptr(), acc.data_ptr(), pos.shape[0], float(dt_kick), float(dt_drift),
                                  _box(lo, size), int(bool(periodic))))


def hot_noalloc_last_error() -> str:
    return _load().hot_noalloc_last_error().decode()


def hot_sort_keys_noalloc(key, perm, key_work, idx_work, stream=None):
    """Allocation-free stable sort (n <= 2^22): key [n] 8-byte integers (sorted in place), perm [n] 4-byte integers
    (out), two work tensors of the same kinds; contiguous CUDA tensors on the current device.  Enqueues on `stream`
    (torch.cuda.Stream; default: torch's current stream) and returns without synchronising."""
    import torch

    n = key.numel()
    for t_, size, name in ((key, 8, "key"), (key_work, 8, "key_work"), (perm, 4, "perm"), (idx_work, 4, "idx_work")):
        if not (t_.is_cuda and t_.is_contiguous() and t_.element_size() == size and not t_.dtype.is_floating_point
                and t_.numel() == n and t_.device.index == torch.cuda.current_device()):
            raise TypeError(f"hot_sort_keys_noalloc wants {name} as a contiguous CUDA tensor of {n} {size}-byte integers on the current device")
    s = torch.cuda.current_stream() if stream is None else stream
    rc = _load().hot_sort_keys_noalloc(key.data_ptr(), perm.data_ptr(), key_work.data_ptr(), idx_work.data_ptr(), n, C.c_void_p(s.cuda_stream))
    if rc != 0:
        raise HotError(rc, hot_noalloc_last_error())


def hot_free():
    _load().hot_free()


def hot_build(pos, mass, lo, size, periodic=False):
    """pos [n,3] / mass [n]: contiguous CUDA float32 tensors on the current device (borrowed for the call)."""
    import torch

    if not (pos.is_cuda and mass.is_cuda and pos.dtype == torch.float32 and mass.dtype == torch.float32):
        raise TypeError("hot_build wants CUDA float32 tensors")
    if not (pos.is_contiguous() and mass.is_contiguous() and pos.dim() == 2 and pos.shape[1] == 3
            and mass.numel() == pos.shape[0]):
        raise TypeError("hot_build wants contiguous pos [n,3] and mass [n]")
    cur = torch.cuda.current_device()
    if pos.device.index != cur or mass.device.index != cur:
        raise TypeError(f"hot_build wants tensors on the current CUDA device (cuda:{cur}): the library works there")
    _check(_load().hot_build(pos.data_ptr(), mass.data_ptr(), pos.shape[0], _box(lo, size), int(bool(periodic))))


def hot_forces_tol(tol, eps, acc=None, pot=None, want_pot=True):
    """hot_forces with the error-bound criterion (absolute acceleration tolerance per interaction, order chosen per
    interaction).  Returns (acc [n,3], pot [n] or None)."""
    import torch

    n = int(hot_stats()["n"])
    dev = torch.device("cuda", torch.cuda.current_device())
    if acc is None:
        acc = torch.empty((max(n, 1), 3), dtype=torch.float32, device=dev)
    elif n:
        _check_out(acc, (n, 3), "acc")
    if pot is None and want_pot:
        pot = torch.empty(max(n, 1), dtype=torch.float32, device=dev)
    elif pot is not None and n:
        _check_out(pot, (n,), "pot")
    _check(_load().hot_forces_tol(float(tol), float(eps), acc.data_ptr(), pot.data_ptr() if pot is not None else None))
    return acc, pot


def hot_export_group_orders() -> dict:
    ng = hot_stats()["n_groups"]
    out = dict(mono=np.empty(ng, np.uint64), quad=np.empty(ng, np.uint64), hexa=np.empty(ng, np.uint64))
    got = C.c_int64()
    _check(_load().hot_export_group_orders(out["mono"].ctypes.data, out["quad"].ctypes.data, out["hexa"].ctypes.data, ng, C.byref(got)))
    return out


def _check_out(t, shape, name):
    import torch

    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
            and tuple(t.shape) == shape and t.device.index == torch.cuda.current_device()):
        raise TypeError(f"hot_forces wants {name} as a contiguous CUDA float32 tensor of shape {shape} on the current device")


def hot_forces(theta, eps, order, acc=None, pot=None, want_pot=True):
    """Returns (acc [n,3], pot [n] or None) as CUDA float32 tensors in the caller's particle order.
    n is the size of the library's current build (hot_stats), whichever call made it."""
    import torch

    n = int(hot_stats()["n"])  # 0 before a build: the library then reports HOT_EORDER
    dev = torch.device("cuda", torch.cuda.current_device())
    if acc is None:
        acc = torch.empty((max(n, 1), 3), dtype=torch.float32, device=dev)
    elif n:
        _check_out(acc, (n, 3), "acc")
    if pot is None and want_pot:
        pot = torch.empty(max(n, 1), dtype=torch.float32, device=dev)
    elif pot is not None and n:
        _check_out(pot, (n,), "pot")
    _check(_load().hot_forces(float(theta), float(eps), int(order), acc.data_ptr(),
                              pot.data_ptr() if pot is not None else None))
    return acc, pot


def hot_stats() -> dict:
    s = hot_stats_t()
    _check(_load().hot_stats(C.byref(s)))
    return {k: getattr(s, k) for k, _ in hot_stats_t._fields_}


def hot_step_host(pos, mass, lo, size, periodic, theta, eps, order, acc=None, pot=None):
    """HOST numpy float32 arrays in, HOST arrays out; copies are inside the call."""
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    mass = np.ascontiguousarray(mass, dtype=np.float32)
    n = pos.shape[0]
    if acc is None:
        acc = np.empty((n, 3), np.float32)
    if pot is None:
        pot = np.empty(n, np.float32)
    _check(_load().hot_step_host(pos.ctypes.data, mass.ctypes.data, n, _box(lo, size), int(bool(periodic)),
                                 float(theta), float(eps), int(order), acc.ctypes.data, pot.ctypes.data))
    return acc, pot


def hot_export_keys():
    n = hot_stats()["n"]
    key = np.empty(n, np.uint64)
    perm = np.empty(n, np.uint32)
    _check(_load().hot_export_keys(key.ctypes.data, perm.ctypes.data))
    return key, perm


def hot_export_cells() -> dict:
    nc = hot_stats()["n_cells"]
    out = dict(key=np.empty(nc, np.uint64), first=np.empty(nc, np.uint32), count=np.empty(nc, np.uint32),
               mask=np.empty(nc, np.uint8), child=np.empty(nc, np.int32), parent=np.empty(nc, np.int32))
    got = C.c_int64()
    _check(_load().hot_export_cells(out["key"].ctypes.data, out["first"].ctypes.data, out["count"].ctypes.data,
                                    out["mask"].ctypes.data, out["child"].ctypes.data, out["parent"].ctypes.data,
                                    nc, C.byref(got)))
    return out


def hot_export_groups() -> dict:
    ng = hot_stats()["n_groups"]
    out = dict(cell=np.empty(ng, np.int32), key=np.empty(ng, np.uint64), first=np.empty(ng, np.uint32),
               count=np.empty(ng, np.uint32), lpc=np.empty(ng, np.uint64), lpp=np.empty(ng, np.uint64))
    got = C.c_int64()
    _check(_load().hot_export_groups(out["cell"].ctypes.data, out["key"].ctypes.data, out["first"].ctypes.data,
                                     out["count"].ctypes.data, out["lpc"].ctypes.data, out["lpp"].ctypes.data,
                                     ng, C.byref(got)))
    return out


def hot_export_lists(group: int) -> dict:
    """Interaction lists of one sink group from the last hot_forces: accepted cells (+ image ids) and listed
    bodies (sorted positions, + image ids; the group's own bodies are not listed)."""
    npc, npp = C.c_int64(), C.c_int64()
    lib = _load()
    _check(lib.hot_export_lists(int(group), None, None, 0, C.byref(npc), None, None, 0, C.byref(npp)))
    out = dict(pc_cell=np.empty(npc.value, np.int32), pc_img=np.empty(npc.value, np.uint8),
               pp_body=np.empty(npp.value, np.uint32), pp_img=np.empty(npp.value, np.uint8))
    _check(lib.hot_export_lists(int(group), out["pc_cell"].ctypes.data, out["pc_img"].ctypes.data, npc.value, C.byref(npc),
                                out["pp_body"].ctypes.data, out["pp_img"].ctypes.data, npp.value, C.byref(npp)))
    return out


def hot_export_moments(order: int) -> dict:
    nc = hot_stats()["n_cells"]
    out = dict(com=np.empty((nc, 3), np.float64), m0=np.empty(nc, np.float32), bmax=np.empty(nc, np.float32))
    m2 = m3 = m4 = None
    if order >= 2:
        out["m2"] = m2 = np.empty((nc, 6), np.float32)
    if order >= 4:
        out["m3"] = m3 = np.empty((nc, 10), np.float32)
        out["m4"] = m4 = np.empty((nc, 15), np.float32)
    p = lambda a: a.ctypes.data if a is not None else None
    _check(_load().hot_export_moments(p(out["com"]), p(out["m0"]), p(out["bmax"]), p(m2), p(m3), p(m4), nc))
    return out


def hot_lookup_keys(keys) -> np.ndarray:
    keys = np.ascontiguousarray(keys, dtype=np.uint64)
    idx = np.empty(keys.shape[0], np.int32)
    _check(_load().hot_lookup_keys(keys.ctypes.data, keys.shape[0], idx.ctypes.data))
    return idx
