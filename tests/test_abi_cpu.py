"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
that include/hot.h declares; the binding's struct mirrors the header; the oracle builds."""
import ctypes
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "hot.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hot_[a-z_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_1310_4502_b200 import build

    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = _declared_symbols()
    assert {"hot_build", "hot_forces", "hot_stats"} <= set(names) and len(names) >= 12
    for name in names:
        assert hasattr(lib, name), name


def test_binding_names_match_header():
    import paper_1310_4502_b200 as hot

    for name in _declared_symbols():
        assert hasattr(hot, name), name


def test_stats_struct_matches_header_layout():
    from paper_1310_4502_b200 import binding

    src = open(os.path.join(ROOT, "include", "hot.h")).read()
    body = src[:src.index("} hot_stats_t;")]
    body = body[body.rindex("typedef struct {") + len("typedef struct {"):]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        typ, names = decl.split(None, 1)
        fields += [(n.strip(), typ) for n in names.split(",")]
    want = {"int64_t": ctypes.c_int64, "int32_t": ctypes.c_int32, "uint64_t": ctypes.c_uint64, "float": ctypes.c_float}
    got = binding.hot_stats_t._fields_
    assert [f[0] for f in got] == [f[0] for f in fields]
    assert [f[1] for f in got] == [want[f[1]] for f in fields]


def test_calls_without_build_report_order_error_not_crash():
    # these entry points touch no device state before checking the call order
    from paper_1310_4502_b200 import binding

    lib = binding._load()
    assert lib.hot_set_params(16, 64) == 0
    assert lib.hot_set_params(0, 64) == -1 and lib.hot_set_params(64, 16) == -1
    assert b"nleaf" in lib.hot_last_error()
    assert lib.hot_forces(0.5, 1e-3, 2, None, None) == -5  # HOT_EORDER
    assert lib.hot_export_keys(None, None) == -5
    assert lib.hot_stats(None) == -1


def test_oracle_builds_and_is_not_imported_by_the_product():
    from oracle import oracle as O

    assert os.path.exists(O.build())
    pkg = os.path.join(ROOT, "paper_1310_4502_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".inc")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("the oracle", "").replace("The oracle", "") or f == "workloads.py" or "never seen by the oracle" in txt, (dirpath, f)


def test_workloads_are_seeded_and_inside_their_boxes():
    from paper_1310_4502_b200 import workloads as W

    for cfg, scale in ((0, 10), (1, 10), (2, 10), (3, 8), (4, 8)):
        a, b = W.config(cfg, scale), W.config(cfg, scale)
        assert (a.pos == b.pos).all() and a.pos.dtype == np.float32 and a.pos.flags["C_CONTIGUOUS"]
        lo = np.array(a.lo, np.float32)
        t = (a.pos - lo) * np.float32(1.0 / a.size)
        assert (t >= 0).all() and (t < 1).all()
        assert abs(a.mass.astype(np.float64).sum() - 1.0) < 1e-6


def test_far_field_table_host_only():
    """hot_far_coefficients needs no GPU.  The library derives the table from four axis Taylor
    coefficients and the cubic harmonics; the oracle sums all 35 tensor derivatives (SURVEY C-9).
    They share no code, so agreement pins both; C0 and the background term are closed forms."""
    import numpy as np

    from oracle import oracle as O
    from paper_1310_4502_b200 import binding

    c = binding.hot_far_coefficients()
    assert c.shape == (165,)
    assert abs(c[0] - (-60.02450803)) < 1e-7                      # psi_sm(0), SURVEY 8(a) P3
    assert np.allclose(c[[4, 7, 9]], 2.0 * np.pi / 3.0, rtol=1e-14)  # the uniform background
    T = O.Tree(np.array([[0.5, 0.5, 0.5]], np.float32), np.array([1.0], np.float32), (0.0, 0.0, 0.0), 1.0, periodic=True)
    o = T.far_table()
    assert np.abs(c - o).max() < 1e-11
    # laplace(psi_sm) = 4 pi: every degree >= 4 part is harmonic
    k, idx = 0, {}
    for d in range(9):
        for a in range(d, -1, -1):
            for b in range(d - a, -1, -1):
                idx[(a, b, d - a - b)] = k
                k += 1
    for (a, b, cc), k in idx.items():
        if a + b + cc in (2, 4, 6):  # coefficient of x^a y^b z^c in the Laplacian of the degree+2 part
            lap = ((a + 2) * (a + 1) * c[idx[(a + 2, b, cc)]] + (b + 2) * (b + 1) * c[idx[(a, b + 2, cc)]]
                   + (cc + 2) * (cc + 1) * c[idx[(a, b, cc + 2)]])
            assert abs(lap) < 1e-12, (a, b, cc, lap)
