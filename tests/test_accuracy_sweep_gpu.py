"""Error-versus-cost at BASELINE.json configs[2] (N = 2^24 clustered mix): the opening-angle sweep of the config
(theta 0.4 / 0.6 / 0.8 x orders 2, 4) beside the error-bound criterion of hot_forces_tol (PAPER.md:86, 238, 303:
"relaxing the error parameter by a factor of 10 ... reduces the operation count").  Errors are rms acceleration errors
against the oracle's direct sum on 1024 seeded sinks x all 2^24 sources.  Run with -s to see the table
(profiles/r02_c2_sweep.md is its output)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_1310_4502_b200 import workloads as W

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def test_error_vs_cost_theta_and_tolerance(hot):
    import torch

    w = W.config(2)
    hot.hot_set_params(16, 256)
    pos = torch.from_numpy(w.pos).cuda(); mass = torch.from_numpy(w.mass).cuda()
    sinks = np.sort(np.random.default_rng(24).choice(w.n, 1024, replace=False))
    ad, _ = O.direct(w.pos, w.mass, w.eps, sinks=sinks)
    arms = float(np.sqrt((ad ** 2).sum(1).mean()))
    rows = []

    def run(label, fn):
        best = 1e30
        for _ in range(2):
            hot.hot_build(pos, mass, w.lo, w.size, False)
            acc, _ = fn()
            st = hot.hot_stats()
            best = min(best, st["ms_build_total"] + st["ms_forces_total"])
        a = acc[torch.from_numpy(sinks).cuda()].cpu().numpy().astype(np.float64)
        err = float(np.sqrt(((a - ad) ** 2).sum() / (ad ** 2).sum()))
        rows.append((label, best, st["ms_walk"], st["ms_eval"], st["pp_interactions"] / w.n, st["pc_monopole"] / w.n,
                     st["pc_quadrupole"] / w.n, st["pc_hexadecapole"] / w.n, err))
        return err, best

    e_theta = {}
    for order in (2, 4):
        for theta in (0.4, 0.6, 0.8):
            e_theta[(order, theta)] = run(f"theta {theta} order {order}", lambda: hot.hot_forces(theta, w.eps, order, want_pot=False))
    e_tol = {}
    for rtol in (1e-2, 1e-3, 1e-4, 1e-5):
        e_tol[rtol] = run(f"tol {rtol:g} x a_rms", lambda: hot.hot_forces_tol(rtol * arms, w.eps, want_pot=False))
    print("\n| criterion | step ms | walk ms | eval ms | P-P / body | mono / body | quad / body | hexa / body | rms error |")
    print("|---|---:|---:|---:|---:|---:|---:|---:|---:|")
    for r in rows:
        print(f"| {r[0]} | {r[1]:.1f} | {r[2]:.1f} | {r[3]:.1f} | {r[4]:.0f} | {r[5]:.0f} | {r[6]:.0f} | {r[7]:.0f} | {r[8]:.2e} |")
    print(f"(a_rms = {arms:.4g}; N = {w.n}; NLEAF 16, NCRIT 256)")
    # BASELINE.json: the error falls with theta at fixed order and with order at fixed theta
    for order in (2, 4):
        assert e_theta[(order, 0.4)][0] < e_theta[(order, 0.6)][0] < e_theta[(order, 0.8)][0]
    for theta in (0.4, 0.6, 0.8):
        assert e_theta[(4, theta)][0] < e_theta[(2, theta)][0]
    # the error-bound criterion: error and cost are monotone in the tolerance, the rms error stays below it
    tols = sorted(e_tol)
    for a, b in zip(tols[:-1], tols[1:]):
        assert e_tol[a][0] < e_tol[b][0] and e_tol[a][1] > e_tol[b][1]
    for rtol in tols:
        assert e_tol[rtol][0] <= 10 * rtol
