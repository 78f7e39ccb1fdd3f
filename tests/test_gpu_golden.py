"""Full-run parity on BASELINE.json configs[3] and configs[4] against stored oracle results (`-m gpu`).

The fp64 oracle needs 11 minutes (config 3) and more than an hour per source (config 4) for the whole multigroup solve to
the 1e-5 tolerance, so `tests/golden/make_goldens.py` (oracle/ + workloads/ only) ran it once and stored, per group: the
sweep counts K[g], max phi_0, a stride sample of all moments and of phi_u, and the 2048 smallest in-mask cells (where the
relative error of an fp32 path peaks) plus the 256 largest.  Here the CUDA path solves the SAME whole problem through the
C ABI in the launch configuration bench.py times — config 4: all 8 sources, 2 chunks of 4 — replaying K (reading R10), and
every stored cell is compared at the 1e-4 gate inside the 1e-6 mask.  A second solve runs the device-side convergence test
and must stop within one sweep of the oracle in every group.
"""
import os

import numpy as np
import pytest

from workloads import make_config
from tests.parity_util import run_gpu

pytestmark = pytest.mark.gpu
TOL = 1e-4
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1910_11335_b200 import build
    build.build()
    import paper_1910_11335_b200 as p
    p.load_library()
    return p


def _golden(cfg, source, closure=1):
    path = os.path.join(GOLDEN, "cfg%d_src%d_closure%d.npz" % (cfg, source, closure))
    assert os.path.exists(path), "%s is missing: run tests/golden/make_goldens.py" % path
    return np.load(path)


def _compare(p, q, gold, wl, report):
    """Scalar flux of problem q against every stored cell; returns the worst relative error inside the mask.
    report rows: (problem, group, worst, cells compared, cells above the gate)."""
    worst = 0.0
    G = wl.G
    for g in range(G):
        got = p.get_flux_moments(q, g, 0)[0].reshape(-1).astype(np.float64)
        floor = 1e-6 * float(gold["phi0_max"][g])
        w_g, n_g, bad_g = 0.0, 0, 0
        for idx, val in ((gold["small_idx"][g], gold["small_phi0"][g]), (gold["large_idx"][g], gold["large_phi0"][g]),
                         (gold["stride_idx"], gold["stride_phi"][g, 0])):
            val = val.astype(np.float64)
            m = val > floor
            if m.any():
                rel = np.abs(got[idx[m]] - val[m]) / val[m]
                w_g = max(w_g, float(rel.max()))
                n_g += int(m.sum())
                bad_g += int((rel > TOL).sum())
        assert n_g > 2000, (g, n_g)
        report.append((q, g, w_g, n_g, bad_g))
        worst = max(worst, w_g)
    return worst


def test_config3_full_solve_against_golden(pkg, capsys):
    """Config 3 (128x128x64, S16 = 288 directions, P3, 19 groups, cone beam), the whole solve with the downscatter chain."""
    gold = _golden(3, 0)
    wl = make_config(3)
    K = gold["iters"][None, :]
    assert K.shape == (1, wl.G) and K.min() >= 7
    p, info = run_gpu(wl, closure=1, fixed_iters=K)
    assert (info["iters"] == K).all()
    report = []
    worst = _compare(p, 0, gold, wl, report)
    # all 16 moments and the uncollided flux on the stride sample
    sidx = gold["stride_idx"]
    for g in (0, 9, 18):
        mom = p.get_flux_moments(0, g, 3).reshape(16, -1)[:, sidx]
        scale = float(gold["phi0_max"][g])
        assert np.abs(mom - gold["stride_phi"][g]).max() / scale < 2e-5, g
        pu = p.get_uncollided_flux(0, g).reshape(-1)[sidx].astype(np.float64)
        ref_u = gold["stride_phi_u"][g].astype(np.float64)
        lit = ref_u > 0
        assert lit.any() and np.array_equal(pu > 0, lit)
        assert (np.abs(pu[lit] - ref_u[lit]) / ref_u[lit]).max() < 1e-5, g
    # per-sweep particle balance of the last sweep, every group
    np.testing.assert_allclose(info["balance"][0], gold["balance"], rtol=5e-5)
    p.close()
    with capsys.disabled():
        print("\n  cfg3 full solve: worst rel err %.3e over %d stored cells; per group max %s" % (
            worst, sum(r[3] for r in report), " ".join("%.1e" % r[2] for r in report)))
    assert worst < TOL, report
    # device-side convergence test: within one sweep of the oracle in every group
    p2, info2 = run_gpu(wl, closure=1)
    assert info2["status"] == 0 and np.abs(info2["iters"].astype(int) - K).max() <= 1, (info2["iters"], K)
    p2.close()


def test_config4_full_solve_against_goldens(pkg, capsys):
    """Config 4 (256x256x128 GRF phantom, 47 groups, P3, S8) as bench.py runs it: 8 cone-beam sources batched in 2 chunks of
    4.  Every source whose golden is committed (0, 3, 5 with all moments; the others lean: scalar flux) replays the oracle's sweep
    counts through all 47 groups and is compared on every stored cell; sources without a golden run the device-side convergence
    test in the same solve."""
    golds = {s: _golden(4, s) for s in (0, 3, 5)}              # required: tests/golden/make_goldens.py writes them
    for s in range(8):                                         # the other sources where their (lean) golden is committed
        if s not in golds and os.path.exists(os.path.join(GOLDEN, "cfg4_src%d_closure1.npz" % s)):
            golds[s] = _golden(4, s)
    wl = make_config(4)
    K = np.zeros((8, wl.G), dtype=np.int32)                   # 0 = stop by the tolerance
    for s, g in golds.items():
        K[s] = g["iters"]
    p, info = run_gpu(wl, closure=1, fixed_iters=K, source_chunk=4)
    assert info["n_chunks"] == 2 and tuple(info["brick"]) == (20, 8, 4)
    report = []
    worst = 0.0
    for s, g in golds.items():
        assert (info["iters"][s] == g["iters"]).all()
        worst = max(worst, _compare(p, s, g, wl, report))
        np.testing.assert_allclose(info["balance"][s], g["balance"], rtol=1e-4)
        sidx = g["stride_idx"]
        for grp in (0, 23, 46):
            pu = p.get_uncollided_flux(s, grp).reshape(-1)[sidx].astype(np.float64)
            ref_u = g["stride_phi_u"][grp].astype(np.float64)
            lit = ref_u > 0
            assert np.array_equal(pu > 0, lit) and (np.abs(pu[lit] - ref_u[lit]) / ref_u[lit]).max() < 1e-5, (s, grp)
    # the five sources that ran to the tolerance needed about as many sweeps, and converged
    others = [s for s in range(8) if s not in golds]
    if others:
        assert (info["residual"][others] < wl.tol).all()
        assert np.abs(info["iters"][others].astype(int).mean(0) - np.mean([g["iters"] for g in golds.values()], 0)).max() <= 2.0
    with capsys.disabled():
        print("\n  cfg4 sources %s full solve (8 sources, 2 chunks of 4): worst rel err %.3e over %d stored cells" % (
            sorted(golds), worst, sum(r[3] for r in report)))
        for s in golds:
            print("   source %d per group max: %s" % (s, " ".join("%.1e" % r[2] for r in report if r[0] == s)))
    assert worst < TOL, [r for r in report if r[2] >= TOL]
    # same solve with the device-side test for every source: counts within one sweep of the oracle
    info2 = p.solve(tol=wl.tol, max_iters=wl.max_iters, closure=1, source_chunk=4)
    for s, g in golds.items():
        assert np.abs(info2["iters"][s].astype(int) - g["iters"]).max() <= 1, (s, info2["iters"][s], g["iters"])
    p.close()


def test_config4_closure0_literal_diamond_difference_against_golden(pkg, capsys):
    """SURVEY row f2 on config 4: the closure the paper names (pure diamond difference, no fix-up), source 0 through
    all 47 groups, against the oracle run with the same closure.  Pure DD produces negative fluxes in the optically thick low
    groups; the test prints, per group, the worst relative error inside the mask and the count of stored cells above 1e-4, and
    asserts the finding recorded in DESIGN.md section 6."""
    gold = _golden(4, 0, closure=0)
    wl = make_config(4, n_sources=1)
    K = gold["iters"][None, :]
    p, info = run_gpu(wl, closure=0, fixed_iters=K)
    report = []
    worst = _compare(p, 0, gold, wl, report)
    p.close()
    with capsys.disabled():
        print("\n  cfg4 source 0, closure 0: worst rel err %.3e; cells above 1e-4: %d of %d stored; oracle cells with phi0 < 0: %d" % (
            worst, sum(r[4] for r in report), sum(r[3] for r in report), int(gold["n_negative"].sum())))
        print("   per group max: %s" % " ".join("%.1e" % r[2] for r in report))
        print("   per group cells > 1e-4: %s" % " ".join("%d" % r[4] for r in report))
    high = [r for r in report if r[1] < 37]                       # groups 0-36 (above ~38 keV): measured <= 2.2e-5
    assert all(r[2] < TOL for r in high), [r for r in high if r[2] >= TOL]
    assert worst < 1e-3 and sum(r[4] for r in report) <= 50, report


def test_config3_closure0_literal_diamond_difference_against_golden(pkg, capsys):
    """SURVEY row f2 on config 3: pure diamond difference, whole 19-group solve, against the oracle run with the
    same closure; per-group worst relative error and count of stored cells above 1e-4 are printed."""
    gold = _golden(3, 0, closure=0)
    wl = make_config(3)
    p, info = run_gpu(wl, closure=0, fixed_iters=gold["iters"][None, :])
    report = []
    worst = _compare(p, 0, gold, wl, report)
    p.close()
    with capsys.disabled():
        print("\n  cfg3 closure 0: worst rel err %.3e; cells above 1e-4: %d of %d stored; oracle cells with phi0 < 0: %d" % (
            worst, sum(r[4] for r in report), sum(r[3] for r in report), int(gold["n_negative"].sum())))
        print("   per group max: %s" % " ".join("%.1e" % r[2] for r in report))
    assert all(r[2] < TOL for r in report if r[1] < 16), report     # groups 0-15 (above 30 keV) hold the gate
    assert worst < 1e-3 and sum(r[4] for r in report) <= 50, report
