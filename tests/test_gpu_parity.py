"""Parity of the CUDA path (through the C ABI) against the fp64 oracle — run with `-m gpu` on a B200.

Bars (BASELINE.json north_star): integer schedules bit-exact; fp32 scalar flux within 1e-4 max
relative error wherever phi > 1e-6 max(phi), per (problem, group), after the oracle's own sweep
counts are replayed on the GPU (reading R10).  Closure per reading R2: configs 0-1 gated with both
closures, configs 2-4 with closure 1.
"""
import dataclasses

import numpy as np
import pytest

from workloads import make_config, single_sweep_case, paper_shaped
from tests.parity_util import compare_workload, run_gpu, tiny_p3_case, masked_rel_err

pytestmark = pytest.mark.gpu
TOL = 1e-4      # north_star: fp32 scalar flux within 1e-4 max relative error inside the mask


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1910_11335_b200 import build
    build.build()
    import paper_1910_11335_b200 as p
    p.load_library()          # raises if the extension is missing: no fallback
    return p


# ---- a3: schedules the kernels consume, bit-exact ---------------------------------------------
@pytest.mark.parametrize("wl_fn,brick", [(lambda: make_config(0), None), (lambda: tiny_p3_case(), None),
                                         (lambda: tiny_p3_case(), (4, 3, 5)), (lambda: make_config(2), None)])
def test_schedule_bit_exact(pkg, orc, wl_fn, brick):
    wl = wl_fn()
    p = pkg.problem_from_workload(wl)
    for level in (0, 1, 2):
        for octant in range(8):
            dims, off, cells = p.debug_schedule(octant, level, brick=brick)
            off_o, cells_o = orc.schedule(dims[0], dims[1], dims[2], octant)
            assert np.array_equal(off, off_o) and np.array_equal(cells, cells_o), (level, octant)
    d0, _, _ = p.debug_schedule(0, 0)
    assert d0 == (wl.nx, wl.ny, wl.nz)
    d1, _, _ = p.debug_schedule(0, 1, brick=brick)
    d2, _, _ = p.debug_schedule(0, 2, brick=brick)
    assert all(d1[a] == -(-d0[a] // d2[a]) for a in range(3))
    p.close()


@pytest.mark.parametrize("brick", [(16, 8, 4), (20, 8, 4), (8, 4, 8), (4, 3, 5), (12, 32, 1), (12, 1, 32), (4, 1, 1), (64, 8, 4)])
def test_device_wavefront_planes_bit_exact(pkg, orc, brick):
    """Level 2 on the device: the step at which the sweep kernel itself updates each cell of a brick
    equals the cell's sub-sweep index of Eq. (8) in the oracle's schedule, for all 8 octants, and every
    plane holds exactly P(S) cells (Eq. 9).  The same launch bounds-checks every shared-memory address of the
    wavefront loop (idle lanes load from their running addresses): the call fails if one leaves the CTA's allocation."""
    p = pkg.problem_from_workload(make_config(0))
    bx, by, bz = brick
    for octant in range(8):
        steps = p.debug_device_brick_steps(brick, octant).reshape(-1)
        off, cells = orc.schedule(bx, by, bz, octant)
        want = np.empty(bx * by * bz, dtype=np.int32)
        for S in range(len(off) - 1):
            want[cells[off[S]:off[S + 1]]] = S
        assert np.array_equal(steps, want), (brick, octant)
        assert np.array_equal(np.bincount(steps, minlength=len(off) - 1),
                              [orc.wavefront_size(bx, by, bz, S) for S in range(len(off) - 1)])
    p.close()


def test_tables_match_oracle(pkg, orc):
    wl = make_config(1)
    p = pkg.problem_from_workload(wl)
    om, w = p.get_quadrature()
    om_o, w_o = orc.level_symmetric(wl.sn)
    M, D = p.debug_tables(3)
    Mo, Do = orc.projection_tables(3, om, w)
    np.testing.assert_allclose(M, Mo, atol=1e-14)
    np.testing.assert_allclose(D, Do.T, atol=1e-14)
    np.testing.assert_allclose(np.sort(w), np.sort(w_o), atol=1e-12)
    p.close()


# ---- config 0 and small ragged cases: every kernel variant ------------------------------------
@pytest.mark.parametrize("closure", [0, 1])
@pytest.mark.parametrize("mode,det", [(0, 0), (0, 1), (1, 0)])
def test_config0(pkg, orc, closure, mode, det):
    wl = make_config(0)
    ref = orc.solve(wl, closure=closure)
    assert (ref["iters"] == 10).all()
    worst = compare_workload(wl, ref, closure=closure, sweep_mode=mode, deterministic=det)
    assert worst < TOL, worst


@pytest.mark.parametrize("closure", [0, 1])
@pytest.mark.parametrize("kind", [1, 2])
@pytest.mark.parametrize("brick", [None, (4, 3, 5), (8, 2, 2), (12, 8, 4), (16, 4, 8), (4, 1, 32)])
def test_ragged_p3(pkg, orc, closure, kind, brick):
    """12x10x9 mesh (px padding, clipped bricks in every axis), 4 materials, P3, S8, point / cone source."""
    wl = tiny_p3_case(kind=kind)
    ref = orc.solve(wl, closure=closure)
    worst = compare_workload(wl, ref, closure=closure, brick=brick)
    assert worst < TOL, worst


@pytest.mark.parametrize("L,sn", [(0, 4), (1, 4), (2, 6), (3, 12)])
def test_orders(pkg, orc, L, sn):
    wl = tiny_p3_case(nx=9, ny=7, nz=6, G=2, sn=sn, L=L, seed=11)
    ref = orc.solve(wl, closure=1)
    worst = compare_workload(wl, ref, closure=1)
    assert worst < TOL, worst
    worst = compare_workload(wl, ref, closure=1, sweep_mode=1)
    assert worst < TOL, worst


@pytest.mark.parametrize("sn,mtiles", [(4, 1), (8, 1), (12, 2), (16, 3)])
@pytest.mark.parametrize("brick", [None, (4, 8, 4), (8, 3, 5)])
def test_projection_paths_p3(pkg, orc, sn, mtiles, brick):
    """P3 projections on the tensor cores (mma TF32, 3-product split; 1, 2, 3 m-tiles of 16 directions)
    and in the fp32 FMA loops: both inside the gate, and within 2e-5 of each other on every moment."""
    wl = tiny_p3_case(nx=13, ny=9, nz=6, G=2, sn=sn, L=3, seed=5)
    ref = orc.solve(wl, closure=1)
    shape = (wl.nz, wl.ny, wl.nx)
    got = {}
    for proj in (2, 1):
        p, info = run_gpu(wl, closure=1, fixed_iters=ref["iters"], brick=brick, projection=proj)
        ncb = info["brick"][0] * info["brick"][1] * info["brick"][2]
        assert info["projection_mtiles"] == (mtiles if proj == 2 and ncb % 8 == 0 else 0)
        got[proj] = np.stack([p.get_flux_moments(0, g, 3) for g in range(wl.G)])
        p.close()
        for g in range(wl.G):
            e, _ = masked_rel_err(got[proj][g, 0], ref["phi"][0, g, 0].reshape(shape))
            assert e < TOL, (proj, g, e)
    scale = np.abs(got[1][:, 0]).max()
    assert np.abs(got[2] - got[1]).max() / scale < 2e-5


def test_degenerate_meshes(pkg, orc):
    for dims in [(1, 1, 1), (1, 7, 3), (5, 1, 1), (17, 2, 1)]:
        wl = tiny_p3_case(nx=dims[0], ny=dims[1], nz=dims[2], G=2, sn=4, L=1, seed=3)
        ref = orc.solve(wl, closure=0)
        worst = compare_workload(wl, ref, closure=0)
        assert worst < TOL, (dims, worst)


def test_higher_moments_and_balance(pkg, orc):
    wl = tiny_p3_case()
    ref = orc.solve(wl, closure=0)
    p, info = run_gpu(wl, closure=0, fixed_iters=ref["iters"])
    shape = (wl.nz, wl.ny, wl.nx)
    for g in range(wl.G):
        got = p.get_flux_moments(0, g, 3)
        want = ref["phi"][0, g].reshape((16,) + shape)
        scale = np.abs(want[0]).max()
        assert np.abs(got - want).max() / scale < 2e-6          # all 16 moments, relative to max phi_00
        # per-sweep particle balance of the last sweep: sum Q00 V = sum sigt phi0 V + leakage
        src, col, leak = info["balance"][0, g]
        assert abs(src - col - leak) < 2e-5 * src
        np.testing.assert_allclose(info["balance"][0, g], ref["balance"][0, g], rtol=2e-5)
    p.close()


def test_device_convergence_matches_oracle_counts(pkg, orc):
    """The device-side test (a6) stops within +-1 sweep of the fp64 oracle (reading R10)."""
    wl = make_config(1)
    ref = orc.solve(wl, closure=1)
    p, info = run_gpu(wl, closure=1)                        # tolerance mode, no replay
    assert info["status"] == 0
    assert np.abs(info["iters"].astype(int) - ref["iters"]).max() <= 1
    assert (info["residual"] < wl.tol).all()
    got = p.get_flux_moments(0, 18, 0)[0]
    e, _ = masked_rel_err(got, ref["phi"][0, 18, 0].reshape(got.shape))
    assert e < 5e-4                                            # counts may differ by one sweep
    p.close()


def test_max_iters_reports_not_converged(pkg):
    wl = make_config(1)
    p = pkg.problem_from_workload(wl)
    info = p.solve(tol=1e-12, max_iters=3, closure=1)
    assert info["status"] == pkg.NOT_CONVERGED and (info["iters"] == 3).all()
    p.close()


def test_batched_sources_and_chunking(pkg, orc):
    """Independent sources batched in one solve = each solved alone; result independent of source_chunk."""
    wl = tiny_p3_case(kind=2)
    s0 = wl.sources[0]
    import copy
    s1 = copy.deepcopy(s0); s1.pos = (0.3, 9.0, 0.2); s1.axis = (0.0, -1.0, 0.0)
    s2 = copy.deepcopy(s0); s2.kind = 1; s2.pos = (2.0, 1.0, 8.0)
    wl.sources = [s0, s1, s2]
    ref = orc.solve(wl, closure=1)
    assert ref["iters"].shape == (3, wl.G)
    for chunk in (0, 1, 2):
        worst = compare_workload(wl, ref, closure=1, source_chunk=chunk)
        assert worst < TOL, (chunk, worst)


def test_summed_sources_mode1(pkg, orc):
    wl = tiny_p3_case(kind=2)
    import copy
    s1 = copy.deepcopy(wl.sources[0]); s1.pos = (0.3, 9.0, 0.2); s1.axis = (0.0, -1.0, 0.0)
    wl.sources = [wl.sources[0], s1]
    wl.mode = 1
    ref = orc.solve(wl, closure=0)
    assert ref["iters"].shape == (1, wl.G)
    worst = compare_workload(wl, ref, closure=0)
    assert worst < TOL, worst


def test_fan_beam_source(pkg, orc):
    """Source kind 3 (fan beam, reading R18): uncollided and collided flux against the oracle, a fan
    tilted against every mesh axis so that all three direction cosines enter the mask; bad fans are refused."""
    from workloads import SourceSpec
    wl = tiny_p3_case(nx=13, ny=11, nz=9, G=2, sn=8, L=3, seed=6)
    fan = SourceSpec(kind=3, pos=(-11.0, 2.0, 1.5), axis=(1.0, -0.15, -0.1), up=(0.1, 0.3, 1.0), half_angle=np.deg2rad(24.0),
                     half_angle2=np.deg2rad(9.0), spectrum=np.full(wl.G, 1.0 / wl.G))
    w2 = dataclasses.replace(wl, sources=[fan])
    ref = orc.solve(w2, closure=1)
    lit = (ref["phi_u"][0, 0] > 0).mean()
    assert 0.05 < lit < 0.9                                      # a real mask: some cells lit, some dark
    worst = compare_workload(w2, ref, closure=1)
    assert worst < TOL, worst
    p = pkg.problem_from_workload(w2)
    for bad in (dataclasses.replace(fan, up=(2.0, -0.3, -0.2)), dataclasses.replace(fan, half_angle2=0.0),
                dataclasses.replace(fan, half_angle2=2.0)):
        with pytest.raises(pkg.DoctorsError):
            p.set_source([bad], 0)
    p.close()


def test_response_hook(pkg, orc):
    """doctors_get_response (PAPER.md:149 post-processing: fluence -> dose-like quantity) against the oracle's definition,
    independent problems and summed sources, with and without the uncollided part."""
    from workloads import SourceSpec
    wl = tiny_p3_case(nx=13, ny=9, nz=6, G=3, sn=8, L=3, seed=4)
    src2 = [wl.sources[0], SourceSpec(kind=2, pos=(0.4, -12.0, 0.3), axis=(0.0, 1.0, 0.0), half_angle=np.deg2rad(30.0),
                                      spectrum=np.full(wl.G, 1.0 / wl.G))]
    resp = np.array([0.25, 1.5, 3.0])
    shape = (wl.nz, wl.ny, wl.nx)
    for mode in (0, 1):
        w2 = dataclasses.replace(wl, sources=src2, mode=mode)
        ref = orc.solve(w2, closure=1)
        p, info = run_gpu(w2, closure=1, fixed_iters=ref["iters"])
        for q in range(ref["iters"].shape[0]):
            for unc in (True, False):
                got = p.get_response(q, resp, include_uncollided=unc)
                want = orc.response(ref, w2, q, resp, include_uncollided=unc).reshape(shape)
                e, _ = masked_rel_err(got, want)
                assert e < TOL, (mode, q, unc, e)
        with pytest.raises(ValueError):
            p.get_response(0, resp[:2])
        p.close()


def test_api_errors(pkg):
    wl = make_config(0)
    p = pkg.Problem()
    with pytest.raises(pkg.DoctorsError) as e:
        p.set_mesh_materials(wl.material, wl.density, (1.0, -1.0, 1.0), 1)
    assert e.value.status == pkg.INVALID_ARG
    p.set_mesh_materials(wl.material, wl.density, (1.0, 1.0, 1.0), 1)
    up = np.zeros((1, 1, 2, 2)); up[0, 0, 1, 0] = 0.1                      # upscatter entry
    with pytest.raises(pkg.DoctorsError):
        p.set_xs(np.full((1, 2), 0.2), up)
    p.set_xs(wl.sigma_t, wl.sigma_s)
    with pytest.raises(pkg.DoctorsError):
        p.set_quadrature(10)
    with pytest.raises(pkg.DoctorsError) as e:
        p.workspace_bytes()                                                # quadrature / source missing
    assert e.value.status == pkg.BAD_STATE
    p.set_quadrature(2)
    p.set_source(wl.sources, 0)
    L = pkg.load_library()
    import ctypes
    buf = np.zeros(wl.cells, dtype=np.float32)
    assert L.doctors_get_flux_moments(p._h, 0, 0, 0, ctypes.c_void_p(buf.ctypes.data), 0) == pkg.BAD_STATE
    p.solve(fixed_iters=2)
    with pytest.raises(pkg.DoctorsError):
        p.get_flux_moments(0, 1, 0)
    p.close()


# ---- the BASELINE configs -----------------------------------------------------------------------
@pytest.mark.parametrize("closure", [0, 1])
def test_config1_full(pkg, orc, closure):
    wl = make_config(1)
    ref = orc.solve(wl, closure=closure)
    worst = compare_workload(wl, ref, closure=closure)
    assert worst < TOL, worst


def test_config2_full_closure1(pkg, orc):
    wl = make_config(2)
    ref = orc.solve(wl, closure=1)
    worst = compare_workload(wl, ref, closure=1)
    assert worst < TOL, worst
    assert ref["phi"][:, :, 0].min() >= 0.0


def test_config3_full_mesh_sampled_groups(pkg, orc):
    """128x128x64, S16 (36 directions per octant), P3: full mesh and quadrature, groups {0, 18}, 3 sweeps."""
    wl = single_sweep_case(3, groups=(0, 18), fixed_iters=3)
    ref = orc.solve(wl, closure=1)
    worst = compare_workload(wl, ref, closure=1)
    assert worst < TOL, worst


def test_config4_full_mesh_one_source(pkg, orc):
    """256x256x128 GRF phantom in the bench's launch configuration: one source, the lowest-energy
    group pair, 2 sweeps each, against the oracle on every cell."""
    wl = single_sweep_case(4, groups=(45, 46), n_sources=1, fixed_iters=2)
    ref = orc.solve(wl, closure=1)
    worst = compare_workload(wl, ref, closure=1)
    assert worst < TOL, worst


def test_config4_batched_properties(pkg):
    """Properties that hold at any size, on the batched 4-source launch the bench times: exact
    per-sweep particle balance, non-negative flux under closure 1, and the rotational symmetry
    that maps source s to s+2 is NOT assumed (random phantom) — instead each problem of the
    batch must equal the same problem solved alone."""
    wl = single_sweep_case(4, groups=(0, 20, 46), n_sources=4, fixed_iters=3)
    p, info = run_gpu(wl, closure=1, fixed_iters=3)
    assert info["brick"][0] % 4 == 0 and info["brick"][1] * info["brick"][2] <= 32
    for q in range(4):
        for g in range(3):
            src, col, leak = info["balance"][q, g]
            assert src > 0 and abs(src - col - leak) < 5e-5 * src, (q, g, src, col, leak)
    batch = [p.get_flux_moments(q, 2, 0)[0].copy() for q in range(4)]
    assert min(b.min() for b in batch) >= 0.0
    p.close()
    import copy
    w1 = copy.copy(wl)
    w1.sources = [wl.sources[2]]
    p1, _ = run_gpu(w1, closure=1, fixed_iters=3)
    alone = p1.get_flux_moments(0, 2, 0)[0]
    e, n = masked_rel_err(batch[2], alone)
    # the two runs differ only in the order of the octants' fp32 reduce-adds (2.5e-5 at the dimmest of 1.5 M masked cells of the
    # lowest group after 3 sweeps; against the oracle the converged config-4 solve sits at 4e-6: tests/test_gpu_golden.py)
    assert n > 1000 and e < 5e-5, e
    p1.close()


def test_paper_shaped_ct_summed(pkg, orc):
    """Row f1: the paper's coarse CT workload shape (64x64x16, S6 P0, 16 cone beams summed), 6 groups."""
    wl = paper_shaped(ct=True, G=6)
    ref = orc.solve(wl, closure=1)
    worst = compare_workload(wl, ref, closure=1)
    assert worst < TOL, worst


# ---- round 2: source inside the object, bit-reproducibility, the literal closure on config 2 ----
def _inside_source(wl, pos):
    from workloads import SourceSpec
    return dataclasses.replace(wl, sources=[SourceSpec(kind=1, pos=pos, spectrum=np.full(wl.G, 1.0 / wl.G))])


@pytest.mark.parametrize("closure", [0, 1])
def test_source_inside_mesh_ragged(pkg, orc, closure):
    """"the source can be positioned anywhere in the geometry, including in the patient's organ".  Point source
    INSIDE the ragged 12x10x9 mesh, off-centre of its cell (the ray tracer's t0 = 0 path; the 1/R^2 field is steepest here and
    the source's own cell carries the largest first-collision source), uncollided and collided flux against the oracle."""
    wl = _inside_source(tiny_p3_case(), (0.9, -0.55, 0.4))
    ref = orc.solve(wl, closure=closure)
    lo = -0.5 * np.array([wl.nx * wl.dx, wl.ny * wl.dy, wl.nz * wl.dz])
    assert ((np.array(wl.sources[0].pos) > lo) & (np.array(wl.sources[0].pos) < -lo)).all()
    assert ref["phi_u"][0, 0].max() > 50.0 * np.median(ref["phi_u"][0, 0])     # the 1/R^2 peak is on the mesh
    worst = compare_workload(wl, ref, closure=closure)
    assert worst < TOL, worst


def test_source_inside_mesh_config1(pkg, orc):
    """Config 1's sphere phantom with the point source inside the water sphere (off-centre of its cell), all 19 groups."""
    wl = _inside_source(make_config(1), (1.1, -0.4, 0.3))
    ref = orc.solve(wl, closure=1)
    worst = compare_workload(wl, ref, closure=1)
    assert worst < TOL, worst


@pytest.mark.parametrize("wl_fn", [lambda: tiny_p3_case(kind=2), lambda: make_config(1)])
def test_deterministic_mode_is_bit_reproducible(pkg, wl_fn):
    """deterministic = 1 (octants one after another, one reduce-add per cell and octant): two solves of the same inputs
    give bit-identical flux moments, every group, every moment."""
    wl = wl_fn()
    runs = []
    for _ in range(2):
        p, info = run_gpu(wl, closure=1, fixed_iters=4, deterministic=1)
        runs.append(np.stack([p.get_flux_moments(0, g, wl.L) for g in range(wl.G)]))
        p.close()
    assert np.array_equal(runs[0], runs[1])
    assert np.abs(runs[0]).max() > 0.0


def test_config2_full_closure0_literal_diamond_difference(pkg, orc, capsys):
    """the closure the paper names (pure diamond difference, no fix-up) on config 2, whole solve.
    The face recurrence runs in fp64 (R17), storage stays fp32.  Reports, per group, the max relative error inside
    the mask and the count of cells above 1e-4 (reading R2 asked for the count where the literal closure misses the gate)."""
    wl = make_config(2)
    ref = orc.solve(wl, closure=0)
    p, info = run_gpu(wl, closure=0, fixed_iters=ref["iters"])
    shape = (wl.nz, wl.ny, wl.nx)
    worst, report = 0.0, []
    for g in range(wl.G):
        got = p.get_flux_moments(0, g, 0)[0].astype(np.float64)
        want = ref["phi"][0, g, 0].reshape(shape)
        m = want > 1e-6 * np.abs(want).max()
        rel = np.abs(got[m] - want[m]) / want[m]
        report.append((g, float(rel.max()), int((rel > TOL).sum()), int((want < 0).sum())))
        worst = max(worst, float(rel.max()))
    p.close()
    with capsys.disabled():
        for g, e, n, neg in report:
            print("  cfg2 closure 0  g %2d  max rel err %.3e  cells > 1e-4: %d  (oracle cells with phi0 < 0: %d)" % (g, e, n, neg))
    # Finding: with the fp64 face recurrence the literal closure holds the 1e-4 gate in groups 0-17 (worst
    # 3.3e-5); in the lowest group (10-16 keV, 2088 cells with negative oracle flux) ONE masked cell of 262144 sits at
    # 1.009e-4 — next to a sign change of phi_0, where fp32 storage of Q, psi and phi limits the sum of +- terms.
    assert all(e < TOL for g, e, n, neg in report if g < 18), report
    g18 = report[18]
    assert g18[1] < 2e-4 and g18[2] <= 3, report
    assert sum(neg for _, _, _, neg in report) > 1000          # the case is the hard one: pure DD goes negative here


def test_pl_exceeds_quadrature_flag(pkg):
    """doctors_solve_info.pl_exceeds_quadrature: P3 with S4 runs but is flagged, P3 with S8 is not."""
    for sn, want in ((4, 1), (8, 0)):
        wl = tiny_p3_case(nx=6, ny=5, nz=4, G=1, sn=sn, L=3, seed=2)
        p, info = run_gpu(wl, closure=1, fixed_iters=2)
        assert info["pl_exceeds_quadrature"] == want and info["timed_sweeps"] == 2
        p.close()


def test_second_solve_reuses_the_device_setup(pkg, orc):
    """The bricked mesh, tables, task list and tensor maps are built by the first solve and kept (plan cache): a second solve
    on unchanged inputs gives the same flux, a changed input (source, cross sections, options) is picked up."""
    import copy
    wl = tiny_p3_case(kind=2)
    ref = orc.solve(wl, closure=1)
    p, _ = run_gpu(wl, closure=1, fixed_iters=ref["iters"], deterministic=1)
    a = np.stack([p.get_flux_moments(0, g, 3) for g in range(wl.G)])
    p.solve(tol=wl.tol, max_iters=wl.max_iters, fixed_iters=ref["iters"], closure=1, deterministic=1)
    b = np.stack([p.get_flux_moments(0, g, 3) for g in range(wl.G)])
    assert np.array_equal(a, b)
    # new source on the same handle
    s1 = copy.deepcopy(wl.sources[0]); s1.pos = (0.3, 9.0, 0.2); s1.axis = (0.0, -1.0, 0.0)
    w2 = dataclasses.replace(wl, sources=[s1])
    ref2 = orc.solve(w2, closure=1)
    p.set_source(w2.sources, 0)
    p.solve(tol=wl.tol, max_iters=wl.max_iters, fixed_iters=ref2["iters"], closure=1)
    shape = (wl.nz, wl.ny, wl.nx)
    for g in range(wl.G):
        e, _ = masked_rel_err(p.get_flux_moments(0, g, 0)[0], ref2["phi"][0, g, 0].reshape(shape))
        assert e < TOL, (g, e)
    # other options on the same handle: closure and brick shape change the kernel and the layout
    ref3 = orc.solve(w2, closure=0)
    p.solve(tol=wl.tol, max_iters=wl.max_iters, fixed_iters=ref3["iters"], closure=0, brick=(4, 3, 5))
    for g in range(wl.G):
        e, _ = masked_rel_err(p.get_flux_moments(0, g, 0)[0], ref3["phi"][0, g, 0].reshape(shape))
        assert e < TOL, (g, e)
    p.close()
