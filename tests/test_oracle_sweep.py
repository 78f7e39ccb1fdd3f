"""Pins for the oracle's sweep, closure and source iteration (SURVEY §8(c) pin table).

The paper prints no flux values, so the sweep is pinned by mathematics:
closed-form 1-D attenuation, exact per-sweep balance, bitwise order independence,
symmetry, linearity, and an INDEPENDENT formulation: the discretised Eq. (2)
(signed streaming form + diamond relations + vacuum inflow, discrete-to-discrete
scattering kernel from Legendre polynomials) assembled as one dense linear system
and handed to numpy.linalg.solve — no sweeping, no upwind logic, no Y_lm tables.
"""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre

from workloads import Workload, SourceSpec, make_config


def _one_dir(om):
    om = np.array([om], dtype=float)
    return om, np.array([1.0]), np.array([[1.0]]), np.array([[1.0]])     # q_n = Q, phi = psi


def test_1d_attenuation_ratio_and_second_order(orc):
    # N_y = N_z = 1 with huge pitch: source-free cells attenuate by exactly (1-h)/(1+h), h = sig*dx/(2 mu)
    mu, sig, Lx = 0.6, 0.8, 4.0
    errs = []
    for n in (16, 32, 64):
        dx = Lx / n
        om, w, M, D = _one_dir([mu, math.sqrt(1 - mu * mu) * 0.6, math.sqrt(1 - mu * mu) * 0.8])
        Q = np.zeros((1, n + 2)); Q[0, 0] = 1.0
        _, _, psi, _ = orc.sweep(n + 2, 1, 1, dx, 1e30, 1e30, np.full(n + 2, sig), Q, om, w, M, D, want_psi=True)
        psi = psi[0]
        h = sig * dx / (2 * mu)
        assert np.allclose(psi[2:] / psi[1:-1], (1 - h) / (1 + h), rtol=1e-13)
        errs.append(abs(psi[n + 1] / psi[1] - math.exp(-sig * Lx / mu)) / math.exp(-sig * Lx / mu))
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.7 < errs[1] / errs[2] < 4.3      # O(h^2)
    assert errs[2] < 4e-3                      # ~ n * (2/3) h^3, h = 0.0417


def test_negative_direction_mirrors(orc):
    # sweeping -x over the mirrored problem gives the mirrored answer
    rng = np.random.default_rng(1)
    nx, ny, nz = 5, 4, 3
    sig = rng.uniform(0.1, 2.0, (nz, ny, nx)); Q = rng.uniform(0, 1, (1, nz, ny, nx))
    om, w, M, D = _one_dir([0.5, 0.7, math.sqrt(1 - 0.25 - 0.49)])
    a = orc.sweep(nx, ny, nz, 0.3, 0.4, 0.5, sig, Q.reshape(1, -1), om, w, M, D, want_psi=True)[2]
    om2 = om * np.array([-1, 1, -1.0])
    b = orc.sweep(nx, ny, nz, 0.3, 0.4, 0.5, sig[::-1, :, ::-1], Q[:, ::-1, :, ::-1].reshape(1, -1),
                  om2, w, M, D, want_psi=True)[2]
    assert np.array_equal(a.reshape(nz, ny, nx), b.reshape(nz, ny, nx)[::-1, :, ::-1])


def test_corner_cell(orc):
    om, w, M, D = _one_dir([0.3, 0.5, math.sqrt(1 - 0.09 - 0.25)])
    nx = ny = nz = 3
    Q = np.full((1, 27), 2.0)
    psi = orc.sweep(nx, ny, nz, 0.5, 0.25, 1.0, np.full(27, 0.7), Q, om, w, M, D, want_psi=True)[2][0]
    c = 2 * om[0] / np.array([0.5, 0.25, 1.0])
    assert abs(psi[0] - 2.0 / (0.7 + c.sum())) < 1e-15


@pytest.mark.parametrize("closure", [0, 1])
@pytest.mark.parametrize("dims", [(3, 4, 5), (6, 2, 3), (1, 5, 4)])
def test_sweep_order_independence_bitwise(orc, closure, dims):
    nx, ny, nz = dims
    rng = np.random.default_rng(3)
    om, w = orc.level_symmetric(4)
    M, D = orc.projection_tables(1, om, w)
    sig = rng.uniform(0.05, 6.0, nx * ny * nz)
    Q = rng.normal(size=(4, nx * ny * nz)) * np.array([[1.0], [0.2], [0.2], [0.2]]) + np.array([[0.5], [0], [0], [0]])
    a = orc.sweep(nx, ny, nz, 0.7, 0.4, 1.1, sig, Q, om, w, M, D, closure, 0, want_psi=True)
    b = orc.sweep(nx, ny, nz, 0.7, 0.4, 1.1, sig, Q, om, w, M, D, closure, 1, want_psi=True)
    assert np.array_equal(a[2], b[2]) and np.array_equal(a[0], b[0])
    assert a[1] == pytest.approx(b[1], rel=1e-13)
    if closure == 1:
        assert a[3] == b[3]


@pytest.mark.parametrize("closure", [0, 1])
def test_per_sweep_particle_balance(orc, closure):
    nx, ny, nz = 7, 5, 6
    dx, dy, dz = 0.5, 0.8, 0.3
    rng = np.random.default_rng(11)
    om, w = orc.level_symmetric(8)
    M, D = orc.projection_tables(3, om, w)
    sig = rng.uniform(0.01, 8.0, nx * ny * nz)
    Q = rng.normal(size=(16, nx * ny * nz)) * 0.1
    Q[0] = rng.uniform(0, 1, nx * ny * nz)
    phi, leak, psi, nfix = orc.sweep(nx, ny, nz, dx, dy, dz, sig, Q, om, w, M, D, closure, want_psi=True)
    V = dx * dy * dz
    src, col = Q[0].sum() * V, (sig * phi[0]).sum() * V
    assert abs(src - col - leak) < 1e-13 * src
    if closure == 1:
        assert nfix > 0


def test_fixup_gives_nonnegative_flux_and_reduces_to_dd(orc):
    nx, ny, nz = 6, 6, 6
    om, w = orc.level_symmetric(4)
    M, D = orc.projection_tables(0, om, w)
    rng = np.random.default_rng(2)
    Q = rng.uniform(0, 1, (1, 216)); Q[0, 100:] = 0.0
    thick = np.full(216, 9.0)
    p0 = orc.sweep(nx, ny, nz, 1, 1, 1, thick, Q, om, w, M, D, 0, want_psi=True)
    p1 = orc.sweep(nx, ny, nz, 1, 1, 1, thick, Q, om, w, M, D, 1, want_psi=True)
    assert p0[2].min() < 0 and p1[2].min() >= 0.0 and p1[3] > 0
    # thin, uniformly driven cells: no outflow goes negative, fix-up must not fire and results are identical
    thin = np.full(216, 0.05)
    Qu = np.ones((1, 216))
    q0 = orc.sweep(nx, ny, nz, 1, 1, 1, thin, Qu, om, w, M, D, 0, want_psi=True)
    q1 = orc.sweep(nx, ny, nz, 1, 1, 1, thin, Qu, om, w, M, D, 1, want_psi=True)
    assert q1[3] == 0 and np.array_equal(q0[2], q1[2])


def _tiny_workload(nx, ny, nz, d, sig_t, sig_s_l, vol, sn, tol=1e-14):
    L = len(sig_s_l) - 1
    mat = np.zeros((nz, ny, nx), dtype=np.uint8)
    rho = np.ones((nz, ny, nx), dtype=np.float32)
    ss = np.array(sig_s_l, dtype=float).reshape(1, L + 1, 1, 1)
    return Workload("tiny", nx, ny, nz, d[0], d[1], d[2], mat, rho, 1, 1, L, sn,
                    np.array([[sig_t]]), ss, [SourceSpec(kind=0, volume=vol.reshape(1, nz, ny, nx).astype(np.float32))],
                    tol=tol, max_iters=5000)


def _dense_eq2_solve(orc, nx, ny, nz, d, sig_t, sig_s_l, vol, sn):
    """Discretised Eq. (2), all directions coupled, as one linear system (see module docstring)."""
    om, w = orc.level_symmetric(sn)
    nd = len(w)
    nc = nx * ny * nz
    nfx, nfy, nfz = (nx + 1) * ny * nz, nx * (ny + 1) * nz, nx * ny * (nz + 1)
    per = nc + nfx + nfy + nfz
    N = nd * per
    A = np.zeros((N, N)); b = np.zeros(N)
    cosm = om @ om.T
    K = np.zeros((nd, nd))
    for l, s in enumerate(sig_s_l):
        K += (2 * l + 1) / (4 * math.pi) * s * legendre.legval(cosm, [0] * l + [1])
    K = K * w[None, :]                                           # K[n][n'] = sigma_s(n'->n) w_n'
    ci = lambda i, j, k: i + nx * (j + ny * k)
    fx = lambda i, j, k: nc + i + (nx + 1) * (j + ny * k)
    fy = lambda i, j, k: nc + nfx + i + nx * (j + (ny + 1) * k)
    fz = lambda i, j, k: nc + nfx + nfy + i + nx * (j + ny * k)
    row = 0
    for n in range(nd):
        o = n * per
        mu, eta, xi = om[n]
        for k in range(nz):
            for j in range(ny):
                for i in range(nx):
                    c = ci(i, j, k)
                    # cell balance: Omega . grad psi integrated over the cell / volume
                    A[row, o + fx(i + 1, j, k)] += mu / d[0]; A[row, o + fx(i, j, k)] -= mu / d[0]
                    A[row, o + fy(i, j + 1, k)] += eta / d[1]; A[row, o + fy(i, j, k)] -= eta / d[1]
                    A[row, o + fz(i, j, k + 1)] += xi / d[2]; A[row, o + fz(i, j, k)] -= xi / d[2]
                    A[row, o + c] += sig_t
                    for n2 in range(nd):
                        A[row, n2 * per + c] -= K[n, n2]
                    b[row] = vol[k, j, i] / (4 * math.pi)
                    row += 1
                    # diamond relations
                    for fa, fb in ((fx(i, j, k), fx(i + 1, j, k)), (fy(i, j, k), fy(i, j + 1, k)), (fz(i, j, k), fz(i, j, k + 1))):
                        A[row, o + c] = 1.0; A[row, o + fa] -= 0.5; A[row, o + fb] -= 0.5
                        row += 1
        # vacuum inflow
        for k in range(nz):
            for j in range(ny):
                A[row, o + fx(0 if mu > 0 else nx, j, k)] = 1.0; row += 1
        for k in range(nz):
            for i in range(nx):
                A[row, o + fy(i, 0 if eta > 0 else ny, k)] = 1.0; row += 1
        for j in range(ny):
            for i in range(nx):
                A[row, o + fz(i, j, 0 if xi > 0 else nz)] = 1.0; row += 1
    assert row == N
    x = np.linalg.solve(A, b)
    psi = np.stack([x[n * per:n * per + nc] for n in range(nd)])
    return (w[:, None] * psi).sum(0), psi, om, w


@pytest.mark.parametrize("case", [
    dict(dims=(3, 2, 2), d=(1.0, 0.7, 1.3), sig_t=0.9, sig_s=[0.5, 0.2], sn=2),
    dict(dims=(2, 3, 2), d=(0.5, 0.5, 0.5), sig_t=2.0, sig_s=[1.2], sn=4),
    dict(dims=(2, 2, 2), d=(1.0, 1.0, 2.0), sig_t=1.0, sig_s=[0.6, 0.3, 0.1], sn=4),
])
def test_converged_iteration_equals_direct_solve_of_eq2(orc, case):
    nx, ny, nz = case["dims"]
    rng = np.random.default_rng(4)
    vol = rng.uniform(0.2, 1.0, (nz, ny, nx))
    phi_direct, psi, om, w = _dense_eq2_solve(orc, nx, ny, nz, case["d"], case["sig_t"], case["sig_s"], vol, case["sn"])
    wl = _tiny_workload(nx, ny, nz, case["d"], case["sig_t"], case["sig_s"], vol, case["sn"])
    wl.density[:] = 1.0
    res = orc.solve(wl, closure=0)
    vol32 = wl.sources[0].volume[0].astype(float)                # the oracle sees the float32-rounded source
    phi_direct32 = _dense_eq2_solve(orc, nx, ny, nz, case["d"], case["sig_t"], case["sig_s"], vol32, case["sn"])[0]
    assert np.abs(res["phi"][0, 0, 0] - phi_direct32).max() < 1e-11 * phi_direct32.max()
    # higher moments against the direct angular flux, using the harmonics only for the projection
    if len(case["sig_s"]) > 1:
        psi32 = _dense_eq2_solve(orc, nx, ny, nz, case["d"], case["sig_t"], case["sig_s"], vol32, case["sn"])[1]
        mom1 = (w[:, None] * om[:, 0:1] * psi32).sum(0)          # moment of mu = Y_{1,+1}, index 3
        assert np.abs(res["phi"][0, 0, 3] - mom1).max() < 1e-11 * phi_direct32.max()


def test_config0_against_survey_probe_and_symmetry(orc):
    # SURVEY.md App. B (an independent throwaway numpy implementation): phi0 max 0.99727, min 4.18e-4,
    # delta_10 = 9.25e-5 (9.3e-5 in App. B), delta_2 = 0.188, no negative phi0
    res = orc.solve(make_config(0), closure=0, keep_history=True)
    p = res["phi"][0, 0, 0].reshape(8, 8, 8)
    assert abs(p.max() - 0.99727) < 1e-5 and abs(p.min() - 4.18e-4) < 1e-6 and p.min() > 0
    hist = res["history"][0][0]
    assert len(hist) == 10 and abs(hist[1] - 0.188) < 5e-4 and abs(hist[9] - 9.25e-5) < 1e-6
    assert all(hist[k + 1] / hist[k] <= 0.9 for k in range(1, 9))   # geometric, rate <= c = 0.9
    # the 48 cube symmetries: axis permutations and flips
    for perm in [(0, 1, 2), (1, 0, 2), (2, 1, 0), (0, 2, 1), (1, 2, 0), (2, 0, 1)]:
        q = p.transpose(perm)
        for fl in range(8):
            r = q[::-1] if fl & 1 else q
            r = r[:, ::-1] if fl & 2 else r
            r = r[:, :, ::-1] if fl & 4 else r
            assert np.abs(r - p).max() < 1e-14
    # per-sweep balance of the last sweep
    src, col, leak = res["balance"][0, 0]
    assert abs(src - col - leak) < 1e-13 * src


def test_linearity_and_scaling_pure_dd(orc):
    rng = np.random.default_rng(9)
    nx, ny, nz = 4, 3, 5
    v1 = rng.uniform(0, 1, (nz, ny, nx)).astype(np.float32).astype(float)
    v2 = rng.uniform(0, 1, (nz, ny, nx)).astype(np.float32).astype(float)
    v12 = (v1.astype(np.float32) + v2.astype(np.float32)).astype(float)
    mk = lambda v: _tiny_workload(nx, ny, nz, (1.0, 1.0, 1.0), 3.0, [1.5, 0.4], v, 4)
    sol = {}
    for name, v in (("a", v1), ("b", v2), ("ab", v12), ("2a", 2 * v1)):
        wl = mk(v); wl.fixed_iters = 6
        sol[name] = orc.solve(wl, closure=0)["phi"][0, 0]
    assert np.abs(sol["ab"] - sol["a"] - sol["b"]).max() < 1e-6 * np.abs(sol["ab"]).max()   # v12 rounded in f32
    assert np.abs(sol["2a"] - 2 * sol["a"]).max() < 1e-13 * np.abs(sol["2a"]).max()


@pytest.mark.parametrize("closure", [0, 1])
def test_infinite_medium_limit(orc, closure):
    # interior of a thick, uniform, uniformly driven block: phi -> S / (sigma_t - sigma_s).
    # Diamond difference in 3-D carries weakly damped oscillatory modes from the vacuum boundary layer
    # (the antisymmetric face modes have amplification -1 per cell), so the centre value approaches the
    # limit only algebraically in the block size: 5.9e-3 at n = 21, 3.0e-3 at n = 41.  A dropped term or a
    # wrong normalisation (4 pi, factor 2) moves it by O(1).
    n = 21
    wl = _tiny_workload(n, n, n, (2.0, 2.0, 2.0), 1.0, [0.5], np.ones((n, n, n)), 2, tol=1e-12)
    res = orc.solve(wl, closure=closure)
    mid = res["phi"][0, 0, 0].reshape(n, n, n)[n // 2, n // 2, n // 2]
    assert abs(mid - 1.0 / 0.5) < 1e-2
    src, col, leak = res["balance"][0, 0]
    assert abs(src - col - leak) < 1e-12 * src


def test_response_hook_definition(orc):
    """orc.response against what fixes it: a unit response picks one group's total fluence, it is linear in the
    response, and a mode-1 problem adds the uncollided flux of every source."""
    from tests.parity_util import tiny_p3_case
    from workloads import SourceSpec
    wl = tiny_p3_case(nx=6, ny=5, nz=4, G=3, sn=4, L=1, seed=2)
    res = orc.solve(wl, closure=1)
    for g in range(wl.G):
        e = np.zeros(wl.G); e[g] = 1.0
        np.testing.assert_allclose(orc.response(res, wl, 0, e), res["phi"][0, g, 0] + res["phi_u"][0, g], rtol=1e-15)
        np.testing.assert_allclose(orc.response(res, wl, 0, e, include_uncollided=False), res["phi"][0, g, 0], rtol=0)
    r1, r2 = np.array([0.3, 1.7, 2.0]), np.array([1.0, -0.5, 0.25])
    np.testing.assert_allclose(orc.response(res, wl, 0, 2.0 * r1 + r2),
                               2.0 * orc.response(res, wl, 0, r1) + orc.response(res, wl, 0, r2), rtol=1e-13, atol=1e-300)
    # summed sources: one problem, the uncollided part is the sum over both sources
    src2 = [wl.sources[0], SourceSpec(kind=1, pos=(0.4, -9.0, 0.3), spectrum=np.full(wl.G, 1.0 / wl.G))]
    import dataclasses
    wl2 = dataclasses.replace(wl, sources=src2, mode=1)
    res2 = orc.solve(wl2, closure=1)
    ones = np.ones(wl.G)
    want = res2["phi"][0, :, 0].sum(0) + res2["phi_u"].sum((0, 1))
    np.testing.assert_allclose(orc.response(res2, wl2, 0, ones), want, rtol=1e-14)

