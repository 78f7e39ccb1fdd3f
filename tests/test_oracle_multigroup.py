"""Pins for the multigroup coupling of `oracle.solve` (Eq. 2 right-hand side: the sum over g' of
sigma_s^{g' -> g}; Eq. 5: the first-collision source) — the two parts of the oracle that rows a2 and g
of SURVEY §8 are compared against.

What fixes them here, none of it taken from the oracle's own formula:
  * the discretised Eq. (2) written as ONE dense linear system per group (signed streaming + diamond relations + vacuum
    inflow) with the discrete-to-discrete scattering kernel sigma_s(n' -> n) = sum_l (2l+1)/(4 pi) sigma_s,l P_l(Omega_n .
    Omega_n') built from numpy's Legendre polynomials — no Y_lm tables, no moment indices, no sweeping — solved group
    after group (block lower-triangular: in-scatter only from higher energy), per-cell density and material;
  * Eq. (5) written directly in angle: S_u(Omega_n) = sum_l (2l+1)/(4 pi) sigma_s,l P_l(Omega_n . u) phi_u, u from the
    geometry of a point source outside a tiny mesh;
  * particle conservation of the converged multigroup solve, group by group;
  * reciprocity of the optical path and analytic sphere chords for the ray tracer (SURVEY §8(c) pin table).
A swapped (g', g) index pair, a dropped density factor, a wrong l per moment index or a wrong Y_lm(u) each fail
at least one test below (checked by mutating oracle.py while writing them; see the commit message).
"""
import dataclasses
import math

import numpy as np
import pytest
from numpy.polynomial import legendre

from workloads import Workload, SourceSpec, make_config


# ---- the dense system ---------------------------------------------------------------------------------------------
def _dense_group_solve(om, w, dims, d, sig_t, sig_s_l, src):
    """Discretised Eq. (2) of ONE group with all directions coupled by within-group scattering.
         sig_t [cells], sig_s_l [L+1][cells] (already multiplied by the density), src [ndir][cells] = angular source
         density per steradian (everything on the right-hand side except within-group scattering).
       Unknowns per direction: cell-centre flux + the fluxes on all x, y, z faces.  Returns psi [ndir][cells]."""
    nx, ny, nz = dims
    nd, nc = len(w), nx * ny * nz
    nfx, nfy, nfz = (nx + 1) * ny * nz, nx * (ny + 1) * nz, nx * ny * (nz + 1)
    per = nc + nfx + nfy + nfz
    N = nd * per
    A = np.zeros((N, N)); b = np.zeros(N)
    cosm = np.clip(om @ om.T, -1.0, 1.0)
    Pl = [legendre.legval(cosm, [0] * l + [1]) for l in range(len(sig_s_l))]
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
                    A[row, o + fx(i + 1, j, k)] += mu / d[0]; A[row, o + fx(i, j, k)] -= mu / d[0]
                    A[row, o + fy(i, j + 1, k)] += eta / d[1]; A[row, o + fy(i, j, k)] -= eta / d[1]
                    A[row, o + fz(i, j, k + 1)] += xi / d[2]; A[row, o + fz(i, j, k)] -= xi / d[2]
                    A[row, o + c] += sig_t[c]
                    for n2 in range(nd):                           # sum_n' sigma_s(n' -> n) psi_n' w_n'
                        kern = sum((2 * l + 1) / (4 * math.pi) * sig_s_l[l][c] * Pl[l][n, n2] for l in range(len(sig_s_l)))
                        A[row, n2 * per + c] -= kern * w[n2]
                    b[row] = src[n, c]
                    row += 1
                    for fa, fb in ((fx(i, j, k), fx(i + 1, j, k)), (fy(i, j, k), fy(i, j + 1, k)), (fz(i, j, k), fz(i, j, k + 1))):
                        A[row, o + c] = 1.0; A[row, o + fa] -= 0.5; A[row, o + fb] -= 0.5
                        row += 1
        for k in range(nz):
            for j in range(ny):
                A[row, o + fx(0 if mu > 0 else nx, j, k)] = 1.0; row += 1      # vacuum inflow
        for k in range(nz):
            for i in range(nx):
                A[row, o + fy(i, 0 if eta > 0 else ny, k)] = 1.0; row += 1
        for j in range(ny):
            for i in range(nx):
                A[row, o + fz(i, j, 0 if xi > 0 else nz)] = 1.0; row += 1
    assert row == N
    x = np.linalg.solve(A, b)
    return np.stack([x[n * per:n * per + nc] for n in range(nd)])


def _inscatter(om, w, sig_s_l, psi_from):
    """Angular in-scatter source of Eq. (2): sum_n' sigma_s(n' -> n) psi_n' w_n', [ndir][cells]."""
    cosm = np.clip(om @ om.T, -1.0, 1.0)
    out = np.zeros_like(psi_from)
    for l, s in enumerate(sig_s_l):
        kern = (2 * l + 1) / (4 * math.pi) * legendre.legval(cosm, [0] * l + [1])      # [n][n']
        out += s[None, :] * (kern @ (w[:, None] * psi_from))
    return out


def _two_material_mesh(nx, ny, nz, seed):
    rng = np.random.default_rng(seed)
    mat = rng.integers(0, 2, (nz, ny, nx)).astype(np.uint8)
    mat.reshape(-1)[0], mat.reshape(-1)[-1] = 0, 1                      # both materials present
    rho = rng.uniform(0.4, 1.9, (nz, ny, nx)).astype(np.float32)
    return mat, rho


def _asymmetric_xs(G, L, seed):
    """Every entry distinct: sigma_t [2][G]; sigma_s [2][L+1][G][G] lower... g_to >= g_from only."""
    rng = np.random.default_rng(seed)
    st = rng.uniform(0.8, 1.6, (2, G))
    ss = np.zeros((2, L + 1, G, G))
    for m in range(2):
        for gf in range(G):
            for gt in range(gf, G):
                s0 = rng.uniform(0.15, 0.35)
                for l in range(L + 1):
                    ss[m, l, gf, gt] = s0 * rng.uniform(0.3, 0.6) ** l * (1.0 if l == 0 else rng.choice([-1.0, 1.0]))
    return st, ss


def _moments_from_psi(om, w, psi):
    """phi_00 and the three l = 1 moments straight from the angular flux: Y_1,-1 = eta, Y_1,0 = xi, Y_1,+1 = mu (R4)."""
    return np.stack([(w[:, None] * psi).sum(0), (w[:, None] * om[:, 1:2] * psi).sum(0),
                     (w[:, None] * om[:, 2:3] * psi).sum(0), (w[:, None] * om[:, 0:1] * psi).sum(0)])


# ---- (a) downscatter: two and three groups, volume sources ---------------------------------------------------------
@pytest.mark.parametrize("G,L,sn,dims", [(2, 1, 4, (2, 2, 2)), (3, 2, 2, (3, 2, 2))])
def test_downscatter_equals_block_triangular_dense_solve(orc, G, L, sn, dims):
    nx, ny, nz = dims
    d = (1.0, 0.8, 1.3)
    mat, rho = _two_material_mesh(nx, ny, nz, 5)
    st, ss = _asymmetric_xs(G, L, 6)
    rng = np.random.default_rng(7)
    vol = rng.uniform(0.2, 1.0, (G, nz, ny, nx)).astype(np.float32)
    wl = Workload("mg", nx, ny, nz, d[0], d[1], d[2], mat, rho, 2, G, L, sn, st, ss,
                  [SourceSpec(kind=0, volume=vol)], tol=1e-14, max_iters=5000)
    res = orc.solve(wl, closure=0)
    om, w = orc.level_symmetric(sn)
    r, m = rho.astype(float).reshape(-1), mat.reshape(-1)
    psi = []
    for g in range(G):
        src = np.broadcast_to(vol[g].astype(float).reshape(-1) / (4 * math.pi), (len(w), nx * ny * nz)).copy()
        for gp in range(g):                                          # Eq. (2) rhs: in-scatter from the groups above
            src += _inscatter(om, w, [r * ss[m, l, gp, g] for l in range(L + 1)], psi[gp])
        psi.append(_dense_group_solve(om, w, dims, d, r * st[m, g], [r * ss[m, l, g, g] for l in range(L + 1)], src))
        want = _moments_from_psi(om, w, psi[g])
        scale = np.abs(want[0]).max()
        assert np.abs(res["phi"][0, g, 0] - want[0]).max() < 1e-10 * scale, g
        assert np.abs(res["phi"][0, g, 1:4] - want[1:4]).max() < 1e-10 * scale, g
    # the coupling is really there: group 1 without in-scatter from group 0 is a different answer
    src1 = np.broadcast_to(vol[1].astype(float).reshape(-1) / (4 * math.pi), (len(w), nx * ny * nz)).copy()
    alone = _dense_group_solve(om, w, dims, d, r * st[m, 1], [r * ss[m, l, 1, 1] for l in range(L + 1)], src1)
    assert np.abs(_moments_from_psi(om, w, alone)[0] - res["phi"][0, 1, 0]).max() > 1e-2 * np.abs(res["phi"][0, 1, 0]).max()


# ---- (b) first-collision source, all moments l <= 3, two groups ----------------------------------------------------
def test_first_collision_moments_equal_angular_eq5(orc):
    nx, ny, nz = 2, 2, 2
    d = (1.0, 1.2, 0.9)
    G, L, sn = 2, 3, 4
    mat, rho = _two_material_mesh(nx, ny, nz, 15)
    st, ss = _asymmetric_xs(G, L, 16)
    pos = (-3.1, 1.7, 0.6)                                            # outside the mesh, no symmetry with the axes
    spec = np.array([0.7, 0.3])
    wl = Workload("fc", nx, ny, nz, d[0], d[1], d[2], mat, rho, 2, G, L, sn, st, ss,
                  [SourceSpec(kind=1, pos=pos, spectrum=spec)], tol=1e-14, max_iters=5000)
    res = orc.solve(wl, closure=0)
    om, w = orc.level_symmetric(sn)
    r, m = rho.astype(float).reshape(-1), mat.reshape(-1)
    # u_c by hand: cell centres of a mesh centred on the origin
    xs = [(np.arange(n) + 0.5) * h - n * h / 2 for n, h in zip((nx, ny, nz), d)]
    rc = np.array([[xs[0][i], xs[1][j], xs[2][k]] for k in range(nz) for j in range(ny) for i in range(nx)])
    u = rc - np.array(pos)
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    phi_u = res["phi_u"][0]                                           # [G][cells]: the ray tracer has its own pins
    cosu = np.clip(om @ u.T, -1.0, 1.0)                               # [n][cells]

    def eq5(g_from, g_to):
        s = np.zeros((len(w), nx * ny * nz))
        for l in range(L + 1):
            s += (2 * l + 1) / (4 * math.pi) * (r * ss[m, l, g_from, g_to] * phi_u[g_from])[None, :] * legendre.legval(cosu, [0] * l + [1])
        return s

    psi0 = _dense_group_solve(om, w, (nx, ny, nz), d, r * st[m, 0], [r * ss[m, l, 0, 0] for l in range(L + 1)], eq5(0, 0))
    src1 = eq5(0, 1) + eq5(1, 1) + _inscatter(om, w, [r * ss[m, l, 0, 1] for l in range(L + 1)], psi0)
    psi1 = _dense_group_solve(om, w, (nx, ny, nz), d, r * st[m, 1], [r * ss[m, l, 1, 1] for l in range(L + 1)], src1)
    for g, psi in ((0, psi0), (1, psi1)):
        want = _moments_from_psi(om, w, psi)
        scale = np.abs(want[0]).max()
        assert np.abs(res["phi"][0, g, 0:4] - want).max() < 1e-10 * scale, g
        # all 16 moments: direction -> moment with the Cartesian forms of reading R4 written out here
        mu, eta, xi = om[:, 0], om[:, 1], om[:, 2]
        Y = [np.ones_like(mu), eta, xi, mu,
             math.sqrt(3) * mu * eta, math.sqrt(3) * xi * eta, 0.5 * (3 * xi ** 2 - 1), math.sqrt(3) * xi * mu, 0.5 * math.sqrt(3) * (mu ** 2 - eta ** 2),
             math.sqrt(5 / 8) * (3 * mu ** 2 * eta - eta ** 3), math.sqrt(15) * xi * mu * eta, math.sqrt(3 / 8) * (5 * xi ** 2 - 1) * eta,
             0.5 * (5 * xi ** 3 - 3 * xi), math.sqrt(3 / 8) * (5 * xi ** 2 - 1) * mu, 0.5 * math.sqrt(15) * xi * (mu ** 2 - eta ** 2),
             math.sqrt(5 / 8) * (mu ** 3 - 3 * mu * eta ** 2)]
        for lm in range(16):
            assert np.abs(res["phi"][0, g, lm] - (w[:, None] * Y[lm][:, None] * psi).sum(0)).max() < 1e-10 * scale, (g, lm)
    # the anisotropic part of Eq. (5) matters here: an isotropic first-collision source gives a different flux
    iso = (r * ss[m, 0, 0, 0] * phi_u[0])[None, :] / (4 * math.pi) * np.ones((len(w), 1))
    psi_iso = _dense_group_solve(om, w, (nx, ny, nz), d, r * st[m, 0], [r * ss[m, l, 0, 0] for l in range(L + 1)], iso)
    assert np.abs(_moments_from_psi(om, w, psi_iso)[3] - res["phi"][0, 0, 3]).max() > 1e-3 * np.abs(res["phi"][0, 0, 0]).max()


# ---- (c) particle conservation of the converged multigroup solve, group by group -----------------------------------
def test_multigroup_particle_balance_config1(orc):
    """Converged Eq. (2) integrated over angle and volume, for every group g of config 1:
         sum_c sigma_t phi_g V + leakage_g = sum_c sum_{g' <= g} sigma_s0(g' -> g) (phi_g' + phi_u,g') V
       (the collided flux is driven by what scatters out of the uncollided beam, Eq. 5, and by in-scatter).  Summed over g
       with the total out-scatter of the synthetic tables, sum_g sigma_s0(g' -> g) = c_g' sigma_t,g': downscatter conserves
       particles, absorption + leakage = first collisions."""
    wl = make_config(1)
    wl.tol = 1e-9
    res = orc.solve(wl, closure=0)
    r, m = wl.density.astype(float).reshape(-1), wl.material.reshape(-1)
    V = wl.dx * wl.dy * wl.dz
    phi0, phi_u = res["phi"][0, :, 0], res["phi_u"][0]
    tot_first = tot_abs = tot_leak = 0.0
    for g in range(wl.G):
        coll = (r * wl.sigma_t[m, g] * phi0[g]).sum() * V
        leak = res["balance"][0, g, 2]
        src = 0.0
        for gp in range(g + 1):
            src += (r * wl.sigma_s[m, 0, gp, g] * (phi_u[gp] + phi0[gp])).sum() * V
        assert abs(coll + leak - src) < 2e-7 * src, (g, coll, leak, src)
        out_scatter = wl.sigma_s[m, 0, g, :].sum(1)                   # sum over destination groups
        tot_first += (r * out_scatter * phi_u[g]).sum() * V
        tot_abs += (r * (wl.sigma_t[m, g] - out_scatter) * phi0[g]).sum() * V
        tot_leak += leak
    assert abs(tot_abs + tot_leak - tot_first) < 2e-7 * tot_first
    assert tot_leak > 0.1 * tot_first and tot_abs > 0.01 * tot_first   # both terms carry weight


# ---- ray tracer: reciprocity and sphere chords (SURVEY §8(c) pin table) --------------------------------------------
def test_raytrace_reciprocity_between_cell_centres(orc):
    """The areal density per material along the segment between two cell centres does not depend on which end holds the
    source.  Heterogeneous 4-material mesh; pairs in general position."""
    from tests.parity_util import tiny_p3_case
    wl = tiny_p3_case(nx=11, ny=9, nz=7, G=1, sn=2, L=0, seed=3)
    xs = [(np.arange(n) + 0.5) * h - n * h / 2 for n, h in zip((wl.nx, wl.ny, wl.nz), (wl.dx, wl.dy, wl.dz))]
    centre = lambda c: (xs[0][c % wl.nx], xs[1][(c // wl.nx) % wl.ny], xs[2][c // (wl.nx * wl.ny)])
    rng = np.random.default_rng(8)
    one = np.array([1.0])
    for a, b in rng.integers(0, wl.cells, (12, 2)):
        if a == b:
            continue
        with np.errstate(divide="ignore", invalid="ignore"):
            _, A_ab = orc.raytrace(wl, SourceSpec(kind=1, pos=centre(a), spectrum=one), want_areal=True)
            _, A_ba = orc.raytrace(wl, SourceSpec(kind=1, pos=centre(b), spectrum=one), want_areal=True)
        assert A_ab[:, b].sum() > 0
        np.testing.assert_allclose(A_ab[:, b], A_ba[:, a], rtol=1e-11, atol=1e-13)


def test_raytrace_sphere_chords_config1(orc):
    """Config 1: water sphere of radius 6 cm in air, point source at (-20, 0, 0).  For cells beyond the sphere the water
    path A_water / rho_water must equal the analytic chord 2 sqrt(R^2 - b^2) of the ray's impact parameter b, up to the
    voxelisation of the sphere (0.5 cm voxels, centre sampling)."""
    wl = make_config(1)
    src = wl.sources[0]
    _, areal = orc.raytrace(wl, src, want_areal=True)
    x = (np.arange(32) + 0.5) * 0.5 - 8.0
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    rc = np.stack([X, Y, Z], -1).reshape(-1, 3)
    dvec = rc - np.array(src.pos)
    R = np.linalg.norm(dvec, axis=1)
    u = dvec / R[:, None]
    tca = -(u @ np.array(src.pos))                                   # distance along the ray to the closest approach
    b2 = (np.array(src.pos) ** 2).sum() - tca ** 2
    chord = 2.0 * np.sqrt(np.maximum(36.0 - b2, 0.0))
    # impact parameter below 5 cm: nearer the limb d(chord)/d(radius) = 2 R / sqrt(R^2 - b^2) blows the voxelisation up
    behind = (b2 < 25.0) & (R > tca + np.sqrt(np.maximum(36.0 - b2, 0.0)) + 0.5) & (np.linalg.norm(rc, axis=1) > 6.5)
    assert behind.sum() > 500
    water = areal[2] / 1.0                                            # material 2 = water, density 1.0
    err = water[behind] - chord[behind]
    assert np.abs(err).max() < 1.0                                    # two voxels
    assert abs(err.mean()) < 0.1 and np.sqrt((err ** 2).mean()) < 0.3
    central = behind & (b2 < 0.3)
    assert central.any() and np.abs(water[central] - 12.0).max() < 0.55
    miss = (b2 > 49.0)
    assert (water[miss] == 0.0).all()


def test_source_iteration_contracts_at_most_at_the_scattering_ratio(orc):
    """SURVEY 8(c) pin table, "Iteration": delta_k decreases geometrically at a rate <= the in-group scattering ratio c =
    sigma_s,gg / sigma_t (source iteration's error contracts by at most c per sweep in any medium; leakage only helps), and the
    sweep count does not depend on how the sources are chunked (the oracle has no chunks: one problem at a time)."""
    wl = make_config(1)
    wl.G = 2
    wl.sigma_t = wl.sigma_t[:, 8:10].copy(); wl.sigma_s = wl.sigma_s[:, :, 8:10, 8:10].copy()
    wl.sources[0].spectrum = np.array([0.5, 0.5])
    wl.tol = 1e-9
    res = orc.solve(wl, closure=0, keep_history=True)
    for g in range(2):
        c = (wl.sigma_s[:, 0, g, g] / wl.sigma_t[:, g]).max()       # the same ratio in every material of the synthetic tables
        h = res["history"][0][g]
        assert len(h) >= 8 and h[-1] < wl.tol
        ratios = [h[k + 1] / h[k] for k in range(2, len(h) - 1)]
        assert max(ratios) <= c + 1e-3, (g, c, max(ratios))
        assert min(ratios) > 0.02                                     # geometric, not erratic
