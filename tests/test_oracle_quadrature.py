"""Pins for the oracle's quadrature and spherical harmonics (SURVEY §8(c) pin table).

What the paper fixes: N(N+2) directions, 8/24/48/80 for S2..S8, and
Eq. (3) as a quadrature of the angular integral.  Everything else is mathematics.
"""
import math
import os

import numpy as np
import pytest
from numpy.polynomial import legendre

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name, key=None):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        t = line.split()
        if key is None:
            out.append(t)
        elif t[0] == key:
            out.append(t[1:])
    return out


@pytest.mark.parametrize("N", [2, 4, 6, 8, 12, 16])
def test_direction_count_and_weight_sum(orc, N):
    om, w = orc.level_symmetric(N)
    assert om.shape == (N * (N + 2), 3)
    assert abs(w.sum() - 4 * math.pi) < 1e-13                 # reading R6
    assert np.allclose(np.linalg.norm(om, axis=1), 1.0, atol=1e-14)
    assert (w > 0).all()


def test_paper_direction_counts(orc):
    for N, n in _rows("paper_facts.txt", "ndir"):
        assert orc.level_symmetric(int(N))[0].shape[0] == int(n)


@pytest.mark.parametrize("N", [2, 4, 6, 8, 12, 16])
def test_tabulated_mu1(orc, N):
    tab = {int(a): float(b) for a, b in _rows("lqn_mu1.txt")}
    om, _ = orc.level_symmetric(N)
    assert abs(np.abs(om).min() - tab[N]) < 1e-6


def test_s8_weights_are_rational(orc):
    # the S8 LQ_N class weights are exactly 49/405, 49/540, 5/54 per octant
    _, w = orc.level_symmetric(8)
    got = sorted(set(np.round(w[:10] * 8 / (4 * math.pi), 12)))
    want = sorted([49 / 540, 5 / 54, 49 / 405])
    assert np.allclose(got, want, atol=1e-12)


@pytest.mark.parametrize("N", [2, 4, 6, 8, 12, 16])
def test_even_and_odd_moments(orc, N):
    om, w = orc.level_symmetric(N)
    for ax in range(3):
        for k in range(0, N // 2 + 1):
            assert abs((w * om[:, ax] ** (2 * k)).sum() - 4 * math.pi / (2 * k + 1)) < 2e-13
        for k in (1, 3, 5):
            assert abs((w * om[:, ax] ** k).sum()) < 1e-13
    assert abs((w * om[:, 0] * om[:, 1]).sum()) < 1e-13


def test_s16_mixed_moments(orc):
    # rule of App. A: the free parameter makes the mixed even moments of degree 12 exact as well
    om, w = orc.level_symmetric(16)
    dfact = lambda n: 1 if n <= 0 else n * dfact(n - 2)
    for a, b, c in [(2, 2, 2), (4, 1, 1), (3, 2, 1), (3, 3, 0), (5, 1, 0), (3, 3, 1), (5, 1, 1), (4, 2, 1)]:
        exact = 4 * math.pi * dfact(2 * a - 1) * dfact(2 * b - 1) * dfact(2 * c - 1) / dfact(2 * (a + b + c) + 1)
        got = (w * om[:, 0] ** (2 * a) * om[:, 1] ** (2 * b) * om[:, 2] ** (2 * c)).sum()
        assert abs(got - exact) < 1e-12, (a, b, c)


def test_octant_ordering(orc):
    om, w = orc.level_symmetric(8)
    M = 10
    for o in range(8):
        blk = om[o * M:(o + 1) * M]
        assert ((blk[:, 0] < 0) == bool(o & 1)).all()
        assert ((blk[:, 1] < 0) == bool(o & 2)).all()
        assert ((blk[:, 2] < 0) == bool(o & 4)).all()
        assert np.allclose(np.abs(blk), om[:M]) and np.allclose(w[o * M:(o + 1) * M], w[:M])


def test_ylm_cartesian_forms(orc):
    # reading R4: the first 16 real harmonics as Cartesian polynomials
    rng = np.random.default_rng(5)
    v = rng.normal(size=(50, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    mu, eta, xi = v.T
    s3, s15 = math.sqrt(3), math.sqrt(15)
    want = np.stack([
        np.ones_like(mu), eta, xi, mu,
        s3 * mu * eta, s3 * xi * eta, (3 * xi ** 2 - 1) / 2, s3 * xi * mu, s3 / 2 * (mu ** 2 - eta ** 2),
        math.sqrt(5 / 8) * (3 * mu ** 2 * eta - eta ** 3), s15 * xi * mu * eta,
        math.sqrt(3 / 8) * (5 * xi ** 2 - 1) * eta, (5 * xi ** 3 - 3 * xi) / 2,
        math.sqrt(3 / 8) * (5 * xi ** 2 - 1) * mu, s15 / 2 * xi * (mu ** 2 - eta ** 2),
        math.sqrt(5 / 8) * (mu ** 3 - 3 * mu * eta ** 2)], axis=1)
    assert np.abs(orc.real_sph_harm(3, v) - want).max() < 1e-14


def test_addition_theorem(orc):
    # sum_m Y_lm(a) Y_lm(b) = P_l(a.b): ties the harmonics to numpy's Legendre polynomials
    rng = np.random.default_rng(7)
    a = rng.normal(size=(40, 3)); a /= np.linalg.norm(a, axis=1, keepdims=True)
    b = rng.normal(size=(40, 3)); b /= np.linalg.norm(b, axis=1, keepdims=True)
    Ya, Yb = orc.real_sph_harm(3, a), orc.real_sph_harm(3, b)
    ll = orc.l_of_lm(3)
    cosab = (a * b).sum(1)
    for l in range(4):
        lhs = (Ya[:, ll == l] * Yb[:, ll == l]).sum(1)
        rhs = legendre.legval(cosab, [0] * l + [1])
        assert np.abs(lhs - rhs).max() < 1e-14


@pytest.mark.parametrize("N,Lmax", [(2, 1), (4, 2), (6, 3), (8, 4), (16, 5)])
def test_discrete_orthogonality(orc, N, Lmax):
    # sum_n w_n Y_lm Y_l'm' = 4 pi/(2l+1) delta for l, l' <= Lmax: P3 is Galerkin-consistent at S8, S16
    om, w = orc.level_symmetric(N)
    Y = orc.real_sph_harm(Lmax, om)
    ll = orc.l_of_lm(Lmax)
    Gm = (Y * w[:, None]).T @ Y
    assert np.abs(Gm - np.diag(4 * math.pi / (2 * ll + 1))).max() < 1e-12


def test_projection_tables_match_eq2_discrete_form(orc):
    """Eq. (2) literally: scattering source of direction n = sum_n' sigma_s(n'->n) psi_n' w_n'
    with sigma_s(n'->n) = sum_l (2l+1)/(4pi) sigma_s,l P_l(Omega_n . Omega_n').  The oracle's moment form
    (Mtab @ diag(sigma_s,l) @ Dtab) must be the same matrix, for any quadrature (addition theorem)."""
    om, w = orc.level_symmetric(6)
    L = 3
    sig_l = np.array([1.0, 0.3, 0.09, 0.027])
    Mtab, Dtab = orc.projection_tables(L, om, w)
    ll = orc.l_of_lm(L)
    K_moment = Mtab @ np.diag(sig_l[ll]) @ Dtab                     # [n][n']
    cosm = om @ om.T
    K_direct = np.zeros_like(cosm)
    for l in range(L + 1):
        K_direct += (2 * l + 1) / (4 * math.pi) * sig_l[l] * legendre.legval(cosm, [0] * l + [1])
    K_direct = K_direct * w[None, :]
    assert np.abs(K_moment - K_direct).max() < 1e-13
    # moment 0 of the table is Eq. (3): phi = sum_n w_n psi_n
    assert np.allclose(Dtab[0], w)
