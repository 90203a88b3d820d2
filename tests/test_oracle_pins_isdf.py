"""Pins of oracle/isdf.py (Eq. 15-17): interpolation property, separable form of the normal equations,
reconstruction error on smooth orbitals and its decay with N_mu, Eq. 16 against direct four-centre quadrature."""
import numpy as np

from oracle import isdf
from paper_2310_20103_b200 import synth


def _setup(n_grid=8, n_orb=6, n_mu=40, seed=1):
    r, phi, w = synth.box_orbitals(n_grid, n_orb)
    idx = synth.stride_points(r.shape[0], n_mu, seed)
    return r, phi, w, idx


def test_orbitals_are_orthonormal_under_the_grid_quadrature():
    r, phi, w, _ = _setup()
    S = w * phi.T @ phi
    assert np.abs(S - np.eye(phi.shape[1])).max() <= 1e-12


def test_interpolation_property_and_normal_equations():
    """zeta_mu(r_nu) = delta_mu,nu whenever C has full row rank (the fit is exact at the interpolation points), and zeta
    solves the normal equations zeta (C C^T) = Z C^T whose two sides have the separable (Hadamard) form
    Z C^T = (Phi Phi_mu^T) o (Phi Phi_mu^T),  C C^T = (Phi_mu Phi_mu^T) o (Phi_mu Phi_mu^T)."""
    r, phi, w, idx = _setup(n_mu=15)                       # 21 distinct pairs of 6 orbitals >= 15 points: full row rank
    zeta = isdf.fit(phi, phi, idx)
    assert np.abs(zeta[idx] - np.eye(len(idx))).max() <= 1e-8
    P = phi @ phi[idx].T
    ZCt, CCt = P * P, P[idx] * P[idx]
    Z = isdf.pair_products(phi, phi)
    assert np.abs(Z @ Z[idx].T - ZCt).max() <= 1e-13 * np.abs(ZCt).max()
    assert np.abs(zeta @ CCt - ZCt).max() <= 1e-9 * np.abs(ZCt).max()


def test_reconstruction_error_decays_with_n_mu():
    """Eq. 15 on smooth orbitals: the relative Frobenius error of the fitted pair products falls as N_mu grows and is
    at rounding level once N_mu reaches the number of distinct pair products."""
    r, phi, w, _ = _setup(n_orb=6)
    Z = isdf.pair_products(phi, phi)
    errs = []
    for n_mu in (6, 12, 21, 40):
        idx = synth.stride_points(r.shape[0], n_mu, 2)
        zeta = isdf.fit(phi, phi, idx)
        errs.append(np.linalg.norm(Z - zeta @ Z[idx]) / np.linalg.norm(Z))
    assert errs[0] > errs[1] > errs[2] and errs[2] <= 1e-8 and errs[3] <= 1e-8
    assert errs[0] > 1e-2


def test_eq16_against_direct_four_centre_quadrature():
    r, phi, w, idx = _setup(n_mu=30)
    G = isdf.coulomb_grid(r, w, 0.5)
    zeta = isdf.fit(phi, phi, idx)
    V = isdf.two_center(zeta, G)
    assert np.abs(V - V.T).max() <= 1e-10 * np.abs(V).max()
    for (k, l, n, m) in [(0, 1, 2, 3), (0, 0, 5, 5), (1, 4, 1, 4), (2, 3, 0, 5)]:
        d = isdf.four_center_direct(phi, G, k, l, n, m)
        a = isdf.four_center_isdf(phi[idx], V, k, l, n, m)
        assert abs(a - d) <= 1e-8 * max(abs(d), 1e-3)
    # (kl|kl) > 0: the softened Coulomb quadrature kernel is positive definite
    assert isdf.four_center_isdf(phi[idx], V, 1, 2, 1, 2) > 0


def test_two_orbital_sets_fit_only_their_cross_pairs():
    """Pairs (v, c) with v in one set and c in another (the Casida pair space): same least squares on fewer columns."""
    r, phi, w, idx = _setup(n_orb=7, n_mu=12)
    pv, pc = phi[:, :3], phi[:, 3:]
    zeta = isdf.fit(pv, pc, idx)
    Z = isdf.pair_products(pv, pc)
    assert np.linalg.norm(Z - zeta @ Z[idx]) <= 1e-8 * np.linalg.norm(Z)       # 12 pairs, 12 points
    Pv, Pc = pv @ pv[idx].T, pc @ pc[idx].T
    assert np.abs(zeta @ (Pv[idx] * Pc[idx]) - Pv * Pc).max() <= 1e-9 * np.abs(Pv * Pc).max()
