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


# ---- interpolation points by weighted k-means (reading Q22) ------------------------------------------------------
def test_cvt_two_cluster_closed_form():
    """Six collinear points in two groups, unit weights, both initial centroids in the left group: Lloyd must end with the
    groups {0,1,2} and {10,11,12}, centroids 1 and 11, i.e. the grid points 1 and 4."""
    x = np.array([0.0, 1.0, 2.0, 10.0, 11.0, 12.0])
    r = np.stack([x, np.zeros(6), np.zeros(6)], axis=1)
    idx, done, obj = isdf.select_points_cvt(r, np.ones(6), np.array([0, 1]), 20)
    assert list(idx) == [1, 4]
    assert abs(obj[-1] - 4.0) <= 1e-12                      # 2 x (1 + 0 + 1)
    # weights move the centroid: heavy point 12 pulls the right centroid to 11.5 -> nearest member is 11 (index 4) or 12 (5): tie -> lowest
    idx_w, _, _ = isdf.select_points_cvt(r, np.array([1, 1, 1, 1, 1, 3.0]), np.array([0, 1]), 20)
    c_right = (10 + 11 + 3 * 12) / 5.0
    assert idx_w[0] == 1 and idx_w[1] == (4 if abs(11 - c_right) <= abs(12 - c_right) else 5)


def test_cvt_objective_decreases_and_points_are_valid():
    r, phi, w, _ = _setup(n_grid=10, n_orb=9)
    dens = (phi ** 2).sum(axis=1)
    init = synth.stride_points(r.shape[0], 24, 5)
    idx, done, obj = isdf.select_points_cvt(r, dens, init, 50)
    assert all(b <= a * (1 + 1e-14) for a, b in zip(obj, obj[1:]))          # Lloyd never increases the weighted objective
    assert done < 50 and len(set(idx.tolist())) == 24 and idx.min() >= 0 and idx.max() < r.shape[0]
    # a converged tessellation is a fixed point: restarting from the selected points' centroids changes nothing further
    idx2, done2, _ = isdf.select_points_cvt(r, dens, init, done + 5)
    assert np.array_equal(idx, idx2) and done2 == done
    # and it serves its purpose: C C^T at these points is far better conditioned than at the seeded random points
    def cond(ix):
        P = phi @ phi[ix].T
        ev = np.linalg.eigvalsh(P[ix] * P[ix])
        return ev[-1] / ev[0]
    assert cond(idx) < 1e-2 * cond(init)


def test_coulomb_grid_reproduces_the_coulomb_energy_of_two_gaussian_charges():
    """Pin of isdf.coulomb_grid (Eq. 17: (alpha|beta) = int int zeta_alpha(r) zeta_beta(r') / |r - r'|) by a
    value the oracle does not compute itself.  Two normalised Gaussian charges of width sigma at distance R have the
    Coulomb energy 14.4 erf(R / (2 sigma)) / R eV (14.4 eV A = e^2 / (4 pi eps_0)).  With the softened kernel
    1/sqrt(d^2 + s^2) = (2/sqrt(pi)) int_0^inf exp(-t^2 (d^2 + s^2)) dt and the Gaussian average
    E[exp(-t^2 d^2)] = (1 + 4 sigma^2 t^2)^(-3/2) exp(-t^2 R^2 / (1 + 4 sigma^2 t^2)) of the relative coordinate
    d ~ N(R, 2 sigma^2), the softened energy is the one-dimensional integral I(s) below; I(0) is the erf formula.
      (1) I(0) = 14.4 erf(R / 2 sigma) / R to 1e-12 (the integral representation is the textbook result), and
          I(s) -> I(0) monotonically as s -> 0;
      (2) rho_1^T G rho_2 with G = coulomb_grid(r, h^3, s) converges to I(s) as h -> 0: the integrand is smooth on the scale
          of s and sigma, so the midpoint rule converges geometrically -- each refinement gains at least a factor 4, and
          the finest grid agrees to 5e-5.
    A weight instead of weight^2 changes the value by 1/h^3, a missing 14.4 by that factor, a softening placed as
    (d + s)^2 or on the diagonal only misses I(s) by per cent."""
    from math import erf

    from scipy.integrate import quad
    sigma, R, soft, box = 0.9, 1.7, 0.9, 11.0

    def softened_energy(s):
        def f(t):
            q = 1.0 + 4.0 * sigma * sigma * t * t
            return np.exp(-t * t * s * s) * q ** -1.5 * np.exp(-t * t * R * R / q)
        return 14.4 * 2.0 / np.sqrt(np.pi) * quad(f, 0.0, np.inf, epsabs=1e-13, epsrel=1e-13)[0]

    exact = 14.4 * erf(R / (2.0 * sigma)) / R
    assert abs(softened_energy(0.0) - exact) <= 1e-12 * exact
    gaps = [exact - softened_energy(s) for s in (0.4, 0.2, 0.1)]
    assert gaps[0] > 2.5 * gaps[1] > 0 and gaps[1] > 2.5 * gaps[2] > 0 and gaps[2] <= 6e-3 * exact

    c1 = np.array([-0.6, 0.1, -0.2])
    u = np.array([1.0, 2.0, -0.5])
    c2 = c1 + R * u / np.linalg.norm(u)                       # a generic direction: no lattice symmetry to help

    def gauss(r, c):
        return (2.0 * np.pi * sigma * sigma) ** -1.5 * np.exp(-((r - c) ** 2).sum(axis=1) / (2.0 * sigma * sigma))

    target = softened_energy(soft)
    errs = []
    for n in (8, 11, 14, 17):
        h = box / n
        x = -0.5 * box + h * (np.arange(n) + 0.5)
        X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
        r = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
        G = isdf.coulomb_grid(r, h ** 3, soft)
        errs.append(abs(gauss(r, c1) @ (G @ gauss(r, c2)) - target) / target)
    assert errs[0] <= 1e-2 and all(errs[i + 1] <= 0.25 * errs[i] for i in range(3)) and errs[3] <= 5e-5, errs
