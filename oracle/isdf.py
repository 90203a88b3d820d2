"""CPU oracle for the interpolative separable density fitting front end, PAPER.md:115-128
(Eq. 15-17) and :319 ("have not yet been accelerated with GPUs" in the paper's code).

TEST INFRASTRUCTURE, NOT PRODUCT (same rules as gw_oracle.py).  Plain NumPy FP64; the least-squares problem of Eq. 15 is
written out with the pair products formed explicitly (tiny sizes only), no separable shortcut.

Notation: Phi [N_r, N] orbitals on the real-space grid r_i (uniform weight w = h^3), interpolation points
r_mu = r[idx[mu]] (a subset of the grid, the ISDF of refs. [62, 63]), pair products Z[r, (n m)] = phi_n(r) phi_m(r),
fitting coefficients C[mu, (n m)] = phi_n(r_mu) phi_m(r_mu) (reading Q4), auxiliary functions zeta [N_r, N_mu].
"""
from __future__ import annotations

import numpy as np


def pair_products(phi_a, phi_b):
    """Z[r, (a b)] = phi_a(r) phi_b(r), b fastest."""
    n_r = phi_a.shape[0]
    return (phi_a[:, :, None] * phi_b[:, None, :]).reshape(n_r, -1)


def fit(phi_a, phi_b, idx):
    """Eq. 15: phi_a(r) phi_b(r) ~ sum_mu zeta_mu(r) C^mu_ab with C^mu_ab = phi_a(r_mu) phi_b(r_mu);
    zeta minimises || Z - zeta C ||_F (least squares, refs. [62, 63]): zeta = Z C^T (C C^T)^{-1}.  Returns zeta [N_r, N_mu]."""
    Z = pair_products(phi_a, phi_b)
    C = Z[np.asarray(idx)]
    zt, *_ = np.linalg.lstsq(C.T, Z.T, rcond=None)          # C^T zeta^T = Z^T in the least-squares sense
    return zt.T


def coulomb_grid(r, weight, soft):
    """Quadrature form of 1/|r - r'| on the grid points, softened at short range (stand-in for the Poisson solve of the
    real-space code): G[i, j] = weight^2 14.4 / sqrt(|r_i - r_j|^2 + soft^2)  (eV Angstrom units as in synth.py).
    Pinned by the Coulomb energy of two Gaussian charges (erf closed form and its softened one-dimensional integral),
    tests/test_oracle_pins_isdf.py::test_coulomb_grid_reproduces_the_coulomb_energy_of_two_gaussian_charges."""
    d = r[:, None, :] - r[None, :, :]
    return weight * weight * 14.4 / np.sqrt(np.einsum("ijk,ijk->ij", d, d) + soft * soft)


def two_center(zeta, G):
    """Eq. 17: (alpha|beta) = int int zeta_alpha(r) zeta_beta(r') / |r - r'| -> zeta^T G zeta."""
    return zeta.T @ (G @ zeta)


def four_center_direct(phi, G, k, l, n, m):
    """(kl|nm) by direct quadrature of the four-centre integral, for checking Eq. 16."""
    return (phi[:, k] * phi[:, l]) @ (G @ (phi[:, n] * phi[:, m]))


def four_center_isdf(phi_mu, V, k, l, n, m):
    """Eq. 16: (kl|nm) ~ sum_ab (alpha|beta) C^alpha_kl C^beta_nm."""
    return (phi_mu[:, k] * phi_mu[:, l]) @ (V @ (phi_mu[:, n] * phi_mu[:, m]))


# --------------------------------------------------------------------------- #
# Interpolation points by centroidal Voronoi tessellation (weighted k-means)   #
# --------------------------------------------------------------------------- #
def select_points_cvt(r, weight, init_idx, iters):
    """Interpolation points for the ISDF (PAPER.md:128 uses "the interpolative separable density fitting (ISDF) method
    ... [13, 62, 63]" and does not say how its points are chosen; reading Q22b: the centroidal-Voronoi / weighted k-means
    choice of the ISDF literature the paper cites).  Lloyd iterations on the grid points r_i with weights w_i (an
    electron-density-like sum of squared orbitals):
      assign   a_i = argmin_mu |r_i - c_mu|^2                      (ties: the lowest mu)
      update   c_mu = sum_{a_i = mu} w_i r_i / sum_{a_i = mu} w_i   (an empty cluster keeps its centroid)
    started from c_mu = r[init_idx[mu]], `iters` times or until no assignment changes; then one more assignment and every
    centroid is replaced by its nearest MEMBER grid point (ties: the lowest i), which makes the points distinct.
    Returns (idx [N_mu] int32, -1 for an empty cluster; iterations done; objective sum_i w_i |r_i - c_{a_i}|^2 per iteration)."""
    r = np.asarray(r, dtype=np.float64)
    w = np.asarray(weight, dtype=np.float64)
    c = r[np.asarray(init_idx)].copy()
    n_mu = c.shape[0]
    prev = None
    obj = []

    def assign(c):
        d = r[:, None, :] - c[None, :, :]
        d2 = (d[:, :, 0] * d[:, :, 0] + d[:, :, 1] * d[:, :, 1]) + d[:, :, 2] * d[:, :, 2]
        return np.argmin(d2, axis=1), d2

    done = 0
    for it in range(iters):
        a, d2 = assign(c)
        obj.append(float(np.sum(w * d2[np.arange(len(a)), a])))
        if prev is not None and np.array_equal(a, prev):
            break
        prev = a
        for mu in range(n_mu):
            sel = a == mu
            ws = w[sel].sum()
            if ws > 0.0:
                c[mu] = (w[sel][:, None] * r[sel]).sum(axis=0) / ws
        done = it + 1
    a, d2 = assign(c)
    idx = np.full(n_mu, -1, dtype=np.int32)
    for mu in range(n_mu):
        members = np.nonzero(a == mu)[0]
        if members.size:
            idx[mu] = members[np.argmin(d2[members, mu])]
    return idx, done, obj
