"""Python face of the polynomial-mode helpers of the C ABI: coefficients of p_g(x) ~ sqrt(x) and the
fitting range for gwl_set_polynomial.  PAPER.md:85, :284, :317 (readings Q12, Q13, Q23).

The arithmetic lives in libgwl.so -- gwl_fit_sqrt_polynomial (the least-squares fit at the Chebyshev nodes, closed form in the
Chebyshev basis) and gwl_sqrt_fit_range (heuristic range, or the Lanczos estimate of gwl_spectrum_bounds) -- so a C caller can
run the paper's route (g = 7, N_iter = 8) without this file.  The functions here only forward.  No oracle code is used.
"""
from __future__ import annotations

import numpy as np


def default_range(eps_v, eps_c):
    """The paper's heuristic [0.8 min Delta^2, 1.25 max Delta^2], Delta = eps_c - eps_v (PAPER.md:284 with reading
    Q12).  Its upper end is NOT a bound on lambda_max(C) once the coupling 2 sqrt(Delta) K^T V K sqrt(Delta) is
    strong (config 2: lambda_max ~ 2321 eV^2 against 1.25 max Delta^2 = 1125): outside [lo, hi] a Chebyshev fit
    diverges.  Use range_from_spectrum unless the spectrum is known to lie inside."""
    d_min = float(np.min(eps_c) - np.max(eps_v))
    d_max = float(np.max(eps_c) - np.min(eps_v))
    return 0.8 * d_min * d_min, 1.25 * d_max * d_max


def range_from_spectrum(ctx, eps_v, eps_c, steps: int = 40, margin: float = 0.02):
    """Fitting range from the operator itself, "One can use standard Lanczos algorithm to determine the extremal
    eigenvalues min(Omega_s^2) and max(Omega_s^2) of C".
    hi = (1 + margin) x max(top Ritz value + its residual norm from gwl_spectrum_bounds, max Delta^2).  max Delta^2 is a
    diagonal entry of C minus a positive-semidefinite coupling part, so it bounds lambda_max from below.  The Lanczos
    figure is an ESTIMATE, not a bound: some eigenvalue lies within the residual of the top Ritz value, but lambda_max
    itself can sit higher until the top Ritz value has converged (it does within a few steps when the upper edge is
    separated, as in the synthetic configs, where the tests find the GPU's and the oracle's estimates, taken from
    different start vectors, within 1e-6 of each other).  The 2 % margin is a heuristic
    cushion for that, not a guarantee: a caller who cannot afford a diverging p_g raises `steps` until two successive
    estimates agree to well inside the margin.
    lo = the paper's 0.8 min Delta^2, which IS a lower bound of C whenever V is positive semidefinite
    (C - diag(Delta^2) is then positive semidefinite).  Call before the chain list is set (the probe replaces it)."""
    return ctx.sqrt_fit_range(steps, margin)            # eps_v, eps_c: the context already holds them (gwl_set_energies)


def sqrt_chebyshev(g: int, lo: float, hi: float, nodes_per_coefficient: int = 4) -> np.ndarray:
    """c[0..g] with p_g(x) = sum_j c_j T_j((2x - hi - lo)/(hi - lo)) the least-squares fit of sqrt(x) at
    M = nodes_per_coefficient (g + 1) Chebyshev nodes of [lo, hi]."""
    if g < 1 or not (hi > lo > 0.0):
        raise ValueError("need g >= 1 and hi > lo > 0")
    if nodes_per_coefficient != 4:
        raise ValueError("gwl_fit_sqrt_polynomial fits at 4 (g + 1) nodes (DESIGN.md Q13)")
    from . import gwl
    return gwl.fit_sqrt_polynomial(g, lo, hi)
