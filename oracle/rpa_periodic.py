"""CPU oracle for the complex-orbital (periodic) RPA variant of the Lanczos GW method: the pole sum the paper prints for
periodic systems (Supplemental Material section 1) and a Lanczos method "designed for pseudo-Hermitian
matrices" that reaches it.  SURVEY.md 8(f)-3, second step.

TEST INFRASTRUCTURE, NOT PRODUCT (same rules as gw_oracle.py): plain NumPy/SciPy complex128, no code shared with
paper_2310_20103_b200/, imports nothing from it.  Pins: tests/test_oracle_pins_rpa_periodic.py.

What the paper fixes (one transferred momentum q; pair index j = (k, v, c), c fastest; N = N_k N_v N_c):
  C^RPA(q) = [[A, B], [-B^*, -A^*]]
  A = diag(Delta) + K^H V K,   B = K^H V conj(K),  K[mu, j] = conj(psi_vk(mu)) psi_ck+q(mu)
  C^RPA [[X, Y^*], [Y, X^*]] = [[X, Y^*], [Y, X^*]] diag(Omega, -Omega)
  Sigma(omega) = 2/(N_q N_k) sum_n sum_q sum_s |W^s|^2 / (omega - eps_n + eta_n (Omega_s - i delta))
  W^s = sum_j [ (n k-q, m k | v'k', c'k'+q) X^s_j + (n k-q, m k | c'k'+q, v'k') Y^s_j ]
with s over the N POSITIVE excitation energies and the usual normalisation X^H X - Y^H Y = 1 (the one under which the real
one-k-point case is Eq. 7 of the main text; pinned).  `sigma_chain_exact_rpa` is that definition written out.

What the paper leaves open, and the reading taken (Q24): PAPER.md:159 only names "a Lanczos-based method designed
for pseudo-Hermitian matrices [34, 36, 74]".  H = C^RPA = F Omega^ with F = diag(1, -1) and Omega^ = [[A, B], [B^*, A^*]]
Hermitian positive definite (V positive semidefinite, Delta > 0), so H is self-adjoint in the inner product
<a, b>_O = a^H Omega^ b and an ordinary three-term Lanczos in that inner product gives a REAL symmetric tridiagonal T whose
Ritz values approximate +-Omega_s.  With d = conj([P1; P2]) (P1, P2 the printed elements) W^s = d^H v_s for the right
eigenvector v_s = [X^s; Y^s], and because <v_s, F d>_O = lambda_s d^H v_s and <v_s, v_s>_O = |lambda_s|,
  sum_{s: lambda_s > 0} |W^s|^2 g(Omega_s) = <u, f(H) u>_O,   u = F d,   f(lambda) = theta(lambda) g(lambda) / lambda.
The spectrum has a gap around 0, so f is smooth on it and the Lanczos (Gauss) quadrature
  <u, f(H) u>_O ~ <u, u>_O sum_{i: theta_i > 0} w_i g(theta_i) / theta_i      (theta_i, w_i: Ritz values / first components^2)
converges like the Ritz evaluation of Eq. 11 in direct mode; at L = 2N with reorthogonalisation it is exact (pinned).
One step costs ONE product with Omega^ (two K, one V, two K^H products), twice a Tamm-Dancoff step.
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla

from . import tda_periodic as tdp

BREAKDOWN_TOL = 1e-12


def omega_hat_dense(A, B):
    """Omega^ = F C^RPA = [[A, B], [B^*, A^*]] (Hermitian: A = A^H, B = B^T)."""
    return np.block([[A, B], [B.conj(), A.conj()]])


def omega_hat_factored(psi_v, psi_cq, V, delta, X, Y):
    """[X'; Y'] = Omega^ [X; Y] without forming K, A or B.  X, Y [nvec, N] complex.
    A x + B y = Delta x + K^H V (K x + conj(K) y),  B^* x + A^* y = Delta y + K^T V (K x + conj(K) y)  (V real)."""
    n_k, n_mu, n_v = psi_v.shape
    n_c = psi_cq.shape[2]
    X = np.asarray(X, dtype=np.complex128).reshape(-1, n_k, n_v, n_c)
    Y = np.asarray(Y, dtype=np.complex128).reshape(-1, n_k, n_v, n_c)
    nvec = X.shape[0]
    T = (np.einsum("kmv,kmc,bkvc->mb", psi_v.conj(), psi_cq, X, optimize=True)
         + np.einsum("kmv,kmc,bkvc->mb", psi_v, psi_cq.conj(), Y, optimize=True))
    W = V @ T
    U1 = np.einsum("kmv,kmc,mb->bkvc", psi_v, psi_cq.conj(), W, optimize=True)       # K^H W
    U2 = np.einsum("kmv,kmc,mb->bkvc", psi_v.conj(), psi_cq, W, optimize=True)       # K^T W
    return (delta[None, :] * X.reshape(nvec, -1) + U1.reshape(nvec, -1),
            delta[None, :] * Y.reshape(nvec, -1) + U2.reshape(nvec, -1))


def printed_elements(psi_v, psi_cq, V, kn, n_idx, km, m_idx):
    """The two families of integrals in W^s, in the notation of tda_periodic ((a,b|c,d) =
    sum conj(psi_b) psi_a V psi_d conj(psi_c)):
      P1_j = (n k-q, m k | v'k', c'k'+q) = sum_mu g(mu) K[mu, j],   P2_j = (n k-q, m k | c'k'+q, v'k') = sum_mu g(mu) conj(K[mu, j]),
    g = V (conj(psi_m) psi_n)."""
    rho = np.conj(tdp.orbital(psi_v, psi_cq, km, m_idx)) * tdp.orbital(psi_v, psi_cq, kn, n_idx)
    g = V.T @ rho
    P1 = np.einsum("kmv,kmc,m->kvc", psi_v.conj(), psi_cq, g, optimize=True).reshape(-1)
    P2 = np.einsum("kmv,kmc,m->kvc", psi_v, psi_cq.conj(), g, optimize=True).reshape(-1)
    return P1, P2


def rpa_eig(A, B):
    """Positive excitation energies Omega_s and (X^s, Y^s) of C^RPA(q) by a general eigensolver,
    normalised to X^H X - Y^H Y = 1.  Raises if the spectrum is not N real +- pairs (Omega^ not positive definite)."""
    n = A.shape[0]
    lam, vec = sla.eig(tdp.casida_rpa_block(A, B))
    if np.abs(lam.imag).max() > 1e-8 * np.abs(lam).max():
        raise ValueError("C^RPA has complex eigenvalues: Omega^ is not positive definite")
    order = np.argsort(-lam.real)[:n]
    order = order[np.argsort(lam.real[order])]
    om = lam.real[order]
    if om.min() <= 0.0:
        raise ValueError("fewer than N positive eigenvalues")
    X, Y = vec[:n, order], vec[n:, order]
    fnorm = np.einsum("js,js->s", X.conj(), X).real - np.einsum("js,js->s", Y.conj(), Y).real
    if fnorm.min() <= 0.0:
        raise ValueError("a positive-energy eigenvector has non-positive F-norm")
    sc = 1.0 / np.sqrt(fnorm)
    return om, X * sc[None, :], Y * sc[None, :]


def sigma_chain_exact_rpa(om, X, Y, P1, P2, omega, eps_n, sgn_n, dlt, prefactor):
    """The printed pole sum: prefactor sum_s |W^s|^2 / (omega - eps_n + eta_n (Omega_s - i delta)),
    W^s = sum_j (P1_j X^s_j + P2_j Y^s_j) (bilinear, no conjugation of P)."""
    W = P1 @ X + P2 @ Y
    den = np.asarray(omega)[:, None] - eps_n + sgn_n * (om[None, :] - 1j * dlt)
    return prefactor * ((np.abs(W) ** 2)[None, :] / den).sum(axis=1)


def start_vector_rpa(P1, P2):
    """u = F d with d = conj([P1; P2]): the Lanczos start vector (module docstring).  Returns (u1, u2)."""
    return np.conj(P1), -np.conj(P2)


def lanczos_pseudo_hermitian(apply_omega_hat, u1, u2, steps, reorth=False):
    """Three-term Lanczos for H = F Omega^ in the inner product <a, b>_O = a^H Omega^ b, started from u = [u1; u2].
    apply_omega_hat(x, y) -> (x', y').  Per step, with q_k normalised (<q_k, q_k>_O = 1) and s_k = Omega^ q_k carried along:
      h = F s_k (= H q_k),  a_k = <q_k, h>_O = s_k^H F s_k (real),  t = Omega^ h,
      w = h - a_k q_k - b_k q_{k-1},  Omega^ w = t - a_k s_k - b_k s_{k-1},  b_{k+1} = sqrt(w^H Omega^ w),
      q_{k+1} = w / b_{k+1},  s_{k+1} = Omega^ w / b_{k+1}.
    reorth: two passes of w -= sum_j q_j <q_j, w>_O (complex coefficients s_j^H w), Omega^ w updated with the same coefficients.
    Returns alpha[steps], beta[steps] (beta[k] = b_{k+1}), norm2 = <u, u>_O, length (breakdown reading Q9)."""
    n = u1.size
    q = np.concatenate([np.asarray(u1, dtype=np.complex128), np.asarray(u2, dtype=np.complex128)])
    sx, sy = apply_omega_hat(q[:n], q[n:])
    s = np.concatenate([sx, sy])
    norm2 = float(np.vdot(q, s).real)
    alpha = np.zeros(steps)
    beta = np.zeros(steps)
    if norm2 <= 0.0:
        return alpha, beta, max(norm2, 0.0), 0
    q = q / np.sqrt(norm2)
    s = s / np.sqrt(norm2)
    q_prev = np.zeros_like(q)
    s_prev = np.zeros_like(s)
    b_prev = 0.0
    scale = 0.0
    Qb, Sb = [], []
    length = steps
    sign = np.concatenate([np.ones(n), -np.ones(n)])
    for k in range(steps):
        if reorth:
            Qb.append(q)
            Sb.append(s)
        h = sign * s
        a = float(np.vdot(s, h).real)
        tx, ty = apply_omega_hat(h[:n], h[n:])
        t = np.concatenate([tx, ty])
        w = h - a * q - b_prev * q_prev
        sw = t - a * s - b_prev * s_prev
        if reorth:
            Qm, Sm = np.array(Qb), np.array(Sb)
            for _ in range(2):
                c = Sm.conj() @ w
                w = w - Qm.T @ c
                sw = sw - Sm.T @ c
        b2 = float(np.vdot(w, sw).real)
        b = float(np.sqrt(b2)) if b2 > 0.0 else 0.0
        alpha[k] = a
        beta[k] = b
        scale = max(scale, abs(a) + b)
        if b <= BREAKDOWN_TOL * scale:
            beta[k] = 0.0
            length = k + 1
            break
        q_prev, s_prev, b_prev = q, s, b
        q, s = w / b, sw / b
    return alpha, beta, norm2, length


def ritz(alpha, beta, length):
    """Eigenvalues theta_i of T_L and weights w_i = (first eigenvector component)^2."""
    L = int(length)
    if L == 0:
        return np.zeros(0), np.zeros(0)
    if L == 1:
        return np.array([alpha[0]]), np.array([1.0])
    th, Z = sla.eigh_tridiagonal(alpha[:L], beta[:L - 1])
    return th, Z[0] ** 2


def sigma_chain_rpa(alpha, beta, norm2, length, omega, eps_n, sgn_n, dlt, prefactor):
    """prefactor <u, u>_O sum_{i: theta_i > 0} w_i / (theta_i (omega - eps_n + eta_n (theta_i - i delta)))  (module docstring)."""
    th, w = ritz(alpha, beta, length)
    omega = np.asarray(omega, dtype=np.float64)
    out = np.zeros(omega.shape, dtype=np.complex128)
    for t, wi in zip(th, w):
        if t > 0.0:
            out += wi / (t * (omega - eps_n + sgn_n * (t - 1j * dlt)))
    return prefactor * norm2 * out


def resolvent_chain(alpha, beta, norm2, length, zeta):
    """<u|(zeta - H)^{-1}|u>_O by Eq. 14 on the tridiagonal of lanczos_pseudo_hermitian: both branches +-Omega_s."""
    return tdp.continued_fraction(alpha, beta, norm2, zeta, length)


def resolvent_exact_rpa(A, B, u1, u2, zeta):
    """The same matrix element by dense solves: u^H Omega^ (zeta - F Omega^)^{-1} u."""
    n = A.shape[0]
    Oh = omega_hat_dense(A, B)
    H = tdp.casida_rpa_block(A, B)
    u = np.concatenate([u1, u2])
    out = np.zeros(len(zeta), dtype=np.complex128)
    for i, z in enumerate(np.asarray(zeta, dtype=np.complex128)):
        out[i] = np.vdot(u, Oh @ np.linalg.solve(z * np.eye(2 * n) - H, u))
    return out


def run_chains_rpa(psi_v, psi_cq, eps_v, eps_cq, V, chains, steps, omega, dlt, n_q=1, reorth=False):
    """S1-S7 for chains [(kn, n_idx, km, m_idx), ...] in the RPA with complex orbitals."""
    delta = tdp.delta_kvc(eps_v, eps_cq)
    pf = tdp.prefactor(n_q, psi_v.shape[0])

    def op(x, y):
        a, b = omega_hat_factored(psi_v, psi_cq, V, delta, x[None], y[None])
        return a[0], b[0]

    n = len(chains)
    out = dict(alpha=np.zeros((n, steps)), beta=np.zeros((n, steps)), norm2=np.zeros(n),
               len=np.zeros(n, dtype=np.int32), sigma=np.zeros((n, len(omega)), dtype=np.complex128))
    for j, (kn, n_idx, km, m_idx) in enumerate(chains):
        P1, P2 = printed_elements(psi_v, psi_cq, V, int(kn), int(n_idx), int(km), int(m_idx))
        u1, u2 = start_vector_rpa(P1, P2)
        a, b, n2, ln = lanczos_pseudo_hermitian(op, u1, u2, steps, reorth=reorth)
        e_n, sg = tdp.orbital_energy_sign(eps_v, eps_cq, int(kn), int(n_idx))
        out["alpha"][j], out["beta"][j], out["norm2"][j], out["len"][j] = a, b, n2, ln
        out["sigma"][j] = sigma_chain_rpa(a, b, n2, ln, omega, e_n, sg, dlt, pf)
    out["sigma_sum"] = out["sigma"].sum(axis=0)
    return out
