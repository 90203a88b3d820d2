"""CPU oracle for the complex-orbital (periodic) Tamm-Dancoff variant of the Lanczos GW method,
PAPER.md:157-159 and Supplemental Material section 1.

TEST INFRASTRUCTURE, NOT PRODUCT (same rules as gw_oracle.py): plain NumPy/SciPy complex128, no code shared
with paper_2310_20103_b200/, imports nothing from it.  Pins: tests/test_oracle_pins_periodic.py.

One transferred momentum q is fixed.  For every k-point k of the grid (N_k of them) the caller provides
  psi_v [N_k, N_mu, N_v]    psi_{v k}(r_mu)
  psi_cq[N_k, N_mu, N_c]    psi_{c k+q}(r_mu)     (the conduction orbitals already shifted by q)
  eps_v [N_k, N_v], eps_cq [N_k, N_c]
  V [N_mu, N_mu] real symmetric: the paper needs A(q) Hermitian and B(q) symmetric, which the
     discretised integrals give iff V = V^T = V^* (reading Q21); Eq. 17's (alpha|beta) with real zeta is such a V.
Pair index (k, v, c), c fastest.  Notation of the two-electron integrals, read off the printed A(q):
  (a, b | c, d) = sum_{mu nu} conj(psi_b(mu)) psi_a(mu) V[mu, nu] psi_d(nu) conj(psi_c(nu)).
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla

BREAKDOWN_TOL = 1e-12


def delta_kvc(eps_v, eps_cq):
    """Delta_{vck} = eps_{c k+q} - eps_{v k}, flattened (k, v, c).  PAPER.md:298."""
    return (np.asarray(eps_cq)[:, None, :] - np.asarray(eps_v)[:, :, None]).reshape(-1)


def pair_matrix(psi_v, psi_cq):
    """K[mu, (k, v, c)] = conj(psi_{v k}(mu)) psi_{c k+q}(mu): the density psi_{c'k'+q}(r') psi^*_{v'k'}(r') of the ket
    side of A(q)."""
    n_k, n_mu, _ = psi_v.shape
    K = np.conj(psi_v)[:, :, :, None] * psi_cq[:, :, None, :]            # [k, mu, v, c]
    return np.transpose(K, (1, 0, 2, 3)).reshape(n_mu, -1)


def tda_dense(delta, K, V):
    """A(q) = diag(eps_{ck+q} - eps_{vk}) + (vk, ck+q | v'k', c'k'+q) = diag(Delta) + K^H V K.  PAPER.md:298-300."""
    return np.diag(delta).astype(np.complex128) + K.conj().T @ (V @ K)


def coupling_B(K, V):
    """B(q) = (vk, ck+q | c'k'+q, v'k') = K^H V conj(K).  PAPER.md:301."""
    return K.conj().T @ (V @ K.conj())


def casida_rpa_block(A, B):
    """C^RPA(q) = [[A, B], [-B^*, -A^*]]."""
    return np.block([[A, B], [-B.conj(), -A.conj()]])


def casida_td_block(A):
    """C^TD(q) = [[A, 0], [0, -A^*]]."""
    Z = np.zeros_like(A)
    return np.block([[A, Z], [Z, -A.conj()]])


def tda_matvec_factored(psi_v, psi_cq, V, delta, X):
    """Y = A(q) X = Delta o X + K^H ( V ( K X ) ) without forming K.  X [nvec, N_k N_v N_c] complex."""
    n_k, n_mu, n_v = psi_v.shape
    n_c = psi_cq.shape[2]
    X = np.asarray(X, dtype=np.complex128).reshape(-1, n_k, n_v, n_c)
    T = np.einsum("kmv,kmc,bkvc->mb", psi_v.conj(), psi_cq, X, optimize=True)
    W = V @ T
    U = np.einsum("kmv,kmc,mb->bkvc", psi_v, psi_cq.conj(), W, optimize=True)
    return (delta[None, :] * X.reshape(X.shape[0], -1) + U.reshape(X.shape[0], -1))


def orbital(psi_v, psi_cq, k, idx):
    """Orbital `idx` of slot k: idx < N_v is psi_{v k}, else the conduction orbital stored in slot k (momentum k+q)."""
    n_v = psi_v.shape[2]
    return psi_v[k][:, idx] if idx < n_v else psi_cq[k][:, idx - n_v]


def orbital_energy_sign(eps_v, eps_cq, k, idx):
    n_v = eps_v.shape[1]
    return (float(eps_v[k, idx]), 1) if idx < n_v else (float(eps_cq[k, idx - n_v]), -1)


def start_vector_printed(psi_v, psi_cq, V, kn, n_idx, km, m_idx):
    """P_{nmk}(q)_{v'c'k'} = (n k-q, m k | v'k', c'k'+q) as printed, PAPER.md:313:
    sum_{mu nu} conj(psi_m(mu)) psi_n(mu) V[mu, nu] K[nu, (k'v'c')]."""
    rho = np.conj(orbital(psi_v, psi_cq, km, m_idx)) * orbital(psi_v, psi_cq, kn, n_idx)
    w = V.T @ rho
    n_k, n_mu, n_v = psi_v.shape
    return np.einsum("kmv,kmc,m->kvc", psi_v.conj(), psi_cq, w, optimize=True).reshape(-1)


def start_vector(psi_v, psi_cq, V, kn, n_idx, km, m_idx):
    """The ket |P> that the resolvent form of PAPER.md:310 needs (reading Q20): the pole strengths are
    |W^s|^2 with W^s = sum_{v'c'k'} (n k-q, m k | v'k', c'k'+q) X^s_{v'c'k'} (TDA: Y = 0), a BILINEAR
    form in the printed elements, so |W^s|^2 = |<P|X^s>|^2 holds for |P> = conj(printed elements)
    = K^H (V rho~), rho~(mu) = psi_m(mu) conj(psi_n(mu)).  For real orbitals the two coincide."""
    return np.conj(start_vector_printed(psi_v, psi_cq, V, kn, n_idx, km, m_idx))


def lanczos_hermitian(apply_op, p, steps, reorth=False):
    """Standard Lanczos for a Hermitian matrix (Eq. 13): a_k = <q_k|A q_k> (real), b_{k+1} real > 0.
    Same conventions as gw_oracle.lanczos (steps = dimension of T, breakdown reading Q9)."""
    p = np.asarray(p, dtype=np.complex128)
    norm2 = float(np.vdot(p, p).real)
    alpha = np.zeros(steps)
    beta = np.zeros(steps)
    if norm2 == 0.0:
        return alpha, beta, norm2, 0
    q = p / np.sqrt(norm2)
    q_prev = np.zeros_like(q)
    b_prev = 0.0
    scale = 0.0
    basis = []
    length = steps
    for k in range(steps):
        if reorth:
            basis.append(q)
        w = apply_op(q)
        a = float(np.vdot(q, w).real)
        w = w - a * q - b_prev * q_prev
        if reorth:
            Q = np.array(basis)
            for _ in range(2):
                w = w - Q.T @ (Q.conj() @ w)
        b = float(np.sqrt(np.vdot(w, w).real))
        alpha[k] = a
        beta[k] = b
        scale = max(scale, abs(a) + b)
        if b <= BREAKDOWN_TOL * scale:
            beta[k] = 0.0
            length = k + 1
            break
        q_prev, q, b_prev = q, w / b, b
    return alpha, beta, norm2, length


def continued_fraction(alpha, beta, norm2, zeta, length):
    """Eq. 14, readings Q5/Q7, as in gw_oracle.continued_fraction."""
    L = int(length)
    zeta = np.asarray(zeta, dtype=np.complex128)
    if L == 0:
        return np.zeros_like(zeta)
    f = zeta - alpha[L - 1]
    for k in range(L - 2, -1, -1):
        f = zeta - alpha[k] - (beta[k] * beta[k]) / f
    return norm2 / f


def sigma_chain(alpha, beta, norm2, length, omega, eps_n, sgn_n, dlt, prefactor):
    """prefactor <P| 1/(omega - eps_{n k-q} + eta_n (A(q) - i delta)) |P>
    = -eta_n prefactor R_A(-eta_n z_n), z_n = omega - eps_n - i eta_n delta, R_A by Eq. 14."""
    z = np.asarray(omega, dtype=np.float64) - eps_n - 1j * sgn_n * dlt
    return -sgn_n * prefactor * continued_fraction(alpha, beta, norm2, -sgn_n * z, length)


def sigma_chain_exact(lam, X, P_printed, omega, eps_n, sgn_n, dlt, prefactor):
    """The pole sum of PAPER.md:288 in the TDA (Y = 0): prefactor sum_s |W^s|^2 / (omega - eps_n + eta_n (Omega_s - i delta)),
    W^s = sum_{v'c'k'} P_printed X^s (bilinear), (Omega_s, X^s) = eig(A(q))."""
    W = P_printed @ X
    den = np.asarray(omega)[:, None] - eps_n + sgn_n * (lam[None, :] - 1j * dlt)
    return prefactor * ((np.abs(W) ** 2)[None, :] / den).sum(axis=1)


def prefactor(n_q, n_k):
    """2 / (N_q N_k)."""
    return 2.0 / (n_q * n_k)


def run_chains(psi_v, psi_cq, eps_v, eps_cq, V, chains, steps, omega, dlt, n_q=1, reorth=False):
    """S1-S7 for chains [(kn, n_idx, km, m_idx), ...]: start vector, Hermitian Lanczos on A(q), Eq. 14."""
    delta = delta_kvc(eps_v, eps_cq)
    n_k = psi_v.shape[0]
    pf = prefactor(n_q, n_k)

    def op(x):
        return tda_matvec_factored(psi_v, psi_cq, V, delta, x[None])[0]

    n = len(chains)
    out = dict(alpha=np.zeros((n, steps)), beta=np.zeros((n, steps)), norm2=np.zeros(n),
               len=np.zeros(n, dtype=np.int32), sigma=np.zeros((n, len(omega)), dtype=np.complex128))
    for j, (kn, n_idx, km, m_idx) in enumerate(chains):
        P = start_vector(psi_v, psi_cq, V, int(kn), int(n_idx), int(km), int(m_idx))
        a, b, n2, ln = lanczos_hermitian(op, P, steps, reorth=reorth)
        e_n, sg = orbital_energy_sign(eps_v, eps_cq, int(kn), int(n_idx))
        out["alpha"][j], out["beta"][j], out["norm2"][j], out["len"][j] = a, b, n2, ln
        out["sigma"][j] = sigma_chain(a, b, n2, ln, omega, e_n, sg, dlt, pf)
    out["sigma_sum"] = out["sigma"].sum(axis=0)
    return out


def eig_tda(A):
    """(Omega_s(q), X^s(q)) of the Hermitian A(q)."""
    return sla.eigh(A)
