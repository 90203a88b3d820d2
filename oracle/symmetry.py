"""CPU oracle for the point-group symmetry blocks of the Casida matrix: "one can further exploit the point-group symmetries
to make the Casida matrix C block diagonal and simplify the calculation of matrix-vector products [64]".
SURVEY.md 8(f)-4, second part.

TEST INFRASTRUCTURE, NOT PRODUCT (same rules as gw_oracle.py): plain NumPy, no code shared with paper_2310_20103_b200/,
imports nothing from it.  Pins: tests/test_oracle_pins_symmetry.py (block diagonality of the FULL C of gw_oracle on the unfolded
problem, equality of every block with the reduced operator below, equality of Sigma with the unreduced run).

Reading (Q25; the paper gives only the sentence above and ref. [64]): an abelian point group G of order g whose
irreducible representations are one-dimensional and real (D_2h and its subgroups, what real-space codes use); an irrep is a bit
mask, its character at the element h (also a bit mask) is chi_Gamma(h) = (-1)^popcount(Gamma & h), products of irreps are XORs.
  - every orbital carries an irrep Gamma_n: phi_n(h r) = chi_{Gamma_n}(h) phi_n(r);
  - the pair v c transforms as gamma = Gamma_v ^ Gamma_c, (vc|v'c') vanishes between different gamma (the Coulomb operator is
    invariant), so C splits into g blocks and |P_nm> lives in the block gamma = Gamma_n ^ Gamma_m: a chain never leaves it;
  - with fitting points closed under G (wedge points r_mu and their images h r_mu) K[h mu, vc] = chi_gamma(h) K[mu, vc], so
    within block gamma
        K^T V K = Kw^T Vg Kw,   Kw = K on the wedge,   Vg[mu, nu] = g sum_h chi_gamma(h) V(r_mu, h r_nu)
    (V(g mu, g' nu) = V(mu, g^-1 g' nu) for an invariant kernel): the block operator is a Casida operator on N_mu / g points
    and ~ N_vc / g pairs -- a factor ~ g^2 fewer flop per chain-step in the two Khatri-Rao contractions.
Pairs of block gamma are ordered by the irrep a of v (ascending), then v, then c over the irrep a ^ gamma.
"""
from __future__ import annotations

import numpy as np

from . import gw_oracle as orc


def character(gamma, h):
    """chi_gamma(h) = (-1)^popcount(gamma & h)."""
    return -1.0 if bin(int(gamma) & int(h)).count("1") & 1 else 1.0


def unfold_orbitals(phi_w, irrep, g):
    """Orbital values at all g n_w points from the wedge values: phi(h r_mu) = chi_Gamma(h) phi(r_mu); row h n_w + mu."""
    n_w, n = phi_w.shape
    out = np.empty((g * n_w, n))
    for h in range(g):
        ch = np.array([character(irrep[j], h) for j in range(n)])
        out[h * n_w:(h + 1) * n_w] = phi_w * ch[None, :]
    return out


def pair_block(irrep_v, irrep_c, gamma):
    """(v indices, c indices) of the pairs of block gamma in block order."""
    vs, cs = [], []
    for v in range(len(irrep_v)):
        for c in range(len(irrep_c)):
            if int(irrep_v[v]) ^ int(irrep_c[c]) == int(gamma):
                vs.append(v)
                cs.append(c)
    return np.array(vs, dtype=np.int64), np.array(cs, dtype=np.int64)


def reduced_kernel(V_wf, gamma):
    """Vg[mu, nu] = g sum_h chi_gamma(h) V(r_mu, h r_nu); V_wf [n_w][g][n_w]."""
    g = V_wf.shape[1]
    out = np.zeros((V_wf.shape[0], V_wf.shape[2]))
    for h in range(g):
        out += character(gamma, h) * V_wf[:, h, :]
    return g * out


def block_delta(eps_v, eps_c, vs, cs):
    return np.asarray(eps_c)[cs] - np.asarray(eps_v)[vs]


def block_pair_matrix(phi_v_w, phi_c_w, vs, cs):
    """Kw[mu, j] = phi_v(r_mu) phi_c(r_mu) for the pairs j of the block, on the wedge."""
    return phi_v_w[:, vs] * phi_c_w[:, cs]


def casida_block_dense(phi_v_w, phi_c_w, eps_v, eps_c, irrep_v, irrep_c, V_wf, gamma):
    """C restricted to block gamma = diag(Delta^2) + 2 sqrt(Delta) Kw^T Vg Kw sqrt(Delta)  (Eq. 4 with the reduction above)."""
    vs, cs = pair_block(irrep_v, irrep_c, gamma)
    d = block_delta(eps_v, eps_c, vs, cs)
    Kw = block_pair_matrix(phi_v_w, phi_c_w, vs, cs)
    sq = np.sqrt(d)
    return np.diag(d * d) + 2.0 * (sq[:, None] * (Kw.T @ (reduced_kernel(V_wf, gamma) @ Kw)) * sq[None, :])


def block_matvec(phi_v_w, phi_c_w, eps_v, eps_c, irrep_v, irrep_c, V_wf, gamma, X):
    """Y = C_gamma X for X [nvec, n_pairs(gamma)] without forming Kw: one Khatri-Rao contraction per irrep a of v
    (v in a, c in a ^ gamma), summed into T; then Vg; then back, block by block."""
    g = V_wf.shape[1]
    X = np.atleast_2d(np.asarray(X, dtype=np.float64))
    vs, cs = pair_block(irrep_v, irrep_c, gamma)
    d = block_delta(eps_v, eps_c, vs, cs)
    sq = np.sqrt(d)
    xs = X * sq[None, :]
    T = np.zeros((phi_v_w.shape[0], X.shape[0]))
    off = 0
    spans = []
    for a in range(g):
        va = np.nonzero(np.asarray(irrep_v) == a)[0]
        cb = np.nonzero(np.asarray(irrep_c) == (a ^ int(gamma)))[0]
        n = len(va) * len(cb)
        spans.append((off, va, cb))
        if n:
            xa = xs[:, off:off + n].reshape(-1, len(va), len(cb))
            T += np.einsum("mv,mc,bvc->mb", phi_v_w[:, va], phi_c_w[:, cb], xa, optimize=True)
        off += n
    W = reduced_kernel(V_wf, gamma) @ T
    U = np.zeros_like(X)
    for (o, va, cb) in spans:
        n = len(va) * len(cb)
        if n:
            U[:, o:o + n] = np.einsum("mv,mc,mb->bvc", phi_v_w[:, va], phi_c_w[:, cb], W, optimize=True).reshape(X.shape[0], n)
    return (d * d)[None, :] * X + 2.0 * sq[None, :] * U


def orbital_w(phi_v_w, phi_c_w, idx):
    n_v = phi_v_w.shape[1]
    return phi_v_w[:, idx] if idx < n_v else phi_c_w[:, idx - n_v]


def orbital_irrep(irrep_v, irrep_c, idx):
    n_v = len(irrep_v)
    return int(irrep_v[idx]) if idx < n_v else int(irrep_c[idx - n_v])


def start_vector_block(phi_v_w, phi_c_w, eps_v, eps_c, irrep_v, irrep_c, V_wf, n_idx, m_idx):
    """(gamma, P): P_j = sqrt(Delta_j) (nm|vc)_j on the pairs j of the block gamma = Gamma_n ^ Gamma_m, with
    (nm|vc) = Kw^T Vg rho_w, rho_w = phi_n phi_m on the wedge (PAPER.md:67 with the reduction)."""
    gamma = orbital_irrep(irrep_v, irrep_c, n_idx) ^ orbital_irrep(irrep_v, irrep_c, m_idx)
    vs, cs = pair_block(irrep_v, irrep_c, gamma)
    rho = orbital_w(phi_v_w, phi_c_w, n_idx) * orbital_w(phi_v_w, phi_c_w, m_idx)
    w = reduced_kernel(V_wf, gamma) @ rho
    P = np.sqrt(block_delta(eps_v, eps_c, vs, cs)) * (block_pair_matrix(phi_v_w, phi_c_w, vs, cs).T @ w)
    return gamma, P


def run_chains_sym(phi_v_w, phi_c_w, eps_v, eps_c, irrep_v, irrep_c, V_wf, n_idx, m_idx, steps, omega, dlt, reorth=False):
    """S1-S7 chain by chain inside the symmetry blocks (direct mode): Lanczos on C_gamma from |P_nm>, Eq. 11 on the Ritz
    pairs (gw_oracle.sigma_direct)."""
    n = len(n_idx)
    out = dict(alpha=np.zeros((n, steps)), beta=np.zeros((n, steps)), norm2=np.zeros(n), len=np.zeros(n, dtype=np.int32),
               gamma=np.zeros(n, dtype=np.int32), sigma=np.zeros((n, len(omega)), dtype=np.complex128))
    for j in range(n):
        gamma, P = start_vector_block(phi_v_w, phi_c_w, eps_v, eps_c, irrep_v, irrep_c, V_wf, int(n_idx[j]), int(m_idx[j]))

        def op(x, gamma=gamma):
            return block_matvec(phi_v_w, phi_c_w, eps_v, eps_c, irrep_v, irrep_c, V_wf, gamma, x[None])[0]

        a, b, n2, ln = orc.lanczos(op, P, steps, reorth=reorth)
        e_n, sg = orc.orbital_energy_sign(eps_v, eps_c, int(n_idx[j]))
        out["alpha"][j], out["beta"][j], out["norm2"][j], out["len"][j], out["gamma"][j] = a, b, n2, ln, gamma
        out["sigma"][j] = orc.sigma_direct(a, b, n2, ln, omega, e_n, sg, dlt)
    out["sigma_sum"] = out["sigma"].sum(axis=0)
    return out
