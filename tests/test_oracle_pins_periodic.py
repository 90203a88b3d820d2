"""Pins of oracle/tda_periodic.py (complex-orbital Tamm-Dancoff variant) against what the
paper and the mathematics fix: structure of A(q) and B(q), the block spectrum of C^TD, the printed pole sum by full
diagonalisation, a 1x1 closed form, gauge invariance, and the real one-k-point limit (gw_oracle's TDA functions)."""
import numpy as np
import scipy.linalg as sla

from oracle import gw_oracle as orc
from oracle import tda_periodic as tdp
from paper_2310_20103_b200 import synth

DLT = 0.1


def _dense(p):
    delta = tdp.delta_kvc(p.eps_v, p.eps_cq)
    K = tdp.pair_matrix(p.psi_v, p.psi_cq)
    A = tdp.tda_dense(delta, K, p.V)
    return delta, K, A


def test_A_hermitian_B_symmetric_and_brute_force_integrals():
    """A(q) Hermitian, B(q) symmetric; entries against the printed integrals written as explicit sums."""
    p = synth.make_periodic(2, 2, 3, 10, seed=5)
    delta, K, A = _dense(p)
    B = tdp.coupling_B(K, p.V)
    assert np.abs(A - A.conj().T).max() <= 1e-13 * np.abs(A).max()
    assert np.abs(B - B.T).max() <= 1e-13 * np.abs(B).max()
    assert np.abs(A.imag).max() > 1e-3 * np.abs(A).max()                    # genuinely complex
    n_v, n_c = p.n_v, p.n_c

    def flat(k, v, c):
        return (k * n_v + v) * n_c + c

    for (k, v, c, k2, v2, c2) in [(0, 0, 0, 1, 1, 2), (1, 0, 2, 1, 0, 2), (0, 1, 1, 0, 0, 2)]:
        acc_a = acc_b = 0.0
        for mu in range(p.n_mu):
            for nu in range(p.n_mu):
                bra = np.conj(p.psi_cq[k, mu, c]) * p.psi_v[k, mu, v]                     # psi*_{ck+q}(r) psi_{vk}(r)
                acc_a += bra * p.V[mu, nu] * p.psi_cq[k2, nu, c2] * np.conj(p.psi_v[k2, nu, v2])
                acc_b += bra * p.V[mu, nu] * np.conj(p.psi_cq[k2, nu, c2]) * p.psi_v[k2, nu, v2]
        i, j = flat(k, v, c), flat(k2, v2, c2)
        assert abs(A[i, j] - (acc_a + (delta[i] if i == j else 0.0))) <= 1e-12 * abs(A[i, j])
        assert abs(B[i, j] - acc_b) <= 1e-12 * abs(B[i, j])


def test_td_block_spectrum_and_rpa_block_structure():
    """C^TD = [[A, 0], [0, -A^*]] has the eigenvalues +-eig(A); the RPA block matrix has a
    spectrum symmetric about zero."""
    p = synth.make_periodic(2, 2, 2, 8, seed=6)
    delta, K, A = _dense(p)
    lam = sla.eigvalsh(A)
    ev = np.sort(sla.eigvals(tdp.casida_td_block(A)).real)
    assert np.abs(ev - np.sort(np.concatenate([-lam, lam]))).max() <= 1e-10 * np.abs(lam).max()
    er = sla.eigvals(tdp.casida_rpa_block(A, tdp.coupling_B(K, p.V)))
    assert np.abs(er.imag).max() <= 1e-8 * np.abs(er).max()
    er = np.sort(er.real)
    assert np.abs(er + er[::-1]).max() <= 1e-9 * np.abs(er).max()


def test_factored_matvec_equals_dense():
    p = synth.make_periodic(3, 2, 4, 12, seed=7)
    delta, K, A = _dense(p)
    X = synth.random_complex_block(delta.size, 3)
    Y = tdp.tda_matvec_factored(p.psi_v, p.psi_cq, p.V, delta, X)
    ref = X @ A.T
    assert np.abs(Y - ref).max() <= 1e-13 * np.abs(ref).max()


def test_resolvent_needs_the_conjugated_printed_vector():
    """Reading Q20.  Full-length reorthogonalised Lanczos from |P> = conj(printed elements) reproduces the printed pole
    sum sum_s |W^s|^2 / (...) with the bilinear W^s = sum P_printed X^s (TDA); started from the
    printed elements themselves it does not (complex orbitals)."""
    p = synth.make_periodic(2, 2, 3, 10, seed=8)
    delta, K, A = _dense(p)
    lam, X = tdp.eig_tda(A)
    pf = tdp.prefactor(1, p.n_k)
    for (kn, n_idx, km, m_idx) in [(0, 0, 0, 1), (1, 3, 0, 1)]:
        Pp = tdp.start_vector_printed(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
        e_n, sg = tdp.orbital_energy_sign(p.eps_v, p.eps_cq, kn, n_idx)
        exact = tdp.sigma_chain_exact(lam, X, Pp, p.omega, e_n, sg, DLT, pf)
        a, b, n2, ln = tdp.lanczos_hermitian(lambda x: A @ x, np.conj(Pp), delta.size, reorth=True)
        sig = tdp.sigma_chain(a, b, n2, ln, p.omega, e_n, sg, DLT, pf)
        assert np.abs(sig - exact).max() <= 1e-10 * np.abs(exact).max()
        a, b, n2, ln = tdp.lanczos_hermitian(lambda x: A @ x, Pp, delta.size, reorth=True)
        wrong = tdp.sigma_chain(a, b, n2, ln, p.omega, e_n, sg, DLT, pf)
        assert np.abs(wrong - exact).max() > 1e-2 * np.abs(exact).max()
        # the direct resolvent <P| (omega - eps + eta (A - i delta))^-1 |P> of PAPER.md:310 by a dense solve
        P = np.conj(Pp)
        for w in p.omega[::25]:
            M = (w - e_n) * np.eye(delta.size) + sg * (A - 1j * DLT * np.eye(delta.size))
            direct = pf * np.vdot(P, np.linalg.solve(M, P))
            k = int(np.argmin(np.abs(p.omega - w)))
            assert abs(direct - exact[k]) <= 1e-10 * abs(exact[k])


def test_one_by_one_closed_form():
    """N_k = N_v = N_c = 1: A = Delta + rho^H V rho (real), Sigma = (2 / (N_q N_k)) |P|^2 / (omega - eps_n + eta_n (A - i delta))."""
    p = synth.make_periodic(1, 1, 1, 6, seed=9, n_chains=2)
    delta, K, A = _dense(p)
    rho = np.conj(p.psi_v[0, :, 0]) * p.psi_cq[0, :, 0]
    a00 = (p.eps_cq[0, 0] - p.eps_v[0, 0]) + np.vdot(rho, p.V @ rho).real
    assert abs(A[0, 0] - a00) <= 1e-13 * abs(a00) and abs(A[0, 0].imag) <= 1e-15
    r = tdp.run_chains(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, 1, p.omega, DLT, n_q=3)
    for j, (kn, n_idx, km, m_idx) in enumerate(p.chains):
        Pp = tdp.start_vector_printed(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
        e_n, sg = tdp.orbital_energy_sign(p.eps_v, p.eps_cq, kn, n_idx)
        ref = (2.0 / 3.0) * abs(Pp[0]) ** 2 / (p.omega - e_n + sg * (a00 - 1j * DLT))
        assert abs(r["alpha"][j, 0] - a00) <= 1e-12 * a00
        assert np.abs(r["sigma"][j] - ref).max() <= 1e-12 * np.abs(ref).max()


def test_gauge_invariance():
    """A random phase on every orbital changes A by a diagonal unitary similarity and |P> by the same unitary times a
    global phase: alpha, beta, <P|P> and Sigma do not change.  Catches a misplaced complex conjugate anywhere."""
    p = synth.make_periodic(2, 2, 3, 10, seed=10)
    rng = np.random.default_rng(3)
    pv = np.exp(2j * np.pi * rng.random((p.n_k, 1, p.n_v)))
    pc = np.exp(2j * np.pi * rng.random((p.n_k, 1, p.n_c)))
    r0 = tdp.run_chains(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, 8, p.omega, DLT, reorth=True)
    r1 = tdp.run_chains(p.psi_v * pv, p.psi_cq * pc, p.eps_v, p.eps_cq, p.V, p.chains, 8, p.omega, DLT, reorth=True)
    assert np.abs(r0["alpha"] - r1["alpha"]).max() <= 1e-10 * np.abs(r0["alpha"]).max()
    assert np.abs(r0["beta"] - r1["beta"]).max() <= 1e-10 * np.abs(r0["alpha"]).max()
    assert np.abs(r0["norm2"] - r1["norm2"]).max() <= 1e-12 * np.abs(r0["norm2"]).max()
    assert np.abs(r0["sigma"] - r1["sigma"]).max() <= 1e-9 * np.abs(r0["sigma"]).max()


def test_real_one_k_point_limit_is_the_real_tda_oracle():
    """Real orbitals, N_k = 1: A(q) is gw_oracle.tda_dense, the start vector is gw_oracle.tda_start_vector, and Sigma
    is prefactor x gw_oracle.run_chains_tda (whose reading Q19 keeps prefactor 1)."""
    p = synth.make_periodic(1, 3, 4, 14, seed=11, real_orbitals=True)
    delta, K, A = _dense(p)
    phi_v, phi_c = p.psi_v[0].real, p.psi_cq[0].real
    d_real = orc.delta_vc(p.eps_v[0], p.eps_cq[0])
    A_real = orc.tda_dense(d_real, orc.coupling_dense(orc.khatri_rao(phi_v, phi_c), p.V))
    assert np.abs(A.imag).max() == 0.0 and np.abs(A.real - A_real).max() <= 1e-13 * np.abs(A_real).max()
    n_idx, m_idx = p.chains[:, 1], p.chains[:, 3]
    rr = orc.run_chains_tda(phi_v, phi_c, p.eps_v[0], p.eps_cq[0], p.V, n_idx, m_idx, 9, p.omega, DLT, reorth=True)
    rc = tdp.run_chains(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, 9, p.omega, DLT, reorth=True)
    assert np.abs(rc["alpha"] - rr["alpha"]).max() <= 1e-10 * np.abs(rr["alpha"]).max()
    assert np.abs(rc["beta"] - rr["beta"]).max() <= 1e-10 * np.abs(rr["alpha"]).max()
    assert np.abs(rc["sigma"] - tdp.prefactor(1, 1) * rr["sigma"]).max() <= 1e-9 * np.abs(rr["sigma"]).max()


def test_moments_of_the_tridiagonal():
    """e_1^T T^j e_1 = <P|A^j|P> / <P|P> for j <= 2L-1 (complex Hermitian A)."""
    p = synth.make_periodic(2, 2, 3, 10, seed=12)
    delta, K, A = _dense(p)
    P = tdp.start_vector(p.psi_v, p.psi_cq, p.V, 0, 0, 0, 1)
    L = 4
    a, b, n2, ln = tdp.lanczos_hermitian(lambda x: A @ x, P, L)
    T = np.diag(a[:L]) + np.diag(b[:L - 1], 1) + np.diag(b[:L - 1], -1)
    s = P / np.sqrt(n2)
    v, Tj = s.copy(), np.eye(L)
    for j in range(2 * L):
        m_A = np.vdot(s, v).real
        assert abs(Tj[0, 0] - m_A) <= 1e-11 * max(abs(m_A), 1.0), j
        v = A @ v
        Tj = Tj @ T
