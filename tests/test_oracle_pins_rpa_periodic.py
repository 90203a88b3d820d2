"""Pins of oracle/rpa_periodic.py (complex orbitals, full RPA: the pole sum of PAPER.md:286-304 and the pseudo-Hermitian
Lanczos of PAPER.md:159, reading Q24) against what the paper and the mathematics fix: the printed block structure of the
eigenvectors, a 1x1 closed form, the real one-k-point limit (= Eq. 7 of the main text through gw_oracle), the B = 0 limit
(= the Tamm-Dancoff oracle), exactness of the Lanczos quadrature at full length, the moment identity, gauge invariance."""
import numpy as np
import scipy.linalg as sla

from oracle import gw_oracle as orc
from oracle import rpa_periodic as rpa
from oracle import tda_periodic as tdp
from paper_2310_20103_b200 import synth

DLT = 0.1


def _dense(p):
    delta = tdp.delta_kvc(p.eps_v, p.eps_cq)
    K = tdp.pair_matrix(p.psi_v, p.psi_cq)
    A = tdp.tda_dense(delta, K, p.V)
    B = tdp.coupling_B(K, p.V)
    return delta, K, A, B


def test_omega_hat_factored_equals_dense_and_is_positive_definite():
    p = synth.make_periodic(3, 2, 4, 12, seed=21)
    delta, K, A, B = _dense(p)
    Oh = rpa.omega_hat_dense(A, B)
    assert np.abs(Oh - Oh.conj().T).max() <= 1e-13 * np.abs(Oh).max()
    assert sla.eigvalsh(Oh).min() >= delta.min() * (1 - 1e-12)              # Omega^ = diag(Delta) + [K^H; K^T] V [K, K^*] >= Delta
    X = synth.random_complex_block(delta.size, 3, seed=2)
    Y = synth.random_complex_block(delta.size, 3, seed=3)
    X1, Y1 = rpa.omega_hat_factored(p.psi_v, p.psi_cq, p.V, delta, X, Y)
    ref = np.concatenate([X, Y], axis=1) @ Oh.T
    n = delta.size
    assert np.abs(X1 - ref[:, :n]).max() <= 1e-13 * np.abs(ref).max()
    assert np.abs(Y1 - ref[:, n:]).max() <= 1e-13 * np.abs(ref).max()


def test_eigenvector_block_structure_as_printed():
    """C^RPA [[X, Y^*], [Y, X^*]] = [[X, Y^*], [Y, X^*]] diag(Omega, -Omega); plus the normalisation
    X^H X - Y^H Y = 1, X^T Y - Y^T X = 0 and the completeness that the quadrature argument uses."""
    p = synth.make_periodic(2, 2, 3, 10, seed=22)
    delta, K, A, B = _dense(p)
    om, X, Y = rpa.rpa_eig(A, B)
    n = delta.size
    C = tdp.casida_rpa_block(A, B)
    Vp = np.concatenate([X, Y], axis=0)
    Vm = np.concatenate([Y.conj(), X.conj()], axis=0)
    assert np.abs(C @ Vp - Vp * om[None, :]).max() <= 1e-10 * om.max()
    assert np.abs(C @ Vm + Vm * om[None, :]).max() <= 1e-10 * om.max()
    F = np.diag(np.concatenate([np.ones(n), -np.ones(n)]))
    assert np.abs(Vp.conj().T @ F @ Vp - np.eye(n)).max() <= 1e-9
    assert np.abs(Vp.conj().T @ F @ Vm).max() <= 1e-9
    # resolution of the identity in the Omega^ inner product: sum_s v_s v_s^H Omega^ / |lambda_s| = 1
    Oh = rpa.omega_hat_dense(A, B)
    allv = np.concatenate([Vp, Vm], axis=1)
    lam = np.concatenate([om, om])
    assert np.abs((allv / lam[None, :]) @ allv.conj().T @ Oh - np.eye(2 * n)).max() <= 1e-8


def test_one_by_one_closed_form():
    """N = 1: A = a (real), B = b (complex): Omega = sqrt(a^2 - |b|^2), Y = -(a - Omega) X / b, |X|^2 = 1 / (1 - (a - Omega)^2 / |b|^2),
    W = P1 X + P2 Y.  Checks the exact pole sum AND the one-step... two-step Lanczos (L = 2N = 2 is the full space)."""
    p = synth.make_periodic(1, 1, 1, 6, seed=23, n_chains=2)
    delta, K, A, B = _dense(p)
    a, b = A[0, 0].real, B[0, 0]
    om = np.sqrt(a * a - abs(b) ** 2)
    x2 = 1.0 / (1.0 - (a - om) ** 2 / abs(b) ** 2)
    r = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, 2, p.omega, DLT, n_q=3, reorth=True)
    for j, (kn, n_idx, km, m_idx) in enumerate(p.chains):
        P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
        w2 = x2 * abs(P1[0] - P2[0] * (a - om) / b) ** 2
        e_n, sg = tdp.orbital_energy_sign(p.eps_v, p.eps_cq, kn, n_idx)
        ref = (2.0 / 3.0) * w2 / (p.omega - e_n + sg * (om - 1j * DLT))
        omx, X, Y = rpa.rpa_eig(A, B)
        ex = rpa.sigma_chain_exact_rpa(omx, X, Y, P1, P2, p.omega, e_n, sg, DLT, 2.0 / 3.0)
        assert abs(omx[0] - om) <= 1e-12 * om
        assert np.abs(ex - ref).max() <= 1e-11 * np.abs(ref).max()
        assert np.abs(r["sigma"][j] - ref).max() <= 1e-10 * np.abs(ref).max()


def test_real_one_k_point_limit_is_eq7_of_the_main_text():
    """Real orbitals, N_k = 1: the printed periodic pole sum (X, Y of the 2N x 2N problem) equals prefactor x Eq. 7
    (eigenpairs of C = (A-B)^{1/2}(A+B)(A-B)^{1/2}, |P> = (nm|vc) sqrt(Delta)) computed by gw_oracle: two independent
    routes through the paper (SM section 1 against main text Eq. 1-9)."""
    p = synth.make_periodic(1, 3, 4, 14, seed=24, real_orbitals=True)
    delta, K, A, B = _dense(p)
    om, X, Y = rpa.rpa_eig(A, B)
    phi_v, phi_c = p.psi_v[0].real, p.psi_cq[0].real
    d_real = orc.delta_vc(p.eps_v[0], p.eps_cq[0])
    C = orc.casida_dense(d_real, orc.coupling_dense(orc.khatri_rao(phi_v, phi_c), p.V))
    lam, Z = orc.eig_casida(C)
    assert np.abs(np.sqrt(lam) - om).max() <= 1e-10 * om.max()
    pf = tdp.prefactor(1, 1)
    for (kn, n_idx, km, m_idx) in p.chains:
        P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
        e_n, sg = tdp.orbital_energy_sign(p.eps_v, p.eps_cq, kn, n_idx)
        ex = rpa.sigma_chain_exact_rpa(om, X, Y, P1, P2, p.omega, e_n, sg, DLT, pf)
        P = orc.start_vector(phi_v, phi_c, p.V, d_real, int(n_idx), int(m_idx))
        ref = pf * orc.sigma_exact_eq7(lam, Z, P, p.omega, e_n, sg, DLT)
        assert np.abs(ex - ref).max() <= 1e-9 * np.abs(ref).max()
    # and the Lanczos route against gw_oracle's direct mode at full length
    r = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains[:2], 2 * delta.size, p.omega, DLT, reorth=True)
    rr = orc.run_chains(phi_v, phi_c, p.eps_v[0], p.eps_cq[0], p.V, p.chains[:2, 1], p.chains[:2, 3], delta.size, p.omega, DLT,
                        reorth=True)
    assert np.abs(r["sigma"] - pf * rr["sigma"]).max() <= 1e-8 * np.abs(rr["sigma"]).max()


def test_B_zero_limit_is_the_tamm_dancoff_oracle():
    p = synth.make_periodic(2, 2, 3, 10, seed=25)
    delta, K, A, B = _dense(p)
    om, X, Y = rpa.rpa_eig(A, np.zeros_like(B))
    lam, Xt = tdp.eig_tda(A)
    assert np.abs(om - lam).max() <= 1e-10 * lam.max() and np.abs(Y).max() <= 1e-10
    P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, 1, 3, 0, 1)
    ex = rpa.sigma_chain_exact_rpa(om, X, Y, P1, P2, p.omega, -1.0, -1, DLT, 1.0)
    ref = tdp.sigma_chain_exact(lam, Xt, P1, p.omega, -1.0, -1, DLT, 1.0)
    assert np.abs(ex - ref).max() <= 1e-9 * np.abs(ref).max()
    assert np.abs(P1 - tdp.start_vector_printed(p.psi_v, p.psi_cq, p.V, 1, 3, 0, 1)).max() == 0.0


def test_printed_elements_brute_force():
    """P1, P2 of PAPER.md:290 as explicit double sums over the fitting points."""
    p = synth.make_periodic(2, 2, 2, 7, seed=26)
    kn, n_idx, km, m_idx = 1, 2, 0, 1
    P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
    psi_n = tdp.orbital(p.psi_v, p.psi_cq, kn, n_idx)
    psi_m = tdp.orbital(p.psi_v, p.psi_cq, km, m_idx)
    for (k, v, c) in [(0, 0, 1), (1, 1, 0)]:
        a1 = a2 = 0.0
        for mu in range(p.n_mu):
            for nu in range(p.n_mu):
                bra = np.conj(psi_m[mu]) * psi_n[mu] * p.V[mu, nu]
                a1 += bra * p.psi_cq[k, nu, c] * np.conj(p.psi_v[k, nu, v])          # (.., .. | v'k', c'k'+q)
                a2 += bra * p.psi_v[k, nu, v] * np.conj(p.psi_cq[k, nu, c])          # (.., .. | c'k'+q, v'k')
        j = (k * p.n_v + v) * p.n_c + c
        assert abs(P1[j] - a1) <= 1e-12 * abs(a1) and abs(P2[j] - a2) <= 1e-12 * abs(a2)


def test_full_length_lanczos_reproduces_the_printed_pole_sum():
    """Reading Q24: at L = 2N with reorthogonalisation the Ritz quadrature restricted to theta_i > 0 IS the printed pole sum
    (complex orbitals); with a wrong start vector (no F, or no conjugation) it is not."""
    p = synth.make_periodic(2, 2, 3, 10, seed=27)
    delta, K, A, B = _dense(p)
    Oh = rpa.omega_hat_dense(A, B)
    n = delta.size
    om, X, Y = rpa.rpa_eig(A, B)
    pf = tdp.prefactor(1, p.n_k)

    def op(x, y):
        r = Oh @ np.concatenate([x, y])
        return r[:n], r[n:]

    for (kn, n_idx, km, m_idx) in [(0, 0, 0, 1), (1, 3, 0, 1)]:
        P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
        e_n, sg = tdp.orbital_energy_sign(p.eps_v, p.eps_cq, kn, n_idx)
        exact = rpa.sigma_chain_exact_rpa(om, X, Y, P1, P2, p.omega, e_n, sg, DLT, pf)
        u1, u2 = rpa.start_vector_rpa(P1, P2)
        a, b, n2, ln = rpa.lanczos_pseudo_hermitian(op, u1, u2, 2 * n, reorth=True)
        th, w = rpa.ritz(a, b, ln)
        assert abs(w.sum() - 1.0) <= 1e-10
        pos = np.sort(th[th > 0])
        assert np.abs(pos - om).max() <= 1e-8 * om.max()                          # Ritz values = +-Omega_s
        sig = rpa.sigma_chain_rpa(a, b, n2, ln, p.omega, e_n, sg, DLT, pf)
        assert np.abs(sig - exact).max() <= 1e-8 * np.abs(exact).max()
        for (w1, w2) in [(np.conj(P1), np.conj(P2)), (P1, -P2)]:
            a, b, n2, ln = rpa.lanczos_pseudo_hermitian(op, w1, w2, 2 * n, reorth=True)
            wrong = rpa.sigma_chain_rpa(a, b, n2, ln, p.omega, e_n, sg, DLT, pf)
            assert np.abs(wrong - exact).max() > 1e-2 * np.abs(exact).max()


def test_moments_of_the_tridiagonal_in_the_omega_hat_inner_product():
    """<u,u>_O e_1^T T^j e_1 = u^H Omega^ H^j u for j <= 2L-1 (H = F Omega^)."""
    p = synth.make_periodic(2, 2, 3, 10, seed=28)
    delta, K, A, B = _dense(p)
    Oh = rpa.omega_hat_dense(A, B)
    H = tdp.casida_rpa_block(A, B)
    n = delta.size
    P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, 0, 0, 0, 1)
    u1, u2 = rpa.start_vector_rpa(P1, P2)
    L = 4
    a, b, n2, ln = rpa.lanczos_pseudo_hermitian(lambda x, y: tuple(np.split(Oh @ np.concatenate([x, y]), 2)), u1, u2, L)
    u = np.concatenate([u1, u2])
    assert abs(n2 - np.vdot(u, Oh @ u).real) <= 1e-13 * n2
    T = np.diag(a[:L]) + np.diag(b[:L - 1], 1) + np.diag(b[:L - 1], -1)
    v, Tj = u.copy(), np.eye(L)
    for j in range(2 * L):
        m = np.vdot(u, Oh @ v)
        assert abs(m.imag) <= 1e-10 * abs(m) + 1e-14
        assert abs(n2 * Tj[0, 0] - m.real) <= 1e-10 * max(abs(m.real), n2), j
        v = H @ v
        Tj = Tj @ T


def test_gauge_invariance():
    """A random phase on every orbital leaves alpha, beta, <u,u>_O and Sigma unchanged (catches a misplaced conjugate)."""
    p = synth.make_periodic(2, 2, 3, 10, seed=29)
    rng = np.random.default_rng(4)
    pv = np.exp(2j * np.pi * rng.random((p.n_k, 1, p.n_v)))
    pc = np.exp(2j * np.pi * rng.random((p.n_k, 1, p.n_c)))
    r0 = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, 8, p.omega, DLT, reorth=True)
    r1 = rpa.run_chains_rpa(p.psi_v * pv, p.psi_cq * pc, p.eps_v, p.eps_cq, p.V, p.chains, 8, p.omega, DLT, reorth=True)
    assert np.abs(r0["alpha"] - r1["alpha"]).max() <= 1e-10 * np.abs(r0["alpha"]).max()
    assert np.abs(r0["beta"] - r1["beta"]).max() <= 1e-10 * np.abs(r0["alpha"]).max()
    assert np.abs(r0["norm2"] - r1["norm2"]).max() <= 1e-12 * np.abs(r0["norm2"]).max()
    assert np.abs(r0["sigma"] - r1["sigma"]).max() <= 1e-9 * np.abs(r0["sigma"]).max()


def test_short_lanczos_converges_towards_the_pole_sum():
    """The quadrature error falls with L (broadened spectrum, delta = 0.5 eV): L = 24 is closer to the exact sum than L = 6."""
    p = synth.make_periodic(2, 2, 4, 12, seed=30)
    delta, K, A, B = _dense(p)
    om, X, Y = rpa.rpa_eig(A, B)
    kn, n_idx, km, m_idx = p.chains[0]
    P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
    e_n, sg = tdp.orbital_energy_sign(p.eps_v, p.eps_cq, kn, n_idx)
    exact = rpa.sigma_chain_exact_rpa(om, X, Y, P1, P2, p.omega, e_n, sg, 0.5, 1.0)
    errs = []
    for L in (6, 24):
        r = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains[:1], L, p.omega, 0.5, n_q=1, reorth=True)
        errs.append(np.abs(r["sigma"][0] - exact).max())
    assert errs[1] < 0.2 * errs[0]


def test_resolvent_of_the_pseudo_hermitian_matrix_by_eq14():
    """<u|(zeta - H)^-1|u>_O: the continued fraction of the full-length tridiagonal equals the dense solve, and its partial
    fractions carry BOTH branches: sum_s |lambda_s| |d^H v_s|^2 / (zeta - lambda_s) over +Omega_s (v = [X; Y]) and -Omega_s
    (v = [Y^*; X^*])."""
    p = synth.make_periodic(2, 2, 3, 10, seed=31)
    delta, K, A, B = _dense(p)
    n = delta.size
    Oh = rpa.omega_hat_dense(A, B)
    P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, 0, 0, 0, 1)
    u1, u2 = rpa.start_vector_rpa(P1, P2)
    a, b, n2, ln = rpa.lanczos_pseudo_hermitian(lambda x, y: tuple(np.split(Oh @ np.concatenate([x, y]), 2)), u1, u2, 2 * n,
                                                reorth=True)
    zeta = np.array([3.0 + 0.5j, -7.0 + 0.2j, 0.1j, 25.0 - 1.0j])
    cf = rpa.resolvent_chain(a, b, n2, ln, zeta)
    ex = rpa.resolvent_exact_rpa(A, B, u1, u2, zeta)
    assert np.abs(cf - ex).max() <= 1e-9 * np.abs(ex).max()
    om, X, Y = rpa.rpa_eig(A, B)
    d = np.conj(np.concatenate([P1, P2]))
    wp = np.abs(d.conj() @ np.concatenate([X, Y], axis=0)) ** 2
    wm = np.abs(d.conj() @ np.concatenate([Y.conj(), X.conj()], axis=0)) ** 2
    pf = (om[None, :] * wp[None, :] / (zeta[:, None] - om[None, :])).sum(axis=1) \
        + (om[None, :] * wm[None, :] / (zeta[:, None] + om[None, :])).sum(axis=1)
    assert np.abs(pf - ex).max() <= 1e-9 * np.abs(ex).max()
