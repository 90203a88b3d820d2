"""Pins for oracle/gw_oracle.py: every oracle function is checked
against something other than itself -- the paper's defining equations evaluated by
brute force or by a library eigen-solver, closed forms, and algebraic invariants.
CPU only; runs in seconds on config 0 (N_vc = 192) and smaller inputs."""
import numpy as np
import pytest
import scipy.linalg as sla

from oracle import gw_oracle as orc
from paper_2310_20103_b200 import synth

DLT = 0.1


@pytest.fixture(scope="module")
def dense0(cfg0):
    p = cfg0
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    K = orc.khatri_rao(p.phi_v, p.phi_c)
    Kt = orc.coupling_dense(K, p.V)
    C = orc.casida_dense(delta, Kt)
    lam, Z = sla.eigh(C)
    return dict(delta=delta, K=K, Kt=Kt, C=C, lam=lam, Z=Z)


def _tiny(seed=3, n_v=2, n_c=3, n_mu=5):
    return synth.make_custom(n_v, n_c, n_mu, seed=seed)


# ---- definitions by brute force ------------------------------------------------
def test_delta_and_pair_index_bruteforce():
    p = _tiny()
    d = orc.delta_vc(p.eps_v, p.eps_c)
    for v in range(2):
        for c in range(3):
            assert d[v * 3 + c] == p.eps_c[c] - p.eps_v[v]
    assert d.min() > 0


def test_coupling_bruteforce_eq16():
    """(vc|v'c') = sum_ab C^a_vc (a|b) C^b_v'c' with C^mu_vc = phi_v phi_c: explicit loops. PAPER.md:122."""
    p = _tiny()
    K = orc.khatri_rao(p.phi_v, p.phi_c)
    Kt = orc.coupling_dense(K, p.V)
    n_v, n_c, n_mu = 2, 3, 5
    for v in range(n_v):
        for c in range(n_c):
            for v2 in range(n_v):
                for c2 in range(n_c):
                    acc = 0.0
                    for a in range(n_mu):
                        for b in range(n_mu):
                            acc += p.phi_v[a, v] * p.phi_c[a, c] * p.V[a, b] * p.phi_v[b, v2] * p.phi_c[b, c2]
                    assert abs(Kt[v * n_c + c, v2 * n_c + c2] - acc) < 1e-13 * (1 + abs(acc))


def test_start_vector_bruteforce():
    """(P_nm)_vc = (nm|vc) sqrt(eps_c - eps_v), loops; covers valence and conduction n."""
    p = _tiny()
    d = orc.delta_vc(p.eps_v, p.eps_c)
    for n_idx, m_idx in [(0, 2), (1, 4), (3, 1), (4, 4)]:
        P = orc.start_vector(p.phi_v, p.phi_c, p.V, d, n_idx, m_idx)
        phi_all = np.concatenate([p.phi_v, p.phi_c], axis=1)
        for v in range(2):
            for c in range(3):
                acc = 0.0
                for a in range(5):
                    for b in range(5):
                        acc += phi_all[a, n_idx] * phi_all[a, m_idx] * p.V[a, b] * p.phi_v[b, v] * p.phi_c[b, c]
                ref = acc * np.sqrt(p.eps_c[c] - p.eps_v[v])
                assert abs(P[v * 3 + c] - ref) < 1e-13 * (1 + abs(ref))
    assert orc.orbital_energy_sign(p.eps_v, p.eps_c, 1) == (p.eps_v[1], 1)
    assert orc.orbital_energy_sign(p.eps_v, p.eps_c, 3) == (p.eps_c[1], -1)


# ---- P1-P4: the operator ---------------------------------------------------------
def test_P1_symmetric_psd(dense0):
    C, delta, lam = dense0["C"], dense0["delta"], dense0["lam"]
    assert np.abs(C - C.T).max() <= 1e-13 * np.abs(C).max()
    assert lam.min() > 0
    assert lam.min() >= (delta ** 2).min() - 1e-9          # C >= diag(Delta^2) as V is PSD
    rng = np.random.default_rng(5)
    x, y = rng.standard_normal((2, C.shape[0]))
    assert abs(x @ (C @ y) - y @ (C @ x)) <= 1e-12 * abs(x @ (C @ y))


def test_P2_casida_eq1_spectrum(dense0):
    """Positive eigenvalues of [[A,B],[-B,-A]] (Eq. 1) are sqrt(eig(C)) (Eq. 4); fails for Delta instead of Delta^2."""
    A, B = orc.casida_AB(dense0["delta"], dense0["Kt"])
    M = np.block([[A, B], [-B, -A]])
    ev = sla.eigvals(M)
    assert np.abs(ev.imag).max() < 1e-8
    pos = np.sort(ev.real[ev.real > 0])
    assert len(pos) == A.shape[0]
    O = np.sqrt(dense0["lam"])
    assert np.abs(pos - O).max() <= 1e-10 * O.max()
    neg = np.sort(-ev.real[ev.real < 0])
    assert np.abs(neg - O).max() <= 1e-10 * O.max()


def test_P3_sqrtm_form(dense0):
    A, B = orc.casida_AB(dense0["delta"], dense0["Kt"])
    S = sla.sqrtm(A - B).real
    C2 = S @ (A + B) @ S
    assert np.abs(C2 - dense0["C"]).max() <= 1e-13 * np.abs(C2).max()


def test_P4_factored_vs_dense(cfg0, dense0):
    p, C, delta = cfg0, dense0["C"], dense0["delta"]
    X = synth.random_block(p.cfg, 5).reshape(5, -1)
    Y = orc.casida_matvec_factored(p.phi_v, p.phi_c, p.V, delta, X)
    ref = X @ C
    assert np.abs(Y - ref).max() <= 1e-13 * np.abs(ref).max()
    # shape [nvec, n_v, n_c] accepted and preserved
    Y3 = orc.casida_matvec_factored(p.phi_v, p.phi_c, p.V, delta, X.reshape(5, p.cfg.n_v, p.cfg.n_c))
    assert Y3.shape == (5, p.cfg.n_v, p.cfg.n_c) and np.array_equal(Y3.reshape(5, -1), Y)
    # per-v matmul loop form
    yl = orc.casida_matvec_loop(p.phi_v, p.phi_c, p.V, delta, X[0])
    assert np.abs(yl - ref[0]).max() <= 1e-13 * np.abs(ref).max()
    # V = 0 -> Delta^2 o x exactly
    Y0 = orc.casida_matvec_factored(p.phi_v, p.phi_c, np.zeros_like(p.V), delta, X)
    assert np.array_equal(Y0, delta ** 2 * X)
    # unit vectors give the columns of C
    E = np.eye(C.shape[0])[[0, 7, 191]]
    Ye = orc.casida_matvec_factored(p.phi_v, p.phi_c, p.V, delta, E)
    assert np.abs(Ye - C[[0, 7, 191]]).max() <= 1e-13 * np.abs(C).max()


# ---- P5: closed form N_v = N_c = 1 ------------------------------------------------
def test_P5_one_by_one_closed_form():
    p = synth.make_custom(1, 1, 7, seed=11)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    rho = p.phi_v[:, 0] * p.phi_c[:, 0]
    k = rho @ p.V @ rho
    Cs = delta[0] ** 2 + 2 * delta[0] * k
    y = orc.casida_matvec_factored(p.phi_v, p.phi_c, p.V, delta, np.ones((1, 1)))
    assert abs(y[0, 0] - Cs) <= 1e-14 * Cs
    P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, 0, 1)      # (n,m) = (v0, c0)
    assert abs(P[0] - k * np.sqrt(delta[0])) <= 1e-14 * abs(P[0])
    a, b, n2, ln = orc.lanczos(lambda x: Cs * x, P, 3)
    assert ln == 1 and abs(a[0] - Cs) <= 1e-14 * Cs and b[0] == 0.0
    om = np.linspace(-20, 20, 9)
    for n_idx in (0, 1):
        eps_n, sgn = orc.orbital_energy_sign(p.eps_v, p.eps_c, n_idx)
        sig = orc.sigma_direct(a, b, n2, ln, om, eps_n, sgn, DLT)
        O = np.sqrt(Cs)
        z = om - eps_n - 1j * sgn * DLT
        ref = P[0] ** 2 * sgn / (O * (O + sgn * z))
        assert np.abs(sig - ref).max() <= 1e-14 * np.abs(ref).max()


# ---- P6-P7: Lanczos ---------------------------------------------------------------
def test_P6_moments(cfg0, dense0):
    C, delta, p = dense0["C"], dense0["delta"], cfg0
    P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, 0, p.cfg.n_v)
    L = 6
    a, b, n2, ln = orc.lanczos(lambda x: C @ x, P, L)
    T = orc.tridiagonal(a, b, ln)
    s = P / np.sqrt(n2)
    e1 = np.zeros(L); e1[0] = 1
    v, t = s.copy(), e1.copy()
    for k in range(2 * L):
        assert abs(e1 @ t - s @ v) <= 1e-12 * abs(s @ v), k
        v, t = C @ v, T @ t
    # the first moment beyond 2L-1 must differ (the fraction is not exact)
    assert abs(e1 @ t - s @ v) > 1e-10 * abs(s @ v)


def test_P7_full_length_lanczos(cfg0, dense0):
    C, delta, p = dense0["C"], dense0["delta"], cfg0
    n = C.shape[0]
    P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, 1, p.cfg.n_v + 1)
    a, b, n2, ln, Q = orc.lanczos(lambda x: C @ x, P, n, reorth=True, return_basis=True)
    assert ln == n
    T = orc.tridiagonal(a, b, ln)
    assert np.abs(Q @ Q.T - np.eye(n)).max() < 1e-12
    assert np.abs(Q @ C @ Q.T - T).max() < 1e-9 * np.abs(C).max()
    assert np.abs(np.sort(sla.eigvalsh(T)) - dense0["lam"]).max() < 1e-9 * dense0["lam"].max()
    assert b[n - 1] < 1e-7 * np.abs(a).max()
    assert abs(n2 - P @ P) == 0


def test_lanczos_three_term_recurrence(cfg0, dense0):
    """C q_k = b_k q_{k-1} + a_k q_k + b_{k+1} q_{k+1} and beta indexing beta[k] = b_{k+1} (Eq. 13, Q6)."""
    C, delta, p = dense0["C"], dense0["delta"], cfg0
    P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, 0, p.cfg.n_v + 1)
    a, b, n2, ln, Q = orc.lanczos(lambda x: C @ x, P, 12, return_basis=True)
    assert np.allclose(Q[0], P / np.linalg.norm(P), rtol=0, atol=1e-15)
    for k in range(1, 11):
        r = C @ Q[k] - b[k - 1] * Q[k - 1] - a[k] * Q[k] - b[k] * Q[k + 1]
        assert np.abs(r).max() < 1e-10 * np.abs(a).max()
    assert np.all(b[:12] > 0)


def test_breakdown_invariant_subspace():
    """Q9: a start vector inside a 3-dimensional invariant subspace stops after 3 steps."""
    d = np.array([1.0, 2.0, 3.0, 4.0, 5.0, 6.0])
    P = np.array([1.0, 0.0, 2.0, 0.0, 0.0, -1.0])
    a, b, n2, ln = orc.lanczos(lambda x: d * x, P, 6)
    assert ln == 3 and np.all(a[3:] == 0) and np.all(b[2:] == 0)
    th, w = orc.ritz(a, b, ln)
    assert np.allclose(th, [1.0, 3.0, 6.0], atol=1e-12)
    assert np.allclose(w * n2, [1.0, 4.0, 1.0], atol=1e-12)


# ---- P8, P11: continued fraction -------------------------------------------------------
def test_P8_continued_fraction_vs_ritz_and_exact(cfg0, dense0):
    C, delta, p, lam, Z = dense0["C"], dense0["delta"], cfg0, dense0["lam"], dense0["Z"]
    P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, 0, p.cfg.n_v)
    zeta = (np.linspace(-50, 900, 23) + 0.37j) ** 1
    for L in (1, 2, 9, 40):
        a, b, n2, ln = orc.lanczos(lambda x: C @ x, P, L, reorth=True)
        th, w = orc.ritz(a, b, ln)
        ref = n2 * (w[None, :] / (zeta[:, None] - th[None, :])).sum(axis=1)
        got = orc.continued_fraction(a, b, n2, zeta, ln)
        assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max(), L
    a, b, n2, ln = orc.lanczos(lambda x: C @ x, P, C.shape[0], reorth=True)
    got = orc.continued_fraction(a, b, n2, zeta, ln)
    ref = orc.resolvent_exact(lam, Z, P, zeta)
    assert np.abs(got - ref).max() <= 1e-9 * np.abs(ref).max()
    # asymptotics: zeta R(zeta) -> <P|P> (the norm factor of Q5)
    big = np.array([1e9 + 1e9j])
    assert abs(big[0] * orc.continued_fraction(a, b, n2, big, 30)[0] - n2) < 1e-5 * n2


def test_P11_diagonal_operator_closed_form():
    rng = np.random.default_rng(2)
    d = rng.uniform(2.0, 9.0, 7) ** 2
    s = rng.standard_normal(7)
    a, b, n2, ln = orc.lanczos(lambda x: d * x, s, 7, reorth=True)
    zeta = np.array([1.0 + 0.5j, -3.0 + 0.1j, 50.0 - 2.0j])
    ref = (s[None, :] ** 2 / (zeta[:, None] - d[None, :])).sum(axis=1)
    got = orc.continued_fraction(a, b, n2, zeta, ln)
    assert np.abs(got - ref).max() <= 1e-10 * np.abs(ref).max()


def test_continued_fraction_two_level_by_hand():
    """L = 2 written out: n2 / (z - a0 - b1^2/(z - a1)); b_2 (beta[1]) must not enter (Q6, Q7)."""
    a = np.array([2.0, 5.0]); b = np.array([0.7, 123.0]); z = np.array([1.0 + 1.0j])
    ref = 3.0 / (z - 2.0 - 0.49 / (z - 5.0))
    assert np.abs(orc.continued_fraction(a, b, 3.0, z) - ref).max() < 1e-15


# ---- P9, P10: self-energy -------------------------------------------------------------
def test_P9_eq7_eq11_eq12(cfg0, dense0):
    C, delta, p, lam, Z = dense0["C"], dense0["delta"], cfg0, dense0["lam"], dense0["Z"]
    om = p.omega
    D = (Z * np.sqrt(lam)[None, :]) @ Z.T                       # exact D, D^2 = C
    assert np.abs(D @ D - C).max() < 1e-10 * np.abs(C).max()
    for n_idx, m_idx in [(0, p.cfg.n_v), (p.cfg.n_v + 2, p.cfg.n_v - 1)]:
        P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, n_idx, m_idx)
        eps_n, sgn = orc.orbital_energy_sign(p.eps_v, p.eps_c, n_idx)
        s7 = orc.sigma_exact_eq7(lam, Z, P, om, eps_n, sgn, DLT)
        s11 = orc.sigma_exact_eq11(lam, Z, P, om, eps_n, sgn, DLT)
        assert np.abs(s7 - s11).max() < 1e-13
        a, b, n2, ln = orc.lanczos(lambda x: D @ x, P, C.shape[0], reorth=True)
        s12 = orc.sigma_poly(a, b, n2, ln, om, eps_n, sgn, DLT)
        assert np.abs(s12 - s7).max() < 1e-11
        # Herglotz: Im Sigma has the sign of sgn_n for every omega
        assert np.all(sgn * s7.imag > 0)


def test_P10_direct_mode_converges_to_eq7(cfg0, dense0):
    C, delta, p, lam, Z = dense0["C"], dense0["delta"], cfg0, dense0["lam"], dense0["Z"]
    for n_idx, m_idx in [(1, p.cfg.n_v + 1), (p.cfg.n_v, 0)]:
        P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, n_idx, m_idx)
        eps_n, sgn = orc.orbital_energy_sign(p.eps_v, p.eps_c, n_idx)
        a, b, n2, ln = orc.lanczos(lambda x: C @ x, P, C.shape[0], reorth=True)
        sd = orc.sigma_direct(a, b, n2, ln, p.omega, eps_n, sgn, DLT)
        s7 = orc.sigma_exact_eq7(lam, Z, P, p.omega, eps_n, sgn, DLT)
        assert np.abs(sd - s7).max() < 1e-11
    # truncated: error decreases with L
    P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, 0, p.cfg.n_v)
    eps_n, sgn = orc.orbital_energy_sign(p.eps_v, p.eps_c, 0)
    s7 = orc.sigma_exact_eq7(lam, Z, P, p.omega, eps_n, sgn, DLT)
    errs = []
    for L in (5, 20, 80):
        a, b, n2, ln = orc.lanczos(lambda x: C @ x, P, L, reorth=True)
        errs.append(np.abs(orc.sigma_direct(a, b, n2, ln, p.omega, eps_n, sgn, DLT) - s7).max())
    assert errs[0] > errs[1] > errs[2]


def test_sigma_sum_eq10():
    s = np.arange(12).reshape(3, 4) * (1 + 2j)
    assert np.array_equal(orc.sigma_sum(s), s[0] + s[1] + s[2])


# ---- polynomial square root ------------------------------------------------------------
def test_poly_matrix_function(cfg0, dense0):
    """p_g(C) x = Z p_g(Omega^2) Z^T x, and the Q12 range contains the spectrum."""
    C, delta, lam, Z = dense0["C"], dense0["delta"], dense0["lam"], dense0["Z"]
    lo, hi = 0.8 * (delta ** 2).min(), 1.25 * (delta ** 2).max()
    assert lo < lam.min() and lam.max() < hi
    rng = np.random.default_rng(8)
    x = rng.standard_normal(C.shape[0])
    for g in (0, 1, 7, 8):
        c = orc.fit_sqrt_chebyshev(g, lo, hi)
        y = orc.poly_apply(lambda v: C @ v, c, lo, hi, x)
        ref = Z @ (orc.poly_eval_scalar(c, lo, hi, lam) * (Z.T @ x))
        assert np.abs(y - ref).max() <= 1e-11 * np.abs(ref).max(), g
        # the scalar evaluator agrees with numpy's own Chebyshev evaluation
        t = (2 * lam - (hi + lo)) / (hi - lo)
        assert np.abs(orc.poly_eval_scalar(c, lo, hi, lam) - np.polynomial.chebyshev.chebval(t, c)).max() < 1e-12


def test_P12_sqrt_fit_trend():
    """the error grows with hi/lo and is largest near lo; g = 8 is already good on [0.1, 10]."""
    errs = {}
    for lo, hi in [(0.1, 10.0), (0.05, 20.0), (0.01, 100.0)]:
        x = np.geomspace(lo, hi, 4001)
        for g in (8, 18, 24):
            c = orc.fit_sqrt_chebyshev(g, lo, hi)
            e = np.abs(orc.poly_eval_scalar(c, lo, hi, x) - np.sqrt(x))
            errs[(lo, g)] = e.max()
            assert x[np.argmax(e)] < lo + 0.05 * (hi - lo)
    assert errs[(0.1, 8)] < errs[(0.05, 8)] < errs[(0.01, 8)]
    assert errs[(0.1, 8)] < 0.05
    assert errs[(0.01, 24)] > 0.2 * errs[(0.01, 18)]       # no systematic improvement from 18 to 24


def test_poly_mode_close_to_exact_on_narrow_spectrum():
    """Poly mode (Eq. 12 + 14 on p_g(C)) approaches Eq. 7 when the fit is good."""
    p = synth.make_custom(3, 4, 24, seed=4)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    K = orc.khatri_rao(p.phi_v, p.phi_c)
    C = orc.casida_dense(delta, orc.coupling_dense(K, p.V))
    lam, Z = sla.eigh(C)
    lo, hi = 0.8 * (delta ** 2).min(), 1.25 * (delta ** 2).max()
    c = orc.fit_sqrt_chebyshev(10, lo, hi)
    P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, 0, 3)
    eps_n, sgn = orc.orbital_energy_sign(p.eps_v, p.eps_c, 0)
    a, b, n2, ln = orc.lanczos(lambda x: orc.poly_apply(lambda v: C @ v, c, lo, hi, x), P, 12, reorth=True)
    s = orc.sigma_poly(a, b, n2, ln, p.omega, eps_n, sgn, DLT)
    s7 = orc.sigma_exact_eq7(lam, Z, P, p.omega, eps_n, sgn, DLT)
    fit_err = np.abs(orc.poly_eval_scalar(c, lo, hi, lam) - np.sqrt(lam)).max()
    assert np.abs(s - s7).max() < 50 * fit_err * np.abs(s7).max() + 1e-12


# ---- the whole path ---------------------------------------------------------------------
def test_run_chains_config0(cfg0, dense0):
    p = cfg0
    out = orc.run_chains(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, p.n_idx, p.m_idx,
                         30, p.omega, DLT, reorth=True)
    C, delta = dense0["C"], dense0["delta"]
    assert list(p.n_idx) == [0, 0, 1, 1] and list(p.m_idx) == [8, 9, 8, 9]       # Q11
    for j in range(4):
        P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, int(p.n_idx[j]), int(p.m_idx[j]))
        a, b, n2, ln = orc.lanczos(lambda x: C @ x, P, 30, reorth=True)
        assert np.abs(out["alpha"][j] - a).max() <= 1e-10 * np.abs(a).max()
        assert np.abs(out["beta"][j] - b).max() <= 1e-10 * np.abs(a).max()
        assert abs(out["norm2"][j] - n2) <= 1e-13 * n2
    assert np.abs(out["sigma_sum"] - out["sigma"].sum(axis=0)).max() == 0


# ---- exchange part, Sigma_mm over all n, quasiparticle equation ------------------
def test_exchange_eq6_bruteforce_and_hadamard_form():
    """Eq. 6: -sum_v (vm|vm) by explicit loops over the fitting points, and the closed form
    -p_m^T (V o (Phi_v Phi_v^T)) p_m (Hadamard product with the occupied density matrix)."""
    p = _tiny(seed=5, n_v=3, n_c=4, n_mu=7)
    for m in (0, 2, 3, 6):
        pm = p.phi_v[:, m] if m < 3 else p.phi_c[:, m - 3]
        brute = 0.0
        for v in range(3):
            for a in range(7):
                for b in range(7):
                    brute -= p.phi_v[a, v] * pm[a] * p.V[a, b] * p.phi_v[b, v] * pm[b]
        had = -pm @ ((p.V * (p.phi_v @ p.phi_v.T)) @ pm)
        got = orc.exchange_eq6(p.phi_v, p.phi_c, p.V, m)
        assert abs(got - brute) <= 1e-13 * abs(brute) and abs(got - had) <= 1e-13 * abs(had)
        assert got < 0                                  # V positive definite: every (vm|vm) > 0


def test_sigma_state_full_length_equals_eq7_summed_over_n():
    """Eq. 10 with one chain per n: at L = N_vc with reorthogonalisation the sum equals Eq. 7 (double sum
    over n and s) evaluated on the exact eigenpairs of C."""
    p = _tiny(seed=11, n_v=2, n_c=3, n_mu=9)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    C = orc.casida_dense(delta, orc.coupling_dense(orc.khatri_rao(p.phi_v, p.phi_c), p.V))
    lam, Z = sla.eigh(C)
    omega = np.linspace(-20, 20, 41)
    for m in (1, 2):
        exact = np.zeros(len(omega), dtype=np.complex128)
        for n in range(5):
            P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, n, m)
            e_n, sg = orc.orbital_energy_sign(p.eps_v, p.eps_c, n)
            exact += orc.sigma_exact_eq7(lam, Z, P, omega, e_n, sg, DLT)
        got = orc.sigma_state(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, m, 6, omega, DLT, reorth=True)
        assert np.abs(got - exact).max() <= 1e-11


def test_qp_solve_linear_selfenergy_closed_form():
    """Sigma(w) = a + b w (exactly representable by the linear interpolant): E = (eps + Sx + a - vxc)/(1 - b),
    Z = 1/(1 - b); Newton on a linear function lands on the root in one step."""
    omega = np.linspace(-20, 20, 201)
    a, b, eps, sx, vxc = -0.7, -0.25, -6.3, -4.1, -5.2
    e, z, it = orc.qp_solve(eps, vxc, sx, (a + b * omega) + 0.3j, omega)
    assert abs(e - (eps + sx + a - vxc) / (1 - b)) <= 1e-12
    assert abs(z - 1 / (1 - b)) <= 1e-12 and it <= 3


def test_qp_solve_is_a_root_of_the_interpolated_equation():
    import scipy.optimize as so
    omega = np.linspace(-20, 20, 401)
    re = 0.8 * np.tanh(0.3 * (omega + 5.0)) - 0.1 * omega
    eps, sx, vxc = -6.0, -3.0, -3.5
    F = lambda w: eps + sx + np.interp(w, omega, re) - vxc - w      # noqa: E731
    root = so.brentq(F, -20, 20, xtol=1e-14)
    e, z, it = orc.qp_solve(eps, vxc, sx, re.astype(np.complex128), omega)
    assert abs(e - root) <= 1e-9 and 0 < z < 1.5 and it < orc.QP_MAX_ITER
    # a root outside the grid is clamped to the grid edge
    e2, _, _ = orc.qp_solve(100.0, 0.0, 0.0, np.zeros(401, dtype=np.complex128), omega)
    assert e2 == omega[-1]


# ---- SURVEY.md §8(f)-3 (first step): Tamm-Dancoff, real Gamma-only ------------------------------------------
def test_tda_operator_spectrum_and_selfenergy(cfg0, dense0):
    """B = 0 in Eq. 1: the eigenvalues of the block matrix [[A, 0], [0, -A]] are +-eig(A); the
    factored product equals the dense A x; Lanczos on A at full length with reorthogonalisation gives the exact
    pole sum (Eq. 7 with B = 0)."""
    p = cfg0
    delta, Kt = dense0["delta"], dense0["Kt"]
    A = orc.tda_dense(delta, Kt)
    assert np.abs(A - A.T).max() <= 1e-14 * np.abs(A).max() and np.abs(np.diag(A) - delta - np.diag(Kt)).max() <= 1e-14 * np.abs(A).max()
    lam, X = sla.eigh(A)
    assert lam.min() >= delta.min()                               # Ktilde is positive semidefinite
    x = np.random.default_rng(2).normal(size=(3, len(delta)))
    y = orc.tda_matvec_factored(p.phi_v, p.phi_c, p.V, delta, x)
    assert np.abs(y - x @ A).max() <= 1e-12 * np.abs(y).max()
    n, m = 1, p.cfg.n_v + 2
    P = orc.tda_start_vector(p.phi_v, p.phi_c, p.V, n, m)
    K = dense0["K"]
    rho = p.phi_v[:, n] * p.phi_c[:, 2]
    assert np.abs(P - K.T @ (p.V @ rho)).max() <= 1e-13 * np.abs(P).max()
    N = len(delta)
    r = orc.run_chains_tda(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, [n, p.cfg.n_v], [m, m], N, p.omega, DLT, reorth=True)
    for j, nn in enumerate([n, p.cfg.n_v]):
        Pj = orc.tda_start_vector(p.phi_v, p.phi_c, p.V, nn, m)
        e_n, sg = orc.orbital_energy_sign(p.eps_v, p.eps_c, nn)
        exact = orc.sigma_tda_exact(lam, X, Pj, p.omega, e_n, sg, DLT)
        assert np.abs(r["sigma"][j] - exact).max() <= 1e-10
        assert (sg * r["sigma"][j].imag > 0).all()                # same Herglotz sign as the RPA case


def test_tda_one_by_one_closed_form():
    """N_v = N_c = 1: A = Delta + k, k = rho^T V rho; Sigma = P^2 / (omega - eps_n + eta (A - i delta))."""
    p = synth.make_custom(1, 1, 6, seed=8)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    rho = p.phi_v[:, 0] * p.phi_c[:, 0]
    k = rho @ p.V @ rho
    om = np.linspace(-5, 5, 11)
    r = orc.run_chains_tda(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, [0, 1], [1, 1], 1, om, DLT)
    assert abs(r["alpha"][0, 0] - (delta[0] + k)) <= 1e-13 * (delta[0] + k)
    for j, (e_n, sg, P2) in enumerate([(p.eps_v[0], 1, k * k), (p.eps_c[0], -1, ((p.phi_c[:, 0] ** 2) @ p.V @ rho) ** 2)]):
        ref = P2 / (om - e_n + sg * (delta[0] + k - 1j * DLT))
        assert np.abs(r["sigma"][j] - ref).max() <= 1e-12 * np.abs(ref).max()


def test_oracle_matches_its_golden_file():
    """Regression pin: tests/golden/cfg0_oracle.txt (written by tests/golden/make_golden.py from the oracle alone; the paper
    prints no worked example).  A deliberate change of the oracle's arithmetic regenerates the file in the same commit."""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    got = {(n, j, k): v for n, j, k, v in mod.compute()}
    stored = {}
    for line in open(os.path.join(here, "cfg0_oracle.txt")):
        if line.startswith("#"):
            continue
        n, j, k, v = line.split()
        stored[(n, int(j), int(k))] = float(v)
    assert set(got) == set(stored)
    for key, v in stored.items():
        assert abs(got[key] - v) <= 1e-9 * max(1.0, abs(v)), key


# ---- thin spots named by the round-1 review ------------------------------------------------------
def test_fit_sqrt_chebyshev_least_squares_optimality():
    """The fit is THE least-squares solution on M = 4(g+1) first-kind Chebyshev nodes of [lo, hi] (PAPER.md:85, :284,
    :317; reading Q13): the residual is orthogonal to T_0..T_g on those nodes (normal equations), rebuilt here from the
    textbook node formula x_k = mid + half cos(pi (2k+1) / (2M)).  A wrong node set, node count or basis fails this."""
    for g, lo, hi in [(1, 2.0, 3.0), (7, 9.4, 997.0), (8, 0.1, 10.0), (12, 7.0, 2600.0)]:
        c = orc.fit_sqrt_chebyshev(g, lo, hi)
        M = 4 * (g + 1)
        k = np.arange(M)
        t = np.cos(np.pi * (2 * k + 1) / (2 * M))
        x = 0.5 * (hi + lo) + 0.5 * (hi - lo) * t
        T = np.cos(np.arange(g + 1)[None, :] * np.arccos(t)[:, None])         # T_j(t_k) = cos(j arccos t_k)
        resid = T @ c - np.sqrt(x)
        assert np.abs(T.T @ resid).max() <= 1e-11 * np.sqrt(hi) * M
        # and it beats any perturbed coefficient vector in the discrete 2-norm
        rng = np.random.default_rng(g)
        for _ in range(5):
            d = 1e-3 * rng.standard_normal(g + 1)
            assert np.linalg.norm(T @ (c + d) - np.sqrt(x)) > np.linalg.norm(resid)
        # discrete orthogonality gives the same coefficients in closed form: c_j = (2/M) sum_k f(x_k) T_j(t_k), c_0 halved
        cf = (2.0 / M) * (T.T @ np.sqrt(x))
        cf[0] *= 0.5
        assert np.abs(c - cf).max() <= 1e-12 * np.abs(cf).max()


def _strongly_coupled_tiny():
    """N_vc = 96 on 16 fitting points in a 3 A box: the coupling dominates, lambda_max(C) ~ 2138 eV^2."""
    p = synth.make_custom(6, 16, 16, box=3.0, seed=3, chains_a=2, chains_b=2)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    C = orc.casida_dense(delta, orc.coupling_dense(orc.khatri_rao(p.phi_v, p.phi_c), p.V))
    lam, Z = sla.eigh(C)
    return p, delta, C, lam, Z


def test_heuristic_fit_range_misses_a_strongly_coupled_spectrum():
    """PAPER.md:284's heuristic range (reading Q12) is not a bound on the spectrum of C: its lower end is
    (lambda_min(C) >= min Delta^2 for V >= 0, pin P1), its upper end is not once 2 sqrt(Delta) K^T V K sqrt(Delta) is
    large, and a Chebyshev fit evaluated outside its interval diverges."""
    p, delta, C, lam, Z = _strongly_coupled_tiny()
    lo, hi = 0.8 * (delta ** 2).min(), 1.25 * (delta ** 2).max()
    assert lo < lam[0] and lam[-1] > 2.0 * hi
    c = orc.fit_sqrt_chebyshev(7, lo, hi)
    assert abs(orc.poly_eval_scalar(c, lo, hi, lam[-1])) > 100.0 * np.sqrt(lam[-1])


def test_spectrum_bounds_lanczos():
    """extremal eigenvalues by Lanczos.  Full length: exact extremes.  Short runs: the upper estimate
    theta_max + r_max has converged from above after a few steps (separated top eigenvalue), the Ritz values stay inside
    the spectrum, and the intervals shrink with the number of steps."""
    p, delta, C, lam, Z = _strongly_coupled_tiny()
    n = delta.size
    lo_f, hi_f = orc.spectrum_bounds_lanczos(lambda x: C @ x, n, n)
    assert abs(hi_f - lam[-1]) <= 1e-9 * lam[-1] and abs(lo_f - lam[0]) <= 1e-7 * lam[-1]
    prev = None
    for steps in (5, 10, 20, 40):
        lo_s, hi_s = orc.spectrum_bounds_lanczos(lambda x: C @ x, n, steps)
        assert hi_s >= lam[-1] * (1 - 1e-12) and lo_s <= lam[0] * (1 + 1e-12)
        if prev is not None:
            assert hi_s <= prev[1] * (1 + 1e-12) and lo_s >= prev[0] - 1e-9
        prev = (lo_s, hi_s)
    assert prev[1] <= lam[-1] * (1 + 1e-9)
    # the factored product gives the same estimate as the dense matrix
    lo_x, hi_x = orc.spectrum_bounds_lanczos(
        lambda x: orc.casida_matvec_factored(p.phi_v, p.phi_c, p.V, delta, x[None])[0], n, 20)
    lo_d, hi_d = orc.spectrum_bounds_lanczos(lambda x: C @ x, n, 20)
    # (the lower estimate is rounding-sensitive once the top Ritz value has converged and the basis loses orthogonality)
    assert abs(hi_x - hi_d) <= 1e-9 * hi_d and abs(lo_x - lo_d) <= 1e-2 * hi_d


def test_run_chains_poly_branch_end_to_end_against_eq7():
    """The poly= branch of run_chains (start vector -> Lanczos on p_g(C) -> sigma_poly dispatch -> Eq. 10 sum) as one
    piece against Eq. 7 by full diagonalisation, on the strongly coupled problem with the range taken from its
    spectrum.  At L = N_vc with reorthogonalisation the only error left is the fit error
    eps = max_s |p_g(Omega_s^2) - Omega_s|, which moves every pole of Eq. 12 by at most eps:
    |dSigma| <= <P|P> eps (1/(Omega_min (Omega_min - eps)) + 1/delta^2) / delta.  The error must also fall with g."""
    p, delta, C, lam, Z = _strongly_coupled_tiny()
    n, dl = delta.size, 0.68
    lo, hi = 0.8 * (delta ** 2).min(), 1.02 * lam[-1]
    o_min = np.sqrt(lam[0])
    worst = []
    for g in (7, 12, 24):
        c = orc.fit_sqrt_chebyshev(g, lo, hi)
        eps = np.abs(orc.poly_eval_scalar(c, lo, hi, lam) - np.sqrt(lam)).max()
        r = orc.run_chains(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, p.n_idx, p.m_idx, n, p.omega, dl, reorth=True,
                           poly=(c, lo, hi))
        errs, tot = [], 0.0
        for j in range(len(p.n_idx)):
            P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, int(p.n_idx[j]), int(p.m_idx[j]))
            e_n, sg = orc.orbital_energy_sign(p.eps_v, p.eps_c, int(p.n_idx[j]))
            exact = orc.sigma_exact_eq7(lam, Z, P, p.omega, e_n, sg, dl)
            bound = (P @ P) * eps * (1.0 / (o_min * (o_min - eps)) + 1.0 / dl ** 2) / dl
            err = np.abs(r["sigma"][j] - exact).max()
            assert err <= bound, (g, j, err, bound)
            errs.append(err / np.abs(exact).max())
            tot = tot + exact
        assert np.abs(r["sigma_sum"] - tot).max() <= sum(errs) * np.abs(tot).max() + 1e-12
        worst.append(max(errs))
    assert worst[0] > worst[1] > worst[2] and worst[2] < 0.01
