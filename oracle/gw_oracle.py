"""CPU oracle for the Lanczos full-frequency GW hot path (arXiv 2310.20103).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py may import this module.  It is
plain NumPy/SciPy FP64, follows the paper step by step in the paper's notation,
shares no code with paper_2310_20103_b200/ (the CUDA path) and imports nothing
from it.  Every function cites the passage of /root/reference/PAPER.md
("PAPER.md:<line>") it restates; readings of silent/garbled passages are the
Q-numbers of SURVEY.md §8(c), listed again in DESIGN.md.

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): P1-P11 of SURVEY.md §8(c) --
Hermiticity/PSD of C, Eq. 1 <-> Eq. 4 spectra, sqrtm form of C, factored vs
dense product, the 1x1 closed form, moment identity, full-length Lanczos vs
eigh, continued fraction vs spectral sum, Eq. 7 == Eq. 11 == Eq. 12, and the
diagonal-operator closed form.  No function here is "parity unpinned".

Notation: N_vc = N_v N_c, pair index vc = v N_c + c (c fastest).
  Phi_v [N_mu, N_v], Phi_c [N_mu, N_c]   orbitals at the fitting points
  K [N_mu, N_vc], K[mu, vc] = Phi_v[mu, v] Phi_c[mu, c]          (Q4)
  V [N_mu, N_mu] symmetric positive definite, stands for (alpha|beta), Eq. 17
  Delta[vc] = eps_c - eps_v > 0
  sgn_n = the paper's eta_n (+1 occupied, -1 empty); dlt = the paper's delta
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla

BREAKDOWN_TOL = 1e-12   # reading Q9


# --------------------------------------------------------------------------- #
# Operator definition                                                          #
# --------------------------------------------------------------------------- #
def delta_vc(eps_v, eps_c):
    """Delta_vc = eps_c - eps_v, flattened with c fastest.  PAPER.md:41 (Eq. 2)."""
    return (np.asarray(eps_c)[None, :] - np.asarray(eps_v)[:, None]).reshape(-1)


def khatri_rao(phi_v, phi_c):
    """K[mu, vc] = phi_v(r_mu) phi_c(r_mu): the ISDF coefficients C^mu_vc of
    PAPER.md:117-123 (Eq. 15-16) under reading Q4."""
    n_mu = phi_v.shape[0]
    return (phi_v[:, :, None] * phi_c[:, None, :]).reshape(n_mu, -1)


def coupling_dense(K, V):
    """Ktilde[vc, v'c'] = (vc|v'c') = sum_ab K[a,vc] (a|b) K[b,v'c'].  PAPER.md:122 (Eq. 16)."""
    return K.T @ (V @ K)


def casida_AB(delta, Ktilde):
    """A = diag(Delta) + (vc|v'c'), B = (vc|c'v') = (vc|v'c') for real orbitals.
    PAPER.md:41-45 (Eq. 2-3); no extra spin factor (Q3)."""
    return np.diag(delta) + Ktilde, Ktilde.copy()


def casida_dense(delta, Ktilde):
    """C = (A-B)^{1/2} (A+B) (A-B)^{1/2} with A-B = diag(Delta):
    C = diag(Delta^2) + 2 diag(sqrt Delta) Ktilde diag(sqrt Delta).  PAPER.md:52 (Eq. 4), Q2."""
    s = np.sqrt(delta)
    return np.diag(delta * delta) + 2.0 * (s[:, None] * Ktilde * s[None, :])


def casida_matvec_factored(phi_v, phi_c, V, delta, X):
    """Y = C X without forming C or K:
    Y = Delta^2 o X + 2 sqrt(Delta) o K^T ( V ( K ( sqrt(Delta) o X ) ) ).
    X: [nvec, N_vc] (or [nvec, N_v, N_c]); returns the same shape."""
    shape = X.shape
    n_v, n_c = phi_v.shape[1], phi_c.shape[1]
    s = np.sqrt(delta).reshape(n_v, n_c)
    d2 = (delta * delta).reshape(n_v, n_c)
    Xb = X.reshape(-1, n_v, n_c)
    Xs = Xb * s[None]
    # T[mu, b] = sum_v phi_v[mu, v] sum_c phi_c[mu, c] Xs[b, v, c]
    G = np.einsum("mc,bvc->mbv", phi_c, Xs, optimize=True)
    T = np.einsum("mv,mbv->mb", phi_v, G)
    W = V @ T
    # U[b, v, c] = sum_mu phi_v[mu, v] phi_c[mu, c] W[mu, b]
    U = np.einsum("mv,mc,mb->bvc", phi_v, phi_c, W, optimize=True)
    Y = d2[None] * Xb + 2.0 * s[None] * U
    return Y.reshape(shape)


def casida_matvec_loop(phi_v, phi_c, V, delta, x):
    """The same product for ONE vector written as explicit per-v matmuls (the
    "2 matrix-vector multiplications" of PAPER.md:383); used to cross-check the einsum form."""
    n_v, n_c = phi_v.shape[1], phi_c.shape[1]
    s = np.sqrt(delta).reshape(n_v, n_c)
    xs = x.reshape(n_v, n_c) * s
    t = np.zeros(phi_v.shape[0])
    for v in range(n_v):
        t += phi_v[:, v] * (phi_c @ xs[v])
    w = V @ t
    u = np.empty((n_v, n_c))
    for v in range(n_v):
        u[v] = phi_c.T @ (phi_v[:, v] * w)
    return ((delta * delta).reshape(n_v, n_c) * x.reshape(n_v, n_c) + 2.0 * s * u).reshape(x.shape)


# --------------------------------------------------------------------------- #
# Start vectors                                                                #
# --------------------------------------------------------------------------- #
def orbital_column(phi_v, phi_c, idx):
    """phi_n at the fitting points; idx < N_v valence, else conduction idx - N_v."""
    n_v = phi_v.shape[1]
    return phi_v[:, idx] if idx < n_v else phi_c[:, idx - n_v]


def orbital_energy_sign(eps_v, eps_c, idx):
    """(eps_n, sgn_n): sgn_n = eta_n = +1 occupied, -1 empty.  PAPER.md:62."""
    n_v = len(eps_v)
    return (float(eps_v[idx]), 1) if idx < n_v else (float(eps_c[idx - n_v]), -1)


def start_vector(phi_v, phi_c, V, delta, n_idx, m_idx):
    """(P_nm)_vc = (nm|vc) (eps_c - eps_v)^{1/2}.  PAPER.md:67; (nm|vc) by Eq. 16
    with rho_nm(mu) = phi_n(r_mu) phi_m(r_mu) (Q4)."""
    rho = orbital_column(phi_v, phi_c, n_idx) * orbital_column(phi_v, phi_c, m_idx)
    w = V @ rho
    n_v, n_c = phi_v.shape[1], phi_c.shape[1]
    eri = np.einsum("mv,mc,m->vc", phi_v, phi_c, w, optimize=True).reshape(n_v * n_c)
    return eri * np.sqrt(delta)


# --------------------------------------------------------------------------- #
# Polynomial square root (optional mode)                                       #
# --------------------------------------------------------------------------- #
def fit_sqrt_chebyshev(g, lo, hi):
    """Least-squares fit of sqrt(x) on [lo, hi] at M = 4(g+1) first-kind Chebyshev
    nodes, in the Chebyshev basis (reading Q13).
    Returns c[0..g] with p_g(x) = sum_j c_j T_j((2x - hi - lo)/(hi - lo))."""
    M = 4 * (g + 1)
    t = np.cos(np.pi * (2.0 * np.arange(M) + 1.0) / (2.0 * M))
    x = 0.5 * (hi + lo) + 0.5 * (hi - lo) * t
    Tm = np.polynomial.chebyshev.chebvander(t, g)
    c, *_ = np.linalg.lstsq(Tm, np.sqrt(x), rcond=None)
    return c


def spectrum_bounds_lanczos(apply_op, n, steps, seed=0):
    """Extremal eigenvalues of the operator for the fitting range: "One can use standard Lanczos algorithm to determine
    the extremal eigenvalues min(Omega_s^2) and max(Omega_s^2) of C".  `steps` Lanczos steps from a
    generic random vector; returns (theta_min - r_min, theta_max + r_max) with theta the extreme eigenvalues of T and
    r_i = b_L |s_L,i| the residual norm of that Ritz pair (an eigenvalue of the operator lies within r_i of theta_i)."""
    p = np.random.default_rng(seed).uniform(-1.0, 1.0, n)
    a, b, _, ln = lanczos(apply_op, p, min(int(steps), n))
    if ln == 1:
        return float(a[0] - b[0]), float(a[0] + b[0])
    theta, S = sla.eigh_tridiagonal(a[:ln], b[:ln - 1])
    r = b[ln - 1] * np.abs(S[-1, :])
    return float(theta[0] - r[0]), float(theta[-1] + r[-1])


def poly_eval_scalar(c, lo, hi, x):
    """p_g(x) for scalars/arrays, by the same three-term recurrence as poly_apply."""
    t = (2.0 * np.asarray(x, dtype=np.float64) - (hi + lo)) / (hi - lo)
    t0 = np.ones_like(t)
    y = c[0] * t0
    if len(c) == 1:
        return y
    t1 = t
    y = y + c[1] * t1
    for j in range(2, len(c)):
        t0, t1 = t1, 2.0 * t * t1 - t0
        y = y + c[j] * t1
    return y


def poly_apply(apply_C, c, lo, hi, x):
    """p_g(C) x = a_0 x + sum_k a_k C^k x, evaluated in the
    Chebyshev basis on Ctilde = (2C - (hi+lo))/(hi-lo): g applications of C (Q13)."""
    def ct(v):
        return (2.0 * apply_C(v) - (hi + lo) * v) / (hi - lo)
    t0 = x
    y = c[0] * t0
    if len(c) == 1:
        return y
    t1 = ct(x)
    y = y + c[1] * t1
    for j in range(2, len(c)):
        t0, t1 = t1, 2.0 * ct(t1) - t0
        y = y + c[j] * t1
    return y


# --------------------------------------------------------------------------- #
# Lanczos                                                                      #
# --------------------------------------------------------------------------- #
def lanczos(apply_op, p, steps, reorth=False, return_basis=False):
    """Standard Lanczos tridiagonalisation started from |P> (Eq. 13).
    steps = number of operator applications = dimension of T (Q6).
    Returns alpha[steps] (a_0..a_{L-1}), beta[steps] with beta[k] = b_{k+1},
    norm2 = <P|P>, len = effective length (Q9: breakdown when
    b_{k+1} <= 1e-12 max_i(|a_i| + b_i); the tail is zero-filled).
    reorth=True: two-pass full reorthogonalisation against all previous q."""
    p = np.asarray(p, dtype=np.float64)
    norm2 = float(p @ p)
    alpha = np.zeros(steps)
    beta = np.zeros(steps)
    basis = []
    if norm2 == 0.0:
        return (alpha, beta, norm2, 0, np.zeros((0, p.size))) if return_basis else (alpha, beta, norm2, 0)
    q = p / np.sqrt(norm2)
    q_prev = np.zeros_like(q)
    b_prev = 0.0
    scale = 0.0
    length = steps
    for k in range(steps):
        if reorth or return_basis:
            basis.append(q)
        w = apply_op(q)
        a = float(q @ w)
        w = w - a * q - b_prev * q_prev
        if reorth:
            Q = np.array(basis)
            for _ in range(2):
                w = w - Q.T @ (Q @ w)
        b = float(np.sqrt(w @ w))
        alpha[k] = a
        beta[k] = b
        scale = max(scale, abs(a) + b)
        if b <= BREAKDOWN_TOL * scale:
            beta[k] = 0.0
            length = k + 1
            break
        q_prev, q, b_prev = q, w / b, b
    if return_basis:
        return alpha, beta, norm2, length, np.array(basis)
    return alpha, beta, norm2, length


def tridiagonal(alpha, beta, length):
    """T_L of Eq. 13 restricted to dimension L = length (Q6): diag a_0..a_{L-1}, off-diag b_1..b_{L-1}."""
    T = np.diag(alpha[:length])
    if length > 1:
        T += np.diag(beta[:length - 1], 1) + np.diag(beta[:length - 1], -1)
    return T


# --------------------------------------------------------------------------- #
# Resolvents and the self-energy                                               #
# --------------------------------------------------------------------------- #
def continued_fraction(alpha, beta, norm2, zeta, length=None):
    """<P|(zeta - Op)^{-1}|P> by the Haydock continued fraction, PAPER.md:92-99 (Eq. 14):
    norm2 / (zeta - a_0 - b_1^2 / (zeta - a_1 - b_2^2 / (... zeta - a_{L-1}))),
    "zeta - a_k" at every level, times <P|P> (Q5), plain truncation (Q7).
    Evaluated bottom-up.  zeta: complex array; returns the same shape."""
    L = len(alpha) if length is None else int(length)
    zeta = np.asarray(zeta, dtype=np.complex128)
    if L == 0:
        return np.zeros_like(zeta)
    f = zeta - alpha[L - 1]
    for k in range(L - 2, -1, -1):
        f = zeta - alpha[k] - (beta[k] * beta[k]) / f
    return norm2 / f


def ritz(alpha, beta, length=None):
    """Eigenvalues theta_i of T_L and weights w_i = (first eigenvector component)^2
    (Gauss quadrature of the spectral measure of |P>; used by direct mode, Q1)."""
    L = len(alpha) if length is None else int(length)
    if L == 0:
        return np.zeros(0), np.zeros(0)
    if L == 1:
        return np.array([alpha[0]]), np.array([1.0])
    theta, S = sla.eigh_tridiagonal(alpha[:L], beta[:L - 1])
    return theta, S[0, :] ** 2


def z_n(omega, eps_n, sgn_n, dlt):
    """z_n = omega - eps_n - i eta_n delta.  PAPER.md:79 (Q8)."""
    return np.asarray(omega, dtype=np.float64) - eps_n - 1j * sgn_n * dlt


def sigma_direct(alpha, beta, norm2, length, omega, eps_n, sgn_n, dlt):
    """Direct mode (Lanczos on C, Q1): Eq. 11 evaluated on the Ritz pairs of T_L,
    Sigma(omega, n) = <P|P> sum_i w_i [1/z (1/O_i - 1/(O_i + sgn z))],  O_i = sqrt(theta_i)
                    = <P|P> sum_i w_i sgn / (O_i (O_i + sgn z))."""
    theta, w = ritz(alpha, beta, length)
    O = np.sqrt(theta)
    z = z_n(omega, eps_n, sgn_n, dlt)
    terms = (w / O)[None, :] * sgn_n / (O[None, :] + sgn_n * z[:, None])
    return norm2 * terms.sum(axis=1)


def sigma_poly(alpha, beta, norm2, length, omega, eps_n, sgn_n, dlt):
    """Poly mode (Lanczos on D ~ p_g(C)): Eq. 12 with Eq. 14,
    Sigma = 1/z [ <P|D^-1|P> - <P|(D + sgn z)^-1|P> ] = 1/z [ R(-sgn z) - R(0) ],
    R(zeta) = <P|(zeta - D)^-1|P>  (Q8)."""
    z = z_n(omega, eps_n, sgn_n, dlt)
    R0 = continued_fraction(alpha, beta, norm2, np.array([0.0 + 0.0j]), length)[0]
    Rz = continued_fraction(alpha, beta, norm2, -sgn_n * z, length)
    return (Rz - R0) / z


def sigma_sum(sig_chains):
    """Sigma_mm(omega) = sum_n Sigma_mm(omega, n).  PAPER.md:73 (Eq. 10)."""
    return np.sum(np.asarray(sig_chains), axis=0)


# --------------------------------------------------------------------------- #
# Exact references (full diagonalisation; tiny sizes only)                     #
# --------------------------------------------------------------------------- #
def eig_casida(C):
    """(Omega_s^2, Z^s) of Eq. 4."""
    return sla.eigh(C)


def sigma_exact_eq7(lam, Z, P, omega, eps_n, sgn_n, dlt):
    """Eq. 7 with Eq. 9: sum_s (<P|Z^s>^2 / O_s) / (omega - eps_n + sgn (O_s - i delta))."""
    O = np.sqrt(lam)
    W2 = (Z.T @ P) ** 2 / O
    den = np.asarray(omega)[:, None] - eps_n + sgn_n * (O[None, :] - 1j * dlt)
    return (W2[None, :] / den).sum(axis=1)


def sigma_exact_eq11(lam, Z, P, omega, eps_n, sgn_n, dlt):
    """Eq. 11 on the exact eigenpairs."""
    O = np.sqrt(lam)
    pz2 = (Z.T @ P) ** 2
    z = z_n(omega, eps_n, sgn_n, dlt)
    br = 1.0 / O[None, :] - 1.0 / (O[None, :] + sgn_n * z[:, None])
    return (pz2[None, :] * br).sum(axis=1) / z


def resolvent_exact(lam, Z, P, zeta, power=1.0):
    """sum_s <P|Z^s>^2 / (zeta - lam_s^power): R_C (power 1) or R_D (power 1/2).  PAPER.md:81."""
    pz2 = (Z.T @ P) ** 2
    zeta = np.asarray(zeta, dtype=np.complex128)
    return (pz2[None, :] / (zeta[:, None] - lam[None, :] ** power)).sum(axis=1)


# --------------------------------------------------------------------------- #
# Whole path for a list of chains (what the parity tests compare against)      #
# --------------------------------------------------------------------------- #
def run_chains(phi_v, phi_c, eps_v, eps_c, V, n_idx, m_idx, steps, omega, dlt,
               reorth=False, poly=None):
    """S1..S7 of SURVEY.md §8(a) for chains (n_j, m_j).  poly = None (direct mode, Op = C)
    or (c, lo, hi) (poly mode, Op = p_g(C)).  Returns dict of alpha, beta, norm2, len, sigma, sigma_sum."""
    delta = delta_vc(eps_v, eps_c)

    def apply_C(x):
        return casida_matvec_factored(phi_v, phi_c, V, delta, x[None])[0]

    if poly is None:
        op = apply_C
    else:
        c, lo, hi = poly

        def op(x):
            return poly_apply(apply_C, c, lo, hi, x)

    n = len(n_idx)
    out = dict(alpha=np.zeros((n, steps)), beta=np.zeros((n, steps)), norm2=np.zeros(n),
               len=np.zeros(n, dtype=np.int32), sigma=np.zeros((n, len(omega)), dtype=np.complex128))
    for j in range(n):
        P = start_vector(phi_v, phi_c, V, delta, int(n_idx[j]), int(m_idx[j]))
        a, b, n2, ln = lanczos(op, P, steps, reorth=reorth)
        eps_n, sgn = orbital_energy_sign(eps_v, eps_c, int(n_idx[j]))
        f = sigma_direct if poly is None else sigma_poly
        out["alpha"][j], out["beta"][j], out["norm2"][j], out["len"][j] = a, b, n2, ln
        out["sigma"][j] = f(a, b, n2, ln, omega, eps_n, sgn, dlt)
    out["sigma_sum"] = sigma_sum(out["sigma"])
    return out


# --------------------------------------------------------------------------- #
# exchange part and the quasiparticle equation              #
# --------------------------------------------------------------------------- #
def exchange_eq6(phi_v, phi_c, V, m_idx):
    """Sigma^ex_mm = - sum_v (vm|vm), PAPER.md:57 (Eq. 6; the printed summation index "m" is read as
    the occupied orbital v, Q15), with (vm|vm) = rho_vm^T V rho_vm, rho_vm(mu) = phi_v(r_mu) phi_m(r_mu)
    (Eq. 16 under Q4)."""
    pm = orbital_column(phi_v, phi_c, m_idx)
    tot = 0.0
    for v in range(phi_v.shape[1]):
        rho = phi_v[:, v] * pm
        tot += rho @ (V @ rho)
    return -tot


def sigma_state(phi_v, phi_c, eps_v, eps_c, V, m_idx, steps, omega, dlt, reorth=False, poly=None):
    """Sigma^corr_mm(omega) = sum over ALL n = 1..N_v+N_c of Sigma^corr_mm(omega, n), PAPER.md:73 (Eq. 10):
    one Lanczos chain per n started from |P_nm>."""
    n_orb = phi_v.shape[1] + phi_c.shape[1]
    n_idx = np.arange(n_orb, dtype=np.int32)
    r = run_chains(phi_v, phi_c, eps_v, eps_c, V, n_idx, np.full(n_orb, m_idx, dtype=np.int32), steps, omega, dlt,
                   reorth=reorth, poly=poly)
    return r["sigma_sum"]


QP_MAX_ITER = 50
QP_TOL = 1e-10   # eV


def qp_solve(eps_m, vxc_m, sigma_x, sigma_c, omega):
    """Quasiparticle equation of: E(omega) = eps_m + <m|Sigma(omega) - V_xc|m> is known on the
    frequency grid; "the Newton-Raphson algorithm is used to get a graphical solution of E(omega) = omega".
    Reading Q18 (the paper gives no more detail): F(w) = eps_m + Re[Sigma^ex + Sigma^corr(w)] - V_xc - w with
    Re Sigma^corr interpolated linearly between grid points; Newton from w_0 = eps_m,
    w <- w - F(w)/F'(w), F' = (slope of the grid interval holding w) - 1, w clamped to the grid range, until
    |step| <= 1e-10 eV or 50 iterations.  Returns (E_qp, Z, iterations), Z = 1/(1 - dReSigma/dw) = -1/F'."""
    omega = np.asarray(omega, dtype=np.float64)
    re = np.real(np.asarray(sigma_c))
    n = len(omega)
    w = min(max(float(eps_m), omega[0]), omega[-1])
    z = 1.0
    it = 0
    for it in range(1, QP_MAX_ITER + 1):
        i = int(np.searchsorted(omega, w, side="right")) - 1      # largest i with omega[i] <= w
        i = min(max(i, 0), n - 2)
        slope = (re[i + 1] - re[i]) / (omega[i + 1] - omega[i])
        s_w = re[i] + slope * (w - omega[i])
        F = eps_m + sigma_x + s_w - vxc_m - w
        dF = slope - 1.0
        z = -1.0 / dF
        step = -F / dF
        w_new = min(max(w + step, omega[0]), omega[-1])
        done = abs(w_new - w) <= QP_TOL
        w = w_new
        if done:
            break
    return w, z, it


# --------------------------------------------------------------------------- #
# SURVEY.md §8(f)-3, first step: Tamm-Dancoff approximation, real Gamma-only   #
# --------------------------------------------------------------------------- #
def tda_dense(delta, Ktilde):
    """A = diag(Delta) + (vc|v'c'): "setting matrix B = 0 in the RPA Casida matrix ... only a Hermitian matrix A
    remains" (Eq. 2).  Real orbitals, one k-point: the Gamma-only restriction of A(q)."""
    return np.diag(delta) + Ktilde


def tda_matvec_factored(phi_v, phi_c, V, delta, X):
    """y = A x = Delta o x + K^T (V (K x)) for a block X [nvec, N_vc], K never formed (same contraction order as
    casida_matvec_factored)."""
    n_v, n_c = phi_v.shape[1], phi_c.shape[1]
    X = np.asarray(X, dtype=np.float64).reshape(-1, n_v * n_c)
    X3 = X.reshape(-1, n_v, n_c)
    T = np.einsum("mv,mc,bvc->mb", phi_v, phi_c, X3, optimize=True)
    W = V @ T
    U = np.einsum("mv,mc,mb->bvc", phi_v, phi_c, W, optimize=True).reshape(X.shape)
    return delta[None, :] * X + U


def tda_start_vector(phi_v, phi_c, V, n_idx, m_idx):
    """P_vc = (nm|vc): the vector of PAPER.md:313 for one k-point (no (eps_c - eps_v)^{1/2} factor in the TDA)."""
    rho = orbital_column(phi_v, phi_c, n_idx) * orbital_column(phi_v, phi_c, m_idx)
    w = V @ rho
    return np.einsum("mv,mc,m->vc", phi_v, phi_c, w, optimize=True).reshape(-1)


def sigma_tda(alpha, beta, norm2, length, omega, eps_n, sgn_n, dlt):
    """Sigma(omega, n) = <P| 1/(omega - eps_n + eta_n (A - i delta)) |P>  (one k-point, prefactor of
    Eq. 7: reading Q19) = -eta_n R_A(-eta_n z_n), z_n = omega - eps_n - i eta_n delta, with the resolvent
    R_A(zeta) = <P|(zeta - A)^{-1}|P> by the continued fraction of Eq. 14."""
    z = z_n(omega, eps_n, sgn_n, dlt)
    return -sgn_n * continued_fraction(alpha, beta, norm2, -sgn_n * z, length)


def sigma_tda_exact(lam, X, P, omega, eps_n, sgn_n, dlt):
    """Eq. 7 with B = 0: sum_s <P|X^s>^2 / (omega - eps_n + eta_n (Omega_s - i delta)), (Omega_s, X^s) = eig(A)."""
    w2 = (X.T @ P) ** 2
    den = np.asarray(omega)[:, None] - eps_n + sgn_n * (lam[None, :] - 1j * dlt)
    return (w2[None, :] / den).sum(axis=1)


def run_chains_tda(phi_v, phi_c, eps_v, eps_c, V, n_idx, m_idx, steps, omega, dlt, reorth=False):
    """run_chains in the Tamm-Dancoff approximation: Lanczos on A started from (nm|vc), Sigma by sigma_tda."""
    delta = delta_vc(eps_v, eps_c)

    def op(x):
        return tda_matvec_factored(phi_v, phi_c, V, delta, x[None])[0]

    n = len(n_idx)
    out = dict(alpha=np.zeros((n, steps)), beta=np.zeros((n, steps)), norm2=np.zeros(n),
               len=np.zeros(n, dtype=np.int32), sigma=np.zeros((n, len(omega)), dtype=np.complex128))
    for j in range(n):
        P = tda_start_vector(phi_v, phi_c, V, int(n_idx[j]), int(m_idx[j]))
        a, b, n2, ln = lanczos(op, P, steps, reorth=reorth)
        eps_n, sgn = orbital_energy_sign(eps_v, eps_c, int(n_idx[j]))
        out["alpha"][j], out["beta"][j], out["norm2"][j], out["len"][j] = a, b, n2, ln
        out["sigma"][j] = sigma_tda(a, b, n2, ln, omega, eps_n, sgn, dlt)
    out["sigma_sum"] = sigma_sum(out["sigma"])
    return out
