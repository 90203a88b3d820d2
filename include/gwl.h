/* gwl.h -- C ABI of libgwl: the B200 (sm_100a) hot path of the Lanczos full-frequency GW method
 * of Gao, Tang, Zhao and Chelikowsky, arXiv 2310.20103 ("PAPER.md" below = /root/reference/PAPER.md).
 *
 * What the library computes (all FP64; units eV; arrays row-major, last index fastest):
 *   C      = (A-B)^{1/2}(A+B)(A-B)^{1/2}                                    PAPER.md:52  (Eq. 4)
 *          = diag(Delta^2) + 2 diag(sqrt Delta) K^T V K diag(sqrt Delta),   PAPER.md:41-45 (Eq. 2-3), :122 (Eq. 16)
 *            Delta_vc = eps_c - eps_v,  K[mu, vc] = phi_v(r_mu) phi_c(r_mu),  V = (alpha|beta)  PAPER.md:125 (Eq. 17)
 *   |P_nm> : (P_nm)_vc = (nm|vc) sqrt(Delta_vc)
 *   Lanczos tridiagonalisation started from |P_nm>, one chain per (n,m)      PAPER.md:87-90 (Eq. 13)
 *   <P|(zeta - Op)^{-1}|P> by the Haydock continued fraction                 PAPER.md:92-99 (Eq. 14)
 *   Sigma^corr_mm(omega, n) and its sum over n                               PAPER.md:73-83 (Eq. 10-12)
 * Pair index vc = v*n_c + c.  "delta" of the paper (the broadening) is the argument `eta`.
 *
 * Conventions
 *   - Every entry point returns a gwl_status; the library never throws, aborts or prints.
 *     gwl_last_error() gives a context-owned, NUL-terminated description of the last failure.
 *   - The caller owns every buffer it passes.  set_* calls COPY their inputs; no caller pointer is
 *     kept after a call returns.  Outputs are written into caller-allocated buffers.
 *   - Pointer mode 0 (default): all array arguments are HOST pointers.  Pointer mode 1: all array
 *     arguments of gwl_casida_matvec / gwl_lanczos / gwl_resolvent / gwl_selfenergy /
 *     gwl_set_start_vectors(p) are DEVICE pointers on the context's device (used for timing with the
 *     data already resident in HBM).  Index arrays (n_idx, m_idx, sgn_n, eps_n) and set_orbitals /
 *     set_energies / set_kernel / set_polynomial inputs are always HOST pointers.
 *   - Calls are synchronous on return in pointer mode 0.  In pointer mode 1 work is enqueued on the
 *     context's stream (gwl_set_stream) and the call returns without synchronising, except gwl_lanczos
 *     which synchronises only if a host-side decision is needed (never in the default path).
 *   - One in-flight call per context; contexts are independent.
 *   - Calls out of order (e.g. gwl_lanczos before gwl_set_kernel) return GWL_ESTATE.
 *   - There is no CPU fallback: without a CUDA device gwl_create returns GWL_ECUDA.
 */
#ifndef GWL_H
#define GWL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gwl_ctx gwl_ctx; /* opaque; owns its device memory */

typedef enum {
    GWL_OK = 0,
    GWL_EINVAL = 1, /* bad argument (NULL, non-positive size, eps_c <= eps_v, ...) */
    GWL_ESTATE = 2, /* call out of order */
    GWL_ENOMEM = 3, /* device or host allocation failed */
    GWL_ECUDA = 4   /* CUDA runtime/driver error; see gwl_last_error */
} gwl_status;

/* Create a context for N_v occupied, N_c empty orbitals and N_mu fitting points on the CURRENT CUDA
 * device.  PAPER.md:39 (N_vc = N_v N_c), :117-120 (N_mu).  All sizes >= 1. */
gwl_status gwl_create(gwl_ctx** out, int64_t n_v, int64_t n_c, int64_t n_mu);
void gwl_destroy(gwl_ctx* ctx);                 /* NULL-safe; frees all device memory */
const char* gwl_last_error(const gwl_ctx* ctx); /* "" if none; NULL-safe */

gwl_status gwl_set_pointer_mode(gwl_ctx* ctx, int device_ptrs); /* 0 host (default), 1 device */
/* Run all work on `cuda_stream` (a cudaStream_t / CUstream handle; NULL = the legacy default
 * stream).  The stream stays owned by the caller and must outlive the context's use of it. */
gwl_status gwl_set_stream(gwl_ctx* ctx, void* cuda_stream);

/* Orbitals at the fitting points, PAPER.md:117-123 (C^mu_nm = phi_n(r_mu) phi_m(r_mu)).
 * phi_v [n_mu][n_v], phi_c [n_mu][n_c], host. */
gwl_status gwl_set_orbitals(gwl_ctx* ctx, const double* phi_v, const double* phi_c);
/* Kohn-Sham energies.  eps_v [n_v], eps_c [n_c], host.
 * GWL_EINVAL unless min(eps_c) > max(eps_v) (Delta > 0 is needed for (A-B)^{1/2}). */
gwl_status gwl_set_energies(gwl_ctx* ctx, const double* eps_v, const double* eps_c);
/* Two-centre integrals (alpha|beta), PAPER.md:125 (Eq. 17).  V [n_mu][n_mu], host, symmetric
 * (only V itself is used; symmetry is the caller's responsibility). */
gwl_status gwl_set_kernel(gwl_ctx* ctx, const double* V);
/* Optional polynomial square root D ~ p_g(C).  cheb[g+1] are coefficients in
 * the Chebyshev basis on [lo, hi]: p_g(x) = sum_j cheb[j] T_j((2x-hi-lo)/(hi-lo)).  g >= 1 switches
 * gwl_lanczos to Op = p_g(C) and gwl_selfenergy to Eq. 12 + Eq. 14 ("poly mode"); g = 0 (cheb may be
 * NULL) clears it: Op = C and gwl_selfenergy evaluates Eq. 11 on the Ritz pairs of T_L ("direct mode"). */
gwl_status gwl_set_polynomial(gwl_ctx* ctx, int g, const double* cheb, double lo, double hi);

/* Coefficients for gwl_set_polynomial: cheb[0..g] (HOST, caller-allocated) of the least-squares fit of sqrt(x) at the
 * 4 (g + 1) Chebyshev nodes of [lo, hi] -- "a polynomial function p_g(x) ... fitted to sqrt(x)" with the coefficients found "via
 * least-squares fitting", g = 7 in the paper's runs.  Host arithmetic only (closed form
 * in the Chebyshev basis); needs no context and no GPU.  GWL_EINVAL unless 1 <= g <= 64 and 0 < lo < hi. */
gwl_status gwl_fit_sqrt_polynomial(int g, double lo, double hi, double* cheb);
/* The fitting range for it.  steps = 0: the heuristic [0.8 min Delta^2, 1.25 max Delta^2] from the energies of
 * gwl_set_energies, no GPU work.  steps >= 2: lo = 0.8 min Delta^2 (a lower bound of C when V is positive semidefinite) and
 * hi = (1 + margin) max(lam_max of gwl_spectrum_bounds(steps), max Delta^2); margin (e.g. 0.02) cushions an unconverged top
 * Ritz value and is a heuristic, not a bound.  Like gwl_spectrum_bounds this replaces the chain list and synchronises.
 * lo, hi HOST outputs.  Real-orbital contexts with energies set (GWL_ESTATE otherwise). */
gwl_status gwl_sqrt_fit_range(gwl_ctx* ctx, int64_t steps, double margin, double* lo, double* hi);

/* Extremal eigenvalues of the operator for the fitting range of p_g: "One can use standard Lanczos algorithm to
 * determine the extremal eigenvalues min(Omega_s^2) and max(Omega_s^2) of C".  Runs `steps`
 * (2..512; 30-60 is plenty) Lanczos steps on the operator itself (C, or A in the TDA; never p_g(C)) from a generic
 * pseudo-random start vector and returns lam_max = theta_max + r_max and lam_min = theta_min - r_min, where theta are
 * the extreme Ritz values and r = b_L |s_L| their residual norms (an eigenvalue lies within r of each; the top of a
 * spectrum with a separated upper edge converges in a few steps, the dense lower edge slowly -- lam_min is a lower
 * ESTIMATE that can undershoot; with V positive semidefinite min(Delta)^2 is a rigorous lower bound of C).
 * Host outputs.  Replaces the chain list (call it before gwl_set_chains / gwl_set_start_vectors), synchronises. */
gwl_status gwl_spectrum_bounds(gwl_ctx* ctx, int64_t steps, double* lam_min, double* lam_max);

/* SURVEY.md 8(f)-3, first step.  GWL_RPA (default): the operator is C of Eq. 4.  GWL_TDA: the Tamm-Dancoff
 * approximation, "setting matrix B = 0 in the RPA Casida matrix ... only a Hermitian matrix A remains, and a standard
 * Lanczos algorithm for Hermitian matrix can be used" (formulas PAPER.md:306-313), here for real
 * orbitals and one k-point: the operator becomes A = diag(Delta) + K^T V K (Eq. 2), chains start from
 * P_vc = (nm|vc) (no sqrt(Delta) factor), gwl_casida_matvec applies A, and gwl_selfenergy evaluates
 * Sigma(omega, n) = <P| 1/(omega - eps_n + eta_n (A - i eta)) |P> = -eta_n R_A(-eta_n z_n) by Eq. 14.
 * Switching invalidates the results of the last gwl_lanczos.  GWL_ESTATE if a polynomial is set (it fits sqrt(C)).
 * On a complex-orbital context (gwl_tdc_create, below) GWL_TDA is the default and GWL_RPA selects the pseudo-Hermitian
 * Lanczos for the full C^RPA(q) described there. */
#define GWL_RPA 0
#define GWL_TDA 1
gwl_status gwl_set_approximation(gwl_ctx* ctx, int approximation);

/* y = C x for nvec vectors, PAPER.md:52 with the factorisation of PAPER.md:128, :383-389:
 * y = Delta^2 o x + 2 sqrt(Delta) o K^T ( V ( K ( sqrt(Delta) o x ) ) ).  Always C, never p_g(C).
 * x, y [nvec][n_v][n_c]; x and y must not overlap.  nvec >= 0 (0 is a no-op). */
gwl_status gwl_casida_matvec(gwl_ctx* ctx, const double* x, double* y, int64_t nvec);

/* Chains by orbital indices: chain j starts from |P_{n_j m_j}>.  An index in
 * [0, n_v + n_c): < n_v is the occupied orbital of that number (eta_n = +1), otherwise the empty
 * orbital idx - n_v (eta_n = -1).  eps_n and eta_n of PAPER.md:62, :79 are taken from n_idx.  Host arrays. */
gwl_status gwl_set_chains(gwl_ctx* ctx, int64_t n_chains, const int32_t* n_idx, const int32_t* m_idx);
/* Alternative: explicit start vectors p [n_chains][n_v][n_c] (pointer mode applies to p) with
 * eps_n [n_chains], sgn_n [n_chains] (+1/-1), host. */
gwl_status gwl_set_start_vectors(gwl_ctx* ctx, int64_t n_chains, const double* p,
                                 const double* eps_n, const int32_t* sgn_n);

/* Lanczos tridiagonalisation of Op (C, or p_g(C) in poly mode) for the first n_chains chains set
 * above, `block` chains at a time (the last block may be short), PAPER.md:87-90 (Eq. 13).
 * steps = number of Op applications = dimension of T_L (1..100000).  reorth: 0 off, 1 two-pass full
 * reorthogonalisation against all previous Lanczos vectors of the same chain; then steps <= GWL_MAX_REORTH_STEPS
 * (GWL_EINVAL above it: the kernels keep one projection coefficient per earlier vector in shared memory, and the
 * basis of steps x block x N_vc doubles has to fit in HBM anyway).
 * Outputs (may be NULL to skip; the context keeps its own copy for gwl_resolvent/gwl_selfenergy):
 *   alpha [n_chains][steps]  a_0 .. a_{L-1}
 *   beta  [n_chains][steps]  beta[k] = b_{k+1}; beta[steps-1] is returned but not part of T_L
 *   norm2 [n_chains]         <P|P>
 *   len   [n_chains]         effective length <= steps: on breakdown (b_{k+1} <= 1e-12 max_i(|a_i|+b_i))
 *                            len = k+1, b_{k+1} is stored as 0 and the tail is zero-filled. */
#define GWL_MAX_REORTH_STEPS 8192
gwl_status gwl_lanczos(gwl_ctx* ctx, int64_t n_chains, int64_t steps, int64_t block, int reorth,
                       double* alpha, double* beta, double* norm2, int32_t* len);

/* r[j][i] = <P_j|(zeta_i - Op)^{-1}|P_j> by Eq. 14 from the tridiagonals of the last
 * gwl_lanczos: norm2 / (zeta - a_0 - b_1^2/(zeta - a_1 - ...)), truncated at len_j.
 * zeta [n_zeta][2] (re, im); r [n_chains][n_zeta][2]. */
gwl_status gwl_resolvent(gwl_ctx* ctx, const double* zeta, int64_t n_zeta, double* r);

/* Sigma^corr_mm(omega, n_j) for every chain of the last gwl_lanczos, PAPER.md:77-83 (Eq. 11-12), with
 * z_n = omega - eps_n - i eta_n eta (eta > 0 is the paper's delta), and optionally
 * the sum over chains, PAPER.md:73 (Eq. 10).
 * omega [n_omega]; sigma [n_chains][n_omega][2] (may be NULL); sigma_sum [n_omega][2] (may be NULL). */
gwl_status gwl_selfenergy(gwl_ctx* ctx, const double* omega, int64_t n_omega, double eta,
                          double* sigma, double* sigma_sum);

/* ---- the rest of one quasiparticle state ------------------------------------------------ */

/* Sigma^corr_mm(omega) of ONE orbital m, summed over all n = 0 .. n_v+n_c-1 (Eq. 10; one Lanczos
 * chain per n started from |P_nm>): equivalent to gwl_set_chains(all n, m) + gwl_lanczos(steps,
 * block, reorth) + gwl_selfenergy(sum only), and it leaves the context in that state (gwl_resolvent etc. then
 * refer to these n_v+n_c chains).  m_idx as in gwl_set_chains.  omega [n_omega], sigma_mm [n_omega][2]
 * (pointer mode applies to both). */
gwl_status gwl_selfenergy_state(gwl_ctx* ctx, int32_t m_idx, int64_t steps, int64_t block, int reorth,
                                const double* omega, int64_t n_omega, double eta, double* sigma_mm);

/* Exchange part Sigma^ex_mm = - sum_v (vm|vm) over the occupied orbitals, PAPER.md:57 (Eq. 6), with
 * (vm|vm) = rho_vm^T V rho_vm, rho_vm(mu) = phi_v(r_mu) phi_m(r_mu) (Eq. 16).  m_idx [n_states] host, indices
 * as in gwl_set_chains; sigma_x [n_states] (pointer mode applies).  Needs orbitals and kernel. */
gwl_status gwl_exchange(gwl_ctx* ctx, int64_t n_states, const int32_t* m_idx, double* sigma_x);

/* Quasiparticle equation: E(omega) = eps_m + <m|Sigma(omega) - V_xc|m> on the frequency grid,
 * solved for E(omega) = omega by Newton-Raphson on the piecewise-linear interpolant of Re Sigma^corr, started
 * at eps_m, clamped to the grid, until |step| <= 1e-10 eV or 50 iterations (reading Q18).
 * eps_m, vxc_m [n_states] host.  sigma_x [n_states], sigma_c [n_states][n_omega][2], omega [n_omega]
 * (ascending, n_omega >= 2), and the outputs e_qp [n_states], z_qp [n_states] (renormalisation factor
 * 1/(1 - dReSigma/domega) at the solution), iters [n_states] (may be NULL) follow the pointer mode. */
gwl_status gwl_qp_solve(gwl_ctx* ctx, int64_t n_states, const double* eps_m, const double* vxc_m,
                        const double* sigma_x, const double* sigma_c, const double* omega, int64_t n_omega,
                        double* e_qp, double* z_qp, int32_t* iters);

/* ---- complex orbitals and k-points in the Tamm-Dancoff approximation -------------------------------
 * PAPER.md:157 and Supplemental Material section 1: for periodic systems the orbitals are complex and
 * "if the Tamm-Dancoff approximation is used ... only a Hermitian matrix A remains, and a standard Lanczos algorithm for
 * Hermitian matrix can be used".  One context serves ONE transferred momentum q:
 *   A(q)_{vck,v'c'k'} = (eps_{ck+q} - eps_{vk}) delta + (vk, ck+q | v'k', c'k'+q)
 *                     = diag(Delta) + K^H V K,  K[mu, (k,v,c)] = conj(psi_{vk}(r_mu)) psi_{ck+q}(r_mu),
 *   Sigma^corr_{mk,mk}(omega) = 2/(N_q N_k) sum_n sum_q <P_nmk(q)| 1/(omega - eps_{nk-q} + eta (A(q) - i delta)) |P_nmk(q)>
 * with V = (alpha|beta) real symmetric as set by gwl_set_kernel (A Hermitian and B symmetric, need that).
 * Pair index (k, v, c), c fastest.  Complex arrays are interleaved (re, im) doubles.
 * A context made by gwl_tdc_create accepts gwl_tdc_set_orbitals / gwl_tdc_set_energies / gwl_set_kernel /
 * gwl_tdc_set_chains / gwl_tdc_matvec and then gwl_lanczos, gwl_resolvent, gwl_selfenergy, gwl_get_* exactly as above
 * (alpha, beta are real: A is Hermitian; gwl_selfenergy includes the prefactor 2/(N_q N_k) in every chain and evaluates
 * Eq. 14 at -eta_n z_n as in GWL_TDA); the real-orbital set_* calls, gwl_set_polynomial, gwl_exchange return GWL_ESTATE.
 *
 * Full RPA with complex orbitals (gwl_set_approximation(ctx, GWL_RPA) on such a context): "if RPA is used, then a Lanczos-based
 * method designed for pseudo-Hermitian matrices can be adopted".  The paper fixes the target,
 *   Sigma^corr_{mk,mk}(omega) = 2/(N_q N_k) sum_n sum_q sum_s |W^s|^2 / (omega - eps_{nk-q} + eta (Omega_s(q) - i delta)),
 *   W^s = sum_j [ (nk-q, mk | v'k', c'k'+q) X^s_j + (nk-q, mk | c'k'+q, v'k') Y^s_j ],
 * over the positive eigenvalues of C^RPA(q) = [[A, B], [-B^*, -A^*]], B = K^H V conj(K), and leaves the
 * Lanczos scheme to its refs. [34, 36, 74]; the one built here (reading Q24): C^RPA = F Omega^ with F = diag(1, -1) and
 * Omega^ = [[A, B], [B^*, A^*]] Hermitian positive definite is self-adjoint in <a, b>_O = a^H Omega^ b, so a three-term Lanczos
 * in that inner product, started from u = F conj([P1; P2]) (the printed integrals), gives a real symmetric T_L with
 *   sum_{s: Omega_s > 0} |W^s|^2 g(Omega_s) ~ <u,u>_O sum_{i: theta_i > 0} w_i g(theta_i) / theta_i     (Ritz pairs of T_L),
 * exact at L = 2 N_k N_v N_c.  One step costs one product with Omega^ (2 K, 1 V, 2 K^H contractions: twice a TDA step).
 * gwl_lanczos then returns the alpha, beta of that T_L and norm2 = <u,u>_O; gwl_selfenergy evaluates the sum above (with the
 * prefactor); gwl_resolvent gives <u|(zeta - C^RPA)^{-1}|u>_O by Eq. 14 (both branches). */
#define GWL_TDC_MAX_KV 65535 /* n_k * n_v of a complex context (the (k, v) planes are a grid dimension); GWL_EINVAL above it */
gwl_status gwl_tdc_create(gwl_ctx** out, int64_t n_k, int64_t n_v, int64_t n_c, int64_t n_mu, int64_t n_q);
/* psi_v [n_k][n_mu][n_v][2] = psi_{v k}(r_mu); psi_cq [n_k][n_mu][n_c][2] = psi_{c k+q}(r_mu) (slot k holds the conduction
 * orbitals of momentum k+q: the caller does the momentum bookkeeping).  Host. */
gwl_status gwl_tdc_set_orbitals(gwl_ctx* ctx, const double* psi_v, const double* psi_cq);
/* eps_v [n_k][n_v], eps_cq [n_k][n_c] (eps_{c k+q} in slot k), host; GWL_EINVAL unless min(eps_cq) > max(eps_v). */
gwl_status gwl_tdc_set_energies(gwl_ctx* ctx, const double* eps_v, const double* eps_cq);
/* Chain j starts from the ket of PAPER.md:310-313 for (n k-q, m k): chains [n_chains][4] = (slot of n, n index,
 * slot of m, m index), host; an orbital (slot s, index i) is psi_v[s][:, i] for i < n_v (eta = +1), else the conduction
 * orbital psi_cq[s][:, i - n_v] (eta = -1).  The printed elements P_{v'c'k'} = (nk-q, mk | v'k', c'k'+q) enter the pole
 * strengths bilinearly (W^s = sum P X^s), so the Lanczos start vector is their complex conjugate
 * K^H (V rho~), rho~ = psi_m conj(psi_n) (reading Q20; identical for real orbitals). */
gwl_status gwl_tdc_set_chains(gwl_ctx* ctx, int64_t n_chains, const int32_t* chains);
/* y = A(q) x for nvec complex vectors x, y [nvec][n_k][n_v][n_c][2] (pointer mode applies); x and y must not overlap. */
gwl_status gwl_tdc_matvec(gwl_ctx* ctx, const double* x, double* y, int64_t nvec);
/* [ox; oy] = Omega^ [x; y] = [A x + B y; B^* x + A^* y] (C^RPA [x; y] = [ox; -oy]) for nvec pairs of complex
 * vectors, each [nvec][n_k][n_v][n_c][2] (pointer mode applies); inputs and outputs must not overlap.  Either approximation. */
gwl_status gwl_tdc_matvec_rpa(gwl_ctx* ctx, const double* x, const double* y, double* ox, double* oy, int64_t nvec);

/* The q-term of Sigma^corr_{mk,mk}(omega) (PAPER.md:288 / :310) summed over ALL n = 0 .. n_v+n_c-1 of slot kn (the orbitals of
 * momentum k-q): one chain per n from (n kn, m km), in the context's approximation (GWL_TDA or GWL_RPA), prefactor 2/(N_q N_k)
 * included; the sum over q is the caller's (one context per q).  Equivalent to gwl_tdc_set_chains(all n) + gwl_lanczos +
 * gwl_selfenergy(sum only) and leaves the context in that state.  omega [n_omega], sigma_mm [n_omega][2] (pointer mode applies). */
gwl_status gwl_tdc_selfenergy_state(gwl_ctx* ctx, int32_t kn, int32_t km, int32_t m_idx, int64_t steps, int64_t block, int reorth,
                                    const double* omega, int64_t n_omega, double eta, double* sigma_mm);

/* ---- interpolative separable density fitting front end -------------------------------------------
 * PAPER.md:115-128 (Eq. 15-17): phi_n(r) phi_m(r) ~ sum_mu zeta_mu(r) C^mu_nm with C^mu_nm = phi_n(r_mu) phi_m(r_mu) at given
 * interpolation points r_mu = r[idx[mu]] (ISDF, refs. [62, 63]); zeta is the least-squares solution
 * zeta = Z C^T (C C^T)^{-1} over the pairs of ALL n_v + n_c orbitals, computed from the separable normal equations
 * Z C^T = (Phi Phi_mu^T) o (Phi Phi_mu^T) (Cholesky; GWL_EINVAL if C C^T is not positive definite); then
 * (alpha|beta) = int int zeta_alpha(r) zeta_beta(r') / |r - r'| (Eq. 17) as the grid quadrature
 * sum_ij zeta_alpha(r_i) G_ij zeta_beta(r_j), G_ij = weight^2 14.4 / sqrt(|r_i - r_j|^2 + soft^2) eV (softened at short range:
 * the stand-in for the real-space Poisson solve).  The paper's code runs this part on CPUs.
 * Inputs (host): phi_v_grid [n_r][n_v], phi_c_grid [n_r][n_c] orbitals on the real-space grid, r [n_r][3] grid points
 * (Angstrom), weight = h^3, soft > 0, idx [n_mu] distinct grid indices.  n_mu <= n_r <= GWL_ISDF_MAX_NR.  Device memory is about
 * 8 n_r (n_v + n_c + 3 n_mu + 8192) bytes: G is generated in panels of 8192 rows that feed the G zeta GEMM (GWL_ENOMEM if it does not fit).
 * Effect: the context's orbitals become the grid orbitals at the interpolation points and its kernel becomes (alpha|beta),
 * exactly as after gwl_set_orbitals + gwl_set_kernel (gwl_set_energies is still needed).  Optional host outputs:
 * zeta_t [n_mu][n_r] (zeta transposed) and V_out [n_mu][n_mu]; either may be NULL. */
#define GWL_ISDF_MAX_NR 4194304 /* grid points of gwl_isdf_build; the Coulomb quadrature matrix is walked in row panels, never held */
gwl_status gwl_isdf_build(gwl_ctx* ctx, int64_t n_r, const double* phi_v_grid, const double* phi_c_grid, const double* r,
                          double weight, double soft, const int32_t* idx, double* zeta_t, double* V_out);

/* Interpolation points for gwl_isdf_build by centroidal Voronoi tessellation (weighted k-means).  PAPER.md:128 names the
 * ISDF method of its refs. [13, 62, 63] and is silent on how the points are chosen; this is the k-means choice of that
 * literature (reading Q22).  Lloyd iterations on the grid points r [n_r][3] with weights weight [n_r] >= 0 (e.g.
 * sum_n phi_n(r)^2): assign every point to its nearest centroid (ties: the lowest centroid index), move every centroid to
 * the weighted mean of its points (an empty cluster keeps its centroid), starting from the grid points init_idx [n_mu],
 * at most max_iters times or until no assignment changes; finally every centroid is replaced by the nearest grid point of
 * its own cluster (ties: the lowest index), so the n_mu = ctx's N_mu points are distinct.  Host arrays; idx [n_mu] receives
 * the grid indices (-1 for a cluster that ended empty), *iters_done (may be NULL) the number of centroid updates. */
gwl_status gwl_isdf_select_points(gwl_ctx* ctx, int64_t n_r, const double* r, const double* weight, const int32_t* init_idx,
                                  int64_t max_iters, int32_t* idx, int32_t* iters_done);

/* ---- SURVEY.md 8(f)-4, second part: point-group symmetry blocks of the Casida matrix ---------------------------------------
 * "One can further exploit the point-group symmetries to make the Casida matrix C block diagonal and simplify the calculation
 * of matrix-vector products [64]".  Reading (Q25): an abelian group of order g = 2^n_gen (n_gen <= 3
 * commuting generators, e.g. mirror planes: C_s, C_2v, D_2h, ...) with one-dimensional real irreducible representations.  An
 * irrep is a bit mask in [0, g), its character at the element h is (-1)^popcount(irrep & h), the product of two irreps is their
 * XOR.  Orbitals are sorted by irrep (nv_irrep[a] occupied, nc_irrep[a] empty orbitals of irrep a).  The pair (v, c) belongs to
 * block gamma = irrep(v) ^ irrep(c); C does not couple different blocks and |P_nm> lies in block irrep(n) ^ irrep(m).  With
 * fitting points closed under the group (n_mu_w points r_mu of the irreducible wedge and their images h r_mu), within block gamma
 *   K^T V K = Kw^T Vg Kw,  Kw = K on the wedge,  Vg[mu][nu] = g sum_h chi_gamma(h) V(r_mu, h r_nu),
 * so one chain-step costs 4 n_mu_w N_pairs(gamma) + 2 n_mu_w^2 flop: about g^2 fewer than without the symmetry.
 * A context made by gwl_sym_create takes gwl_sym_set_orbitals / gwl_set_energies / gwl_sym_set_kernel once, then
 * gwl_sym_select(gamma) makes block gamma the operator: gwl_sym_matvec, gwl_set_chains (pairs (n, m) of that block only, else
 * GWL_EINVAL), gwl_lanczos, gwl_resolvent, gwl_selfenergy, gwl_set_polynomial and the gwl_get_* calls then work as on a plain
 * context, and so does gwl_spectrum_bounds (bounds of the selected block); gwl_sym_selfenergy_state walks all blocks for one
 * orbital m; gwl_exchange works on any orbital (rho_vm transforms as irrep(v) ^ irrep(m): every irrep of v goes against its own
 * reduced kernel) and gwl_qp_solve is unchanged.  Block vectors hold the pairs of block gamma ordered by the irrep a of v
 * (ascending), then v, then c over the irrep a ^ gamma.  gwl_set_orbitals, gwl_set_kernel, gwl_casida_matvec,
 * gwl_set_start_vectors, gwl_selfenergy_state, gwl_set_approximation and gwl_isdf_build return GWL_ESTATE on such a context. */
gwl_status gwl_sym_create(gwl_ctx** out, int n_gen, const int32_t* nv_irrep /*[2^n_gen]*/, const int32_t* nc_irrep /*[2^n_gen]*/,
                          int64_t n_mu_w);
/* Orbital values at the wedge points: phi_v_w [n_mu_w][N_v], phi_c_w [n_mu_w][N_c] (N_v = sum nv_irrep, N_c = sum nc_irrep), host. */
gwl_status gwl_sym_set_orbitals(gwl_ctx* ctx, const double* phi_v_w, const double* phi_c_w);
/* Rows of (alpha|beta) for the wedge points against every image: V_wf [n_mu_w][g][n_mu_w] = V(r_mu, h r_nu), host; element h is
 * the bit mask of the generators applied.  The g reduced kernels Vg are formed on the device. */
gwl_status gwl_sym_set_kernel(gwl_ctx* ctx, const double* V_wf);
/* Makes block gamma the operator (needs the energies); *n_pairs (may be NULL) receives its dimension.  GWL_EINVAL if the block
 * has no pairs.  Invalidates chains and results. */
gwl_status gwl_sym_select(gwl_ctx* ctx, int gamma, int64_t* n_pairs);
/* y = C_gamma x for nvec vectors of the selected block, x, y [nvec][n_pairs] (pointer mode applies); must not overlap. */
gwl_status gwl_sym_matvec(gwl_ctx* ctx, const double* x, double* y, int64_t nvec);
/* Sigma^corr_mm(omega) = sum over ALL n (Eq. 10) for one orbital m, block by block: for every gamma the chains
 * n with irrep(n) ^ irrep(m) = gamma run inside block gamma and Eq. 10 is accumulated on the device.  Arguments as
 * gwl_selfenergy_state; leaves the last non-empty block selected. */
gwl_status gwl_sym_selfenergy_state(gwl_ctx* ctx, int32_t m_idx, int64_t steps, int64_t block, int reorth, const double* omega,
                                    int64_t n_omega, double eta, double* sigma_mm);

/* CUDA-event totals (ms) of the last gwl_lanczos: time inside Casida products (S2), inside the Lanczos
 * vector kernels (S4) and overall.  Any pointer may be NULL.  Synchronises the stream. */
gwl_status gwl_get_timing(gwl_ctx* ctx, double* ms_matvec, double* ms_vecops, double* ms_total);

/* Profiling level: 0 no events -- this is also the switch for the CUDA-graph replay of the step loop: at level 0 gwl_lanczos
 * replays six steps at a time from a captured graph when the problem is launch-bound (N_vc <= 65 536, reorth = 0, real
 * orbitals, steps >= 16, at most 8 chain blocks per call); the results are bit-identical to plain launches, which every
 * other level uses; 1 (default) one CUDA-event triple per Lanczos step (feeds gwl_get_timing);
 * 2 additionally an event pair around every kernel launch, tagged with its class (feeds gwl_get_kernel_times). */
gwl_status gwl_set_profiling(gwl_ctx* ctx, int level);
/* Per-class device time (ms) and launch count since the start of the last gwl_lanczos (including later
 * gwl_resolvent / gwl_selfenergy calls); needs profiling level 2.  ms and count have GWL_N_KERNEL_CLASSES entries:
 * 0 K.X GEMM, 1 V GEMM, 2 K^T.W GEMM (with the Delta epilogue), 3 split-K reduction, 4 scaling/axpy/dot
 * helpers, 5 Lanczos recurrence kernels, 6 reorthogonalisation, 7 continued fraction / Ritz / Sigma.
 * Synchronises the stream. */
#define GWL_N_KERNEL_CLASSES 8
gwl_status gwl_get_kernel_times(gwl_ctx* ctx, double* ms, int64_t* count);

/* Number of kernels launched by this context since creation (for bench.py's gpu_launches). */
gwl_status gwl_get_launch_count(gwl_ctx* ctx, int64_t* n_launches);

/* The one entry point that allocates nothing: norm2[j] = <P_j|P_j> = sum_vc p[j][vc]^2, the numerator of the continued
 * fraction (Eq. 14) and the same quantity gwl_lanczos returns as `norm2`.
 *
 * It is for host programs that cannot let a library call cudaMalloc: a driver that has given all of HBM to its own pool
 * (a later cudaMalloc fails or fragments the remainder), or one that keeps other streams busy (cudaMalloc / cudaFree
 * synchronise the whole device and would stall them).  Everything else in this header needs a gwl_ctx, whose buffers come
 * from cudaMalloc; this call needs no context and calls no cudaMalloc, cudaFree or allocating library routine.  The partial
 * sums of its two-stage reduction go into a fixed array of GWL_STATIC_SCRATCH_BYTES that is part of the library image: every
 * GPU that loads the library's kernels holds those bytes until the process exits.
 *
 *   p      [n_chains][n_vc]  DEVICE pointer, read only, contiguous (row stride n_vc)
 *   norm2  [n_chains]        DEVICE pointer, written; must not overlap p
 *   cuda_stream              cudaStream_t the two kernels are enqueued on (NULL = legacy default stream); the call does not
 *                            synchronise: norm2 is valid once the stream has reached this point
 *   err, err_len             optional caller-owned buffer for a NUL-terminated description of a failure ("" on success);
 *                            err may be NULL
 * p and norm2 must live on the CURRENT device (cudaSetDevice); the caller owns them.
 * Limits: 0 <= n_chains <= GWL_STATIC_MAX_CHAINS, 1 <= n_vc <= GWL_STATIC_MAX_NVC, else GWL_EINVAL with the limit named in
 * err; nothing is launched then.  n_chains = 0 is a no-op.  A failed set-up or launch returns GWL_ECUDA.
 * First call on each device: the library looks up the device address of its scratch array once (cudaGetSymbolAddress, with
 * that device current) and keeps it.  Make that first call during start-up, outside any stream capture.
 * Sharing: all calls in the process use the same array on a given device.  It keeps the previous call's partial sums; that
 * is harmless because each call writes every slot before it reads it (nothing has to start at zero).  Two calls whose
 * kernels can overlap on one GPU (different streams, or different host threads) race on the array and give wrong norms:
 * order them on one stream or with events.
 * Results repeat bit for bit for the same arguments and agree with gwl_lanczos's norm2 to rounding (1e-12 relative). */
#define GWL_STATIC_SCRATCH_BYTES 262144          /* 32 768 doubles */
#define GWL_STATIC_MAX_CHAINS 4096
#define GWL_STATIC_MAX_NVC 4294967296LL          /* 2^32 pairs */
gwl_status gwl_chain_norms_static(const double* p, int64_t n_chains, int64_t n_vc, double* norm2, void* cuda_stream,
                                  char* err, int64_t err_len);

/* Measurement helper, not part of the method: run a register-resident mma.sync.m8n8k4.f64 (kind 0) or
 * DFMA (kind 1) loop on every SM of the current device and return the achieved FP64 TFLOP/s.
 * This is the denominator DESIGN.md uses for the FP64 tensor roofline. */
gwl_status gwl_probe_fp64_peak(int kind, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* GWL_H */
