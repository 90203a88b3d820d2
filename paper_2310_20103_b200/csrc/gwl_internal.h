// Internal declarations shared by the translation units of libgwl.  No torch, no oracle code.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>
#include <vector>

#include "../../include/gwl.h"

namespace gwl {

constexpr int BK = 16;  // doubles per k-tile row = one 128-byte swizzled shared-memory row

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
static inline int64_t ceil_div(int64_t x, int64_t m) { return (x + m - 1) / m; }

// ---------------------------------------------------------------------------------------------
// GEMM layer (kr_gemm.cu).  All three contractions of the Casida product are "TN" GEMMs
//   out[n][m] = sum_k A[m][k] * B[n][k]      (both operands K-contiguous, output M-contiguous)
// with A = the matrix (Phi_c, V, Phi_c^T) and B = the block of vectors.
// ---------------------------------------------------------------------------------------------
enum GemmMode { MODE_FWD = 0, MODE_PLAIN = 1, MODE_BWD = 2 };
enum GemmEpi { EPI_STORE = 0, EPI_CASIDA = 1, EPI_START = 2, EPI_CHEB = 3 };

struct GemmParams {
    const double* A;      // [M][lda]
    int64_t lda;
    const double* B;      // [N][ldb]
    int64_t ldb;
    int M, N;             // valid rows of A / of B
    int kt_total;         // k-tiles (of BK) in the whole reduction
    int a_wrap;           // FWD: k-tiles per v (n_cp / BK); k-tile kt = (c-tile kt / n_v, v = kt % n_v)
    int kt_per_split;     // FWD/PLAIN: k-tiles handled by one blockIdx.z
    const double* scale;  // Phi_v^T [n_v][lds]: FWD row scale (index m), BWD k scale (index k)
    int64_t lds;
    int scale_rows;       // n_v
    double* out;          // EPI_STORE: out[z*out_split_stride + n*ldo + m]; CASIDA/START: out[n*ldo + v*n_c + m]
    int64_t ldo;
    int64_t out_split_stride;
    const double* X;      // EPI_CASIDA: x[n*ldx + v*n_c + m]
    int64_t ldx;
    const double* d2;     // diagonal term [n_vc]: Delta^2 (RPA, operator C) or Delta (TDA, operator A)
    const double* s;      // scaling [n_vc]: sqrt(Delta) (RPA) or 1 (TDA)
    double coupling;      // epilogue: y = d2 x + coupling * s * u; 2 (A+B, RPA) or 1 (A alone, TDA)
    double* dotpart;      // CASIDA: sum_m x*y, START: sum_m p*p ; dotpart[n*dot_stride + v*gridDim.x + blockIdx.x]
    int dot_stride;
    int n_c;
    // EPI_CHEB: one term of the Chebyshev recurrence of p_g(C) fused behind the Casida epilogue:
    //   y = d2 x + coupling s u;  t = ca y + cb x + cc t0;  w = first ? c0 x + cw t : w + cw t;
    //   out = t, xs_out = s o t (padded layout, the next K.X operand), dotpart = sum q w (last term only).
    // x, t0, w, q and out share ldx; t0 may alias out (every element is read and written by the same thread).
    const double* T0;     // t_{j-2} or NULL (then cc is ignored)
    double* Wacc;         // running sum p_g(C) q
    const double* Q;      // Lanczos vector for the alpha dots, or NULL
    double* xs_out;       // [N][n_v][n_cp] or NULL
    int64_t ldxs;
    int n_cp;
    double ca, cb, cc, cw, c0;
    int first;
    // BWD (persistent stream-K grid, kr_gemm.cu): tile grid, partial-tile workspace and hand-over flags
    int tiles_m, tiles_n, n_tiles;  // filled by launch_gemm
    double* ws;                     // [grid][BM*BN] partial accumulators, >= gemm_bwd_ws_bytes()
    unsigned* flags;                // [grid], flags[cta] == epoch once that CTA's partial of THIS launch is visible
    unsigned epoch;                 // differs from every earlier launch that used the same flags (never 0)
    int n_sm;
};

struct GemmPlan {
    int bm, bn;       // CTA tile
    int splits;       // grid.z for FWD/PLAIN
    int kt_per_split;
};

// Chooses tile and split so that the grid is close to a multiple of the SM count.
GemmPlan plan_gemm(int mode, int M, int N, int kt_total, int a_wrap, int n_sm);
// Bytes of GemmParams::ws / ::flags a BWD launch may touch on a device with n_sm SMs.
size_t gemm_bwd_ws_bytes(int n_sm);
size_t gemm_bwd_flag_bytes(int n_sm);
// Launches; returns cudaGetLastError().  `nz` = splits (FWD/PLAIN) or n_v (BWD).
cudaError_t launch_gemm(int mode, int epi, const GemmPlan& plan, const GemmParams& p, int nz, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// Complex GEMM layer (kr_gemm_c.cu): the two Khatri-Rao contractions of the periodic Tamm-Dancoff operator
// A(q) = diag(Delta) + K^H V K, K[mu, (k,v,c)] = conj(psi_vk(mu)) psi_ck+q(mu).  All arrays planar.
// ---------------------------------------------------------------------------------------------
struct GemmParamsC {
    const double* A;       // FWD: psi_cq planar [2][n_mu][lda = n_k*n_cp]; BWD: psi_cq^T planar [2][a_rows = n_k*n_c][lda = n_mup]
    int64_t lda, a_plane;  // a_plane: elements between the real and the imaginary plane
    int a_rows;
    const double* B;       // FWD: x [N][ldb = 2*n_kv*n_cp], planes side by side; BWD: W planar [2][N][ldb]
    int64_t ldb, b_plane;
    int b_plane_cols;      // FWD: column offset of the imaginary plane (n_kv * n_cp)
    int M, N;              // FWD: M = n_mu; BWD: M = n_c (rows of one k-point's conduction block)
    int kt_total;          // FWD: n_kv * (n_cp / 16); BWD: n_mup / 16
    int a_wrap;            // FWD: k-tiles per (k, v) = n_cp / 16
    int kt_per_split;      // FWD: k-tiles per blockIdx.z
    int n_v, n_c;          // occupied orbitals per k-point; conduction orbitals per k-point
    const double* scale;   // psi_v^T planar [2][scale_rows = n_kv][lds]
    int64_t lds, s_plane;
    int scale_rows;
    double* out;           // STORE: out[z*out_split_stride + n*ldo + m] (+ o_plane: imaginary); BWD: out[n*ldo + kv*n_c + m]
    int64_t ldo, o_plane, out_split_stride;
    const double* X;       // CASIDA: x[n*ldx + kv*n_c + m] (+ x_plane)
    int64_t ldx, x_plane;
    const double* d2;      // diagonal term [n_kv*n_c]
    double coupling;
    double* dotpart;       // [n*dot_stride + kv*tiles_m + m-tile]
    int dot_stride;
};
int gemm_c_tiles_m(int M);  // m-tiles of a BWD launch (dot partials per kv)
GemmPlan plan_gemm_c(int M, int N, int kt_total, int n_sm);  // split-K plan of the FWD product
cudaError_t launch_gemm_c(int mode, int epi, const GemmParamsC& p, int nz, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// Vector kernels (vec_kernels.cu).  Block vectors are [nb][n_vc]; partial sums are [nb][npart].
// ---------------------------------------------------------------------------------------------
constexpr int VEC_THREADS = 256;
int vec_parts(int64_t n_vc);  // number of partial-sum blocks per column used by the kernels below

// tda = 0: d2 = Delta^2, s = sqrt(Delta);  tda = 1: d2 = Delta, s = 1
cudaError_t launch_build_delta(const double* eps_v, const double* eps_c, int n_v, int n_c, double* d2, double* s,
                               int tda, cudaStream_t st);
// x[i] = pseudo-random uniform in [-1, 1), a function of (seed, i) only
cudaError_t launch_fill_hash(double* x, int64_t n, unsigned long long seed, cudaStream_t st);
// xs[b][v][c_pad] = s[vc] * x[b][vc] * (colscale ? colscale[b] : 1)
cudaError_t launch_prescale(const double* x, int64_t ldx, double* xs, int64_t ldxs, const double* s, int n_v, int n_c,
                            int n_cp, int nb, cudaStream_t st);
// t[b][m] = sum_z part[z][b][m]
cudaError_t launch_splitk_reduce(const double* part, int64_t split_stride, int splits, double* t, int64_t ld, int m,
                                 int nb, cudaStream_t st);
// dst[r][c] = src[c][r]  (src [rows][cols] -> dst [cols][ld_dst]), for Phi^T copies
cudaError_t launch_transpose(const double* src, int rows, int cols, double* dst, int64_t ld_dst, cudaStream_t st);
cudaError_t launch_copy_pad(const double* src, int rows, int cols, double* dst, int64_t ld_dst, cudaStream_t st);
// rho[b][mu] = phi_{n_b}(mu) * phi_{m_b}(mu), orbitals taken from PhiV^T / PhiC^T
cudaError_t launch_rho(const double* phivT, const double* phicT, int64_t ldt, int n_v, int n_mu, const int32_t* n_idx,
                       const int32_t* m_idx, double* rho, int64_t ld_rho, int nb, cudaStream_t st);
// The same two passes for complex planar vectors [re (n_vc/2) | im (n_vc/2)] with COMPLEX projection coefficients;
// npart = reorth_parts(n_vc / 2), coef partials [nb][nslots][2][npart]
cudaError_t launch_reorth_dots_c(const double* basis, int64_t slot_stride, int nslots, const double* w, int64_t n_vc,
                                 int nb, double* coefpart, int npart, cudaStream_t st);
cudaError_t launch_reorth_apply_c(const double* basis, int64_t slot_stride, int nslots, double* w, int64_t n_vc, int nb,
                                  const double* coefpart, int npart, double* normpart, cudaStream_t st);
// Planar copies of complex (interleaved re, im) input: dst_{r,i}[k*stride_k + m*stride_m + o*stride_o] = src[k][m][o]
cudaError_t launch_scatter_complex(const double* src, int n_k, int n_m, int n_o, double* dst_r, double* dst_i,
                                   int64_t stride_k, int64_t stride_m, int64_t stride_o, cudaStream_t st);
// x interleaved [nvec][n][2] <-> planar [nvec][2][n]
cudaError_t launch_deinterleave(const double* src, int64_t n, int nvec, double* dst, cudaStream_t st);
cudaError_t launch_interleave(const double* src, int64_t n, int nvec, double* dst, cudaStream_t st);
// rho~_j(mu) = psi_m(mu) conj(psi_n(mu)) (planar, rows j and nb + j of rho), orbitals from the planar psi_v^T / psi_cq^T;
// chains[j] = (k slot of n, n index, k slot of m, m index)
cudaError_t launch_rho_c(const double* psivT, int64_t pv_plane, const double* psicT, int64_t pc_plane, int64_t ldt, int n_v,
                         int n_c, int n_mu, const int32_t* chains, double* rho, int64_t ld_rho, int nb, cudaStream_t st);
// d2[(part, k, v, c)] = eps_cq[k][c] - eps_v[k][v], s = 1, both planes
cudaError_t launch_build_delta_c(const double* eps_v, const double* eps_cq, int n_k, int n_v, int n_c, double* d2,
                                 double* s, cudaStream_t st);
// part[b][blk] = sum over the block's slice of x[b]*y[b]
cudaError_t launch_dot_partials(const double* x, const double* y, int64_t ld, int64_t n, int nb, double* part,
                                int npart, cudaStream_t st);

struct LanczosState {       // device arrays, one entry per chain of the current block
    double* alpha;          // [nb][steps]  (points into the context's per-chain arrays)
    double* beta;           // [nb][steps]
    double* norm2;          // [nb]
    int32_t* len;           // [nb]
    double* scale;          // [nb] running max(|a|+b)
    int32_t* alive;         // [nb]
    int steps;
    const int* kbase = nullptr;  // device step counter added to the kernel's step argument (CUDA-graph replay), or NULL
};
// *p = v / *p += d (one thread): the step counter of the graph replay
cudaError_t launch_set_int(int* p, int v, cudaStream_t st);
cudaError_t launch_add_int(int* p, int d, cudaStream_t st);
// q0 = p/||p|| in place, xs = s o q0; norm2 from partials; dead if norm2 == 0.
cudaError_t launch_lanczos_init(double* p, int64_t n_vc, int nb, const double* normpart, int npart, LanczosState st_,
                                double* xs, int64_t ldxs, const double* s, int n_v, int n_c, int n_cp,
                                cudaStream_t st);
// alpha_k = sum(dotpart); w = w - alpha q - beta_{k} q_prev (in place in w); norm partials of the new w.
cudaError_t launch_lanczos_update1(double* w, const double* q, const double* q_prev, int64_t n_vc, int nb,
                                   const double* dotpart, int ndot, int dot_stride, LanczosState st_, int k,
                                   double* normpart, int npart, cudaStream_t st);
// beta_{k+1} = sqrt(sum normpart); breakdown test; q_next = w / beta in place; xs = s o q_next.
cudaError_t launch_lanczos_update2(double* w, int64_t n_vc, int nb, const double* normpart, int npart,
                                   LanczosState st_, int k, double* xs, int64_t ldxs, const double* s, int n_v,
                                   int n_c, int n_cp, cudaStream_t st);
// update1 + update2 in one pass (reorth off) when one chain fits in the registers of a thread-block cluster.
bool lanczos_fused_fits(int64_t n_vc);
cudaError_t launch_lanczos_fused(double* w, const double* q, const double* q_prev, int64_t n_vc, int nb,
                                 const double* dotpart, int ndot, int dot_stride, LanczosState st_, int k, double* xs,
                                 int64_t ldxs, const double* s, int n_v, int n_c, int n_cp, cudaStream_t st);
int reorth_parts(int64_t n_vc);  // partial sums per chain of the two kernels below (their `npart`)
// Full reorthogonalisation pass (classical Gram-Schmidt against basis vectors 0..k of each chain).
// basis: [k+1 slots][nb][n_vc] with slot stride `slot_stride`; coef partials [nb][k+1][npart].
cudaError_t launch_reorth_dots(const double* basis, int64_t slot_stride, int nslots, const double* w, int64_t n_vc,
                               int nb, double* coefpart, int npart, cudaStream_t st);
cudaError_t launch_reorth_apply(const double* basis, int64_t slot_stride, int nslots, double* w, int64_t n_vc, int nb,
                                const double* coefpart, int npart, double* normpart, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// Pseudo-Hermitian RPA Lanczos for complex orbitals (prpa_kernels.cu, reading Q24).
// A chain is the real vector [x_re | x_im | z_re | z_im] of n4 = 4 n_kvc doubles, z = conj(y) of the pair [x; y].
// ---------------------------------------------------------------------------------------------
int prpa_parts(int64_t n4);  // partial sums per chain of the kernels below
// Tc[j] = T[2j] + conj(T[2j+1]); T planar [2][2 nb][ld], Tc planar [2][nb][ld]
cudaError_t launch_prpa_combine(const double* T, int64_t ld, int nb, int n_mu, double* Tc, cudaStream_t st);
// W[2j] = Wc[j], W[2j+1] = sign conj(Wc[j]); Wc planar [2][nb][ld], W planar [2][2 nb][ld]
cudaError_t launch_prpa_expand(const double* Wc, int64_t ld, int nb, int n_mu, double sign, double* W, cudaStream_t st);
// q_0 = u / sqrt(u . su), s_0 = su / sqrt(u . su) in place (normpart: partials of u . su); xs = F s_0; apart [nb][prpa_parts]
cudaError_t launch_prpa_init(double* u, double* su, int64_t n4, int nb, const double* normpart, int npart_in, LanczosState st_,
                             double* xs, int64_t ldxs, int n_c, int n_cp, double* apart, cudaStream_t st);
// a_k = sum(apart); h = F s; w = h - a q - b_k q_prev -> wq; t (= K^H W part of Omega^ h on entry) <- t + d2 o h - a s - b_k s_prev;
// normpart [nb][prpa_parts] = partials of w . t
cudaError_t launch_prpa_update1(double* t, double* wq, const double* q, const double* q_prev, const double* s,
                                const double* s_prev, const double* d2, int64_t n4, int nb, const double* apart, LanczosState st_,
                                int k, double* normpart, cudaStream_t st);
// b_{k+1}, breakdown, q_{k+1} = wq / b, s_{k+1} = sw / b in place, xs = F s_{k+1}, apart for the next a
cudaError_t launch_prpa_update2(double* wq, double* sw, int64_t n4, int nb, const double* normpart, LanczosState st_, int k,
                                double* xs, int64_t ldxs, int n_c, int n_cp, double* apart, cudaStream_t st);
// complex coefficients c_j = s_j^H w, j < nslots: coefpart [nb][nslots][2][prpa_parts]
cudaError_t launch_prpa_reorth_dots(const double* sbasis, int64_t slot_stride, int nslots, const double* w, int64_t n4, int nb,
                                    double* coefpart, cudaStream_t st);
// w -= sum c_j q_j, sw -= sum c_j s_j; normpart (may be NULL) = partials of w . sw
cudaError_t launch_prpa_reorth_apply(const double* qbasis, const double* sbasis, int64_t slot_stride, int nslots, double* w,
                                     double* sw, int64_t n4, int nb, const double* coefpart, double* normpart, cudaStream_t st);

// interleaved pairs x, y [nvec][n][2] <-> stored chains [nvec][x_re | x_im | Re y | -Im y]
cudaError_t launch_prpa_pack(const double* x, const double* y, int64_t n, int nvec, double* out, cudaStream_t st);
cudaError_t launch_prpa_unpack(const double* in, int64_t n, int nvec, double* x, double* y, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// Spectral kernels (spectral_kernels.cu): Eq. 14, Ritz pairs of T_L, Eq. 11 / Eq. 12, Eq. 10.
// ---------------------------------------------------------------------------------------------
cudaError_t launch_contfrac(const double* alpha, const double* beta, const double* norm2, const int32_t* len, int steps,
                            int n_chains, const double* zeta, int n_zeta, double* r, cudaStream_t st);
// theta[chain][steps], wgt[chain][steps] (first `len` entries valid); work: 3*n_chains*steps doubles
cudaError_t launch_ritz(const double* alpha, const double* beta, const int32_t* len, int steps, int n_chains,
                        double* theta, double* wgt, double* work, int32_t* info, cudaStream_t st);
// Same outputs by divide and conquer, one CTA per chain (ritz_dc.cu); steps must satisfy ritz_dc_fits().
bool ritz_dc_fits(int steps);
cudaError_t launch_ritz_dc(const double* alpha, const double* beta, const int32_t* len, int steps, int n_chains,
                           double* theta, double* wgt, int32_t* info, cudaStream_t st);
// linear = 0: Eq. 11 on the Ritz pairs of C (Omega_i = sqrt(theta_i)); linear = 1: pseudo-Hermitian RPA (Omega_i = theta_i,
// Ritz values theta_i <= 0 -- the negative branch of C^RPA -- are left out); Sigma is multiplied by prefactor
cudaError_t launch_sigma_direct(const double* theta, const double* wgt, const double* norm2, const int32_t* len,
                                int steps, int n_chains, const double* eps_n, const int32_t* sgn_n,
                                const double* omega, int n_omega, double eta, int linear, double prefactor, double* sigma,
                                cudaStream_t st);
cudaError_t launch_sigma_poly(const double* alpha, const double* beta, const double* norm2, const int32_t* len,
                              int steps, int n_chains, const double* eps_n, const int32_t* sgn_n, const double* omega,
                              int n_omega, double eta, double* sigma, cudaStream_t st);
// TDA: Sigma = -sgn R_A(-sgn z), R_A by Eq. 14
cudaError_t launch_sigma_tda(const double* alpha, const double* beta, const double* norm2, const int32_t* len,
                             int steps, int n_chains, const double* eps_n, const int32_t* sgn_n, const double* omega,
                             int n_omega, double eta, double prefactor, double* sigma, cudaStream_t st);
// sigma_sum[w] (+)= sum over the chains (Eq. 10), fixed order; accumulate = 1 adds to what sigma_sum holds
cudaError_t launch_sigma_sum(const double* sigma, int n_chains, int n_omega, double* sigma_sum, int accumulate,
                             cudaStream_t st);
// out[0] = (first ? 0 : out[0]) - sum(part[0..count)) in a fixed order (Eq. 6 accumulation)
cudaError_t launch_accum_neg(const double* part, int count, double* out, int first, cudaStream_t st);
// Newton-Raphson solve of E(omega) = omega on the grid, one thread per state
cudaError_t launch_qp_solve(int n_states, const double* eps_m, const double* vxc_m, const double* sigma_x,
                            const double* sigma_c, const double* omega, int n_omega, double* e_qp, double* z_qp,
                            int32_t* iters, cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// ISDF front end (isdf.cu): gathers, Hadamard product, Coulomb quadrature matrix, Cholesky factorisation and solves.
// ---------------------------------------------------------------------------------------------
cudaError_t launch_gather_rows(const double* src, int64_t ld_src, int n_cols, const int32_t* idx, int n_mu, double* dst,
                               int64_t ld_dst, cudaStream_t st);
cudaError_t launch_hadamard(double* y, const double* x, int64_t n, cudaStream_t st);
cudaError_t launch_gather_cols(const double* Y, int64_t ld_y, const int32_t* idx, int n_mu, double* S, int64_t ld_s,
                               cudaStream_t st);
cudaError_t launch_coulomb_grid(const double* r, int n_r, int i0, int rows, double weight, double soft, double* G, int64_t ld,
                                cudaStream_t st);  // rows i0 .. i0+rows-1 of the quadrature matrix into G[0..rows-1][*], rows <= 65535
// S = L L^T in place (lower triangle, upper zeroed inside the diagonal blocks); *info (zero on entry) = 1-based index of the
// first pivot that is not above 1e-13 max_i S_ii (scale: one device double of scratch)
cudaError_t launch_cholesky(double* S, int64_t ld, int n, double* scale, int* info, cudaStream_t st);
// X <- (L L^T)^{-1} X for X [n][ldx] with n_r columns
cudaError_t launch_cholesky_solve(const double* L, int64_t ldl, int n, double* X, int64_t ldx, int n_r, cudaStream_t st);

// Weighted k-means (centroidal Voronoi) selection of the interpolation points: nearest-centroid assignment (sets *changed
// when an assignment differs from the stored one), deterministic centroid update, snap to the nearest member grid point
cudaError_t launch_cvt_assign(const double* r, int n_r, const double* c, int n_mu, int32_t* assign, int* changed,
                              cudaStream_t st);
cudaError_t launch_cvt_update(const double* r, const double* w, int n_r, const int32_t* assign, int n_mu, double* c,
                              cudaStream_t st);
cudaError_t launch_cvt_snap(const double* r, int n_r, const int32_t* assign, const double* c, int n_mu, int32_t* idx,
                            cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// Point-group symmetry blocks (sym_kernels.cu, reading Q25)
// ---------------------------------------------------------------------------------------------
// vg[gamma][mu][nu] (row stride ld) = g sum_h chi_gamma(h) vwf[mu][h][nu], all gamma < g <= 8
cudaError_t launch_sym_reduce_kernel(const double* vwf, int n_w, int g, double* vg, int64_t ld, cudaStream_t st);
// d2 = Delta^2, s = sqrt(Delta) of one [nv][ncp] rectangle (columns >= nc are padding: d2 = s = 1)
cudaError_t launch_sym_build_delta(const double* eps_v, const double* eps_c, int nv, int nc, int ncp, double* d2, double* s,
                                   cudaStream_t st);
// one rectangle of nvec block vectors: dir 0 api [nv][nc] -> padded [nv][ncp] (zero fill), dir 1 back
cudaError_t launch_sym_copy_rect(double* api, int64_t ld_api, double* padded, int64_t ld_pad, int nv, int nc, int ncp, int nvec,
                                 int dir, cudaStream_t st);

// zero the padding columns c >= nc of one [nv][ncp] rectangle of nvec block vectors (row stride ld)
cudaError_t launch_sym_zero_pad(double* x, int64_t ld, int nv, int nc, int ncp, int nvec, cudaStream_t st);

// probe.cu
cudaError_t probe_fp64_peak(int kind, double* tflops);

// ---------------------------------------------------------------------------------------------
// Programmatic dependent launch.  The kernels of the Lanczos step loop are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization: the next kernel's CTAs are dispatched, and run their
// prologue (mbarrier init, tensor-map prefetch, index arithmetic), while the previous kernel drains; pdl_wait()
// then blocks until every earlier kernel of the stream has completed and its writes are visible.  EVERY kernel
// launched through launch_pdl() calls pdl_trigger(); pdl_wait(); in all threads before it touches global memory
// (that also makes the ordering transitive along the stream).
// ---------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;\n" ::: "memory"); }
#endif
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              unsigned cluster_x, Args... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    unsigned n = 0;
    attr[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[n].val.programmaticStreamSerializationAllowed = 1;
    ++n;
    if (cluster_x > 1) {
        attr[n].id = cudaLaunchAttributeClusterDimension;
        attr[n].val.clusterDim.x = cluster_x;
        attr[n].val.clusterDim.y = 1;
        attr[n].val.clusterDim.z = 1;
        ++n;
    }
    cfg.attrs = attr;
    cfg.numAttrs = n;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of a function ON a device: one instance of this per
// kernel remembers, per device, the largest size already configured (contexts on several GPUs in one process).
struct SmemAttr {
    std::atomic<size_t> configured[64] = {};
    template <class K>
    cudaError_t ensure(K kern, size_t bytes) {
        if (bytes <= 48 * 1024) return cudaSuccess;
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        if (dev < 0 || dev >= 64) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (configured[dev].load(std::memory_order_relaxed) >= bytes) return cudaSuccess;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e == cudaSuccess) configured[dev].store(bytes, std::memory_order_relaxed);
        return e;
    }
};

// SM count of the current device (cached per device); grids of the streaming kernels are sized from it.
inline int device_sm_count() {
    static std::atomic<int> cached[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    int n = cached[dev].load(std::memory_order_relaxed);
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cached[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

// Every launch_* bumps this counter once per kernel launched (read by gwl_get_launch_count).
extern thread_local int64_t* g_launch_counter;
inline void count_launch(int n = 1) {
    if (g_launch_counter) *g_launch_counter += n;
}

}  // namespace gwl
