// Resolvent and self-energy kernels: Haydock continued fraction (Eq. 14), Ritz pairs of the
// Lanczos tridiagonal T_L (Eq. 13), Sigma^corr(omega, n) by Eq. 11 (direct mode) or Eq. 12 + Eq. 14 (poly
// mode), and the sum over chains (Eq. 10).  Complex FP64 on the plain FP64 ALUs; tiny next to the GEMMs.
#include <algorithm>

#include "gwl_internal.h"

namespace gwl {

namespace {

struct cplx {
    double re, im;
};
__device__ __forceinline__ cplx cdiv(cplx a, cplx b) {
    const double d = b.re * b.re + b.im * b.im;
    return cplx{(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d};
}
__device__ __forceinline__ cplx crecip_scaled(double num, cplx b) {  // num / b
    const double d = b.re * b.re + b.im * b.im;
    return cplx{num * b.re / d, -num * b.im / d};
}

// <P|(zeta - T)^{-1}|P> = norm2 / (zeta - a_0 - b_1^2/(zeta - a_1 - ... )), bottom-up, L levels.
__device__ __forceinline__ cplx contfrac_eval(const double* __restrict__ a, const double* __restrict__ b, int L,
                                              double norm2, cplx zeta) {
    if (L <= 0) return cplx{0.0, 0.0};
    cplx f{zeta.re - a[L - 1], zeta.im};
    for (int k = L - 2; k >= 0; --k) {
        const cplx t = crecip_scaled(b[k] * b[k], f);
        f = cplx{zeta.re - a[k] - t.re, zeta.im - t.im};
    }
    return crecip_scaled(norm2, f);
}

__global__ void k_contfrac(const double* __restrict__ alpha, const double* __restrict__ beta,
                           const double* __restrict__ norm2, const int32_t* __restrict__ len, int steps,
                           const double* __restrict__ zeta, int n_zeta, double* __restrict__ r) {
    const int j = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_zeta) return;
    const cplx z{zeta[2 * i], zeta[2 * i + 1]};
    const cplx v = contfrac_eval(alpha + (int64_t)j * steps, beta + (int64_t)j * steps, len[j], norm2[j], z);
    r[((int64_t)j * n_zeta + i) * 2] = v.re;
    r[((int64_t)j * n_zeta + i) * 2 + 1] = v.im;
}

// Golub-Welsch: eigenvalues of the symmetric tridiagonal T_L by the implicit QL iteration with Wilkinson
// shifts; the same rotations are applied to e_1^T so that z_i = first component of eigenvector i.
// One chain per block; lane 0 runs the (inherently sequential) sweeps on shared-memory copies.
__global__ void k_ritz(const double* __restrict__ alpha, const double* __restrict__ beta,
                       const int32_t* __restrict__ len, int steps, double* __restrict__ theta,
                       double* __restrict__ wgt, int32_t* __restrict__ info) {
    extern __shared__ double shm[];
    double* d = shm;
    double* e = shm + steps;
    double* z = shm + 2 * steps;
    const int j = blockIdx.x;
    const int n = len[j];
    // Scale T by a power of two (exact) so that f^2 + g^2 below can neither overflow nor lose its small terms.
    __shared__ double sh_max[32];
    double mx = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        mx = fmax(mx, fabs(alpha[(int64_t)j * steps + i]));
        if (i + 1 < n) mx = fmax(mx, fabs(beta[(int64_t)j * steps + i]));
    }
    sh_max[threadIdx.x] = mx;
    __syncthreads();
    mx = 0.0;
    for (int i = 0; i < (int)blockDim.x; ++i) mx = fmax(mx, sh_max[i]);
    int ex = 0;
    if (mx > 0.0) frexp(mx, &ex);
    const double sc = ldexp(1.0, -ex), unsc = ldexp(1.0, ex);
    for (int i = threadIdx.x; i < steps; i += blockDim.x) {
        d[i] = (i < n) ? sc * alpha[(int64_t)j * steps + i] : 0.0;
        e[i] = (i + 1 < n) ? sc * beta[(int64_t)j * steps + i] : 0.0;
        z[i] = (i == 0) ? 1.0 : 0.0;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int fail = 0;
        const double eps = 2.220446049250313e-16;
        for (int l = 0; l < n && !fail; ++l) {
            int iter = 0;
            while (true) {
                int m = l;
                for (; m < n - 1; ++m) {
                    const double dd = fabs(d[m]) + fabs(d[m + 1]);
                    if (fabs(e[m]) <= eps * dd) break;
                }
                if (m == l) break;
                if (++iter > 80) {
                    fail = 1;
                    break;
                }
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                double r = sqrt(g * g + 1.0);
                g = d[m] - d[l] + e[l] / (g + copysign(r, g));
                double s = 1.0, c = 1.0, p = 0.0;
                bool underflow = false;
                // The rotation chain is one long dependency; rsqrt (one MUFU + Newton steps) replaces the
                // sqrt-then-divide pair on that critical path.  e[i], d[i] of the next rotation are fetched early.
                double ei = e[m - 1], di = d[m - 1], dn = d[m];
                double zf = z[m], zi = z[m - 1];  // zf: the (already rotated) entry i+1, carried in a register
                for (int i = m - 1; i >= l; --i) {
                    const double f = s * ei;
                    const double bq = c * ei;
                    const double h = f * f + g * g;
                    const bool more = i > l;
                    const double e_nx = more ? e[i - 1] : 0.0, d_nx = more ? d[i - 1] : 0.0, z_nx = more ? z[i - 1] : 0.0;
                    if (h == 0.0) {
                        e[i + 1] = 0.0;
                        d[i + 1] = dn - p;
                        z[i + 1] = zf;
                        e[m] = 0.0;
                        underflow = true;
                        break;
                    }
                    const double rinv = rsqrt(h);
                    e[i + 1] = h * rinv;
                    s = f * rinv;
                    c = g * rinv;
                    g = dn - p;
                    r = (di - g) * s + 2.0 * c * bq;
                    p = s * r;
                    d[i + 1] = g + p;
                    g = c * r - bq;
                    z[i + 1] = s * zi + c * zf;
                    zf = c * zi - s * zf;
                    ei = e_nx;
                    dn = di;
                    di = d_nx;
                    zi = z_nx;
                }
                if (underflow) continue;
                z[l] = zf;
                d[l] -= p;
                e[l] = g;
                e[m] = 0.0;
            }
        }
        if (info != nullptr) info[j] = fail;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < steps; i += blockDim.x) {
        theta[(int64_t)j * steps + i] = (i < n) ? unsc * d[i] : 0.0;
        wgt[(int64_t)j * steps + i] = (i < n) ? z[i] * z[i] : 0.0;
    }
}

// Eq. 11 on the Ritz pairs: Sigma_j(omega) = norm2 * sum_i w_i * sgn / (O_i (O_i + sgn z)), O_i = sqrt(theta_i),
// z = omega - eps_n - i sgn eta.
__global__ void k_sigma_direct(const double* __restrict__ theta, const double* __restrict__ wgt,
                               const double* __restrict__ norm2, const int32_t* __restrict__ len, int steps,
                               const double* __restrict__ eps_n, const int32_t* __restrict__ sgn_n,
                               const double* __restrict__ omega, int n_omega, double eta, int linear,
                               double prefactor, double* __restrict__ sigma) {
    extern __shared__ double shm[];
    double* O = shm;
    double* wo = shm + steps;
    const int j = blockIdx.y;
    const int n = len[j];
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double th = theta[(int64_t)j * steps + i];
        if (linear) {  // pseudo-Hermitian RPA: the Ritz values approximate +-Omega_s; only the positive branch enters
            O[i] = th > 0.0 ? th : 1.0;
            wo[i] = th > 0.0 ? wgt[(int64_t)j * steps + i] / th : 0.0;
        } else {
            const double o = sqrt(fmax(th, 1e-300));
            O[i] = o;
            wo[i] = wgt[(int64_t)j * steps + i] / o;
        }
    }
    __syncthreads();
    const int iw = blockIdx.x * blockDim.x + threadIdx.x;
    if (iw >= n_omega) return;
    const double sg = (double)sgn_n[j];
    const double zre = omega[iw] - eps_n[j], zim = -sg * eta;
    double sre = 0.0, sim = 0.0;
    for (int i = 0; i < n; ++i) {
        const cplx den{O[i] + sg * zre, sg * zim};
        const cplx t = crecip_scaled(wo[i], den);
        sre += t.re;
        sim += t.im;
    }
    const double f = prefactor * norm2[j] * sg;
    sigma[((int64_t)j * n_omega + iw) * 2] = f * sre;
    sigma[((int64_t)j * n_omega + iw) * 2 + 1] = f * sim;
}

// Eq. 12 with Eq. 14: Sigma = (1/z) [ R(-sgn z) - R(0) ],  R(zeta) = <P|(zeta - D)^{-1}|P>.
__global__ void k_sigma_poly(const double* __restrict__ alpha, const double* __restrict__ beta,
                             const double* __restrict__ norm2, const int32_t* __restrict__ len, int steps,
                             const double* __restrict__ eps_n, const int32_t* __restrict__ sgn_n,
                             const double* __restrict__ omega, int n_omega, double eta, double* __restrict__ sigma) {
    const int j = blockIdx.y;
    const int iw = blockIdx.x * blockDim.x + threadIdx.x;
    if (iw >= n_omega) return;
    const double sg = (double)sgn_n[j];
    const cplx z{omega[iw] - eps_n[j], -sg * eta};
    const double* a = alpha + (int64_t)j * steps;
    const double* b = beta + (int64_t)j * steps;
    const cplx r0 = contfrac_eval(a, b, len[j], norm2[j], cplx{0.0, 0.0});
    const cplx rz = contfrac_eval(a, b, len[j], norm2[j], cplx{-sg * z.re, -sg * z.im});
    const cplx v = cdiv(cplx{rz.re - r0.re, rz.im - r0.im}, z);
    sigma[((int64_t)j * n_omega + iw) * 2] = v.re;
    sigma[((int64_t)j * n_omega + iw) * 2 + 1] = v.im;
}

// Tamm-Dancoff (B = 0): Sigma = <P| 1/(omega - eps_n + sgn (A - i eta)) |P> = -sgn R_A(-sgn z)  (Eq. 14).
__global__ void k_sigma_tda(const double* __restrict__ alpha, const double* __restrict__ beta,
                            const double* __restrict__ norm2, const int32_t* __restrict__ len, int steps,
                            const double* __restrict__ eps_n, const int32_t* __restrict__ sgn_n,
                            const double* __restrict__ omega, int n_omega, double eta, double prefactor,
                            double* __restrict__ sigma) {
    const int j = blockIdx.y;
    const int iw = blockIdx.x * blockDim.x + threadIdx.x;
    if (iw >= n_omega) return;
    const double sg = (double)sgn_n[j];
    const cplx z{omega[iw] - eps_n[j], -sg * eta};
    const cplx r = contfrac_eval(alpha + (int64_t)j * steps, beta + (int64_t)j * steps, len[j], norm2[j],
                                 cplx{-sg * z.re, -sg * z.im});
    sigma[((int64_t)j * n_omega + iw) * 2] = -sg * prefactor * r.re;
    sigma[((int64_t)j * n_omega + iw) * 2 + 1] = -sg * prefactor * r.im;
}

__global__ void k_sigma_sum(const double* __restrict__ sigma, int n_chains, int n_omega,
                            double* __restrict__ sigma_sum, int accumulate) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;  // over 2*n_omega reals
    if (i >= 2 * n_omega) return;
    double acc = accumulate ? sigma_sum[i] : 0.0;
    for (int j = 0; j < n_chains; ++j) acc += sigma[(int64_t)j * n_omega * 2 + i];
    sigma_sum[i] = acc;
}

// Sigma^ex accumulation: one block, fixed-order tree.
__global__ void k_accum_neg(const double* __restrict__ part, int count, double* __restrict__ out, int first) {
    __shared__ double sh[256];
    double t = 0.0;
    for (int i = threadIdx.x; i < count; i += 256) t += part[i];
    sh[threadIdx.x] = t;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = (first ? 0.0 : out[0]) - sh[0];
}

// E(omega) = eps_m + Re[Sigma^ex + Sigma^corr(omega)] - V_xc = omega by Newton-Raphson on the piecewise-linear
// interpolant of Re Sigma^corr (reading Q18): start at eps_m, clamp to the grid, stop at
// |step| <= 1e-10 eV or after 50 iterations.
__global__ void k_qp_solve(int n_states, const double* __restrict__ eps_m, const double* __restrict__ vxc_m,
                           const double* __restrict__ sigma_x, const double* __restrict__ sigma_c,
                           const double* __restrict__ omega, int n_omega, double* __restrict__ e_qp,
                           double* __restrict__ z_qp, int32_t* __restrict__ iters) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_states) return;
    const double* sc = sigma_c + (int64_t)j * n_omega * 2;
    const double e0 = eps_m[j], vxc = vxc_m[j], sx = sigma_x[j];
    const double wlo = omega[0], whi = omega[n_omega - 1];
    double w = fmin(fmax(e0, wlo), whi);
    double z = 1.0;
    int it = 0;
    for (it = 1; it <= 50; ++it) {
        int lo = 0, hi = n_omega;  // first index with omega[idx] > w
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (omega[mid] <= w) lo = mid + 1; else hi = mid;
        }
        int i = lo - 1;
        i = min(max(i, 0), n_omega - 2);
        const double r0 = sc[2 * i], r1 = sc[2 * (i + 1)];
        const double slope = (r1 - r0) / (omega[i + 1] - omega[i]);
        const double s_w = r0 + slope * (w - omega[i]);
        const double F = e0 + sx + s_w - vxc - w;
        const double dF = slope - 1.0;
        z = -1.0 / dF;
        const double w_new = fmin(fmax(w + (-F / dF), wlo), whi);
        const bool done = fabs(w_new - w) <= 1e-10;
        w = w_new;
        if (done) break;
    }
    e_qp[j] = w;
    z_qp[j] = z;
    if (iters != nullptr) iters[j] = it > 50 ? 50 : it;
}

}  // namespace

constexpr int MAX_GRID_Y = 65535;  // chains go to grid.y: longer lists are cut into launches of at most this many

cudaError_t launch_contfrac(const double* alpha, const double* beta, const double* norm2, const int32_t* len, int steps,
                            int n_chains, const double* zeta, int n_zeta, double* r, cudaStream_t st) {
    if (n_chains <= 0 || n_zeta <= 0) return cudaSuccess;
    for (int j0 = 0; j0 < n_chains; j0 += MAX_GRID_Y) {
        const int nc = std::min(MAX_GRID_Y, n_chains - j0);
        dim3 grid((unsigned)ceil_div(n_zeta, 128), (unsigned)nc);
        k_contfrac<<<grid, 128, 0, st>>>(alpha + (int64_t)j0 * steps, beta + (int64_t)j0 * steps, norm2 + j0, len + j0, steps,
                                         zeta, n_zeta, r + (int64_t)j0 * n_zeta * 2);
        count_launch();
    }
    return cudaGetLastError();
}

cudaError_t launch_ritz(const double* alpha, const double* beta, const int32_t* len, int steps, int n_chains,
                        double* theta, double* wgt, double* work, int32_t* info, cudaStream_t st) {
    (void)work;
    if (n_chains <= 0) return cudaSuccess;
    const size_t sm = (size_t)3 * steps * sizeof(double);
    static SmemAttr attr;
    cudaError_t ea = attr.ensure(k_ritz, sm);
    if (ea != cudaSuccess) return ea;
    k_ritz<<<(unsigned)n_chains, 32, sm, st>>>(alpha, beta, len, steps, theta, wgt, info);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_sigma_direct(const double* theta, const double* wgt, const double* norm2, const int32_t* len,
                                int steps, int n_chains, const double* eps_n, const int32_t* sgn_n,
                                const double* omega, int n_omega, double eta, int linear, double prefactor, double* sigma,
                                cudaStream_t st) {
    if (n_chains <= 0 || n_omega <= 0) return cudaSuccess;
    const size_t sm = (size_t)2 * steps * sizeof(double);
    static SmemAttr attr;
    cudaError_t ea = attr.ensure(k_sigma_direct, sm);
    if (ea != cudaSuccess) return ea;
    for (int j0 = 0; j0 < n_chains; j0 += MAX_GRID_Y) {
        const int nc = std::min(MAX_GRID_Y, n_chains - j0);
        dim3 grid((unsigned)ceil_div(n_omega, 128), (unsigned)nc);
        k_sigma_direct<<<grid, 128, sm, st>>>(theta + (int64_t)j0 * steps, wgt + (int64_t)j0 * steps, norm2 + j0, len + j0, steps,
                                              eps_n + j0, sgn_n + j0, omega, n_omega, eta, linear, prefactor,
                                              sigma + (int64_t)j0 * n_omega * 2);
        count_launch();
    }
    return cudaGetLastError();
}

cudaError_t launch_sigma_poly(const double* alpha, const double* beta, const double* norm2, const int32_t* len,
                              int steps, int n_chains, const double* eps_n, const int32_t* sgn_n, const double* omega,
                              int n_omega, double eta, double* sigma, cudaStream_t st) {
    if (n_chains <= 0 || n_omega <= 0) return cudaSuccess;
    for (int j0 = 0; j0 < n_chains; j0 += MAX_GRID_Y) {
        const int nc = std::min(MAX_GRID_Y, n_chains - j0);
        dim3 grid((unsigned)ceil_div(n_omega, 128), (unsigned)nc);
        k_sigma_poly<<<grid, 128, 0, st>>>(alpha + (int64_t)j0 * steps, beta + (int64_t)j0 * steps, norm2 + j0, len + j0, steps,
                                  eps_n + j0, sgn_n + j0, omega, n_omega, eta, sigma + (int64_t)j0 * n_omega * 2);
        count_launch();
    }
    return cudaGetLastError();
}

cudaError_t launch_sigma_tda(const double* alpha, const double* beta, const double* norm2, const int32_t* len,
                             int steps, int n_chains, const double* eps_n, const int32_t* sgn_n, const double* omega,
                             int n_omega, double eta, double prefactor, double* sigma, cudaStream_t st) {
    if (n_chains <= 0 || n_omega <= 0) return cudaSuccess;
    for (int j0 = 0; j0 < n_chains; j0 += MAX_GRID_Y) {
        const int nc = std::min(MAX_GRID_Y, n_chains - j0);
        dim3 grid((unsigned)ceil_div(n_omega, 128), (unsigned)nc);
        k_sigma_tda<<<grid, 128, 0, st>>>(alpha + (int64_t)j0 * steps, beta + (int64_t)j0 * steps, norm2 + j0, len + j0, steps,
                                  eps_n + j0, sgn_n + j0, omega, n_omega, eta, prefactor, sigma + (int64_t)j0 * n_omega * 2);
        count_launch();
    }
    return cudaGetLastError();
}

cudaError_t launch_sigma_sum(const double* sigma, int n_chains, int n_omega, double* sigma_sum, int accumulate,
                             cudaStream_t st) {
    if (n_omega <= 0) return cudaSuccess;
    k_sigma_sum<<<(unsigned)ceil_div(2 * n_omega, 128), 128, 0, st>>>(sigma, n_chains, n_omega, sigma_sum, accumulate);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_accum_neg(const double* part, int count, double* out, int first, cudaStream_t st) {
    k_accum_neg<<<1, 256, 0, st>>>(part, count, out, first);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_qp_solve(int n_states, const double* eps_m, const double* vxc_m, const double* sigma_x,
                            const double* sigma_c, const double* omega, int n_omega, double* e_qp, double* z_qp,
                            int32_t* iters, cudaStream_t st) {
    if (n_states <= 0) return cudaSuccess;
    k_qp_solve<<<(unsigned)ceil_div(n_states, 64), 64, 0, st>>>(n_states, eps_m, vxc_m, sigma_x, sigma_c, omega, n_omega,
                                                               e_qp, z_qp, iters);
    count_launch();
    return cudaGetLastError();
}

}  // namespace gwl
