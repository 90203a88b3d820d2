// Interpolative separable density fitting front end, PAPER.md:115-128 (Eq. 15-17) and :319:
//   phi_n(r) phi_m(r) ~ sum_mu zeta_mu(r) C^mu_nm,  C^mu_nm = phi_n(r_mu) phi_m(r_mu)                         (Eq. 15)
//   zeta = Z C^T (C C^T)^{-1}  (least squares at given interpolation points r_mu = r[idx[mu]], refs. [62, 63]) with the
//   separable normal equations  Z C^T = (Phi Phi_mu^T) o (Phi Phi_mu^T),  C C^T = the same at the interpolation points,
//   (alpha|beta) = int int zeta_alpha(r) zeta_beta(r') / |r - r'|  -> zeta^T G zeta on the grid quadrature        (Eq. 17)
// The dense contractions (Gram products, G zeta, zeta^T (G zeta)) run on the DMMA GEMM of kr_gemm.cu (MODE_PLAIN); this
// file holds what is left: gathers, the Hadamard product, the Coulomb quadrature matrix, and a blocked Cholesky
// factorisation with its two triangular solves for N_r right-hand sides.  Everything FP64; zeta is kept transposed,
// zeta_t[mu][r], which is both the GEMM operand layout and the row-block layout of the solves.
#include <algorithm>

#include "gwl_internal.h"

namespace gwl {

namespace {

constexpr int NB = 32;  // Cholesky / solve block size

__global__ void k_gather_rows(const double* __restrict__ src, int64_t ld_src, int n_cols, const int32_t* __restrict__ idx,
                              double* __restrict__ dst, int64_t ld_dst) {
    const int mu = blockIdx.x;
    const double* s = src + (int64_t)idx[mu] * ld_src;
    for (int j = threadIdx.x; j < n_cols; j += blockDim.x) dst[(int64_t)mu * ld_dst + j] = s[j];
}

// y[mu][r] *= x[mu][r]
__global__ void k_hadamard(double* __restrict__ y, const double* __restrict__ x, int64_t n) {
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) y[i] *= x[i];
}

// S[mu][nu] = Y[mu][idx[nu]]   (C C^T = Z C^T sampled at the interpolation points)
__global__ void k_gather_cols(const double* __restrict__ Y, int64_t ld_y, const int32_t* __restrict__ idx, int n_mu,
                              double* __restrict__ S, int64_t ld_s) {
    const int mu = blockIdx.x;
    for (int nu = threadIdx.x; nu < n_mu; nu += blockDim.x) S[(int64_t)mu * ld_s + nu] = Y[(int64_t)mu * ld_y + idx[nu]];
}

// G[i][j] = w^2 * 14.4 / sqrt(|r_i - r_j|^2 + soft^2): the grid quadrature of 1/|r - r'| (eV Angstrom)
// One launch fills the row panel i0 .. i0 + gridDim.y - 1 into G[0 .. gridDim.y - 1][*]: the full N_r x N_r matrix is never
// held (gwl_isdf_build walks it in panels that feed the G zeta GEMM).
__global__ void k_coulomb_grid(const double* __restrict__ r, int n_r, int i0, double w2, double soft2, double* __restrict__ G,
                               int64_t ld) {
    const int i = i0 + blockIdx.y;
    const double xi = r[3 * i], yi = r[3 * i + 1], zi = r[3 * i + 2];
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_r; j += gridDim.x * blockDim.x) {
        const double dx = xi - r[3 * j], dy = yi - r[3 * j + 1], dz = zi - r[3 * j + 2];
        G[(int64_t)blockIdx.y * ld + j] = w2 * 14.4 / sqrt(dx * dx + dy * dy + dz * dz + soft2);
    }
}

// ---- blocked right-looking Cholesky, lower triangle in place: S = L L^T ---------------------------------------------
// (a) diagonal block: one CTA of NB x NB threads, column by column in shared memory
// scale[0] = max_i S[i][i]: pivots below 1e-13 of it count as "not positive definite" (an exactly singular C C^T
// leaves pivots of either sign at rounding level)
__global__ void k_max_diag(const double* __restrict__ S, int64_t ld, int n, double* __restrict__ scale) {
    __shared__ double sh[256];
    double m = 0.0;
    for (int i = threadIdx.x; i < n; i += 256) m = fmax(m, S[(int64_t)i * ld + i]);
    sh[threadIdx.x] = m;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) scale[0] = sh[0];
}

__global__ void k_chol_diag(double* __restrict__ S, int64_t ld, int n, int k0, const double* __restrict__ scale,
                            int* __restrict__ info) {
    __shared__ double a[NB][NB + 1];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int nb = min(NB, n - k0);
    a[ty][tx] = (ty < nb && tx < nb) ? S[(int64_t)(k0 + ty) * ld + k0 + tx] : (ty == tx ? 1.0 : 0.0);
    __syncthreads();
    for (int j = 0; j < nb; ++j) {
        if (tx == 0 && ty == 0) {
            const double d = a[j][j];
            if (!(d > 1e-13 * scale[0])) {
                if (*info == 0) *info = k0 + j + 1;
                a[j][j] = 1.0;
            } else {
                a[j][j] = sqrt(d);
            }
        }
        __syncthreads();
        if (tx == 0 && ty > j) a[ty][j] /= a[j][j];
        __syncthreads();
        if (tx > j && ty >= tx) a[ty][tx] -= a[ty][j] * a[tx][j];
        __syncthreads();
    }
    if (ty < nb && tx < nb) S[(int64_t)(k0 + ty) * ld + k0 + tx] = (tx <= ty) ? a[ty][tx] : 0.0;
}

// (b) panel below the diagonal block: L_ik = A_ik L_kk^{-T}, one row per thread
__global__ void k_chol_panel(double* __restrict__ S, int64_t ld, int n, int k0) {
    __shared__ double l[NB][NB + 1];
    const int nb = min(NB, n - k0);
    for (int t = threadIdx.x; t < NB * NB; t += blockDim.x) {
        const int i = t / NB, j = t % NB;
        l[i][j] = (i < nb && j < nb) ? S[(int64_t)(k0 + i) * ld + k0 + j] : (i == j ? 1.0 : 0.0);
    }
    __syncthreads();
    const int row = k0 + nb + blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= n) return;
    double x[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) x[j] = j < nb ? S[(int64_t)row * ld + k0 + j] : 0.0;
#pragma unroll
    for (int j = 0; j < NB; ++j) {
        double v = x[j];
#pragma unroll
        for (int t = 0; t < NB; ++t)
            if (t < j) v -= x[t] * l[j][t];
        x[j] = v / l[j][j];
    }
#pragma unroll
    for (int j = 0; j < NB; ++j)
        if (j < nb) S[(int64_t)row * ld + k0 + j] = x[j];
}

// (c) trailing update of the lower triangle: A_ij -= sum_t L_it L_jt, 32 x 32 tile per CTA
__global__ void k_chol_update(double* __restrict__ S, int64_t ld, int n, int k0) {
    const int nb = min(NB, n - k0);
    const int bi = blockIdx.y, bj = blockIdx.x;
    if (bj > bi) return;
    const int base = k0 + nb;
    __shared__ double li[NB][NB + 1], lj[NB][NB + 1];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int ri = base + bi * NB + ty, rj = base + bj * NB + ty;
    li[ty][tx] = (ri < n && tx < nb) ? S[(int64_t)ri * ld + k0 + tx] : 0.0;
    lj[ty][tx] = (rj < n && tx < nb) ? S[(int64_t)rj * ld + k0 + tx] : 0.0;
    __syncthreads();
    const int i = base + bi * NB + ty, j = base + bj * NB + tx;
    if (i >= n || j >= n || j > i) return;
    double acc = 0.0;
#pragma unroll
    for (int t = 0; t < NB; ++t) acc += li[ty][t] * lj[tx][t];
    S[(int64_t)i * ld + j] -= acc;
}

// ---- triangular solves with n_r right-hand sides, X[mu][r] in place -------------------------------------------------
// forward (L Z = Y), block row k: Z_k = L_kk^{-1} (Y_k - sum_{j<k} L_kj Z_j); one column r per thread, NB accumulators
__global__ void k_trsm_fwd(const double* __restrict__ L, int64_t ldl, int n, double* __restrict__ X, int64_t ldx, int n_r,
                           int k0) {
    __shared__ double l[NB][NB + 1];
    const int nb = min(NB, n - k0);
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    double acc[NB];
#pragma unroll
    for (int i = 0; i < NB; ++i) acc[i] = (i < nb && c < n_r) ? X[(int64_t)(k0 + i) * ldx + c] : 0.0;
    for (int j0 = 0; j0 < k0; j0 += NB) {
        __syncthreads();
        for (int t = threadIdx.x; t < NB * NB; t += blockDim.x) {
            const int i = t / NB, j = t % NB;
            l[i][j] = i < nb ? L[(int64_t)(k0 + i) * ldl + j0 + j] : 0.0;
        }
        __syncthreads();
        if (c < n_r) {
#pragma unroll 4
            for (int j = 0; j < NB; ++j) {
                const double xj = X[(int64_t)(j0 + j) * ldx + c];
#pragma unroll
                for (int i = 0; i < NB; ++i) acc[i] -= l[i][j] * xj;
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < NB * NB; t += blockDim.x) {
        const int i = t / NB, j = t % NB;
        l[i][j] = (i < nb && j < nb) ? L[(int64_t)(k0 + i) * ldl + k0 + j] : (i == j ? 1.0 : 0.0);
    }
    __syncthreads();
    if (c >= n_r) return;
#pragma unroll
    for (int i = 0; i < NB; ++i) {
        double v = acc[i];
#pragma unroll
        for (int t = 0; t < NB; ++t)
            if (t < i) v -= l[i][t] * acc[t];
        acc[i] = v / l[i][i];
    }
#pragma unroll
    for (int i = 0; i < NB; ++i)
        if (i < nb) X[(int64_t)(k0 + i) * ldx + c] = acc[i];
}

// backward (L^T X = Z), block row k from the bottom: X_k = L_kk^{-T} (Z_k - sum_{j>k} L_jk^T X_j)
__global__ void k_trsm_bwd(const double* __restrict__ L, int64_t ldl, int n, double* __restrict__ X, int64_t ldx, int n_r,
                           int k0) {
    __shared__ double l[NB][NB + 1];
    const int nb = min(NB, n - k0);
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    double acc[NB];
#pragma unroll
    for (int i = 0; i < NB; ++i) acc[i] = (i < nb && c < n_r) ? X[(int64_t)(k0 + i) * ldx + c] : 0.0;
    for (int j0 = k0 + nb; j0 < n; j0 += NB) {
        const int njb = min(NB, n - j0);
        __syncthreads();
        for (int t = threadIdx.x; t < NB * NB; t += blockDim.x) {
            const int j = t / NB, i = t % NB;  // l[j][i] = L[j0 + j][k0 + i]
            l[j][i] = (j < njb && i < nb) ? L[(int64_t)(j0 + j) * ldl + k0 + i] : 0.0;
        }
        __syncthreads();
        if (c < n_r) {
            for (int j = 0; j < njb; ++j) {
                const double xj = X[(int64_t)(j0 + j) * ldx + c];
#pragma unroll
                for (int i = 0; i < NB; ++i) acc[i] -= l[j][i] * xj;
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < NB * NB; t += blockDim.x) {
        const int i = t / NB, j = t % NB;
        l[i][j] = (i < nb && j < nb) ? L[(int64_t)(k0 + i) * ldl + k0 + j] : (i == j ? 1.0 : 0.0);
    }
    __syncthreads();
    if (c >= n_r) return;
#pragma unroll
    for (int i = NB - 1; i >= 0; --i) {
        double v = acc[i];
#pragma unroll
        for (int t = 0; t < NB; ++t)
            if (t > i) v -= l[t][i] * acc[t];
        acc[i] = v / l[i][i];
    }
#pragma unroll
    for (int i = 0; i < NB; ++i)
        if (i < nb) X[(int64_t)(k0 + i) * ldx + c] = acc[i];
}


// ---- interpolation points by centroidal Voronoi tessellation (weighted k-means, Lloyd) -------------------------------
// assign: a_i = argmin_mu |r_i - c_mu|^2, ties to the lowest mu; d2 = (dx dx + dy dy) + dz dz in that order
__global__ void k_cvt_assign(const double* __restrict__ r, int n_r, const double* __restrict__ c, int n_mu,
                             int32_t* __restrict__ assign, int* __restrict__ changed) {
    extern __shared__ double cs[];  // centroids, chunk of up to 1024
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double x = 0.0, y = 0.0, z = 0.0;
    if (i < n_r) {
        x = r[3 * i];
        y = r[3 * i + 1];
        z = r[3 * i + 2];
    }
    double best = INFINITY;
    int arg = 0;
    for (int m0 = 0; m0 < n_mu; m0 += 1024) {
        const int nm = min(1024, n_mu - m0);
        __syncthreads();
        for (int t = threadIdx.x; t < 3 * nm; t += blockDim.x) cs[t] = c[3 * m0 + t];
        __syncthreads();
        for (int m = 0; m < nm; ++m) {
            const double dx = x - cs[3 * m], dy = y - cs[3 * m + 1], dz = z - cs[3 * m + 2];
            const double d2 = (dx * dx + dy * dy) + dz * dz;
            if (d2 < best) {
                best = d2;
                arg = m0 + m;
            }
        }
    }
    if (i < n_r) {
        if (assign[i] != arg) *changed = 1;
        assign[i] = arg;
    }
}

// update: one CTA per cluster walks all points in index order (fixed slices, fixed tree: deterministic);
// c_mu = sum w r / sum w over its members, unchanged if the cluster is empty
__global__ void k_cvt_update(const double* __restrict__ r, const double* __restrict__ w, int n_r,
                             const int32_t* __restrict__ assign, double* __restrict__ c) {
    __shared__ double sh[4][256];
    const int mu = blockIdx.x;
    double sw = 0.0, sx = 0.0, sy = 0.0, sz = 0.0;
    for (int i = threadIdx.x; i < n_r; i += 256) {
        if (assign[i] == mu) {
            const double wi = w[i];
            sw += wi;
            sx += wi * r[3 * i];
            sy += wi * r[3 * i + 1];
            sz += wi * r[3 * i + 2];
        }
    }
    sh[0][threadIdx.x] = sw;
    sh[1][threadIdx.x] = sx;
    sh[2][threadIdx.x] = sy;
    sh[3][threadIdx.x] = sz;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o)
            for (int q = 0; q < 4; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0 && sh[0][0] > 0.0) {
        c[3 * mu] = sh[1][0] / sh[0][0];
        c[3 * mu + 1] = sh[2][0] / sh[0][0];
        c[3 * mu + 2] = sh[3][0] / sh[0][0];
    }
}

// snap: idx_mu = the member grid point nearest to c_mu (ties: the lowest i); -1 for an empty cluster
__global__ void k_cvt_snap(const double* __restrict__ r, int n_r, const int32_t* __restrict__ assign,
                           const double* __restrict__ c, int32_t* __restrict__ idx) {
    __shared__ double bd[256];
    __shared__ int bi[256];
    const int mu = blockIdx.x;
    const double cx = c[3 * mu], cy = c[3 * mu + 1], cz = c[3 * mu + 2];
    double best = INFINITY;
    int arg = -1;
    for (int i = threadIdx.x; i < n_r; i += 256) {
        if (assign[i] == mu) {
            const double dx = r[3 * i] - cx, dy = r[3 * i + 1] - cy, dz = r[3 * i + 2] - cz;
            const double d2 = (dx * dx + dy * dy) + dz * dz;
            if (d2 < best) {  // i ascends within a thread: the first minimum is the lowest index
                best = d2;
                arg = i;
            }
        }
    }
    bd[threadIdx.x] = best;
    bi[threadIdx.x] = arg;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            const double d = bd[threadIdx.x + o];
            const int j = bi[threadIdx.x + o];
            if (j >= 0 && (bi[threadIdx.x] < 0 || d < bd[threadIdx.x] || (d == bd[threadIdx.x] && j < bi[threadIdx.x]))) {
                bd[threadIdx.x] = d;
                bi[threadIdx.x] = j;
            }
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) idx[mu] = bi[0];
}

}  // namespace

cudaError_t launch_gather_rows(const double* src, int64_t ld_src, int n_cols, const int32_t* idx, int n_mu, double* dst,
                               int64_t ld_dst, cudaStream_t st) {
    k_gather_rows<<<(unsigned)n_mu, 128, 0, st>>>(src, ld_src, n_cols, idx, dst, ld_dst);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_hadamard(double* y, const double* x, int64_t n, cudaStream_t st) {
    const unsigned g = (unsigned)std::max<int64_t>(1, std::min<int64_t>(ceil_div(n, 1024), (int64_t)device_sm_count() * 16));
    k_hadamard<<<g, 256, 0, st>>>(y, x, n);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_gather_cols(const double* Y, int64_t ld_y, const int32_t* idx, int n_mu, double* S, int64_t ld_s,
                               cudaStream_t st) {
    k_gather_cols<<<(unsigned)n_mu, 128, 0, st>>>(Y, ld_y, idx, n_mu, S, ld_s);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_coulomb_grid(const double* r, int n_r, int i0, int rows, double weight, double soft, double* G, int64_t ld,
                                cudaStream_t st) {
    if (rows <= 0) return cudaSuccess;
    if (rows > 65535 || i0 < 0 || i0 + rows > n_r) return cudaErrorInvalidValue;
    dim3 grid((unsigned)std::min<int64_t>(ceil_div(n_r, 256), 64), (unsigned)rows);
    k_coulomb_grid<<<grid, 256, 0, st>>>(r, n_r, i0, weight * weight, soft * soft, G, ld);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_cholesky(double* S, int64_t ld, int n, double* scale, int* info, cudaStream_t st) {
    k_max_diag<<<1, 256, 0, st>>>(S, ld, n, scale);
    count_launch();
    for (int k0 = 0; k0 < n; k0 += NB) {
        const int nb = std::min(NB, n - k0);
        k_chol_diag<<<1, dim3(NB, NB), 0, st>>>(S, ld, n, k0, scale, info);
        const int rest = n - k0 - nb;
        if (rest > 0) {
            k_chol_panel<<<(unsigned)ceil_div(rest, 128), 128, 0, st>>>(S, ld, n, k0);
            const unsigned nt = (unsigned)ceil_div(rest, NB);
            k_chol_update<<<dim3(nt, nt), dim3(NB, NB), 0, st>>>(S, ld, n, k0);
            count_launch(2);
        }
        count_launch();
    }
    return cudaGetLastError();
}

cudaError_t launch_cholesky_solve(const double* L, int64_t ldl, int n, double* X, int64_t ldx, int n_r, cudaStream_t st) {
    const unsigned g = (unsigned)ceil_div(n_r, 128);
    for (int k0 = 0; k0 < n; k0 += NB) {
        k_trsm_fwd<<<g, 128, 0, st>>>(L, ldl, n, X, ldx, n_r, k0);
        count_launch();
    }
    for (int k0 = (n - 1) / NB * NB; k0 >= 0; k0 -= NB) {
        k_trsm_bwd<<<g, 128, 0, st>>>(L, ldl, n, X, ldx, n_r, k0);
        count_launch();
    }
    return cudaGetLastError();
}

cudaError_t launch_cvt_assign(const double* r, int n_r, const double* c, int n_mu, int32_t* assign, int* changed,
                              cudaStream_t st) {
    k_cvt_assign<<<(unsigned)ceil_div(n_r, 256), 256, 3 * 1024 * sizeof(double), st>>>(r, n_r, c, n_mu, assign, changed);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_cvt_update(const double* r, const double* w, int n_r, const int32_t* assign, int n_mu, double* c,
                              cudaStream_t st) {
    k_cvt_update<<<(unsigned)n_mu, 256, 0, st>>>(r, w, n_r, assign, c);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_cvt_snap(const double* r, int n_r, const int32_t* assign, const double* c, int n_mu, int32_t* idx,
                            cudaStream_t st) {
    k_cvt_snap<<<(unsigned)n_mu, 256, 0, st>>>(r, n_r, assign, c, idx);
    count_launch();
    return cudaGetLastError();
}

}  // namespace gwl
