// Ritz pairs of the Lanczos tridiagonal T_L (Eq. 13) for the direct-mode self-energy
// (Eq. 11 evaluated as a Gauss quadrature: theta_i = eigenvalues, w_i = squared first eigenvector components).
//
// Divide and conquer (Cuppen) restricted to what the quadrature needs: besides the eigenvalues of a sub-block only
// the FIRST and LAST rows of its eigenvector matrix are carried (the last row of the left block and the first row of
// the right block form the rank-one update vector of a merge; the first row of the top block gives the weights).
// T is torn at every off-diagonal (leaves are 1x1: d_i = a_i - b_i - b_{i+1}), then merged level by level; the
// segments of one level are independent and every step inside a merge is parallel over the roots except one short
// deflation scan.  A merge of blocks with eigenvalues D (sorted), update vector z (normalised) and rho > 0:
//   1. deflation: rho |z_j| <= tol keeps (D_j, rows) as they are; neighbours with |(D_k - D_j) c s| <= tol are
//      rotated so that one z vanishes (this is what absorbs the clusters of "ghost" Ritz values of a Lanczos run
//      without reorthogonalisation);
//   2. the roots of the secular equation 1 + rho sum_j z_j^2 / (D_j - mu) = 0, one per thread, as an offset tau from
//      the nearer pole (keeps mu - D_j accurate), by rational interpolation through both neighbouring poles,
//      safeguarded by a bisection bracket;
//   3. Gu-Eisenstat: z is recomputed from the roots so that the eigenvectors v_i = zhat / (D - mu_i) are orthogonal to
//      working accuracy;
//   4. new first/last rows = old rows times v_i / ||v_i||.
// One CTA per chain.  The implicit-QL kernel (spectral_kernels.cu) is inherently sequential: ~L^2 rotations of
// ~300 cycles each, 5.9 ms at L = 200; this kernel does the same job in parallel in about 0.1 ms.
#include "gwl_internal.h"

namespace gwl {

namespace {

constexpr int RT = 256;  // threads per CTA
constexpr double DC_EPS = 2.220446049250313e-16;

// 1/x to ~1 ulp: MUFU.RCP64H seed (about 2^-22) and two Newton steps.  The secular solver stops at
// |w| <= 4 eps (1 + |psi| + |phi|) and every quotient below is one factor of a long product or sum, so correct
// rounding (the ~30-instruction div.rn.f64 sequence, 60 % of this kernel's samples in the first profile) buys nothing.
// x is finite and nonzero at every call site (distinct poles, offsets strictly inside a bracket).
__device__ __forceinline__ double fast_rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}

struct DcShared {
    double *Ad, *Af, *Al;          // eigen-data of the current segments: value, first-row entry, last-row entry
    double *BD, *Bz, *BF, *BL;     // a merge's inputs in sorted order
    double *CD, *Cz2, *Cz, *CF, *CL;  // the non-deflated ones, compacted per segment
    double *org, *tau, *zh;        // root i: mu_i = org_i + tau_i; zh = Gu-Eisenstat vector
    double *rho;                   // per segment (at its first position)
    int *nd, *kcount;              // compacted -> sorted position; non-deflated count per segment
    unsigned char* defl;
};

__device__ __forceinline__ DcShared carve(unsigned char* base, int n) {
    DcShared s;
    double* d = reinterpret_cast<double*>(base);
    s.Ad = d; s.Af = d + n; s.Al = d + 2 * n;
    s.BD = d + 3 * n; s.Bz = d + 4 * n; s.BF = d + 5 * n; s.BL = d + 6 * n;
    s.CD = d + 7 * n; s.Cz2 = d + 8 * n; s.Cz = d + 9 * n; s.CF = d + 10 * n; s.CL = d + 11 * n;
    s.org = d + 12 * n; s.tau = d + 13 * n; s.zh = d + 14 * n; s.rho = d + 15 * n;
    int* ip = reinterpret_cast<int*>(d + 16 * n);
    s.nd = ip; s.kcount = ip + n;
    s.defl = reinterpret_cast<unsigned char*>(ip + 2 * n);
    return s;
}

// segment s of depth t covers [floor(s n / 2^t), floor((s+1) n / 2^t))
__device__ __forceinline__ void segment_of(int i, int n, int t, int& lo, int& hi, int& mid) {
    const long long p = 1ll << t;
    const long long sidx = ((long long)(i + 1) * p + n - 1) / n - 1;
    lo = (int)(sidx * n / p);
    hi = (int)((sidx + 1) * n / p);
    mid = (int)((2 * sidx + 1) * n / (2 * p));
}

// Steps 1-2 of a level: sort the two children of every segment together, then the deflation scan (one thread per segment).
__device__ void dc_sort_and_deflate(const DcShared& s, const double* __restrict__ beta_j, int n, int t) {
    for (int i = threadIdx.x; i < n; i += RT) {
        int lo, hi, mid;
        segment_of(i, n, t, lo, hi, mid);
        if (mid == lo || mid == hi) continue;  // an empty child: nothing to merge
        const double x = s.Ad[i];
        int rank = 0;
        for (int j = lo; j < hi; ++j) {
            const double y = s.Ad[j];
            rank += (y < x || (y == x && j < i)) ? 1 : 0;
        }
        const int pos = lo + rank;
        const bool left = i < mid;
        s.BD[pos] = x;
        s.Bz[pos] = left ? s.Al[i] : s.Af[i];
        s.BF[pos] = left ? s.Af[i] : 0.0;
        s.BL[pos] = left ? 0.0 : s.Al[i];
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += RT) {
        int lo, hi, mid;
        segment_of(i, n, t, lo, hi, mid);
        if (i != lo || mid == lo || mid == hi) continue;
        double rho = beta_j[mid - 1];
        double z2 = 0.0, dmax = 0.0;
        for (int k = lo; k < hi; ++k) {
            z2 += s.Bz[k] * s.Bz[k];
            dmax = fmax(dmax, fabs(s.BD[k]));
        }
        int K = 0;
        if (!(rho > 0.0) || !(z2 > 0.0)) {  // exact split: the children's pairs are the parent's pairs
            for (int k = lo; k < hi; ++k) s.defl[k] = 1;
        } else {
            const double zinv = rsqrt(z2);
            rho *= z2;
            double zmax = 0.0;
            for (int k = lo; k < hi; ++k) {
                s.Bz[k] *= zinv;
                zmax = fmax(zmax, fabs(s.Bz[k]));
            }
            const double tol = 8.0 * DC_EPS * fmax(dmax, zmax);
            int prev = -1;
            for (int k = lo; k < hi; ++k) {
                const double zk = s.Bz[k];
                if (rho * fabs(zk) <= tol) {
                    s.defl[k] = 1;
                    continue;
                }
                s.defl[k] = 0;
                if (prev >= 0) {
                    const int j = prev;
                    const double zj = s.Bz[j];
                    const double t2 = zj * zj + zk * zk;
                    if (fabs((s.BD[k] - s.BD[j]) * zj * zk) <= tol * t2) {
                        const double tt = sqrt(t2);
                        const double c = zk / tt, sn = -zj / tt;
                        s.Bz[k] = tt;
                        s.Bz[j] = 0.0;
                        const double dj = s.BD[j], dk = s.BD[k];
                        s.BD[j] = dj * c * c + dk * sn * sn;
                        s.BD[k] = dj * sn * sn + dk * c * c;
                        const double fj = s.BF[j], fk = s.BF[k];
                        s.BF[j] = c * fj + sn * fk;
                        s.BF[k] = -sn * fj + c * fk;
                        const double lj = s.BL[j], lk = s.BL[k];
                        s.BL[j] = c * lj + sn * lk;
                        s.BL[k] = -sn * lj + c * lk;
                        s.defl[j] = 1;
                    }
                }
                prev = k;
            }
            for (int k = lo; k < hi; ++k) {
                if (s.defl[k]) continue;
                const int c = lo + K;
                s.nd[c] = k;
                s.CD[c] = s.BD[k];
                s.Cz[c] = s.Bz[k];
                s.Cz2[c] = s.Bz[k] * s.Bz[k];
                s.CF[c] = s.BF[k];
                s.CL[c] = s.BL[k];
                ++K;
            }
        }
        s.kcount[lo] = K;
        s.rho[lo] = rho;
    }
    __syncthreads();
}

// Root r of the secular equation of one segment: K poles CD[0..K) (ascending), weights Cz2, rho > 0.
// Returns the origin pole value and the offset tau (mu = org + tau).
__device__ void dc_secular_root(const double* __restrict__ CD, const double* __restrict__ Cz2, int K, double rho, int r,
                                double& org_out, double& tau_out) {
    double lo, hi;
    int o;
    if (r < K - 1) {
        const double mid = 0.5 * (CD[r + 1] - CD[r]);
        double g = 0.0;
        for (int j = 0; j < K; ++j) g += Cz2[j] * fast_rcp((CD[j] - CD[r]) - mid);
        g = 1.0 + rho * g;
        if (g >= 0.0) {
            o = r;
            lo = 0.0;
            hi = mid;
        } else {
            o = r + 1;
            lo = -mid;
            hi = 0.0;
        }
    } else {
        double zs = 0.0;
        for (int j = 0; j < K; ++j) zs += Cz2[j];
        o = r;
        lo = 0.0;
        hi = rho * zs;
    }
    const double dorg = CD[o];
    double t = 0.5 * (lo + hi);
    for (int it = 0; it < 80; ++it) {
        double psi = 0.0, dpsi = 0.0, phi = 0.0, dphi = 0.0;
        {   // two independent accumulator sets per side: the sums are latency-bound (2 warps per scheduler)
            double p1 = 0.0, d1 = 0.0;
            int j = 0;
            for (; j + 1 <= r; j += 2) {
                const double i0 = fast_rcp((CD[j] - dorg) - t), i1 = fast_rcp((CD[j + 1] - dorg) - t);
                const double q0 = Cz2[j] * i0, q1 = Cz2[j + 1] * i1;
                psi += q0;
                p1 += q1;
                dpsi = fma(q0, i0, dpsi);
                d1 = fma(q1, i1, d1);
            }
            if (j <= r) {
                const double i0 = fast_rcp((CD[j] - dorg) - t);
                const double q0 = Cz2[j] * i0;
                psi += q0;
                dpsi = fma(q0, i0, dpsi);
            }
            psi += p1;
            dpsi += d1;
            p1 = d1 = 0.0;
            j = r + 1;
            for (; j + 1 < K; j += 2) {
                const double i0 = fast_rcp((CD[j] - dorg) - t), i1 = fast_rcp((CD[j + 1] - dorg) - t);
                const double q0 = Cz2[j] * i0, q1 = Cz2[j + 1] * i1;
                phi += q0;
                p1 += q1;
                dphi = fma(q0, i0, dphi);
                d1 = fma(q1, i1, d1);
            }
            if (j < K) {
                const double i0 = fast_rcp((CD[j] - dorg) - t);
                const double q0 = Cz2[j] * i0;
                phi += q0;
                dphi = fma(q0, i0, dphi);
            }
            phi += p1;
            dphi += d1;
        }
        psi *= rho;
        dpsi *= rho;
        phi *= rho;
        dphi *= rho;
        const double w = 1.0 + psi + phi;
        if (w >= 0.0) hi = t; else lo = t;
        if (fabs(w) <= 4.0 * DC_EPS * (1.0 + fabs(psi) + fabs(phi))) break;
        const double Di = (CD[r] - dorg) - t;
        double best = 0.0;
        bool have = false;
        auto consider = [&](double eta) {
            const double tn = t + eta;
            if (tn > lo && tn < hi && (!have || fabs(eta) < fabs(best))) {
                best = eta;
                have = true;
            }
        };
        if (r < K - 1) {
            // model 1 + [s + S/(d_r - x)] + [u + R/(d_{r+1} - x)] matched in value and slope at t ("middle way")
            const double Dj = (CD[r + 1] - dorg) - t;
            const double c = w - Di * dpsi - Dj * dphi;
            const double B = c * (Di + Dj) + Di * Di * dpsi + Dj * Dj * dphi;
            const double b0 = Di * Dj * w;
            const double disc = B * B - 4.0 * c * b0;
            if (disc >= 0.0) {
                const double sq = sqrt(disc);
                if (B + sq != 0.0) consider(2.0 * b0 / (B + sq));
                if (B - sq != 0.0) consider(2.0 * b0 / (B - sq));
                if (c != 0.0) {
                    consider((B + sq) / (2.0 * c));
                    consider((B - sq) / (2.0 * c));
                }
            }
        } else {
            const double c = w - Di * dpsi;
            if (c != 0.0) consider(Di + Di * Di * dpsi / c);
        }
        double tn = have ? t + best : 0.5 * (lo + hi);
        if (tn == t || !(tn > lo && tn < hi)) {
            tn = 0.5 * (lo + hi);
            if (tn == lo || tn == hi) break;
        }
        t = tn;
    }
    org_out = dorg;
    tau_out = t;
}

// Steps 3-5 of a level.
__device__ void dc_solve_and_update(const DcShared& s, int n, int t) {
    for (int i = threadIdx.x; i < n; i += RT) {
        int lo, hi, mid;
        segment_of(i, n, t, lo, hi, mid);
        if (mid == lo || mid == hi) continue;
        const int K = s.kcount[lo], r = i - lo;
        if (r >= K) continue;
        double o, tau;
        dc_secular_root(s.CD + lo, s.Cz2 + lo, K, s.rho[lo], r, o, tau);
        s.org[i] = o;
        s.tau[i] = tau;
    }
    __syncthreads();
    // Gu-Eisenstat: zhat_j^2 = prod_i (mu_i - d_j) / (rho prod_{i != j} (d_i - d_j)), as a product of positive ratios
    for (int i = threadIdx.x; i < n; i += RT) {
        int lo, hi, mid;
        segment_of(i, n, t, lo, hi, mid);
        if (mid == lo || mid == hi) continue;
        const int K = s.kcount[lo], j = i - lo;
        if (j >= K) continue;
        const double dj = s.CD[i];
        double prod = ((s.org[i] - dj) + s.tau[i]) / s.rho[lo];
        for (int k = 0; k < K; ++k) {
            if (k == j) continue;
            prod *= ((s.org[lo + k] - dj) + s.tau[lo + k]) * fast_rcp(s.CD[lo + k] - dj);
        }
        s.zh[i] = copysign(sqrt(fabs(prod)), s.Cz[i]);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += RT) {
        int lo, hi, mid;
        segment_of(i, n, t, lo, hi, mid);
        if (mid == lo || mid == hi) continue;
        if (s.defl[i]) {  // deflated pairs pass through (possibly rotated)
            s.Ad[i] = s.BD[i];
            s.Af[i] = s.BF[i];
            s.Al[i] = s.BL[i];
        }
        const int K = s.kcount[lo], r = i - lo;
        if (r >= K) continue;
        const double o = s.org[i], tau = s.tau[i];
        double nrm = 0.0, sf = 0.0, sl = 0.0;
        for (int k = 0; k < K; ++k) {
            const double v = s.zh[lo + k] * fast_rcp((s.CD[lo + k] - o) - tau);
            nrm += v * v;
            sf += s.CF[lo + k] * v;
            sl += s.CL[lo + k] * v;
        }
        const double inv = rsqrt(nrm);
        const int pos = s.nd[i];
        s.Ad[pos] = o + tau;
        s.Af[pos] = sf * inv;
        s.Al[pos] = sl * inv;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(RT) k_ritz_dc(const double* __restrict__ alpha, const double* __restrict__ beta,
                                                const int32_t* __restrict__ len, int steps, double* __restrict__ theta,
                                                double* __restrict__ wgt, int32_t* __restrict__ info) {
    extern __shared__ __align__(16) unsigned char dc_smem[];
    const int j = blockIdx.x;
    const int n = len[j];
    const double* a = alpha + (int64_t)j * steps;
    const double* b = beta + (int64_t)j * steps;  // b[i] couples rows i and i+1
    if (n > 0) {
        const DcShared s = carve(dc_smem, n);
        for (int i = threadIdx.x; i < n; i += RT) {
            double d = a[i];
            if (i > 0) d -= b[i - 1];
            if (i + 1 < n) d -= b[i];
            s.Ad[i] = d;
            s.Af[i] = 1.0;
            s.Al[i] = 1.0;
        }
        __syncthreads();
        int T = 0;
        while ((1 << T) < n) ++T;
        for (int t = T - 1; t >= 0; --t) {
            dc_sort_and_deflate(s, b, n, t);
            dc_solve_and_update(s, n, t);
        }
        for (int i = threadIdx.x; i < n; i += RT) {
            theta[(int64_t)j * steps + i] = s.Ad[i];
            wgt[(int64_t)j * steps + i] = s.Af[i] * s.Af[i];
        }
    }
    for (int i = n + threadIdx.x; i < steps; i += RT) {
        theta[(int64_t)j * steps + i] = 0.0;
        wgt[(int64_t)j * steps + i] = 0.0;
    }
    if (info != nullptr && threadIdx.x == 0) info[j] = 0;
}

}  // namespace

size_t ritz_dc_smem_bytes(int steps) { return (size_t)steps * (16 * sizeof(double) + 2 * sizeof(int) + 1) + 16; }

bool ritz_dc_fits(int steps) { return ritz_dc_smem_bytes(steps) <= 200 * 1024; }

cudaError_t launch_ritz_dc(const double* alpha, const double* beta, const int32_t* len, int steps, int n_chains,
                           double* theta, double* wgt, int32_t* info, cudaStream_t st) {
    if (n_chains <= 0) return cudaSuccess;
    const size_t sm = ritz_dc_smem_bytes(steps);
    static SmemAttr attr;
    cudaError_t ea = attr.ensure(k_ritz_dc, sm);
    if (ea != cudaSuccess) return ea;
    k_ritz_dc<<<(unsigned)n_chains, RT, sm, st>>>(alpha, beta, len, steps, theta, wgt, info);
    count_launch();
    return cudaGetLastError();
}

}  // namespace gwl
