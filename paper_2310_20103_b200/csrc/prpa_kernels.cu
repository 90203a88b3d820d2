// Vector kernels of the pseudo-Hermitian RPA Lanczos for complex orbitals (PAPER.md:159 with the pole sum of
// PAPER.md:286-304; reading Q24, second step).
//
// H = C^RPA(q) = F Omega^, F = diag(1, -1), Omega^ = [[A, B], [B^*, A^*]] Hermitian positive definite.  A pair [x; y] is stored
// as (x, z = conj(y)), planar: one chain = [x_re | x_im | z_re | z_im], each of n_kvc doubles.  In these variables
//   Omega^ (x, z) = ( Delta x + K^H W,  Delta z + K^H conj(W) ),   W = V ( K x + conj(K z) ),
// i.e. the SAME Tamm-Dancoff contractions (kr_gemm_c.cu) on the 2 nb columns x_0, z_0, x_1, z_1, ... with the two small
// kernels below between them, F flips the sign of the z half, and real inner products of pairs are plain dot products of
// the stacked real vectors.  The Lanczos recurrence runs in the inner product <a, b>_O = a^H Omega^ b (three-term, real
// symmetric T); s_k = Omega^ q_k is carried along so that one product with Omega^ per step suffices:
//   h = F s_k,  a_k = s_k . F s_k,  t = Omega^ h,  w = h - a_k q_k - b_k q_{k-1},  Omega^ w = t - a_k s_k - b_k s_{k-1},
//   b_{k+1} = sqrt(w . Omega^ w),  q_{k+1} = w / b_{k+1},  s_{k+1} = Omega^ w / b_{k+1}.
// All reductions: fixed slices, fixed trees, partials re-reduced in a fixed order (deterministic, chain j independent of its block).
#include "gwl_internal.h"

namespace gwl {

namespace {

constexpr int NT = VEC_THREADS;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double block_sum(double v, double* sh /*[NT/32 + 1]*/) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) sh[w] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int i = 0; i < NT / 32; ++i) t += sh[i];
        sh[NT / 32] = t;
    }
    __syncthreads();
    return sh[NT / 32];
}

__device__ __forceinline__ double block_sum_array(const double* a, int cnt, double* sh) {
    double t = 0.0;
    for (int i = threadIdx.x; i < cnt; i += NT) t += a[i];
    return block_sum(t, sh);
}

__device__ __forceinline__ void slice_of(int64_t n, int npart, int blk, int64_t& lo, int64_t& hi) {
    const int64_t per = (n + npart - 1) / npart;
    lo = (int64_t)blk * per;
    hi = lo + per < n ? lo + per : n;
    if (lo > n) lo = n;
}

// position of element i (0 .. 2 n_vc) of a chain in the padded K.x operand xs [2 nb][n_v rows][n_cp]: column 2b + i / n_vc
__device__ __forceinline__ int64_t xs_pos(int64_t i, int64_t n_vc, int64_t ldxs, int n_c, int n_cp) {
    const int64_t col = i >= n_vc ? 1 : 0;
    const int64_t r = i - col * n_vc;
    const int64_t v = r / n_c;
    return col * ldxs + v * n_cp + (r - v * n_c);
}

// Tc[j] = T[2j] + conj(T[2j+1])  (K x + conj(K z)); T planar [2][2 nb][ld] -> Tc planar [2][nb][ld]
__global__ void k_prpa_combine(const double* __restrict__ T, int64_t ld, int nb, int n_mu, double* __restrict__ Tc) {
    pdl_trigger();
    pdl_wait();
    const int j = blockIdx.y;
    const double* tr = T;
    const double* ti = T + (int64_t)2 * nb * ld;
    for (int m = blockIdx.x * NT + threadIdx.x; m < n_mu; m += gridDim.x * NT) {
        Tc[(int64_t)j * ld + m] = tr[(int64_t)(2 * j) * ld + m] + tr[(int64_t)(2 * j + 1) * ld + m];
        Tc[(int64_t)(nb + j) * ld + m] = ti[(int64_t)(2 * j) * ld + m] - ti[(int64_t)(2 * j + 1) * ld + m];
    }
}

// W[2j] = Wc[j], W[2j+1] = sign conj(Wc[j]); Wc planar [2][nb][ld] -> W planar [2][2 nb][ld]
__global__ void k_prpa_expand(const double* __restrict__ Wc, int64_t ld, int nb, int n_mu, double sign, double* __restrict__ W) {
    pdl_trigger();
    pdl_wait();
    const int j = blockIdx.y;
    double* wr = W;
    double* wi = W + (int64_t)2 * nb * ld;
    for (int m = blockIdx.x * NT + threadIdx.x; m < n_mu; m += gridDim.x * NT) {
        const double re = Wc[(int64_t)j * ld + m], im = Wc[(int64_t)(nb + j) * ld + m];
        wr[(int64_t)(2 * j) * ld + m] = re;
        wi[(int64_t)(2 * j) * ld + m] = im;
        wr[(int64_t)(2 * j + 1) * ld + m] = sign * re;
        wi[(int64_t)(2 * j + 1) * ld + m] = -sign * im;
    }
}

// q_0 = u / sqrt(<u,u>_O), s_0 = Omega^ u / sqrt(<u,u>_O) in place; xs = F s_0; apart = partials of s_0 . F s_0
__global__ void k_prpa_init(double* __restrict__ u, double* __restrict__ su, int64_t n4, int nb,
                            const double* __restrict__ normpart, int npart_in, LanczosState st, double* __restrict__ xs,
                            int64_t ldxs, int n_c, int n_cp, double* __restrict__ apart) {
    pdl_trigger();
    pdl_wait();
    __shared__ double sh[NT / 32 + 1];
    const int b = blockIdx.y;
    const double n2 = block_sum_array(normpart + (int64_t)b * npart_in, npart_in, sh);
    const bool ok = n2 > 0.0;
    const double r = ok ? 1.0 / sqrt(n2) : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        st.norm2[b] = ok ? n2 : 0.0;
        st.len[b] = ok ? st.steps : 0;
        st.scale[b] = 0.0;
        st.alive[b] = ok ? 1 : 0;
    }
    int64_t lo, hi;
    slice_of(n4, gridDim.x, blockIdx.x, lo, hi);
    const int64_t half = n4 / 2;
    double* ub = u + (int64_t)b * n4;
    double* sb = su + (int64_t)b * n4;
    double* xsb = xs + (int64_t)(2 * b) * ldxs;
    double acc = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += NT) {
        const double sg = i < half ? 1.0 : -1.0;
        const double qv = ok ? ub[i] * r : 0.0;
        const double sv = ok ? sb[i] * r : 0.0;
        ub[i] = qv;
        sb[i] = sv;
        xsb[xs_pos(i, half, ldxs, n_c, n_cp)] = sg * sv;
        acc += sg * sv * sv;
    }
    acc = block_sum(acc, sh);
    if (threadIdx.x == 0) apart[(int64_t)b * gridDim.x + blockIdx.x] = acc;
}

// a_k = sum(apart);  h = F s;  w = h - a q - b_k q_prev -> wq;  t holds the coupling part K^H W of Omega^ h on entry:
// Omega^ w = (t + Delta o h) - a s - b_k s_prev (in place in t; d2 = Delta [n4 / 2], the same for x and z);  partials of w . Omega^ w
__global__ void k_prpa_update1(double* __restrict__ t, double* __restrict__ wq, const double* __restrict__ q,
                               const double* __restrict__ q_prev, const double* __restrict__ s,
                               const double* __restrict__ s_prev, const double* __restrict__ d2, int64_t n4, int nb,
                               const double* __restrict__ apart, int napart, LanczosState st, int k,
                               double* __restrict__ normpart) {
    pdl_trigger();
    pdl_wait();
    __shared__ double sh[NT / 32 + 1];
    const int b = blockIdx.y;
    const int par = k & 1;
    const bool alive = st.alive[par * nb + b] != 0;
    double a = block_sum_array(apart + (int64_t)b * napart, napart, sh);
    if (!alive) a = 0.0;
    const double bprev = (k > 0) ? st.beta[(int64_t)b * st.steps + k - 1] : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) st.alpha[(int64_t)b * st.steps + k] = a;
    int64_t lo, hi;
    slice_of(n4, gridDim.x, blockIdx.x, lo, hi);
    const int64_t half = n4 / 2;
    const int64_t off = (int64_t)b * n4;
    double acc = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += NT) {
        const double sg = i < half ? 1.0 : -1.0;
        const double sv = s[off + i], qv = q[off + i];
        const double h = sg * sv;
        double w = h - a * qv;
        double sw = (t[off + i] + d2[i < half ? i : i - half] * h) - a * sv;
        if (k > 0) {
            w -= bprev * q_prev[off + i];
            sw -= bprev * s_prev[off + i];
        }
        wq[off + i] = w;
        t[off + i] = sw;
        acc += w * sw;
    }
    acc = block_sum(acc, sh);
    if (threadIdx.x == 0) normpart[(int64_t)b * gridDim.x + blockIdx.x] = acc;
}

// b_{k+1} = sqrt(sum normpart) (0 if the sum is not positive); breakdown test (reading Q9); q_{k+1} = w / b, s_{k+1} = Omega^ w / b in
// place; xs = F s_{k+1}; apart = partials of s_{k+1} . F s_{k+1} (the next a)
__global__ void k_prpa_update2(double* __restrict__ wq, double* __restrict__ sw, int64_t n4, int nb,
                               const double* __restrict__ normpart, int npart_in, LanczosState st, int k,
                               double* __restrict__ xs, int64_t ldxs, int n_c, int n_cp, double* __restrict__ apart) {
    pdl_trigger();
    pdl_wait();
    __shared__ double sh[NT / 32 + 1];
    const int b = blockIdx.y;
    const int par = k & 1;
    const double n2 = block_sum_array(normpart + (int64_t)b * npart_in, npart_in, sh);
    const double beta = n2 > 0.0 ? sqrt(n2) : 0.0;
    const bool alive = st.alive[par * nb + b] != 0;
    const double a = st.alpha[(int64_t)b * st.steps + k];
    const double sc_old = st.scale[par * nb + b];
    const double sc_new = fmax(sc_old, fabs(a) + beta);
    const bool broken = !alive || !(beta > 1e-12 * sc_new);
    const double rbeta = broken ? 0.0 : 1.0 / beta;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        st.beta[(int64_t)b * st.steps + k] = broken ? 0.0 : beta;
        st.scale[(par ^ 1) * nb + b] = sc_new;
        st.alive[(par ^ 1) * nb + b] = broken ? 0 : 1;
        if (alive && broken) st.len[b] = k + 1;
    }
    int64_t lo, hi;
    slice_of(n4, gridDim.x, blockIdx.x, lo, hi);
    const int64_t half = n4 / 2;
    const int64_t off = (int64_t)b * n4;
    double* xsb = xs + (int64_t)(2 * b) * ldxs;
    double acc = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += NT) {
        const double sg = i < half ? 1.0 : -1.0;
        const double qv = broken ? 0.0 : wq[off + i] * rbeta;
        const double sv = broken ? 0.0 : sw[off + i] * rbeta;
        wq[off + i] = qv;
        sw[off + i] = sv;
        xsb[xs_pos(i, half, ldxs, n_c, n_cp)] = sg * sv;
        acc += sg * sv * sv;
    }
    acc = block_sum(acc, sh);
    if (threadIdx.x == 0) apart[(int64_t)b * gridDim.x + blockIdx.x] = acc;
}

// Full reorthogonalisation in the Omega^ inner product: c_j = <q_j, w>_O = s_j^H w (complex) for the slots j = 0..nslots-1.
// In (x, z) variables s^H w = conj(s_x) . w_x + conj( conj(s_z) . w_z ).  coefpart [nb][nslots][2][npart].
__global__ void k_prpa_reorth_dots(const double* __restrict__ sbasis, int64_t slot_stride, const double* __restrict__ w,
                                   int64_t n4, double* __restrict__ coefpart, int npart) {
    pdl_trigger();
    pdl_wait();
    __shared__ double sh[NT / 32 + 1];
    const int blk = blockIdx.x, j = blockIdx.y, b = blockIdx.z;
    const int nslots = gridDim.y;
    const int64_t nq = n4 / 4;
    int64_t lo, hi;
    slice_of(nq, npart, blk, lo, hi);
    const double* sj = sbasis + (int64_t)j * slot_stride + (int64_t)b * n4;
    const double* wb = w + (int64_t)b * n4;
    double cre = 0.0, cim = 0.0;
    for (int64_t e = lo + threadIdx.x; e < hi; e += NT) {
        const double sxr = sj[e], sxi = sj[nq + e], szr = sj[2 * nq + e], szi = sj[3 * nq + e];
        const double wxr = wb[e], wxi = wb[nq + e], wzr = wb[2 * nq + e], wzi = wb[3 * nq + e];
        cre += (sxr * wxr + sxi * wxi) + (szr * wzr + szi * wzi);
        cim += (sxr * wxi - sxi * wxr) - (szr * wzi - szi * wzr);
    }
    cre = block_sum(cre, sh);
    cim = block_sum(cim, sh);
    if (threadIdx.x == 0) {
        double* cp = coefpart + (((int64_t)b * nslots + j) * 2) * npart;
        cp[blk] = cre;
        cp[npart + blk] = cim;
    }
}

// w -= sum_j c_j q_j and Omega^ w -= sum_j c_j s_j, where c [x; y] = (c x, conj(c) z) in the stored variables;
// normpart (may be NULL) = partials of the new w . Omega^ w
__global__ void k_prpa_reorth_apply(const double* __restrict__ qbasis, const double* __restrict__ sbasis, int64_t slot_stride,
                                    int nslots, double* __restrict__ w, double* __restrict__ sw, int64_t n4,
                                    const double* __restrict__ coefpart, int npart, double* __restrict__ normpart) {
    pdl_trigger();
    pdl_wait();
    extern __shared__ double coef[];  // [nslots][2]
    __shared__ double sh[NT / 32 + 1];
    const int blk = blockIdx.x, b = blockIdx.y;
    for (int t = threadIdx.x; t < 2 * nslots; t += NT) {
        const double* cp = coefpart + ((int64_t)b * nslots * 2 + t) * npart;
        double acc = 0.0;
        for (int i = 0; i < npart; ++i) acc += cp[i];
        coef[t] = acc;
    }
    __syncthreads();
    const int64_t nq = n4 / 4;
    int64_t lo, hi;
    slice_of(nq, gridDim.x, blk, lo, hi);
    double* wb = w + (int64_t)b * n4;
    double* swb = sw + (int64_t)b * n4;
    double acc = 0.0;
    for (int64_t e = lo + threadIdx.x; e < hi; e += NT) {
        double wv[4], sv[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            wv[c] = wb[c * nq + e];
            sv[c] = swb[c * nq + e];
        }
        for (int j = 0; j < nslots; ++j) {
            const double cr = coef[2 * j], ci = coef[2 * j + 1];
            const double* qj = qbasis + (int64_t)j * slot_stride + (int64_t)b * n4;
            const double* sj = sbasis + (int64_t)j * slot_stride + (int64_t)b * n4;
            const double qxr = qj[e], qxi = qj[nq + e], qzr = qj[2 * nq + e], qzi = qj[3 * nq + e];
            const double sxr = sj[e], sxi = sj[nq + e], szr = sj[2 * nq + e], szi = sj[3 * nq + e];
            wv[0] -= cr * qxr - ci * qxi;   // c q_x
            wv[1] -= cr * qxi + ci * qxr;
            wv[2] -= cr * qzr + ci * qzi;   // conj(c) q_z
            wv[3] -= cr * qzi - ci * qzr;
            sv[0] -= cr * sxr - ci * sxi;
            sv[1] -= cr * sxi + ci * sxr;
            sv[2] -= cr * szr + ci * szi;
            sv[3] -= cr * szi - ci * szr;
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            wb[c * nq + e] = wv[c];
            swb[c * nq + e] = sv[c];
            acc += wv[c] * sv[c];
        }
    }
    if (normpart != nullptr) {
        acc = block_sum(acc, sh);
        if (threadIdx.x == 0) normpart[(int64_t)b * gridDim.x + blk] = acc;
    }
}

// host-facing pairs [x; y] (interleaved complex, [nvec][n][2] each) <-> stored chains [x_re | x_im | Re y | -Im y]
__global__ void k_prpa_pack(const double* __restrict__ x, const double* __restrict__ y, int64_t n, double* __restrict__ out) {
    const int b = blockIdx.y;
    for (int64_t e = blockIdx.x * (int64_t)NT + threadIdx.x; e < n; e += (int64_t)gridDim.x * NT) {
        double* o = out + (int64_t)b * 4 * n;
        o[e] = x[((int64_t)b * n + e) * 2];
        o[n + e] = x[((int64_t)b * n + e) * 2 + 1];
        o[2 * n + e] = y[((int64_t)b * n + e) * 2];
        o[3 * n + e] = -y[((int64_t)b * n + e) * 2 + 1];
    }
}

__global__ void k_prpa_unpack(const double* __restrict__ in, int64_t n, double* __restrict__ x, double* __restrict__ y) {
    const int b = blockIdx.y;
    for (int64_t e = blockIdx.x * (int64_t)NT + threadIdx.x; e < n; e += (int64_t)gridDim.x * NT) {
        const double* o = in + (int64_t)b * 4 * n;
        x[((int64_t)b * n + e) * 2] = o[e];
        x[((int64_t)b * n + e) * 2 + 1] = o[n + e];
        y[((int64_t)b * n + e) * 2] = o[2 * n + e];
        y[((int64_t)b * n + e) * 2 + 1] = -o[3 * n + e];
    }
}

}  // namespace

cudaError_t launch_prpa_pack(const double* x, const double* y, int64_t n, int nvec, double* out, cudaStream_t st) {
    if (nvec <= 0) return cudaSuccess;
    dim3 grid((unsigned)std::min<int64_t>(ceil_div(n, NT), 1024), (unsigned)nvec);
    k_prpa_pack<<<grid, NT, 0, st>>>(x, y, n, out);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_prpa_unpack(const double* in, int64_t n, int nvec, double* x, double* y, cudaStream_t st) {
    if (nvec <= 0) return cudaSuccess;
    dim3 grid((unsigned)std::min<int64_t>(ceil_div(n, NT), 1024), (unsigned)nvec);
    k_prpa_unpack<<<grid, NT, 0, st>>>(in, n, x, y);
    count_launch();
    return cudaGetLastError();
}

int prpa_parts(int64_t n4) { return (int)std::max<int64_t>(1, std::min<int64_t>(64, ceil_div(n4, 8192))); }

cudaError_t launch_prpa_combine(const double* T, int64_t ld, int nb, int n_mu, double* Tc, cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    dim3 grid((unsigned)std::min<int64_t>(ceil_div(n_mu, NT), 64), (unsigned)nb);
    count_launch();
    return launch_pdl(k_prpa_combine, grid, dim3(NT), 0, st, 1, T, ld, nb, n_mu, Tc);
}

cudaError_t launch_prpa_expand(const double* Wc, int64_t ld, int nb, int n_mu, double sign, double* W, cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    dim3 grid((unsigned)std::min<int64_t>(ceil_div(n_mu, NT), 64), (unsigned)nb);
    count_launch();
    return launch_pdl(k_prpa_expand, grid, dim3(NT), 0, st, 1, Wc, ld, nb, n_mu, sign, W);
}

cudaError_t launch_prpa_init(double* u, double* su, int64_t n4, int nb, const double* normpart, int npart_in, LanczosState st_,
                             double* xs, int64_t ldxs, int n_c, int n_cp, double* apart, cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    dim3 grid((unsigned)prpa_parts(n4), (unsigned)nb);
    count_launch();
    return launch_pdl(k_prpa_init, grid, dim3(NT), 0, st, 1, u, su, n4, nb, normpart, npart_in, st_, xs, ldxs, n_c, n_cp, apart);
}

cudaError_t launch_prpa_update1(double* t, double* wq, const double* q, const double* q_prev, const double* s,
                                const double* s_prev, const double* d2, int64_t n4, int nb, const double* apart, LanczosState st_,
                                int k, double* normpart, cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    const int np = prpa_parts(n4);
    dim3 grid((unsigned)np, (unsigned)nb);
    count_launch();
    return launch_pdl(k_prpa_update1, grid, dim3(NT), 0, st, 1, t, wq, q, q_prev, s, s_prev, d2, n4, nb, apart, np, st_, k,
                      normpart);
}

cudaError_t launch_prpa_update2(double* wq, double* sw, int64_t n4, int nb, const double* normpart, LanczosState st_, int k,
                                double* xs, int64_t ldxs, int n_c, int n_cp, double* apart, cudaStream_t st) {
    if (nb <= 0) return cudaSuccess;
    const int np = prpa_parts(n4);
    dim3 grid((unsigned)np, (unsigned)nb);
    count_launch();
    return launch_pdl(k_prpa_update2, grid, dim3(NT), 0, st, 1, wq, sw, n4, nb, normpart, np, st_, k, xs, ldxs, n_c, n_cp, apart);
}

cudaError_t launch_prpa_reorth_dots(const double* sbasis, int64_t slot_stride, int nslots, const double* w, int64_t n4, int nb,
                                    double* coefpart, cudaStream_t st) {
    if (nb <= 0 || nslots <= 0) return cudaSuccess;
    const int np = prpa_parts(n4);
    for (int b0 = 0; b0 < nb; b0 += 65535) {  // grid.z limit
        const int nz = std::min(65535, nb - b0);
        dim3 grid((unsigned)np, (unsigned)nslots, (unsigned)nz);
        count_launch();
        cudaError_t e = launch_pdl(k_prpa_reorth_dots, grid, dim3(NT), 0, st, 1, sbasis + (int64_t)b0 * n4, slot_stride,
                                   w + (int64_t)b0 * n4, n4, coefpart + (int64_t)b0 * nslots * 2 * np, np);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_prpa_reorth_apply(const double* qbasis, const double* sbasis, int64_t slot_stride, int nslots, double* w,
                                     double* sw, int64_t n4, int nb, const double* coefpart, double* normpart, cudaStream_t st) {
    if (nb <= 0 || nslots <= 0) return cudaSuccess;
    const int np = prpa_parts(n4);
    dim3 grid((unsigned)np, (unsigned)nb);
    const size_t smem = (size_t)2 * nslots * sizeof(double);
    static SmemAttr attr;
    cudaError_t ea = attr.ensure(k_prpa_reorth_apply, smem);
    if (ea != cudaSuccess) return ea;
    count_launch();
    return launch_pdl(k_prpa_reorth_apply, grid, dim3(NT), smem, st, 1, qbasis, sbasis, slot_stride, nslots, w, sw, n4, coefpart, np,
                      normpart);
}

}  // namespace gwl
