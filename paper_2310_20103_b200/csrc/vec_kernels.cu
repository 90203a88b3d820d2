// Streaming (HBM-bound) kernels of the path: Delta scaling, split-K reduction, and the batched Lanczos
// three-term recurrence (Eq. 13) for nb independent chains, with optional two-pass full
// reorthogonalisation.  All reductions are two-stage and deterministic: a fixed slice per block, a fixed
// tree inside the block, and consumers re-reduce the per-block partials in a fixed order.
#include <cooperative_groups.h>

#include "gwl_internal.h"

namespace cg = cooperative_groups;

namespace gwl {

namespace {

constexpr int NT = VEC_THREADS;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block in a fixed order; result valid in every thread.
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

// Fixed-order sum of a global array of `cnt` doubles, same result in every block that calls it.
__device__ __forceinline__ double block_sum_array(const double* a, int cnt, double* sh) {
    double t = 0.0;
    for (int i = threadIdx.x; i < cnt; i += NT) t += a[i];
    return block_sum(t, sh);
}

__device__ __forceinline__ void slice_of(int64_t n, int npart, int blk, int64_t& lo, int64_t& hi) {
    const int64_t per = ((n + npart - 1) / npart + 1) & ~(int64_t)1;  // even: slices start 16-byte aligned
    lo = (int64_t)blk * per;
    hi = lo + per < n ? lo + per : n;
    if (lo > n) lo = n;
}

__device__ __forceinline__ int64_t xs_index(int64_t vc, int n_c, int n_cp) {
    if (n_c == n_cp) return vc;
    const int64_t v = vc / n_c;
    return v * n_cp + (vc - v * n_c);
}

__global__ void k_build_delta(const double* __restrict__ eps_v, const double* __restrict__ eps_c, int n_v, int n_c,
                              double* __restrict__ d2, double* __restrict__ s, int tda) {
    const int64_t n = (int64_t)n_v * n_c;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int v = (int)(i / n_c), c = (int)(i - (int64_t)v * n_c);
        const double d = eps_c[c] - eps_v[v];
        d2[i] = tda ? d : d * d;
        s[i] = tda ? 1.0 : sqrt(d);
    }
}

__global__ void k_prescale(const double* __restrict__ x, int64_t ldx, double* __restrict__ xs, int64_t ldxs,
                           const double* __restrict__ s, int n_c, int n_cp, int64_t n_vc) {
    pdl_trigger();
    pdl_wait();
    const int b = blockIdx.y;
    const double* xb = x + (int64_t)b * ldx;
    double* xsb = xs + (int64_t)b * ldxs;
    for (int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x; i < n_vc; i += (int64_t)gridDim.x * NT)
        xsb[xs_index(i, n_c, n_cp)] = s[i] * xb[i];
}

__global__ void k_splitk_reduce(const double* __restrict__ part, int64_t split_stride, int splits,
                                double* __restrict__ t, int64_t ld, int m) {
    pdl_trigger();
    pdl_wait();
    const int b = blockIdx.y;
    for (int i = blockIdx.x * NT + threadIdx.x; i < m; i += gridDim.x * NT) {
        const double* p = part + (int64_t)b * ld + i;
        double acc = 0.0;
        for (int z = 0; z < splits; ++z) acc += p[(int64_t)z * split_stride];
        t[(int64_t)b * ld + i] = acc;
    }
}

__global__ void k_transpose(const double* __restrict__ src, int rows, int cols, double* __restrict__ dst,
                            int64_t ld_dst) {
    __shared__ double tile[32][33];
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    for (int i = threadIdx.y; i < 32; i += blockDim.y) {
        const int r = r0 + i, c = c0 + threadIdx.x;
        if (r < rows && c < cols) tile[i][threadIdx.x] = src[(int64_t)r * cols + c];
    }
    __syncthreads();
    for (int i = threadIdx.y; i < 32; i += blockDim.y) {
        const int c = c0 + i, r = r0 + threadIdx.x;
        if (r < rows && c < cols) dst[(int64_t)c * ld_dst + r] = tile[threadIdx.x][i];
    }
}

__global__ void k_copy_pad(const double* __restrict__ src, int rows, int cols, double* __restrict__ dst,
                           int64_t ld_dst) {
    const int64_t n = (int64_t)rows * cols;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / cols, c = i - r * cols;
        dst[r * ld_dst + c] = src[i];
    }
}

__global__ void k_rho(const double* __restrict__ phivT, const double* __restrict__ phicT, int64_t ldt, int n_v,
                      int n_mu, const int32_t* __restrict__ n_idx, const int32_t* __restrict__ m_idx,
                      double* __restrict__ rho, int64_t ld_rho) {
    pdl_trigger();
    pdl_wait();
    const int b = blockIdx.y;
    const int n = n_idx[b], m = m_idx[b];
    const double* pn = n < n_v ? phivT + (int64_t)n * ldt : phicT + (int64_t)(n - n_v) * ldt;
    const double* pm = m < n_v ? phivT + (int64_t)m * ldt : phicT + (int64_t)(m - n_v) * ldt;
    for (int i = blockIdx.x * NT + threadIdx.x; i < n_mu; i += gridDim.x * NT)
        rho[(int64_t)b * ld_rho + i] = pn[i] * pm[i];
}

__global__ void k_dot_partials(const double* __restrict__ x, const double* __restrict__ y, int64_t ld, int64_t n,
                               double* __restrict__ part, int npart) {
    pdl_trigger();
    pdl_wait();
    __shared__ double sh[NT / 32 + 1];
    const int b = blockIdx.y;
    int64_t lo, hi;
    slice_of(n, npart, blockIdx.x, lo, hi);
    const double* xb = x + (int64_t)b * ld;
    const double* yb = y + (int64_t)b * ld;
    double acc = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += NT) acc += xb[i] * yb[i];
    acc = block_sum(acc, sh);
    if (threadIdx.x == 0) part[(int64_t)b * npart + blockIdx.x] = acc;
}

// state parity: arrays scale/alive hold two copies [2][nb]; step k reads copy k&1 and writes copy (k+1)&1,
// so that blocks of one launch never read what another block of the same launch writes.
__global__ void k_lanczos_init(double* __restrict__ p, int64_t n_vc, int nb, const double* __restrict__ normpart,
                               int npart, LanczosState st, double* __restrict__ xs, int64_t ldxs,
                               const double* __restrict__ s, int n_c, int n_cp) {
    pdl_trigger();
    pdl_wait();
    __shared__ double sh[NT / 32 + 1];
    const int b = blockIdx.y;
    const double n2 = block_sum_array(normpart + (int64_t)b * npart, npart, sh);
    const bool ok = n2 > 0.0;
    // one division per thread, then a multiply per element (the normalised vector differs from w / ||w|| by <= 1 ulp
    // per element; a per-element div.rn.f64 costs ~30 FP64 instructions and made update2 ALU- rather than HBM-bound)
    const double rnrm = ok ? 1.0 / sqrt(n2) : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        st.norm2[b] = n2;
        st.len[b] = ok ? st.steps : 0;
        st.scale[b] = 0.0;
        st.alive[b] = ok ? 1 : 0;
    }
    int64_t lo, hi;
    slice_of(n_vc, gridDim.x, blockIdx.x, lo, hi);
    double* pb = p + (int64_t)b * n_vc;
    double* xsb = xs + (int64_t)b * ldxs;
    for (int64_t i = lo + threadIdx.x; i < hi; i += NT) {
        const double qv = ok ? pb[i] * rnrm : 0.0;
        pb[i] = qv;
        xsb[xs_index(i, n_c, n_cp)] = s[i] * qv;
    }
}

__global__ void k_lanczos_update1(double* __restrict__ w, const double* __restrict__ q,
                                  const double* __restrict__ q_prev, int64_t n_vc, int nb,
                                  const double* __restrict__ dotpart, int ndot, int dot_stride, LanczosState st, int k,
                                  double* __restrict__ normpart, int npart) {
    pdl_trigger();
    pdl_wait();
    __shared__ double sh[NT / 32 + 1];
    const int b = blockIdx.y;
    const int par = k & 1;
    const bool alive = st.alive[par * nb + b] != 0;
    double a = block_sum_array(dotpart + (int64_t)b * dot_stride, ndot, sh);
    if (!alive) a = 0.0;
    const double bprev = (k > 0) ? st.beta[(int64_t)b * st.steps + k - 1] : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) st.alpha[(int64_t)b * st.steps + k] = a;
    int64_t lo, hi;
    slice_of(n_vc, npart, blockIdx.x, lo, hi);
    double* wb = w + (int64_t)b * n_vc;
    const double* qb = q + (int64_t)b * n_vc;
    double acc = 0.0;
    if (k > 0) {
        const double* qp = q_prev + (int64_t)b * n_vc;
        for (int64_t i = lo + threadIdx.x; i < hi; i += NT) {
            const double v = wb[i] - a * qb[i] - bprev * qp[i];
            wb[i] = v;
            acc += v * v;
        }
    } else {
        for (int64_t i = lo + threadIdx.x; i < hi; i += NT) {
            const double v = wb[i] - a * qb[i];
            wb[i] = v;
            acc += v * v;
        }
    }
    acc = block_sum(acc, sh);
    if (threadIdx.x == 0) normpart[(int64_t)b * npart + blockIdx.x] = acc;
}

__global__ void k_lanczos_update2(double* __restrict__ w, int64_t n_vc, int nb, const double* __restrict__ normpart,
                                  int npart, LanczosState st, int k, double* __restrict__ xs, int64_t ldxs,
                                  const double* __restrict__ s, int n_c, int n_cp) {
    pdl_trigger();
    pdl_wait();
    __shared__ double sh[NT / 32 + 1];
    const int b = blockIdx.y;
    const int par = k & 1;
    const double n2 = block_sum_array(normpart + (int64_t)b * npart, npart, sh);
    const double beta = sqrt(n2);
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
    slice_of(n_vc, gridDim.x, blockIdx.x, lo, hi);
    double* wb = w + (int64_t)b * n_vc;
    double* xsb = xs + (int64_t)b * ldxs;
    if (n_c == n_cp && ((n_vc | ldxs) & 1) == 0) {  // no padding inside xs, every chain 16-byte aligned: 16-byte accesses
        double2* w2 = reinterpret_cast<double2*>(wb);
        double2* x2 = reinterpret_cast<double2*>(xsb);
        const double2* s2 = reinterpret_cast<const double2*>(s);
        for (int64_t i = (lo >> 1) + threadIdx.x; i < ((hi + 1) >> 1); i += NT) {
            double2 v = w2[i];
            const double2 sv = __ldg(s2 + i);
            v.x = broken ? 0.0 : v.x * rbeta;
            v.y = broken ? 0.0 : v.y * rbeta;
            w2[i] = v;
            x2[i] = make_double2(sv.x * v.x, sv.y * v.y);
        }
        return;
    }
    for (int64_t i = lo + threadIdx.x; i < hi; i += NT) {
        const double qv = broken ? 0.0 : wb[i] * rbeta;
        wb[i] = qv;
        xsb[xs_index(i, n_c, n_cp)] = s[i] * qv;
    }
}

// Single-pass Lanczos update for vectors that fit in the registers of one thread-block cluster (reorth off):
//   alpha_k = sum(dotpart);  w <- w - alpha q - beta_k q_prev;  beta_{k+1} = ||w||;  q_next = w / beta_{k+1};  xs = s o q_next
// One cluster of gridDim.x CTAs per chain; each CTA keeps its slice of w in registers between the two phases and
// the norm is reduced across the cluster through distributed shared memory in a fixed order (rank 0..CS-1), so that
// every CTA of the cluster sees the same beta bit for bit.  w, q, q_prev are read once and q_next, xs written once:
// 40 N_vc bytes per chain-step instead of the 64 N_vc of the two-kernel path.
template <int EPT>
__global__ void __launch_bounds__(NT) k_lanczos_fused(double* __restrict__ w, const double* __restrict__ q,
                                                      const double* __restrict__ q_prev, int64_t n_vc, int nb,
                                                      const double* __restrict__ dotpart, int ndot, int dot_stride,
                                                      LanczosState st, int k_arg, double* __restrict__ xs, int64_t ldxs,
                                                      const double* __restrict__ s, int n_c, int n_cp) {
    pdl_trigger();
    pdl_wait();
    const int k = k_arg + (st.kbase != nullptr ? *st.kbase : 0);  // graph replay: the step number lives on the device
    __shared__ double sh[NT / 32 + 1];
    __shared__ double cl_part;  // this CTA's partial of ||w||^2; read by the other CTAs of the cluster
    __shared__ double cl_sum;
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned rank = cluster.block_rank(), cs = cluster.num_blocks();
    const int b = blockIdx.y;
    const int par = k & 1;
    const bool alive = st.alive[par * nb + b] != 0;
    double a = block_sum_array(dotpart + (int64_t)b * dot_stride, ndot, sh);
    if (!alive) a = 0.0;
    const double bprev = (k > 0) ? st.beta[(int64_t)b * st.steps + k - 1] : 0.0;
    int64_t lo, hi;
    slice_of(n_vc, (int)cs, (int)rank, lo, hi);
    double* wb = w + (int64_t)b * n_vc;
    const double* qb = q + (int64_t)b * n_vc;
    const double* qp = q_prev + (int64_t)b * n_vc;
    double v[EPT];
    double acc = 0.0;
#pragma unroll
    for (int j = 0; j < EPT; ++j) {
        const int64_t i = lo + threadIdx.x + (int64_t)j * NT;
        v[j] = 0.0;
        if (i < hi) {
            v[j] = (k > 0) ? wb[i] - a * qb[i] - bprev * qp[i] : wb[i] - a * qb[i];
            acc += v[j] * v[j];
        }
    }
    acc = block_sum(acc, sh);
    if (threadIdx.x == 0) cl_part = acc;
    cluster.sync();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (unsigned r = 0; r < cs; ++r) t += *cluster.map_shared_rank(&cl_part, r);
        cl_sum = t;
    }
    __syncthreads();
    // all remote reads of this cluster are done once every CTA has passed this arrive; the matching wait sits at the end
    asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory");
    const double n2 = cl_sum;
    const double beta = sqrt(n2);
    const double sc_old = st.scale[par * nb + b];
    const double sc_new = fmax(sc_old, fabs(a) + beta);
    const bool broken = !alive || !(beta > 1e-12 * sc_new);
    const double rbeta = broken ? 0.0 : 1.0 / beta;
    if (rank == 0 && threadIdx.x == 0) {
        st.alpha[(int64_t)b * st.steps + k] = a;
        st.beta[(int64_t)b * st.steps + k] = broken ? 0.0 : beta;
        st.scale[(par ^ 1) * nb + b] = sc_new;
        st.alive[(par ^ 1) * nb + b] = broken ? 0 : 1;
        if (alive && broken) st.len[b] = k + 1;
    }
    double* xsb = xs + (int64_t)b * ldxs;
#pragma unroll
    for (int j = 0; j < EPT; ++j) {
        const int64_t i = lo + threadIdx.x + (int64_t)j * NT;
        if (i < hi) {
            const double qv = broken ? 0.0 : v[j] * rbeta;
            wb[i] = qv;
            xsb[xs_index(i, n_c, n_cp)] = s[i] * qv;
        }
    }
    asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}

// ---- full reorthogonalisation (classical Gram-Schmidt, run twice): c = Q^T w, w -= Q c ---------------------------
// HBM-bound: every pass streams the k+1 basis vectors of each chain twice (dots, apply).  Slices of RSLICE
// elements per block (reorth_parts(n_vc) of them) so that a few blocks per SM keep enough loads in flight.
// dots: the slice of w is staged in shared memory once; each WARP then takes basis vectors i = warp, warp + 8, ...
// and reduces its dot by shuffles -- no block-wide barrier inside the loop over basis vectors.
// coefpart[(b*nslots + i)*npart + blk] = sum over the slice of basis_i[b] * w[b]
constexpr int RSLICE = 2048;

__global__ void __launch_bounds__(NT) k_reorth_dots(const double* __restrict__ basis, int64_t slot_stride, int nslots,
                                                    const double* __restrict__ w, int64_t n_vc,
                                                    double* __restrict__ coefpart, int npart, int64_t slice) {
    pdl_trigger();
    pdl_wait();
    extern __shared__ double ws[];  // [RSLICE] chunk of w, then [nslots] running sums (one owner warp per basis vector)
    double* accs = ws + RSLICE;
    const int b = blockIdx.y;
    const int64_t lo = (int64_t)blockIdx.x * slice;
    const int64_t len = max((int64_t)0, min(slice, n_vc - lo));
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool vec2 = ((n_vc | slot_stride | slice) & 1) == 0;  // 16-byte alignment of every (slot, chain, slice) start
    for (int i = threadIdx.x; i < nslots; i += NT) accs[i] = 0.0;
    // a slice longer than RSLICE (N_vc > 64 * RSLICE) is walked in chunks; the chunk order is fixed
    for (int64_t c0 = 0; c0 < len; c0 += RSLICE) {
        const int clen = (int)min((int64_t)RSLICE, len - c0);
        const double* wb = w + (int64_t)b * n_vc + lo + c0;
        __syncthreads();  // the previous chunk has been consumed (and accs is initialised)
        for (int j = threadIdx.x; j < clen; j += NT) ws[j] = wb[j];
        __syncthreads();
        for (int i = warp; i < nslots; i += NT / 32) {
            const double* qb = basis + (int64_t)i * slot_stride + (int64_t)b * n_vc + lo + c0;
            double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
            if (vec2) {
                const double2* q2 = reinterpret_cast<const double2*>(qb);
                const double2* w2 = reinterpret_cast<const double2*>(ws);
                const int n2 = clen >> 1;
                int j = lane;
                for (; j + 96 < n2; j += 128) {
                    const double2 x0 = __ldg(q2 + j), x1 = __ldg(q2 + j + 32), x2 = __ldg(q2 + j + 64), x3 = __ldg(q2 + j + 96);
                    const double2 y0 = w2[j], y1 = w2[j + 32], y2 = w2[j + 64], y3 = w2[j + 96];
                    a0 = fma(x0.x, y0.x, fma(x0.y, y0.y, a0));
                    a1 = fma(x1.x, y1.x, fma(x1.y, y1.y, a1));
                    a2 = fma(x2.x, y2.x, fma(x2.y, y2.y, a2));
                    a3 = fma(x3.x, y3.x, fma(x3.y, y3.y, a3));
                }
                for (; j < n2; j += 32) {
                    const double2 x0 = __ldg(q2 + j);
                    const double2 y0 = w2[j];
                    a0 = fma(x0.x, y0.x, fma(x0.y, y0.y, a0));
                }
            } else {
                for (int j = lane; j < clen; j += 32) a0 = fma(__ldg(qb + j), ws[j], a0);
            }
            const double acc = warp_sum((a0 + a1) + (a2 + a3));
            if (lane == 0) accs[i] += acc;  // basis vector i always belongs to this warp
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nslots; i += NT) coefpart[((int64_t)b * nslots + i) * npart + blockIdx.x] = accs[i];
}

// w -= sum_i c_i basis_i, c_i = fixed-order sum of the partials; optionally the partial norms of the new w.
__global__ void __launch_bounds__(NT) k_reorth_apply(const double* __restrict__ basis, int64_t slot_stride, int nslots,
                                                     double* __restrict__ w, int64_t n_vc,
                                                     const double* __restrict__ coefpart, int npart,
                                                     double* __restrict__ normpart, int64_t slice) {
    pdl_trigger();
    pdl_wait();
    extern __shared__ double coef[];  // [nslots] + block_sum scratch
    double* sh = coef + nslots;
    const int b = blockIdx.y;
    for (int i = threadIdx.x; i < nslots; i += NT) {
        const double* cp = coefpart + ((int64_t)b * nslots + i) * npart;
        double t = 0.0;
        for (int j = 0; j < npart; ++j) t += cp[j];
        coef[i] = t;
    }
    __syncthreads();
    const int64_t lo = (int64_t)blockIdx.x * slice;
    const int len = (int)max((int64_t)0, min(slice, n_vc - lo));
    double* wb = w + (int64_t)b * n_vc + lo;
    const double* q0 = basis + (int64_t)b * n_vc + lo;
    const bool vec2 = ((n_vc | slot_stride | slice) & 1) == 0;
    double acc = 0.0;
    if (vec2) {
        const int n2 = len >> 1;
        for (int j = threadIdx.x; j < n2; j += NT) {
            double2 v = reinterpret_cast<double2*>(wb)[j];
            int i = 0;
            for (; i + 3 < nslots; i += 4) {  // four independent 16-byte loads in flight per thread
                const double2 x0 = __ldg(reinterpret_cast<const double2*>(q0 + (int64_t)i * slot_stride) + j);
                const double2 x1 = __ldg(reinterpret_cast<const double2*>(q0 + (int64_t)(i + 1) * slot_stride) + j);
                const double2 x2 = __ldg(reinterpret_cast<const double2*>(q0 + (int64_t)(i + 2) * slot_stride) + j);
                const double2 x3 = __ldg(reinterpret_cast<const double2*>(q0 + (int64_t)(i + 3) * slot_stride) + j);
                const double c0 = coef[i], c1 = coef[i + 1], c2 = coef[i + 2], c3 = coef[i + 3];
                v.x -= c0 * x0.x;
                v.y -= c0 * x0.y;
                v.x -= c1 * x1.x;
                v.y -= c1 * x1.y;
                v.x -= c2 * x2.x;
                v.y -= c2 * x2.y;
                v.x -= c3 * x3.x;
                v.y -= c3 * x3.y;
            }
            for (; i < nslots; ++i) {
                const double2 x0 = __ldg(reinterpret_cast<const double2*>(q0 + (int64_t)i * slot_stride) + j);
                v.x -= coef[i] * x0.x;
                v.y -= coef[i] * x0.y;
            }
            reinterpret_cast<double2*>(wb)[j] = v;
            acc += v.x * v.x + v.y * v.y;
        }
        if ((len & 1) && threadIdx.x == 0) {
            double v = wb[len - 1];
            for (int i = 0; i < nslots; ++i) v -= coef[i] * q0[(int64_t)i * slot_stride + len - 1];
            wb[len - 1] = v;
            acc += v * v;
        }
    } else {
        for (int j = threadIdx.x; j < len; j += NT) {
            double v = wb[j];
            for (int i = 0; i < nslots; ++i) v -= coef[i] * __ldg(q0 + (int64_t)i * slot_stride + j);
            wb[j] = v;
            acc += v * v;
        }
    }
    if (normpart != nullptr) {
        acc = block_sum(acc, sh);
        if (threadIdx.x == 0) normpart[(int64_t)b * npart + blockIdx.x] = acc;
    }
}

// ---- the same for complex (planar) Lanczos vectors of the periodic Tamm-Dancoff variant ------------------------------
// w = [w_r (N) | w_i (N)], N = n_vc / 2.  The projection coefficient on q_j is the COMPLEX <q_j, w> =
// (q_r.w_r + q_i.w_i) + i (q_r.w_i - q_i.w_r): the real dot of the stacked vectors is only its real part, and rounding
// feeds the imaginary part just as much (without it the basis lost orthogonality after ~30 steps at 16 384 pairs).
// coefpart[((b*nslots + i)*2 + part)*npart + blk]; slices run over the N complex elements.
__global__ void __launch_bounds__(NT) k_reorth_dots_c(const double* __restrict__ basis, int64_t slot_stride, int nslots,
                                                      const double* __restrict__ w, int64_t n_vc,
                                                      double* __restrict__ coefpart, int npart, int64_t slice) {
    pdl_trigger();
    pdl_wait();
    extern __shared__ double ws[];  // [RSLICE] w_r chunk, [RSLICE] w_i chunk, [2 nslots] running sums
    double* wi_s = ws + RSLICE;
    double* accs = ws + 2 * RSLICE;
    const int b = blockIdx.y;
    const int64_t N = n_vc >> 1;
    const int64_t lo = (int64_t)blockIdx.x * slice;
    const int64_t len = max((int64_t)0, min(slice, N - lo));
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < 2 * nslots; i += NT) accs[i] = 0.0;
    for (int64_t c0 = 0; c0 < len; c0 += RSLICE) {
        const int clen = (int)min((int64_t)RSLICE, len - c0);
        const double* wb = w + (int64_t)b * n_vc + lo + c0;
        __syncthreads();
        for (int j = threadIdx.x; j < clen; j += NT) {
            ws[j] = wb[j];
            wi_s[j] = wb[N + j];
        }
        __syncthreads();
        for (int i = warp; i < nslots; i += NT / 32) {
            const double* qb = basis + (int64_t)i * slot_stride + (int64_t)b * n_vc + lo + c0;
            double ar0 = 0.0, ar1 = 0.0, ai0 = 0.0, ai1 = 0.0;
            int j = lane;
            for (; j + 32 < clen; j += 64) {
                const double qr0 = __ldg(qb + j), qi0 = __ldg(qb + N + j), qr1 = __ldg(qb + j + 32), qi1 = __ldg(qb + N + j + 32);
                ar0 = fma(qr0, ws[j], fma(qi0, wi_s[j], ar0));
                ai0 = fma(qr0, wi_s[j], fma(-qi0, ws[j], ai0));
                ar1 = fma(qr1, ws[j + 32], fma(qi1, wi_s[j + 32], ar1));
                ai1 = fma(qr1, wi_s[j + 32], fma(-qi1, ws[j + 32], ai1));
            }
            for (; j < clen; j += 32) {
                const double qr0 = __ldg(qb + j), qi0 = __ldg(qb + N + j);
                ar0 = fma(qr0, ws[j], fma(qi0, wi_s[j], ar0));
                ai0 = fma(qr0, wi_s[j], fma(-qi0, ws[j], ai0));
            }
            const double sr = warp_sum(ar0 + ar1), si = warp_sum(ai0 + ai1);
            if (lane == 0) {
                accs[2 * i] += sr;
                accs[2 * i + 1] += si;
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * nslots; i += NT) coefpart[((int64_t)b * 2 * nslots + i) * npart + blockIdx.x] = accs[i];
}

__global__ void __launch_bounds__(NT) k_reorth_apply_c(const double* __restrict__ basis, int64_t slot_stride, int nslots,
                                                       double* __restrict__ w, int64_t n_vc,
                                                       const double* __restrict__ coefpart, int npart,
                                                       double* __restrict__ normpart, int64_t slice) {
    pdl_trigger();
    pdl_wait();
    extern __shared__ double coef[];  // [2 nslots] (re, im) + block_sum scratch
    double* sh = coef + 2 * nslots;
    const int b = blockIdx.y;
    const int64_t N = n_vc >> 1;
    for (int i = threadIdx.x; i < 2 * nslots; i += NT) {
        const double* cp = coefpart + ((int64_t)b * 2 * nslots + i) * npart;
        double t = 0.0;
        for (int j = 0; j < npart; ++j) t += cp[j];
        coef[i] = t;
    }
    __syncthreads();
    const int64_t lo = (int64_t)blockIdx.x * slice;
    const int len = (int)max((int64_t)0, min(slice, N - lo));
    double* wb = w + (int64_t)b * n_vc + lo;
    const double* q0 = basis + (int64_t)b * n_vc + lo;
    double acc = 0.0;
    for (int j = threadIdx.x; j < len; j += NT) {
        double vr = wb[j], vi = wb[N + j];
        for (int i = 0; i < nslots; ++i) {
            const double qr = __ldg(q0 + (int64_t)i * slot_stride + j), qi = __ldg(q0 + (int64_t)i * slot_stride + N + j);
            const double cr = coef[2 * i], ci = coef[2 * i + 1];
            vr -= cr * qr - ci * qi;
            vi -= cr * qi + ci * qr;
        }
        wb[j] = vr;
        wb[N + j] = vi;
        acc += vr * vr + vi * vi;
    }
    if (normpart != nullptr) {
        acc = block_sum(acc, sh);
        if (threadIdx.x == 0) normpart[(int64_t)b * npart + blockIdx.x] = acc;
    }
}

// ---- complex (planar) helpers of the periodic Tamm-Dancoff variant -------------------------------------------------
__global__ void k_scatter_complex(const double* __restrict__ src, int n_k, int n_m, int n_o, double* __restrict__ dst_r,
                                  double* __restrict__ dst_i, int64_t stride_k, int64_t stride_m, int64_t stride_o) {
    const int64_t n = (int64_t)n_k * n_m * n_o;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t o = i % n_o, m = (i / n_o) % n_m, k = i / ((int64_t)n_o * n_m);
        const int64_t d = k * stride_k + m * stride_m + o * stride_o;
        dst_r[d] = src[2 * i];
        dst_i[d] = src[2 * i + 1];
    }
}

__global__ void k_deinterleave(const double* __restrict__ src, int64_t n, double* __restrict__ dst) {
    const int b = blockIdx.y;
    const double2* s2 = reinterpret_cast<const double2*>(src) + (int64_t)b * n;
    double* d = dst + (int64_t)b * 2 * n;
    for (int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x; i < n; i += (int64_t)gridDim.x * NT) {
        const double2 v = s2[i];
        d[i] = v.x;
        d[n + i] = v.y;
    }
}

__global__ void k_interleave(const double* __restrict__ src, int64_t n, double* __restrict__ dst) {
    const int b = blockIdx.y;
    const double* s = src + (int64_t)b * 2 * n;
    double2* d2 = reinterpret_cast<double2*>(dst) + (int64_t)b * n;
    for (int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x; i < n; i += (int64_t)gridDim.x * NT)
        d2[i] = make_double2(s[i], s[n + i]);
}

__global__ void k_rho_c(const double* __restrict__ psivT, int64_t pv_plane, const double* __restrict__ psicT,
                        int64_t pc_plane, int64_t ldt, int n_v, int n_c, int n_mu, const int32_t* __restrict__ chains,
                        double* __restrict__ rho, int64_t ld_rho, int nb) {
    pdl_trigger();
    pdl_wait();
    const int b = blockIdx.y;
    const int kn = chains[4 * b], n = chains[4 * b + 1], km = chains[4 * b + 2], m = chains[4 * b + 3];
    const double* pn = n < n_v ? psivT + ((int64_t)kn * n_v + n) * ldt : psicT + ((int64_t)kn * n_c + (n - n_v)) * ldt;
    const double* pm = m < n_v ? psivT + ((int64_t)km * n_v + m) * ldt : psicT + ((int64_t)km * n_c + (m - n_v)) * ldt;
    const int64_t pln = n < n_v ? pv_plane : pc_plane, plm = m < n_v ? pv_plane : pc_plane;
    for (int i = blockIdx.x * NT + threadIdx.x; i < n_mu; i += gridDim.x * NT) {
        const double nr = pn[i], ni = pn[pln + i], mr = pm[i], mi = pm[plm + i];
        // psi_m conj(psi_n)
        rho[(int64_t)b * ld_rho + i] = mr * nr + mi * ni;
        rho[(int64_t)(nb + b) * ld_rho + i] = mi * nr - mr * ni;
    }
}

__global__ void k_build_delta_c(const double* __restrict__ eps_v, const double* __restrict__ eps_cq, int n_k, int n_v,
                                int n_c, double* __restrict__ d2, double* __restrict__ s) {
    const int64_t n = (int64_t)n_k * n_v * n_c;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int c = (int)(i % n_c), v = (int)((i / n_c) % n_v), k = (int)(i / ((int64_t)n_c * n_v));
        const double d = eps_cq[(int64_t)k * n_c + c] - eps_v[(int64_t)k * n_v + v];
        d2[i] = d;
        d2[n + i] = d;
        s[i] = 1.0;
        s[n + i] = 1.0;
    }
}

// x[i] = uniform in [-1, 1) from a counter-based hash (splitmix64 finaliser) of (seed, i): a generic start vector
__global__ void k_set_int(int* p, int v) {
    pdl_trigger();
    pdl_wait();
    *p = v;
}

__global__ void k_add_int(int* p, int d) {
    pdl_trigger();
    pdl_wait();
    *p += d;
}

__global__ void k_fill_hash(double* __restrict__ x, int64_t n, unsigned long long seed) {
    for (int64_t i = blockIdx.x * (int64_t)NT + threadIdx.x; i < n; i += (int64_t)gridDim.x * NT) {
        unsigned long long z = seed + 0x9E3779B97F4A7C15ull * (unsigned long long)(i + 1);
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        z ^= z >> 31;
        x[i] = (double)(z >> 11) * (2.0 / 9007199254740992.0) - 1.0;
    }
}

inline unsigned grid1d(int64_t n, int per_thread = 4) {
    int64_t g = ceil_div(n, (int64_t)NT * per_thread);
    return (unsigned)std::max<int64_t>(1, std::min<int64_t>(g, (int64_t)device_sm_count() * 32));
}

}  // namespace

int vec_parts(int64_t n_vc) { return (int)std::max<int64_t>(1, std::min<int64_t>(64, ceil_div(n_vc, 8192))); }

cudaError_t launch_build_delta(const double* eps_v, const double* eps_c, int n_v, int n_c, double* d2, double* s,
                               int tda, cudaStream_t st) {
    k_build_delta<<<grid1d((int64_t)n_v * n_c, 1), NT, 0, st>>>(eps_v, eps_c, n_v, n_c, d2, s, tda);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_scatter_complex(const double* src, int n_k, int n_m, int n_o, double* dst_r, double* dst_i,
                                   int64_t stride_k, int64_t stride_m, int64_t stride_o, cudaStream_t st) {
    k_scatter_complex<<<grid1d((int64_t)n_k * n_m * n_o, 1), NT, 0, st>>>(src, n_k, n_m, n_o, dst_r, dst_i, stride_k, stride_m,
                                                                          stride_o);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_deinterleave(const double* src, int64_t n, int nvec, double* dst, cudaStream_t st) {
    dim3 grid(std::min<unsigned>(grid1d(n), 1024u), (unsigned)nvec);
    k_deinterleave<<<grid, NT, 0, st>>>(src, n, dst);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_interleave(const double* src, int64_t n, int nvec, double* dst, cudaStream_t st) {
    dim3 grid(std::min<unsigned>(grid1d(n), 1024u), (unsigned)nvec);
    k_interleave<<<grid, NT, 0, st>>>(src, n, dst);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_rho_c(const double* psivT, int64_t pv_plane, const double* psicT, int64_t pc_plane, int64_t ldt, int n_v,
                         int n_c, int n_mu, const int32_t* chains, double* rho, int64_t ld_rho, int nb, cudaStream_t st) {
    dim3 grid((unsigned)ceil_div(n_mu, NT), (unsigned)nb);
    cudaError_t le = launch_pdl(k_rho_c, grid, dim3(NT), (size_t)0, st, 1u, psivT, pv_plane, psicT, pc_plane, ldt, n_v, n_c,
                                n_mu, chains, rho, ld_rho, nb);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_build_delta_c(const double* eps_v, const double* eps_cq, int n_k, int n_v, int n_c, double* d2,
                                 double* s, cudaStream_t st) {
    k_build_delta_c<<<grid1d((int64_t)n_k * n_v * n_c, 1), NT, 0, st>>>(eps_v, eps_cq, n_k, n_v, n_c, d2, s);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_set_int(int* p, int v, cudaStream_t st) {
    cudaError_t e = launch_pdl(k_set_int, dim3(1), dim3(1), 0, st, 1u, p, v);
    count_launch();
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_add_int(int* p, int d, cudaStream_t st) {
    cudaError_t e = launch_pdl(k_add_int, dim3(1), dim3(1), 0, st, 1u, p, d);
    count_launch();
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_fill_hash(double* x, int64_t n, unsigned long long seed, cudaStream_t st) {
    k_fill_hash<<<grid1d(n), NT, 0, st>>>(x, n, seed);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_prescale(const double* x, int64_t ldx, double* xs, int64_t ldxs, const double* s, int n_v, int n_c,
                            int n_cp, int nb, cudaStream_t st) {
    const int64_t n_vc = (int64_t)n_v * n_c;
    dim3 grid(std::min<unsigned>(grid1d(n_vc), 1024u), (unsigned)nb);
    cudaError_t le = launch_pdl(k_prescale, dim3(grid), dim3(NT), (size_t)(0), st, 1u, x, ldx, xs, ldxs, s, n_c, n_cp, n_vc);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_splitk_reduce(const double* part, int64_t split_stride, int splits, double* t, int64_t ld, int m,
                                 int nb, cudaStream_t st) {
    dim3 grid((unsigned)ceil_div(m, NT), (unsigned)nb);
    cudaError_t le = launch_pdl(k_splitk_reduce, dim3(grid), dim3(NT), (size_t)(0), st, 1u, part, split_stride, splits, t, ld, m);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_transpose(const double* src, int rows, int cols, double* dst, int64_t ld_dst, cudaStream_t st) {
    dim3 grid((unsigned)ceil_div(cols, 32), (unsigned)ceil_div(rows, 32));
    k_transpose<<<grid, dim3(32, 8), 0, st>>>(src, rows, cols, dst, ld_dst);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_copy_pad(const double* src, int rows, int cols, double* dst, int64_t ld_dst, cudaStream_t st) {
    k_copy_pad<<<grid1d((int64_t)rows * cols, 1), NT, 0, st>>>(src, rows, cols, dst, ld_dst);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_rho(const double* phivT, const double* phicT, int64_t ldt, int n_v, int n_mu, const int32_t* n_idx,
                       const int32_t* m_idx, double* rho, int64_t ld_rho, int nb, cudaStream_t st) {
    dim3 grid((unsigned)ceil_div(n_mu, NT), (unsigned)nb);
    cudaError_t le = launch_pdl(k_rho, dim3(grid), dim3(NT), (size_t)(0), st, 1u, phivT, phicT, ldt, n_v, n_mu, n_idx, m_idx, rho, ld_rho);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_dot_partials(const double* x, const double* y, int64_t ld, int64_t n, int nb, double* part,
                                int npart, cudaStream_t st) {
    dim3 grid((unsigned)npart, (unsigned)nb);
    cudaError_t le = launch_pdl(k_dot_partials, dim3(grid), dim3(NT), (size_t)(0), st, 1u, x, y, ld, n, part, npart);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_lanczos_init(double* p, int64_t n_vc, int nb, const double* normpart, int npart, LanczosState st_,
                                double* xs, int64_t ldxs, const double* s, int n_v, int n_c, int n_cp,
                                cudaStream_t st) {
    (void)n_v;
    dim3 grid((unsigned)vec_parts(n_vc), (unsigned)nb);
    cudaError_t le = launch_pdl(k_lanczos_init, dim3(grid), dim3(NT), (size_t)(0), st, 1u, p, n_vc, nb, normpart, npart, st_, xs, ldxs, s, n_c, n_cp);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_lanczos_update1(double* w, const double* q, const double* q_prev, int64_t n_vc, int nb,
                                   const double* dotpart, int ndot, int dot_stride, LanczosState st_, int k,
                                   double* normpart, int npart, cudaStream_t st) {
    dim3 grid((unsigned)npart, (unsigned)nb);
    cudaError_t le = launch_pdl(k_lanczos_update1, dim3(grid), dim3(NT), (size_t)(0), st, 1u, w, q, q_prev, n_vc, nb, dotpart, ndot, dot_stride, st_, k, normpart, npart);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_lanczos_update2(double* w, int64_t n_vc, int nb, const double* normpart, int npart,
                                   LanczosState st_, int k, double* xs, int64_t ldxs, const double* s, int n_v,
                                   int n_c, int n_cp, cudaStream_t st) {
    (void)n_v;
    dim3 grid((unsigned)vec_parts(n_vc), (unsigned)nb);
    cudaError_t le = launch_pdl(k_lanczos_update2, dim3(grid), dim3(NT), (size_t)(0), st, 1u, w, n_vc, nb, normpart, npart, st_, k, xs, ldxs, s, n_c, n_cp);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

bool lanczos_fused_fits(int64_t n_vc) { return n_vc <= (int64_t)8 * NT * 32; }

cudaError_t launch_lanczos_fused(double* w, const double* q, const double* q_prev, int64_t n_vc, int nb,
                                 const double* dotpart, int ndot, int dot_stride, LanczosState st_, int k, double* xs,
                                 int64_t ldxs, const double* s, int n_v, int n_c, int n_cp, cudaStream_t st) {
    (void)n_v;
    if (!lanczos_fused_fits(n_vc)) return cudaErrorInvalidValue;
    const int ept = n_vc <= (int64_t)8 * NT * 8 ? 8 : 32;
    int cs = 1;
    while ((int64_t)cs * NT * ept < n_vc) cs *= 2;  // 1, 2, 4 or 8: a function of n_vc alone (chain j does not
                                                    // depend on what else is in its block)
    if (q_prev == nullptr) q_prev = q;  // never read at k = 0
    const dim3 grid((unsigned)cs, (unsigned)nb);
    cudaError_t e;
    if (ept == 8)
        e = launch_pdl(k_lanczos_fused<8>, grid, dim3(NT), 0, st, (unsigned)cs, w, q, q_prev, n_vc, nb, dotpart, ndot,
                       dot_stride, st_, k, xs, ldxs, s, n_c, n_cp);
    else
        e = launch_pdl(k_lanczos_fused<32>, grid, dim3(NT), 0, st, (unsigned)cs, w, q, q_prev, n_vc, nb, dotpart, ndot,
                       dot_stride, st_, k, xs, ldxs, s, n_c, n_cp);
    count_launch();
    return e != cudaSuccess ? e : cudaGetLastError();
}

// Slices of the reorthogonalisation kernels: RSLICE elements, at most 64 per chain (even length: 16-byte loads).
int reorth_parts(int64_t n_vc) { return (int)std::max<int64_t>(1, std::min<int64_t>(64, ceil_div(n_vc, RSLICE))); }
static int64_t reorth_slice(int64_t n_vc) { return round_up(ceil_div(n_vc, reorth_parts(n_vc)), 2); }

cudaError_t launch_reorth_dots(const double* basis, int64_t slot_stride, int nslots, const double* w, int64_t n_vc,
                               int nb, double* coefpart, int npart, cudaStream_t st) {
    if (npart != reorth_parts(n_vc)) return cudaErrorInvalidValue;
    const int64_t slice = reorth_slice(n_vc);
    const size_t sm = (size_t)(RSLICE + nslots) * sizeof(double);
    static SmemAttr attr;
    cudaError_t ea = attr.ensure(k_reorth_dots, sm);
    if (ea != cudaSuccess) return ea;
    cudaError_t le = launch_pdl(k_reorth_dots, dim3((unsigned)npart, (unsigned)nb), dim3(NT), sm, st, 1u, basis,
                                slot_stride, nslots, w, n_vc, coefpart, npart, slice);
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_reorth_apply(const double* basis, int64_t slot_stride, int nslots, double* w, int64_t n_vc, int nb,
                                const double* coefpart, int npart, double* normpart, cudaStream_t st) {
    if (npart != reorth_parts(n_vc)) return cudaErrorInvalidValue;
    const size_t sm = (size_t)(nslots + NT / 32 + 1) * sizeof(double);
    static SmemAttr attr;
    cudaError_t ea = attr.ensure(k_reorth_apply, sm);
    if (ea != cudaSuccess) return ea;
    cudaError_t le = launch_pdl(k_reorth_apply, dim3((unsigned)npart, (unsigned)nb), dim3(NT), sm, st, 1u, basis,
                                slot_stride, nslots, w, n_vc, coefpart, npart, normpart, reorth_slice(n_vc));
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_reorth_dots_c(const double* basis, int64_t slot_stride, int nslots, const double* w, int64_t n_vc,
                                 int nb, double* coefpart, int npart, cudaStream_t st) {
    const int64_t N = n_vc / 2;
    if (npart != reorth_parts(N)) return cudaErrorInvalidValue;
    const size_t sm = (size_t)(2 * RSLICE + 2 * nslots) * sizeof(double);
    static SmemAttr attr;
    cudaError_t ea = attr.ensure(k_reorth_dots_c, sm);
    if (ea != cudaSuccess) return ea;
    cudaError_t le = launch_pdl(k_reorth_dots_c, dim3((unsigned)npart, (unsigned)nb), dim3(NT), sm, st, 1u, basis,
                                slot_stride, nslots, w, n_vc, coefpart, npart, reorth_slice(N));
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

cudaError_t launch_reorth_apply_c(const double* basis, int64_t slot_stride, int nslots, double* w, int64_t n_vc, int nb,
                                  const double* coefpart, int npart, double* normpart, cudaStream_t st) {
    const int64_t N = n_vc / 2;
    if (npart != reorth_parts(N)) return cudaErrorInvalidValue;
    const size_t sm = (size_t)(2 * nslots + NT / 32 + 1) * sizeof(double);
    static SmemAttr attr;
    cudaError_t ea = attr.ensure(k_reorth_apply_c, sm);
    if (ea != cudaSuccess) return ea;
    cudaError_t le = launch_pdl(k_reorth_apply_c, dim3((unsigned)npart, (unsigned)nb), dim3(NT), sm, st, 1u, basis,
                                slot_stride, nslots, w, n_vc, coefpart, npart, normpart, reorth_slice(N));
    count_launch();
    return le != cudaSuccess ? le : cudaGetLastError();
}

}  // namespace gwl
