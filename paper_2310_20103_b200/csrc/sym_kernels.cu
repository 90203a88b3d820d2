// Small kernels of the point-group symmetry blocks (reading Q25): the reduced kernels
// Vg = g sum_h chi_gamma(h) V(r_mu, h r_nu), the diagonal term of one block in its padded layout, and the copies between
// the caller's block vectors (pairs of block gamma, unpadded) and the padded layout the GEMMs read.
#include "gwl_internal.h"

namespace gwl {

namespace {

__device__ __forceinline__ double chi(int gamma, int h) { return (__popc(gamma & h) & 1) ? -1.0 : 1.0; }

// Vg[gamma][mu][nu] (row stride ld) = g sum_h chi_gamma(h) V_wf[mu][h][nu]; summed in ascending h for every gamma
__global__ void k_sym_reduce_kernel(const double* __restrict__ vwf, int n_w, int g, double* __restrict__ vg, int64_t ld) {
    const int mu = blockIdx.y;
    for (int nu = blockIdx.x * blockDim.x + threadIdx.x; nu < n_w; nu += gridDim.x * blockDim.x) {
        double v[8];
        for (int h = 0; h < g; ++h) v[h] = vwf[((int64_t)mu * g + h) * n_w + nu];
        for (int gamma = 0; gamma < g; ++gamma) {
            double acc = 0.0;
            for (int h = 0; h < g; ++h) acc += chi(gamma, h) * v[h];
            vg[((int64_t)gamma * n_w + mu) * ld + nu] = (double)g * acc;
        }
    }
}

// one (v-irrep a, c-irrep b) rectangle of the block: rows v (nv of them, energies eps_v[v0..]), columns c < ncp (nc valid,
// energies eps_c[c0..]); d2 = Delta^2, s = sqrt(Delta) on valid pairs, 1 on the zero-padded columns (x = 0 there for ever)
__global__ void k_sym_build_delta(const double* __restrict__ eps_v, const double* __restrict__ eps_c, int nv, int nc, int ncp,
                                  double* __restrict__ d2, double* __restrict__ s) {
    const int64_t n = (int64_t)nv * ncp;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int v = (int)(i / ncp), c = (int)(i - (int64_t)v * ncp);
        if (c < nc) {
            const double d = eps_c[c] - eps_v[v];
            d2[i] = d * d;
            s[i] = sqrt(d);
        } else {
            d2[i] = 1.0;
            s[i] = 1.0;
        }
    }
}

// dir = 0: padded[b][v][c < ncp] = (c < nc ? api[b][v][c] : 0);  dir = 1: api[b][v][c] = padded[b][v][c]
__global__ void k_sym_copy_rect(double* __restrict__ api, int64_t ld_api, double* __restrict__ padded, int64_t ld_pad, int nv,
                                int nc, int ncp, int dir) {
    const int b = blockIdx.y;
    const int64_t n = (int64_t)nv * ncp;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int v = (int)(i / ncp), c = (int)(i - (int64_t)v * ncp);
        if (dir == 0)
            padded[(int64_t)b * ld_pad + i] = c < nc ? api[(int64_t)b * ld_api + (int64_t)v * nc + c] : 0.0;
        else if (c < nc)
            api[(int64_t)b * ld_api + (int64_t)v * nc + c] = padded[(int64_t)b * ld_pad + i];
    }
}

// x[b][v][c] = 0 on the padding columns c >= nc of one rectangle
__global__ void k_sym_zero_pad(double* __restrict__ x, int64_t ld, int nv, int nc, int ncp) {
    const int b = blockIdx.y;
    const int npad = ncp - nc;
    const int64_t n = (int64_t)nv * npad;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int v = (int)(i / npad), c = nc + (int)(i - (int64_t)v * npad);
        x[(int64_t)b * ld + (int64_t)v * ncp + c] = 0.0;
    }
}

}  // namespace

cudaError_t launch_sym_zero_pad(double* x, int64_t ld, int nv, int nc, int ncp, int nvec, cudaStream_t st) {
    if (nv <= 0 || ncp <= nc || nvec <= 0) return cudaSuccess;
    dim3 grid((unsigned)std::min<int64_t>(ceil_div((int64_t)nv * (ncp - nc), 256), 1024), (unsigned)nvec);
    k_sym_zero_pad<<<grid, 256, 0, st>>>(x, ld, nv, nc, ncp);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_sym_reduce_kernel(const double* vwf, int n_w, int g, double* vg, int64_t ld, cudaStream_t st) {
    dim3 grid((unsigned)std::min<int64_t>(ceil_div(n_w, 128), 64), (unsigned)n_w);
    k_sym_reduce_kernel<<<grid, 128, 0, st>>>(vwf, n_w, g, vg, ld);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_sym_build_delta(const double* eps_v, const double* eps_c, int nv, int nc, int ncp, double* d2, double* s,
                                   cudaStream_t st) {
    if (nv <= 0 || ncp <= 0) return cudaSuccess;
    k_sym_build_delta<<<(unsigned)std::min<int64_t>(ceil_div((int64_t)nv * ncp, 256), 1024), 256, 0, st>>>(eps_v, eps_c, nv, nc, ncp,
                                                                                                        d2, s);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_sym_copy_rect(double* api, int64_t ld_api, double* padded, int64_t ld_pad, int nv, int nc, int ncp, int nvec,
                                 int dir, cudaStream_t st) {
    if (nv <= 0 || ncp <= 0 || nvec <= 0) return cudaSuccess;
    dim3 grid((unsigned)std::min<int64_t>(ceil_div((int64_t)nv * ncp, 256), 1024), (unsigned)nvec);
    k_sym_copy_rect<<<grid, 256, 0, st>>>(api, ld_api, padded, ld_pad, nv, nc, ncp, dir);
    count_launch();
    return cudaGetLastError();
}

}  // namespace gwl
