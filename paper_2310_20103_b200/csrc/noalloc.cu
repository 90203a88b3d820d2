// gwl_chain_norms_static: <P_j|P_j> of a block of Lanczos start vectors (the numerator of Eq. 14, PAPER.md:96;
// the `norm2` output of gwl_lanczos) for callers that must not allocate device memory.
//
// Who that is.  Every other entry point of this library works on a gwl_ctx, and gwl_create / gwl_lanczos size
// the context's buffers with cudaMalloc.  Two kinds of host program cannot live with that:
//   - an electronic-structure driver (or a PyTorch process) that has already handed all of HBM to its own pool
//     allocator: a cudaMalloc from a library then fails, or succeeds only by fragmenting what the pool left over;
//   - a driver that keeps several streams busy (another k-point, another spin channel, an MPI progress thread):
//     cudaMalloc and cudaFree synchronise the whole device, so a library that allocates in the middle of such a
//     loop stalls work that has nothing to do with it.
// For them this file holds one self-contained entry point.  It takes device pointers to the inputs and the output,
// and the only extra global memory it needs -- the per-block partial sums of the two-stage reduction -- lives in a
// file-scope __device__ array that is part of the library image.  The price: every GPU on which the library's
// kernels have been loaded holds these GWL_STATIC_SCRATCH_BYTES (256 KB) until the process exits, used or not.
//
// The two-stage reduction is the one k_dot_partials / k_lanczos_init of vec_kernels.cu use (a fixed slice per
// block, a fixed tree inside the block, the partials summed again in a fixed order), written out again here so
// that the existing path is untouched.  Results agree with gwl_lanczos's norm2 to rounding (the slice counts
// differ, so the summation order does), and repeat bit for bit from call to call.
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <mutex>

#include "../../include/gwl.h"

namespace {

constexpr int NT = 256;                                              // threads per block of both kernels
constexpr int64_t SCRATCH_DOUBLES = GWL_STATIC_SCRATCH_BYTES / 8;    // 32 768 partial sums
constexpr int MAX_DEVICES = 64;
constexpr int64_t ELEMS_PER_BLOCK = 16384;                           // target slice length of stage one

// The scratch itself.  In host code this name is only a handle for the runtime (cudaGetSymbolAddress below), NOT
// a device address; device code could name it directly, but the kernels take the resolved pointer as an argument
// so that the launch shows what they write.
static __device__ __align__(256) double g_static_scratch[SCRATCH_DOUBLES];

std::mutex g_setup_mutex;
double* g_scratch_addr[MAX_DEVICES] = {};  // device address of g_static_scratch on each device, NULL until set up

__device__ __forceinline__ double block_sum_fixed(double v, double* sh /*[NT/32]*/) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < NT / 32; ++i) t += sh[i];
    return t;  // valid in thread 0
}

// Stage one: block (s, j) sums p_j[i]^2 over slice s and writes part[j * npart + s].
__global__ void __launch_bounds__(NT) k_static_norm_partials(const double* __restrict__ p, int64_t n_vc, int npart,
                                                             double* __restrict__ part) {
    __shared__ double sh[NT / 32];
    const int64_t per = (n_vc + npart - 1) / npart;
    const int64_t lo = (int64_t)blockIdx.x * per;
    const int64_t hi = lo + per < n_vc ? lo + per : n_vc;
    const double* pj = p + (int64_t)blockIdx.y * n_vc;
    double acc = 0.0;
    for (int64_t i = lo + threadIdx.x; i < hi; i += NT) {
        const double x = pj[i];
        acc = fma(x, x, acc);
    }
    acc = block_sum_fixed(acc, sh);
    if (threadIdx.x == 0) part[(int64_t)blockIdx.y * npart + blockIdx.x] = acc;
}

// Stage two: block j sums its npart partials in a fixed order and writes norm2[j].
__global__ void __launch_bounds__(NT) k_static_norm_final(const double* __restrict__ part, int npart,
                                                          double* __restrict__ norm2) {
    __shared__ double sh[NT / 32];
    const double* row = part + (int64_t)blockIdx.x * npart;
    double acc = 0.0;
    for (int i = threadIdx.x; i < npart; i += NT) acc += row[i];
    acc = block_sum_fixed(acc, sh);
    if (threadIdx.x == 0) norm2[blockIdx.x] = acc;
}

gwl_status fail(gwl_status st, char* err, int64_t err_len, const char* fmt, long long a = 0, long long b = 0) {
    if (err && err_len > 0) snprintf(err, (size_t)err_len, fmt, a, b);
    return st;
}

// Device address of the scratch array on the CURRENT device; resolved once per device.
cudaError_t scratch_on_current_device(double** out, int* dev_out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *dev_out = dev;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
        double* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" gwl_status gwl_chain_norms_static(const double* p, int64_t n_chains, int64_t n_vc, double* norm2,
                                             void* cuda_stream, char* err, int64_t err_len) {
    if (err && err_len > 0) err[0] = '\0';
    if (n_chains < 0 || n_vc < 1)
        return fail(GWL_EINVAL, err, err_len, "gwl_chain_norms_static: n_chains = %lld must be >= 0 and n_vc = %lld >= 1",
                    (long long)n_chains, (long long)n_vc);
    if (n_chains > GWL_STATIC_MAX_CHAINS)
        return fail(GWL_EINVAL, err, err_len,
                    "gwl_chain_norms_static: n_chains = %lld exceeds GWL_STATIC_MAX_CHAINS = %lld (the static scratch "
                    "array cannot grow; split the block or use gwl_lanczos on a context)",
                    (long long)n_chains, (long long)GWL_STATIC_MAX_CHAINS);
    if (n_vc > GWL_STATIC_MAX_NVC)
        return fail(GWL_EINVAL, err, err_len, "gwl_chain_norms_static: n_vc = %lld exceeds GWL_STATIC_MAX_NVC = %lld",
                    (long long)n_vc, (long long)GWL_STATIC_MAX_NVC);
    if (n_chains == 0) return GWL_OK;
    if (!p || !norm2) return fail(GWL_EINVAL, err, err_len, "gwl_chain_norms_static: p and norm2 must not be NULL");

    double* scratch = nullptr;
    int dev = -1;
    cudaError_t e = scratch_on_current_device(&scratch, &dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        if (err && err_len > 0)
            snprintf(err, (size_t)err_len, "gwl_chain_norms_static: set-up of the static scratch on device %d failed: %s", dev,
                     cudaGetErrorString(e));
        return GWL_ECUDA;
    }

    // Slices per chain: about ELEMS_PER_BLOCK elements each, at most what the scratch holds for this many chains.
    int64_t npart = (n_vc + ELEMS_PER_BLOCK - 1) / ELEMS_PER_BLOCK;
    const int64_t cap = SCRATCH_DOUBLES / n_chains;  // >= 8 because n_chains <= GWL_STATIC_MAX_CHAINS
    if (npart > cap) npart = cap;
    if (npart > 2048) npart = 2048;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    k_static_norm_partials<<<dim3((unsigned)npart, (unsigned)n_chains), NT, 0, st>>>(p, n_vc, (int)npart, scratch);
    e = cudaGetLastError();
    if (e == cudaSuccess) {
        k_static_norm_final<<<(unsigned)n_chains, NT, 0, st>>>(scratch, (int)npart, norm2);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (err && err_len > 0)
            snprintf(err, (size_t)err_len, "gwl_chain_norms_static: kernel launch failed: %s", cudaGetErrorString(e));
        return GWL_ECUDA;
    }
    return GWL_OK;
}
