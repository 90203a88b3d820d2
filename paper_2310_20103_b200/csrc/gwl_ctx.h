// The context behind the opaque gwl_ctx of include/gwl.h, the status / launch-timing macros and the host driver helpers
// shared by the translation units of the C ABI (gwl_api.cu: the path; gwl_tdc.cu: complex orbitals; gwl_sym.cu: symmetry
// blocks; gwl_isdf_api.cu: ISDF front end; gwl_driver.cu: the contractions and the pseudo-Hermitian Lanczos driver).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "gwl_internal.h"

namespace gwl {

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
    cudaError_t ensure(size_t need, cudaStream_t st) {
        if (need <= bytes && p != nullptr) return cudaSuccess;
        if (p) {
            cudaError_t e0 = cudaStreamSynchronize(st);
            if (e0 != cudaSuccess) return e0;
            cudaFree(p);
            p = nullptr;
            bytes = 0;
        }
        if (need == 0) need = 8;
        cudaError_t e = cudaMalloc(&p, need);
        if (e != cudaSuccess) {
            p = nullptr;
            cudaGetLastError();  // clear it: the caller reports GWL_ENOMEM and the context stays usable
            return e;
        }
        bytes = need;
        return cudaMemsetAsync(p, 0, need, st);
    }
    void release() {
        if (p) cudaFree(p);
        p = nullptr;
        bytes = 0;
    }
    template <class T>
    T* as() const {
        return static_cast<T*>(p);
    }
};

}  // namespace gwl

struct gwl_ctx {
    using DevBuf = gwl::DevBuf;
    int n_v = 0, n_c = 0, n_mu = 0;
    int64_t n_vc = 0;
    int n_cp = 0, n_mup = 0;
    int n_sm = 148;
    int device = 0;
    // complex-orbital (periodic Tamm-Dancoff) contexts, gwl_tdc_create: Lanczos vectors are planar [re | im], so the
    // vector layout has n_v = 2 * n_kv "rows" of n_c and n_vc = 2 * n_k * nv_k * n_c real entries
    bool cplx = false;
    int n_k = 1, nv_k = 0, n_kv = 0, n_q = 1;
    // symmetry-block contexts (gwl_sym_create, Q25): irreps are bit masks, products are XORs.  After
    // gwl_sym_select(gamma) the vector kernels see one padded block vector (n_c = n_cp = 16, n_v = n_vc / 16) and the GEMM
    // drivers walk the rectangles (v in irrep a) x (c in irrep a ^ gamma), every irrep's conduction count padded to 16 columns
    bool sym = false;
    int sym_g = 1, sym_gamma = -1;
    int sym_nv[8] = {}, sym_nc[8] = {}, sym_ncp[8] = {}, sym_voff[8] = {}, sym_coff[8] = {}, sym_cpoff[8] = {};
    int sym_nv_tot = 0, sym_nc_tot = 0, sym_ncp_tot = 0;
    int64_t sym_vecoff[8] = {}, sym_apioff[8] = {}, sym_npairs = 0;
    int64_t v_sel = 0;          // element offset of the selected kernel inside V (V holds the g reduced kernels)
    bool sig_accumulate = false;  // gwl_selfenergy adds to sigma_sum instead of overwriting it (gwl_sym_selfenergy_state)
    // CUDA graphs of the step loop for small problems (launch-bound: the fused-update path, N_vc <= 65 536): six consecutive
    // Lanczos steps are captured once (slot rotation has period 3, state parity period 2) and replayed; the step number comes
    // from a device counter.  Runs on an internal stream (the caller's may be the legacy default stream, which cannot capture).
    struct StepGraph {
        uint64_t key = 0;
        cudaGraphExec_t exec = nullptr;
        int launches = 0;
        unsigned max_epoch = 0;
        uint64_t stamp = 0;
    };
    std::vector<StepGraph> graphs;
    uint64_t graph_stamp = 0;
    bool graph_off = false;       // set after a failed capture: plain launches from then on
    cudaStream_t gstream = nullptr;
    cudaEvent_t ev_gin = nullptr, ev_gout = nullptr;
    DevBuf kbase;
    cudaStream_t stream = nullptr;
    int device_ptrs = 0;
    std::string err;
    int64_t launches = 0;

    bool have_orb = false, have_eps = false, have_V = false;
    DevBuf phi_c, phi_cT, phi_vT, V, eps_v, eps_c, d2, s;
    std::vector<double> h_eps_v, h_eps_c;

    int approx = 0;  // 0 RPA (operator C), 1 Tamm-Dancoff (operator A)
    int g = 0;
    std::vector<double> cheb;
    double lo = 0.0, hi = 0.0;

    int chain_mode = 0;  // 0 none, 1 indices, 2 explicit vectors
    int64_t n_chains_set = 0;
    DevBuf d_nidx, d_midx, d_start, d_eps_n, d_sgn_n;

    // results of the last gwl_lanczos
    int64_t run_chains = 0;
    int run_steps = 0;
    int run_poly = 0;
    DevBuf alpha, beta, norm2, len, scale, alive;

    // workspaces.  The GEMM scratch (T, W, split-K partials, stream-K hand-over) exists twice: set 0 serves the context's
    // stream, set 1 the side stream on which gwl_lanczos builds the start vectors of the NEXT block (S1) under the step
    // loop of the current one.
    struct WorkSet {
        DevBuf T, W, part, sk_ws, sk_flags;
        unsigned sk_epoch = 0;
    } wset[2];
    int cur = 0;
    cudaStream_t stream2 = nullptr;
    cudaEvent_t ev_consumed = nullptr, ev_s1 = nullptr;
    WorkSet& ws() { return wset[cur]; }
    cudaStream_t lstream() const { return cur ? stream2 : stream; }
    DevBuf xs, dotpart, normpart, basis, coefpart, tA, tB, pnext, pnext_part;
    DevBuf sbasis, prpa_tc, prpa_wc, prpa_apart;  // pseudo-Hermitian RPA Lanczos (complex contexts, GWL_RPA)
    DevBuf x_nidx, x_midx, x_part, x_sig, x_eps, x_vxc, x_sc, x_e, x_z, x_it;  // gwl_exchange / gwl_qp_solve staging
    DevBuf stage;            // gwl_set_orbitals staging
    DevBuf isdf_phi, isdf_phimu, isdf_y, isdf_s, isdf_g, isdf_u;  // gwl_isdf_build
    DevBuf theta, wgt, ritz_info, d_omega, d_zeta, d_sigma, d_sigsum, io_x, io_y;

    // timing: per-step event triples (op start, op end, step end) and, at profiling level 2,
    // an event pair around every kernel launch tagged with its class
    std::vector<cudaEvent_t> ev;
    size_t ev_used = 0;
    int prof_level = 1;
    std::vector<cudaEvent_t> kev;
    size_t kev_used = 0;
    std::vector<int> kev_class;

    gwl_status fail(gwl_status st, const std::string& msg) {
        err = msg;
        return st;
    }
    gwl_status cuda_fail(cudaError_t e, const char* where) {
        err = std::string(where) + ": " + cudaGetErrorString(e);
        return e == cudaErrorMemoryAllocation ? GWL_ENOMEM : GWL_ECUDA;
    }
    cudaEvent_t next_event() {
        if (ev_used == ev.size()) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            ev.push_back(e);
        }
        return ev[ev_used++];
    }
    cudaEvent_t next_kevent() {
        if (kev_used == kev.size()) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            kev.push_back(e);
        }
        return kev[kev_used++];
    }
};

// Event pair around one kernel launch when profiling level 2 is on (gwl_set_profiling).
struct KernelTimer {
    gwl_ctx* c;
    bool on;
    KernelTimer(gwl_ctx* ctx, int cls) : c(ctx), on(ctx->prof_level >= 2) {
        if (on) {
            c->kev_class.push_back(cls);
            cudaEventRecord(c->next_kevent(), c->lstream());
        }
    }
    ~KernelTimer() {
        if (on) cudaEventRecord(c->next_kevent(), c->lstream());
    }
};
#define CKL(cls, call)                                            \
    do {                                                          \
        KernelTimer kt__(ctx, cls);                               \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return ctx->cuda_fail(e__, #call); \
    } while (0)

#define CK(call)                                                  \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return ctx->cuda_fail(e__, #call); \
    } while (0)

namespace gwl {

// Makes the context's device current for the duration of an entry point and restores the caller's device after.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const gwl_ctx* c) {
        if (c != nullptr && cudaGetDevice(&prev) == cudaSuccess && prev != c->device)
            switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};

// A new operator or chain list makes the tridiagonals of the last gwl_lanczos meaningless.
inline void invalidate_run(gwl_ctx* ctx) {
    ctx->run_chains = 0;
    ctx->run_steps = 0;
}

struct LaunchScope {
    explicit LaunchScope(gwl_ctx* c) { g_launch_counter = &c->launches; }
    ~LaunchScope() { g_launch_counter = nullptr; }
};

// ---- host driver (gwl_driver.cu) ---------------------------------------------------------------------------------------
// One term of the Chebyshev recurrence fused into the K^T.W epilogue (EPI_CHEB, kr_gemm.cu)
struct ChebTerm {
    const double* t0;  // t_{j-2} or NULL
    double* w;         // running sum
    const double* q;   // NULL except on the last term (alpha dots)
    double* xs_out;    // NULL on the last term
    double ca, cb, cc, cw, c0;
    int first;
};
gwl_status ensure_workspace(gwl_ctx* ctx, int nb);
// T[b][mu] = sum_vc K[mu, vc] xs[b][vc]; W = V T; u = K^T W with the fused epilogue (real, complex and symmetry-block contexts)
gwl_status gemm_kx(gwl_ctx* ctx, int nb);
gwl_status gemm_v(gwl_ctx* ctx, int nb);
gwl_status gemm_ktw(gwl_ctx* ctx, const double* x, int64_t ldx, double* y, int64_t ldy, int nb, double* dotpart, int dot_stride,
                    const ChebTerm* cheb = nullptr);
// out[n][m] = sum_k A[m][k] B[n][k] on the DMMA GEMM (MODE_PLAIN) with its split-K reduction
gwl_status plain_gemm(gwl_ctx* ctx, const double* A, int64_t lda, const double* B, int64_t ldb, int M, int N, int k_tiles,
                      double* out, int64_t ldo, int cls);
// y = Op x for a block whose scaled copy xs is ready
gwl_status apply_casida_core(gwl_ctx* ctx, const double* x, int64_t ldx, double* y, int64_t ldy, int nb, double* dotpart,
                             int dot_stride);
int casida_ndot(const gwl_ctx* ctx, int nb);
// S1: start vectors of the index chains j0 .. j0 + nb
gwl_status build_start_vectors(gwl_ctx* ctx, int64_t j0, int nb, double* P, double* normpart, int dot_stride);
bool ready(const gwl_ctx* ctx);
// pseudo-Hermitian RPA for complex orbitals (Q24)
bool prpa(const gwl_ctx* ctx);
gwl_status prpa_workspace(gwl_ctx* ctx, int nb);
gwl_status prpa_apply(gwl_ctx* ctx, const double* h, double* out, int nb);
gwl_status lanczos_prpa(gwl_ctx* ctx, int64_t n_chains, int L, int nbmax, int reorth);
// context creation shared by gwl_create / gwl_tdc_create / gwl_sym_create; padded and transposed orbital copies
gwl_status create_common(gwl_ctx** out, int64_t n_k, int64_t n_v, int64_t n_c, int64_t n_mu, bool cplx, int64_t n_q);
gwl_status install_orbitals(gwl_ctx* ctx, const double* d_phi_v, const double* d_phi_c);

}  // namespace gwl
