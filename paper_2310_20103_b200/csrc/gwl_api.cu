// C ABI of libgwl (include/gwl.h): context, input staging, and the host driver that strings the kernels
// together.  There is no host<->device traffic and no host synchronisation inside the Lanczos step loop:
// alpha/beta/len live on the device and are copied out once at the end.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "gwl_internal.h"

using namespace gwl;

namespace {

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

}  // namespace

struct gwl_ctx {
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

namespace {

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
void invalidate_run(gwl_ctx* ctx) {
    ctx->run_chains = 0;
    ctx->run_steps = 0;
}

struct LaunchScope {
    explicit LaunchScope(gwl_ctx* c) { g_launch_counter = &c->launches; }
    ~LaunchScope() { g_launch_counter = nullptr; }
};

gwl_status ensure_workspace(gwl_ctx* ctx, int nb) {
    cudaStream_t st = ctx->stream;
    const int64_t ldxs = (int64_t)ctx->n_v * ctx->n_cp;
    if (ctx->cur == 0) CK(ctx->xs.ensure((size_t)nb * ldxs * 8, st));
    const int rows = ctx->cplx ? 2 * nb : nb;  // complex: T and W hold a real and an imaginary plane of nb rows each
    CK(ctx->ws().T.ensure((size_t)rows * ctx->n_mup * 8, st));
    CK(ctx->ws().W.ensure((size_t)rows * ctx->n_mup * 8, st));
    const int kt_f = ctx->n_v * (ctx->n_cp / BK), kt_v = ctx->n_mup / BK;
    const GemmPlan pf = ctx->cplx ? plan_gemm_c(ctx->n_mu, nb, ctx->n_kv * (ctx->n_cp / BK), ctx->n_sm)
                                  : plan_gemm(MODE_FWD, ctx->n_mu, nb, kt_f, ctx->n_cp / BK, ctx->n_sm);
    const GemmPlan pv = plan_gemm(MODE_PLAIN, ctx->n_mu, rows, kt_v, kt_v, ctx->n_sm);
    const int smax = std::max(pf.splits, pv.splits);
    CK(ctx->ws().part.ensure((size_t)smax * rows * ctx->n_mup * 8, st));
    const int npart = vec_parts(ctx->n_vc);
    const int64_t ndot = std::max<int64_t>((int64_t)ctx->n_v * ceil_div(ctx->n_c, 128), npart);
    CK(ctx->dotpart.ensure((size_t)nb * ndot * 8, st));
    CK(ctx->normpart.ensure((size_t)nb * std::max(npart, reorth_parts(ctx->n_vc)) * 8, st));
    CK(ctx->ws().sk_ws.ensure(gemm_bwd_ws_bytes(ctx->n_sm), st));
    CK(ctx->ws().sk_flags.ensure(gemm_bwd_flag_bytes(ctx->n_sm), st));
    return GWL_OK;
}

// ---- the three contractions (kr_gemm.cu), each with its split-K reduction where the planner asks for one ---------
// T[b][mu] = sum_vc K[mu, vc] xs[b][vc]   (xs = scaled input in the padded [nb][n_v][n_cp] layout)
// complex (planar) K.x of the periodic Tamm-Dancoff operator: T[2][nb][n_mup] (kr_gemm_c.cu)
gwl_status gemm_kx_c(gwl_ctx* ctx, int nb) {
    cudaStream_t st = ctx->lstream();
    const int kt_c = ctx->n_cp / BK, kt_f = ctx->n_kv * kt_c;
    const int64_t ldm = ctx->n_mup;
    const GemmPlan pl = plan_gemm_c(ctx->n_mu, nb, kt_f, ctx->n_sm);
    GemmParamsC p{};
    p.A = ctx->phi_c.as<double>();
    p.lda = (int64_t)ctx->n_k * ctx->n_cp;
    p.a_plane = (int64_t)ctx->n_mu * p.lda;
    p.B = ctx->xs.as<double>();
    p.ldb = (int64_t)ctx->n_v * ctx->n_cp;
    p.b_plane_cols = ctx->n_kv * ctx->n_cp;
    p.M = ctx->n_mu;
    p.N = nb;
    p.kt_total = kt_f;
    p.a_wrap = kt_c;
    p.kt_per_split = pl.kt_per_split;
    p.n_v = ctx->nv_k;
    p.n_c = ctx->n_c;
    p.scale = ctx->phi_vT.as<double>();
    p.lds = ldm;
    p.s_plane = (int64_t)ctx->n_kv * ldm;
    p.scale_rows = ctx->n_kv;
    if (pl.splits > 1) CK(ctx->ws().part.ensure((size_t)pl.splits * 2 * nb * ldm * 8, st));
    p.out = pl.splits == 1 ? ctx->ws().T.as<double>() : ctx->ws().part.as<double>();
    p.ldo = ldm;
    p.o_plane = (int64_t)nb * ldm;
    p.out_split_stride = (int64_t)2 * nb * ldm;
    CKL(0, launch_gemm_c(MODE_FWD, EPI_STORE, p, pl.splits, st));
    if (pl.splits > 1)
        CKL(3, launch_splitk_reduce(ctx->ws().part.as<double>(), (int64_t)2 * nb * ldm, pl.splits, ctx->ws().T.as<double>(), ldm,
                                    ctx->n_mu, 2 * nb, st));
    return GWL_OK;
}

gwl_status gemm_kx_sym(gwl_ctx* ctx, int nb);
gwl_status gemm_kx(gwl_ctx* ctx, int nb) {
    if (ctx->cplx) return gemm_kx_c(ctx, nb);
    if (ctx->sym) return gemm_kx_sym(ctx, nb);
    cudaStream_t st = ctx->lstream();
    const int kt_c = ctx->n_cp / BK, kt_f = ctx->n_v * kt_c;
    const int64_t ldm = ctx->n_mup;
    const GemmPlan pl = plan_gemm(MODE_FWD, ctx->n_mu, nb, kt_f, kt_c, ctx->n_sm);
    GemmParams p{};
    p.A = ctx->phi_c.as<double>();
    p.lda = ctx->n_cp;
    p.B = ctx->xs.as<double>();
    p.ldb = (int64_t)ctx->n_v * ctx->n_cp;
    p.M = ctx->n_mu;
    p.N = nb;
    p.kt_total = kt_f;
    p.a_wrap = kt_c;
    p.kt_per_split = pl.kt_per_split;
    p.scale = ctx->phi_vT.as<double>();
    p.lds = ldm;
    p.scale_rows = ctx->n_v;
    if (pl.splits > 1) CK(ctx->ws().part.ensure((size_t)pl.splits * nb * ldm * 8, st));
    p.out = pl.splits == 1 ? ctx->ws().T.as<double>() : ctx->ws().part.as<double>();
    p.ldo = ldm;
    p.out_split_stride = (int64_t)nb * ldm;
    CKL(0, launch_gemm(MODE_FWD, EPI_STORE, pl, p, pl.splits, st));
    if (pl.splits > 1)
        CKL(3, launch_splitk_reduce(ctx->ws().part.as<double>(), (int64_t)nb * ldm, pl.splits, ctx->ws().T.as<double>(), ldm, ctx->n_mu,
                                nb, st));
    return GWL_OK;
}

// out[n][m] = sum_k A[m][k] B[n][k] on the DMMA GEMM (MODE_PLAIN): A [M][lda], B [N][ldb], both K-contiguous with k_tiles
// tiles of 16 valid (zero-padded) columns; split-K partials reduced in a fixed order by k_splitk_reduce
gwl_status plain_gemm(gwl_ctx* ctx, const double* A, int64_t lda, const double* B, int64_t ldb, int M, int N, int k_tiles,
                      double* out, int64_t ldo, int cls) {
    cudaStream_t st = ctx->lstream();
    const GemmPlan pl = plan_gemm(MODE_PLAIN, M, N, k_tiles, k_tiles, ctx->n_sm);
    GemmParams p{};
    p.A = A;
    p.lda = lda;
    p.B = B;
    p.ldb = ldb;
    p.M = M;
    p.N = N;
    p.kt_total = k_tiles;
    p.a_wrap = k_tiles;
    p.kt_per_split = pl.kt_per_split;
    if (pl.splits > 1) CK(ctx->ws().part.ensure((size_t)pl.splits * N * ldo * 8, st));
    p.out = pl.splits == 1 ? out : ctx->ws().part.as<double>();
    p.ldo = ldo;
    p.out_split_stride = (int64_t)N * ldo;
    CKL(cls, launch_gemm(MODE_PLAIN, EPI_STORE, pl, p, pl.splits, st));
    if (pl.splits > 1)
        CKL(3, launch_splitk_reduce(ctx->ws().part.as<double>(), (int64_t)N * ldo, pl.splits, out, ldo, M, N, st));
    return GWL_OK;
}

// W[b][mu] = sum_nu V[mu][nu] T[b][nu]
gwl_status gemm_v(gwl_ctx* ctx, int nb) {
    if (ctx->cplx) nb *= 2;  // V is real: the two planes of T are 2 nb independent columns
    return plain_gemm(ctx, ctx->V.as<double>() + ctx->v_sel, ctx->n_mup, ctx->ws().T.as<double>(), ctx->n_mup, ctx->n_mu, nb,
                      ctx->n_mup / BK, ctx->ws().W.as<double>(), ctx->n_mup, 1);
}

// u = K^T W with the epilogue fused:  x != NULL: y = d2 o x + coupling s o u and the partial dots sum(x y);
// x == NULL (start vectors): y = s o u and the partial dots sum(y y).
// One term of the Chebyshev recurrence fused into the K^T.W epilogue (EPI_CHEB, kr_gemm.cu)
struct ChebTerm {
    const double* t0;  // t_{j-2} or NULL
    double* w;         // running sum
    const double* q;   // NULL except on the last term (alpha dots)
    double* xs_out;    // NULL on the last term
    double ca, cb, cc, cw, c0;
    int first;
};

// complex (planar) K^H.W with the epilogue y = Delta o x + u (or y = u for start vectors), kr_gemm_c.cu
gwl_status gemm_ktw_c(gwl_ctx* ctx, const double* x, int64_t ldx, double* y, int64_t ldy, int nb, double* dotpart,
                      int dot_stride) {
    const int64_t ldm = ctx->n_mup;
    const int64_t n_kvc = (int64_t)ctx->n_kv * ctx->n_c;
    GemmParamsC p{};
    p.A = ctx->phi_cT.as<double>();
    p.lda = ldm;
    p.a_rows = ctx->n_k * ctx->n_c;
    p.a_plane = (int64_t)p.a_rows * ldm;
    p.B = ctx->ws().W.as<double>();
    p.ldb = ldm;
    p.b_plane = (int64_t)nb * ldm;
    p.M = ctx->n_c;
    p.N = nb;
    p.kt_total = ctx->n_mup / BK;
    p.n_v = ctx->nv_k;
    p.n_c = ctx->n_c;
    p.scale = ctx->phi_vT.as<double>();
    p.lds = ldm;
    p.s_plane = (int64_t)ctx->n_kv * ldm;
    p.scale_rows = ctx->n_kv;
    p.out = y;
    p.ldo = ldy;
    p.o_plane = n_kvc;
    p.X = x;
    p.ldx = ldx;
    p.x_plane = n_kvc;
    p.d2 = ctx->d2.as<double>();
    p.coupling = 1.0;
    p.dotpart = dotpart;
    p.dot_stride = dot_stride;
    CKL(2, launch_gemm_c(MODE_BWD, x != nullptr ? EPI_CASIDA : EPI_START, p, ctx->n_kv, ctx->lstream()));
    return GWL_OK;
}

// One rectangle of the K^T.W product: conduction rows [c_row0, c_row0 + n_c_rows) of Phi_c^T, occupied orbitals
// [v0, v0 + n_v_rows), output / x / Delta / Chebyshev vectors shifted by vec_off inside every chain.  The whole product of an
// ordinary context is the rectangle (0, N_c, 0, N_v, 0); a symmetry block is one rectangle per irrep of v.
struct KtwRect {
    int c_row0, n_c_rows, v0, n_v_rows;
    int64_t vec_off;
};

gwl_status gemm_ktw_rect(gwl_ctx* ctx, const KtwRect& r, const double* x, int64_t ldx, double* y, int64_t ldy, int nb,
                         double* dotpart, int dot_stride, const ChebTerm* cheb);

gwl_status gemm_ktw(gwl_ctx* ctx, const double* x, int64_t ldx, double* y, int64_t ldy, int nb, double* dotpart,
                    int dot_stride, const ChebTerm* cheb = nullptr) {
    if (ctx->cplx) {
        if (cheb != nullptr) return ctx->fail(GWL_EINVAL, "internal: no polynomial mode for complex orbitals");
        return gemm_ktw_c(ctx, x, ldx, y, ldy, nb, dotpart, dot_stride);
    }
    if (ctx->sym) {  // block gamma: rectangles (v in irrep a) x (c in irrep a ^ gamma), dot partials one after the other
        int dbase = 0;
        for (int a = 0; a < ctx->sym_g; ++a) {
            const int b = a ^ ctx->sym_gamma;
            if (ctx->sym_nv[a] == 0 || ctx->sym_nc[b] == 0) continue;
            const KtwRect r{ctx->sym_cpoff[b], ctx->sym_ncp[b], ctx->sym_voff[a], ctx->sym_nv[a], ctx->sym_vecoff[a]};
            gwl_status rs = gemm_ktw_rect(ctx, r, x, ldx, y, ldy, nb, dotpart != nullptr ? dotpart + dbase : nullptr, dot_stride, cheb);
            if (rs != GWL_OK) return rs;
            dbase += ctx->sym_nv[a] * (int)ceil_div(ctx->sym_ncp[b], 128);
        }
        return GWL_OK;
    }
    const KtwRect r{0, ctx->n_c, 0, ctx->n_v, 0};
    return gemm_ktw_rect(ctx, r, x, ldx, y, ldy, nb, dotpart, dot_stride, cheb);
}

gwl_status gemm_ktw_rect(gwl_ctx* ctx, const KtwRect& r, const double* x, int64_t ldx, double* y, int64_t ldy, int nb,
                         double* dotpart, int dot_stride, const ChebTerm* cheb) {
    const int kt_v = ctx->n_mup / BK;
    const int64_t ldm = ctx->n_mup;
    const GemmPlan pl = plan_gemm(MODE_BWD, r.n_c_rows, nb, kt_v, kt_v, ctx->n_sm);
    GemmParams p{};
    p.A = ctx->phi_cT.as<double>() + (int64_t)r.c_row0 * ldm;
    p.lda = ldm;
    p.B = ctx->ws().W.as<double>();
    p.ldb = ldm;
    p.M = r.n_c_rows;
    p.N = nb;
    p.kt_total = kt_v;
    p.a_wrap = kt_v;
    p.kt_per_split = kt_v;
    p.scale = ctx->phi_vT.as<double>() + (int64_t)r.v0 * ldm;
    p.lds = ldm;
    p.scale_rows = r.n_v_rows;
    p.out = y + r.vec_off;
    p.ldo = ldy;
    p.X = x != nullptr ? x + r.vec_off : nullptr;
    p.ldx = ldx;
    p.d2 = ctx->d2.as<double>() + r.vec_off;
    p.s = ctx->s.as<double>() + r.vec_off;
    p.dotpart = dotpart;
    p.dot_stride = dot_stride;
    p.n_c = r.n_c_rows;
    p.coupling = ctx->approx ? 1.0 : 2.0;
    p.ws = ctx->ws().sk_ws.as<double>();
    p.flags = ctx->ws().sk_flags.as<unsigned>();
    if (++ctx->ws().sk_epoch == 0) ++ctx->ws().sk_epoch;
    p.epoch = ctx->ws().sk_epoch;
    p.n_sm = ctx->n_sm;
    int epi = x != nullptr ? EPI_CASIDA : EPI_START;
    if (cheb != nullptr) {
        if (x == nullptr || ldx != ldy) return ctx->fail(GWL_EINVAL, "internal: EPI_CHEB needs x and a common leading dimension");
        epi = EPI_CHEB;
        p.T0 = cheb->t0 != nullptr ? cheb->t0 + r.vec_off : nullptr;
        p.Wacc = cheb->w + r.vec_off;
        p.Q = cheb->q != nullptr ? cheb->q + r.vec_off : nullptr;
        p.xs_out = cheb->xs_out != nullptr ? cheb->xs_out + r.vec_off : nullptr;  // sym: padded layout = vector layout
        p.ldxs = (int64_t)ctx->n_v * ctx->n_cp;
        p.n_cp = ctx->sym ? r.n_c_rows : ctx->n_cp;
        p.ca = cheb->ca;
        p.cb = cheb->cb;
        p.cc = cheb->cc;
        p.cw = cheb->cw;
        p.c0 = cheb->c0;
        p.first = cheb->first;
    }
    CKL(2, launch_gemm(MODE_BWD, epi, pl, p, r.n_v_rows, ctx->lstream()));
    return GWL_OK;
}

// K.X of a symmetry block: one launch per rectangle, all partials (rectangles x their split-K) reduced together
gwl_status gemm_kx_sym(gwl_ctx* ctx, int nb) {
    cudaStream_t st = ctx->lstream();
    const int64_t ldm = ctx->n_mup;
    GemmPlan plans[8];
    int total = 0;
    for (int a = 0; a < ctx->sym_g; ++a) {
        const int b = a ^ ctx->sym_gamma;
        if (ctx->sym_nv[a] == 0 || ctx->sym_nc[b] == 0) continue;
        const int kt_c = ctx->sym_ncp[b] / BK;
        plans[a] = plan_gemm(MODE_FWD, ctx->n_mu, nb, ctx->sym_nv[a] * kt_c, kt_c, ctx->n_sm);
        total += plans[a].splits;
    }
    CK(ctx->ws().part.ensure((size_t)std::max(total, 1) * nb * ldm * 8, st));
    int zbase = 0;
    for (int a = 0; a < ctx->sym_g; ++a) {
        const int b = a ^ ctx->sym_gamma;
        if (ctx->sym_nv[a] == 0 || ctx->sym_nc[b] == 0) continue;
        const int kt_c = ctx->sym_ncp[b] / BK;
        GemmParams p{};
        p.A = ctx->phi_c.as<double>() + ctx->sym_cpoff[b];
        p.lda = ctx->sym_ncp_tot;
        p.B = ctx->xs.as<double>() + ctx->sym_vecoff[a];
        p.ldb = ctx->n_vc;
        p.M = ctx->n_mu;
        p.N = nb;
        p.kt_total = ctx->sym_nv[a] * kt_c;
        p.a_wrap = kt_c;
        p.kt_per_split = plans[a].kt_per_split;
        p.scale = ctx->phi_vT.as<double>() + (int64_t)ctx->sym_voff[a] * ldm;
        p.lds = ldm;
        p.scale_rows = ctx->sym_nv[a];
        p.out = ctx->ws().part.as<double>() + (int64_t)zbase * nb * ldm;
        p.ldo = ldm;
        p.out_split_stride = (int64_t)nb * ldm;
        CKL(0, launch_gemm(MODE_FWD, EPI_STORE, plans[a], p, plans[a].splits, st));
        zbase += plans[a].splits;
    }
    CKL(3, launch_splitk_reduce(ctx->ws().part.as<double>(), (int64_t)nb * ldm, zbase, ctx->ws().T.as<double>(), ldm, ctx->n_mu, nb, st));
    return GWL_OK;
}

// y = Op x for a block whose scaled copy xs is ready: K, V, K^T with the Casida / TDA epilogue.
gwl_status apply_casida_core(gwl_ctx* ctx, const double* x, int64_t ldx, double* y, int64_t ldy, int nb,
                             double* dotpart, int dot_stride) {
    gwl_status rs = gemm_kx(ctx, nb);
    if (rs == GWL_OK) rs = gemm_v(ctx, nb);
    if (rs == GWL_OK) rs = gemm_ktw(ctx, x, ldx, y, ldy, nb, dotpart, dot_stride);
    return rs;
}

// alpha / norm partials written by the K^T.W epilogue: one per (v, m-tile) of the plan used for a block of nb
int casida_ndot(const gwl_ctx* ctx, int nb) {
    if (ctx->cplx) return ctx->n_kv * gemm_c_tiles_m(ctx->n_c);
    if (ctx->sym) {
        int n = 0;
        for (int a = 0; a < ctx->sym_g; ++a)
            if (ctx->sym_nv[a] > 0 && ctx->sym_nc[a ^ ctx->sym_gamma] > 0)
                n += ctx->sym_nv[a] * (int)ceil_div(ctx->sym_ncp[a ^ ctx->sym_gamma], 128);
        return std::max(n, 1);
    }
    const GemmPlan pl = plan_gemm(MODE_BWD, ctx->n_c, nb, ctx->n_mup / BK, ctx->n_mup / BK, ctx->n_sm);
    return ctx->n_v * (int)ceil_div(ctx->n_c, pl.bm);
}

// S1: P_j = sqrt(Delta) o K^T (V rho_j) for index chains j0..j0+nb; writes P and sum(P^2) partials.
gwl_status build_start_vectors(gwl_ctx* ctx, int64_t j0, int nb, double* P, double* normpart, int dot_stride) {
    const int64_t ldm = ctx->n_mup;
    if (ctx->cplx)  // rho~ = psi_m conj(psi_n): the ket of PAPER.md:310 is the conjugate of the printed elements (Q20)
        CKL(4, launch_rho_c(ctx->phi_vT.as<double>(), (int64_t)ctx->n_kv * ldm, ctx->phi_cT.as<double>(),
                            (int64_t)ctx->n_k * ctx->n_c * ldm, ldm, ctx->nv_k, ctx->n_c, ctx->n_mu,
                            ctx->d_nidx.as<int32_t>() + 4 * j0, ctx->ws().T.as<double>(), ldm, nb, ctx->lstream()));
    else
        CKL(4, launch_rho(ctx->phi_vT.as<double>(), ctx->phi_cT.as<double>(), ldm, ctx->sym ? ctx->sym_nv_tot : ctx->n_v, ctx->n_mu,
                      ctx->d_nidx.as<int32_t>() + j0, ctx->d_midx.as<int32_t>() + j0, ctx->ws().T.as<double>(), ldm, nb,
                      ctx->lstream()));
    gwl_status rs = gemm_v(ctx, nb);
    if (rs == GWL_OK) rs = gemm_ktw(ctx, nullptr, ctx->n_vc, P, ctx->n_vc, nb, normpart, dot_stride);
    return rs;
}

bool ready(const gwl_ctx* ctx) { return ctx->have_orb && ctx->have_eps && ctx->have_V; }

// ---- pseudo-Hermitian RPA for complex orbitals (Q24; prpa_kernels.cu) ------------------
bool prpa(const gwl_ctx* ctx) { return ctx->cplx && ctx->approx == GWL_RPA; }

gwl_status prpa_workspace(gwl_ctx* ctx, int nb) {
    cudaStream_t st = ctx->stream;
    gwl_status rs = ensure_workspace(ctx, 2 * nb);  // 2 nb GEMM columns: x_0, z_0, x_1, z_1, ...
    if (rs != GWL_OK) return rs;
    CK(ctx->prpa_tc.ensure((size_t)2 * nb * ctx->n_mup * 8, st));
    CK(ctx->prpa_wc.ensure((size_t)2 * nb * ctx->n_mup * 8, st));
    const int np = prpa_parts(2 * ctx->n_vc);
    CK(ctx->prpa_apart.ensure((size_t)nb * np * 8, st));
    CK(ctx->normpart.ensure((size_t)2 * nb * std::max(np, vec_parts(2 * ctx->n_vc)) * 8, st));
    return GWL_OK;
}

// Coupling part of Omega^ on nb pairs whose padded copy is in xs:  out (x, z) = ( K^H W, K^H conj(W) ),  W = V ( K x + conj(K z) );
// with h != NULL the diagonal term is added in the epilogue: out = Delta o h + coupling part (h = the unpadded vectors in xs).
gwl_status prpa_apply(gwl_ctx* ctx, const double* h, double* out, int nb) {
    const int64_t ldm = ctx->n_mup;
    gwl_status rs = gemm_kx_c(ctx, 2 * nb);
    if (rs != GWL_OK) return rs;
    CKL(4, launch_prpa_combine(ctx->ws().T.as<double>(), ldm, nb, ctx->n_mu, ctx->prpa_tc.as<double>(), ctx->lstream()));
    rs = plain_gemm(ctx, ctx->V.as<double>(), ldm, ctx->prpa_tc.as<double>(), ldm, ctx->n_mu, 2 * nb, ctx->n_mup / BK,
                    ctx->prpa_wc.as<double>(), ldm, 1);
    if (rs != GWL_OK) return rs;
    CKL(4, launch_prpa_expand(ctx->prpa_wc.as<double>(), ldm, nb, ctx->n_mu, 1.0, ctx->ws().W.as<double>(), ctx->lstream()));
    return gemm_ktw_c(ctx, h, ctx->n_vc, out, ctx->n_vc, 2 * nb, nullptr, 0);
}

// S1 in the RPA: u = F conj([P1; P2]) of PAPER.md:290 = ( K^H g~, -K^H conj(g~) ) in the stored variables, g~ = V (psi_m conj(psi_n))
gwl_status prpa_start_vectors(gwl_ctx* ctx, int64_t j0, int nb, double* u) {
    const int64_t ldm = ctx->n_mup;
    CKL(4, launch_rho_c(ctx->phi_vT.as<double>(), (int64_t)ctx->n_kv * ldm, ctx->phi_cT.as<double>(),
                        (int64_t)ctx->n_k * ctx->n_c * ldm, ldm, ctx->nv_k, ctx->n_c, ctx->n_mu,
                        ctx->d_nidx.as<int32_t>() + 4 * j0, ctx->prpa_tc.as<double>(), ldm, nb, ctx->lstream()));
    gwl_status rs = plain_gemm(ctx, ctx->V.as<double>(), ldm, ctx->prpa_tc.as<double>(), ldm, ctx->n_mu, 2 * nb, ctx->n_mup / BK,
                               ctx->prpa_wc.as<double>(), ldm, 1);
    if (rs != GWL_OK) return rs;
    CKL(4, launch_prpa_expand(ctx->prpa_wc.as<double>(), ldm, nb, ctx->n_mu, -1.0, ctx->ws().W.as<double>(), ctx->lstream()));
    return gemm_ktw_c(ctx, nullptr, ctx->n_vc, u, ctx->n_vc, 2 * nb, nullptr, 0);
}

// gwl_lanczos for complex contexts in the RPA: three-term Lanczos of H = F Omega^ in the Omega^ inner product.
gwl_status lanczos_prpa(gwl_ctx* ctx, int64_t n_chains, int L, int nbmax, int reorth) {
    cudaStream_t st = ctx->stream;
    const int64_t n_vc = ctx->n_vc, n4 = 2 * n_vc;
    const int64_t ldxs = (int64_t)ctx->n_v * ctx->n_cp;
    const int np = prpa_parts(n4);
    gwl_status rs = prpa_workspace(ctx, nbmax);
    if (rs != GWL_OK) return rs;
    CK(ctx->scale.ensure((size_t)2 * nbmax * 8, st));
    CK(ctx->alive.ensure((size_t)2 * nbmax * 4, st));
    const int nslots = reorth ? L + 1 : 3;
    CK(ctx->basis.ensure((size_t)nslots * nbmax * n4 * 8, st));
    CK(ctx->sbasis.ensure((size_t)nslots * nbmax * n4 * 8, st));
    if (reorth) CK(ctx->coefpart.ensure((size_t)nbmax * L * 2 * np * 8, st));
    for (int64_t j0 = 0; j0 < n_chains; j0 += nbmax) {
        const int nb = (int)std::min<int64_t>(nbmax, n_chains - j0);
        const int64_t slot_stride = (int64_t)nb * n4;
        auto slot_of = [&](int k) { return (int64_t)(reorth ? k : ((k % 3) + 3) % 3) * slot_stride; };
        double* qb = ctx->basis.as<double>();
        double* sb = ctx->sbasis.as<double>();
        LanczosState S;
        S.alpha = ctx->alpha.as<double>() + j0 * L;
        S.beta = ctx->beta.as<double>() + j0 * L;
        S.norm2 = ctx->norm2.as<double>() + j0;
        S.len = ctx->len.as<int32_t>() + j0;
        S.scale = ctx->scale.as<double>();
        S.alive = ctx->alive.as<int32_t>();
        S.steps = L;
        double* normpart = ctx->normpart.as<double>();
        double* apart = ctx->prpa_apart.as<double>();
        double* xs = ctx->xs.as<double>();
        // ---- S1: u, Omega^ u, <u,u>_O ----
        double* u = qb + slot_of(0);
        double* su = sb + slot_of(0);
        rs = prpa_start_vectors(ctx, j0, nb, u);
        if (rs != GWL_OK) return rs;
        CKL(4, launch_prescale(u, n_vc, xs, ldxs, ctx->s.as<double>(), ctx->n_v, ctx->n_c, ctx->n_cp, 2 * nb, st));
        rs = prpa_apply(ctx, u, su, nb);
        if (rs != GWL_OK) return rs;
        CKL(4, launch_dot_partials(u, su, n4, n4, nb, normpart, np, st));
        CKL(5, launch_prpa_init(u, su, n4, nb, normpart, np, S, xs, ldxs, ctx->n_c, ctx->n_cp, apart, st));
        // ---- the step loop: one product with Omega^ per step, nothing touches the host ----
        for (int k = 0; k < L; ++k) {
            const double* q = qb + slot_of(k);
            const double* s = sb + slot_of(k);
            double* wq = qb + slot_of(k + 1);
            double* t = sb + slot_of(k + 1);
            const double* qp = k > 0 ? qb + slot_of(k - 1) : nullptr;
            const double* sp = k > 0 ? sb + slot_of(k - 1) : nullptr;
            const bool tstep = ctx->prof_level >= 1;
            cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr;
            if (tstep) {
                e0 = ctx->next_event();
                e1 = ctx->next_event();
                e2 = ctx->next_event();
                CK(cudaEventRecord(e0, st));
            }
            rs = prpa_apply(ctx, nullptr, t, nb);  // coupling part of Omega^ (F s_k); the diagonal term is added in update1
            if (rs != GWL_OK) return rs;
            if (tstep) CK(cudaEventRecord(e1, st));
            CKL(5, launch_prpa_update1(t, wq, q, qp, s, sp, ctx->d2.as<double>(), n4, nb, apart, S, k, normpart, st));
            if (reorth) {
                for (int pass = 0; pass < 2; ++pass) {
                    CKL(6, launch_prpa_reorth_dots(sb, slot_stride, k + 1, wq, n4, nb, ctx->coefpart.as<double>(), st));
                    CKL(6, launch_prpa_reorth_apply(qb, sb, slot_stride, k + 1, wq, t, n4, nb, ctx->coefpart.as<double>(),
                                                    pass == 1 ? normpart : nullptr, st));
                }
            }
            CKL(5, launch_prpa_update2(wq, t, n4, nb, normpart, S, k, xs, ldxs, ctx->n_c, ctx->n_cp, apart, st));
            if (tstep) CK(cudaEventRecord(e2, st));
        }
    }
    return GWL_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
extern "C" {

static gwl_status create_common(gwl_ctx** out, int64_t n_k, int64_t n_v, int64_t n_c, int64_t n_mu, bool cplx, int64_t n_q) {
    if (out == nullptr) return GWL_EINVAL;
    *out = nullptr;
    if (n_v < 1 || n_c < 1 || n_mu < 1 || n_k < 1 || n_q < 1 || n_k > 4096 || n_k * n_v > (1 << 20) || n_c > (1 << 20) ||
        n_mu > (1 << 24))
        return GWL_EINVAL;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return GWL_ECUDA;
    }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return GWL_ECUDA;
    }
    if (prop.major != 10) return GWL_ECUDA;  // the kernels are sm_100a code (TMA, DMMA, clusters, PDL): B200 only
    gwl_ctx* ctx = new (std::nothrow) gwl_ctx();
    if (ctx == nullptr) return GWL_ENOMEM;
    ctx->cplx = cplx;
    ctx->n_k = (int)n_k;
    ctx->nv_k = (int)n_v;
    ctx->n_kv = (int)(n_k * n_v);
    ctx->n_q = (int)n_q;
    ctx->n_v = cplx ? 2 * ctx->n_kv : (int)n_v;
    ctx->n_c = (int)n_c;
    ctx->n_mu = (int)n_mu;
    ctx->n_vc = (int64_t)ctx->n_v * n_c;
    ctx->n_cp = (int)round_up(n_c, BK);
    ctx->n_mup = (int)round_up(n_mu, BK);
    ctx->n_sm = prop.multiProcessorCount;
    ctx->device = dev;
    if (cplx) ctx->approx = GWL_TDA;  // Lanczos on the Hermitian A(q)
    *out = ctx;
    return GWL_OK;
}

gwl_status gwl_create(gwl_ctx** out, int64_t n_v, int64_t n_c, int64_t n_mu) {
    return create_common(out, 1, n_v, n_c, n_mu, false, 1);
}

gwl_status gwl_tdc_create(gwl_ctx** out, int64_t n_k, int64_t n_v, int64_t n_c, int64_t n_mu, int64_t n_q) {
    return create_common(out, n_k, n_v, n_c, n_mu, true, n_q);
}

void gwl_destroy(gwl_ctx* ctx) {
    if (ctx == nullptr) return;
    DeviceGuard dg(ctx);
    cudaStreamSynchronize(ctx->stream);
    if (ctx->stream2 != nullptr) cudaStreamSynchronize(ctx->stream2);
    DevBuf* bufs[] = {&ctx->phi_c, &ctx->phi_cT, &ctx->phi_vT, &ctx->V, &ctx->eps_v, &ctx->eps_c, &ctx->d2, &ctx->s,
                      &ctx->d_nidx, &ctx->d_midx, &ctx->d_start, &ctx->d_eps_n, &ctx->d_sgn_n, &ctx->alpha,
                      &ctx->beta, &ctx->norm2, &ctx->len, &ctx->scale, &ctx->alive, &ctx->xs, &ctx->dotpart,
                      &ctx->normpart, &ctx->basis, &ctx->coefpart, &ctx->tA, &ctx->tB, &ctx->pnext, &ctx->pnext_part,
                      &ctx->theta, &ctx->wgt, &ctx->ritz_info, &ctx->d_omega, &ctx->d_zeta, &ctx->d_sigma, &ctx->d_sigsum,
                      &ctx->io_x, &ctx->io_y, &ctx->isdf_phi, &ctx->isdf_phimu, &ctx->isdf_y, &ctx->isdf_s, &ctx->isdf_g,
                      &ctx->isdf_u, &ctx->stage, &ctx->x_nidx, &ctx->x_midx, &ctx->x_part, &ctx->x_sig, &ctx->x_eps,
                      &ctx->x_vxc, &ctx->x_sc, &ctx->x_e, &ctx->x_z, &ctx->x_it};
    for (DevBuf* b : bufs) b->release();
    for (gwl_ctx::WorkSet& w : ctx->wset) {
        DevBuf* wb[] = {&w.T, &w.W, &w.part, &w.sk_ws, &w.sk_flags};
        for (DevBuf* b : wb) b->release();
    }
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    for (cudaEvent_t e : ctx->kev) cudaEventDestroy(e);
    if (ctx->ev_consumed != nullptr) cudaEventDestroy(ctx->ev_consumed);
    if (ctx->ev_s1 != nullptr) cudaEventDestroy(ctx->ev_s1);
    if (ctx->stream2 != nullptr) cudaStreamDestroy(ctx->stream2);
    for (gwl_ctx::StepGraph& g : ctx->graphs)
        if (g.exec != nullptr) cudaGraphExecDestroy(g.exec);
    if (ctx->ev_gin != nullptr) cudaEventDestroy(ctx->ev_gin);
    if (ctx->ev_gout != nullptr) cudaEventDestroy(ctx->ev_gout);
    if (ctx->gstream != nullptr) cudaStreamDestroy(ctx->gstream);
    ctx->kbase.release();
    ctx->sbasis.release();
    ctx->prpa_tc.release();
    ctx->prpa_wc.release();
    ctx->prpa_apart.release();
    delete ctx;
}

const char* gwl_last_error(const gwl_ctx* ctx) { return ctx ? ctx->err.c_str() : ""; }

gwl_status gwl_set_pointer_mode(gwl_ctx* ctx, int device_ptrs) {
    if (ctx == nullptr || (device_ptrs != 0 && device_ptrs != 1)) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    ctx->device_ptrs = device_ptrs;
    return GWL_OK;
}

gwl_status gwl_set_stream(gwl_ctx* ctx, void* cuda_stream) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    return GWL_OK;
}

// Orbitals at the fitting points from compact DEVICE arrays d_phi_v [n_mu][n_v], d_phi_c [n_mu][n_c]: the padded and
// transposed copies the GEMMs read
static gwl_status install_orbitals(gwl_ctx* ctx, const double* d_phi_v, const double* d_phi_c) {
    cudaStream_t st = ctx->stream;
    CK(ctx->phi_c.ensure((size_t)ctx->n_mu * ctx->n_cp * 8, st));
    CK(ctx->phi_cT.ensure((size_t)ctx->n_c * ctx->n_mup * 8, st));
    CK(ctx->phi_vT.ensure((size_t)ctx->n_v * ctx->n_mup * 8, st));
    CK(cudaMemsetAsync(ctx->phi_c.p, 0, ctx->phi_c.bytes, st));
    CK(cudaMemsetAsync(ctx->phi_cT.p, 0, ctx->phi_cT.bytes, st));
    CK(cudaMemsetAsync(ctx->phi_vT.p, 0, ctx->phi_vT.bytes, st));
    CKL(4, launch_copy_pad(d_phi_c, ctx->n_mu, ctx->n_c, ctx->phi_c.as<double>(), ctx->n_cp, st));
    CKL(4, launch_transpose(d_phi_c, ctx->n_mu, ctx->n_c, ctx->phi_cT.as<double>(), ctx->n_mup, st));
    CKL(4, launch_transpose(d_phi_v, ctx->n_mu, ctx->n_v, ctx->phi_vT.as<double>(), ctx->n_mup, st));
    return GWL_OK;
}

gwl_status gwl_set_orbitals(gwl_ctx* ctx, const double* phi_v, const double* phi_c) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_set_orbitals: real-orbital call on a complex (gwl_tdc_create) context");
    if (ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_set_orbitals: symmetry-block (gwl_sym_create) context: use gwl_sym_set_orbitals");
    if (phi_v == nullptr || phi_c == nullptr) return ctx->fail(GWL_EINVAL, "gwl_set_orbitals: NULL input");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const size_t nv = (size_t)ctx->n_mu * ctx->n_v, nc = (size_t)ctx->n_mu * ctx->n_c;
    DevBuf& tmp = ctx->stage;  // kept across calls: no cudaMalloc/cudaFree in a repeated set_orbitals
    CK(tmp.ensure((nv + nc) * 8, st));
    double* dv = tmp.as<double>();
    double* dc = dv + nv;
    CK(cudaMemcpyAsync(dc, phi_c, nc * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(dv, phi_v, nv * 8, cudaMemcpyHostToDevice, st));
    gwl_status rs = install_orbitals(ctx, dv, dc);
    if (rs != GWL_OK) return rs;
    CK(cudaStreamSynchronize(st));
    ctx->have_orb = true;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_set_energies(gwl_ctx* ctx, const double* eps_v, const double* eps_c) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_set_energies: real-orbital call on a complex (gwl_tdc_create) context");
    if (eps_v == nullptr || eps_c == nullptr) return ctx->fail(GWL_EINVAL, "gwl_set_energies: NULL input");
    const int nv_orb = ctx->sym ? ctx->sym_nv_tot : ctx->n_v, nc_orb = ctx->sym ? ctx->sym_nc_tot : ctx->n_c;
    double vmax = -INFINITY, cmin = INFINITY;
    for (int i = 0; i < nv_orb; ++i) {
        if (!std::isfinite(eps_v[i])) return ctx->fail(GWL_EINVAL, "gwl_set_energies: non-finite eps_v");
        vmax = std::max(vmax, eps_v[i]);
    }
    for (int i = 0; i < nc_orb; ++i) {
        if (!std::isfinite(eps_c[i])) return ctx->fail(GWL_EINVAL, "gwl_set_energies: non-finite eps_c");
        cmin = std::min(cmin, eps_c[i]);
    }
    if (!(cmin > vmax)) return ctx->fail(GWL_EINVAL, "gwl_set_energies: need min(eps_c) > max(eps_v)");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    ctx->h_eps_v.assign(eps_v, eps_v + nv_orb);
    ctx->h_eps_c.assign(eps_c, eps_c + nc_orb);
    CK(ctx->eps_v.ensure((size_t)nv_orb * 8, st));
    CK(ctx->eps_c.ensure((size_t)nc_orb * 8, st));
    if (ctx->sym) {  // the diagonal term of a block is built by gwl_sym_select
        CK(cudaMemcpyAsync(ctx->eps_v.p, eps_v, (size_t)nv_orb * 8, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->eps_c.p, eps_c, (size_t)nc_orb * 8, cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));
        ctx->have_eps = true;
        ctx->sym_gamma = -1;
        invalidate_run(ctx);
        ctx->chain_mode = 0;
        ctx->n_chains_set = 0;
        return GWL_OK;
    }
    CK(ctx->d2.ensure((size_t)ctx->n_vc * 8, st));
    CK(ctx->s.ensure((size_t)ctx->n_vc * 8, st));
    CK(cudaMemcpyAsync(ctx->eps_v.p, eps_v, (size_t)ctx->n_v * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->eps_c.p, eps_c, (size_t)ctx->n_c * 8, cudaMemcpyHostToDevice, st));
    CKL(4, launch_build_delta(ctx->eps_v.as<double>(), ctx->eps_c.as<double>(), ctx->n_v, ctx->n_c, ctx->d2.as<double>(),
                          ctx->s.as<double>(), ctx->approx, st));
    CK(cudaStreamSynchronize(st));
    ctx->have_eps = true;
    invalidate_run(ctx);
    if (ctx->chain_mode == 1) {  // eps_n / eta_n of index chains were taken from the old energies
        ctx->chain_mode = 0;
        ctx->n_chains_set = 0;
    }
    return GWL_OK;
}

gwl_status gwl_set_kernel(gwl_ctx* ctx, const double* V) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (V == nullptr) return ctx->fail(GWL_EINVAL, "gwl_set_kernel: NULL input");
    if (ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_set_kernel: symmetry-block (gwl_sym_create) context: use gwl_sym_set_kernel");
    cudaStream_t st = ctx->stream;
    CK(ctx->V.ensure((size_t)ctx->n_mu * ctx->n_mup * 8, st));
    CK(cudaMemsetAsync(ctx->V.p, 0, ctx->V.bytes, st));
    CK(cudaMemcpy2DAsync(ctx->V.p, (size_t)ctx->n_mup * 8, V, (size_t)ctx->n_mu * 8, (size_t)ctx->n_mu * 8,
                         (size_t)ctx->n_mu, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));
    ctx->have_V = true;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_set_polynomial(gwl_ctx* ctx, int g, const double* cheb, double lo, double hi) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_set_polynomial: real-orbital call on a complex (gwl_tdc_create) context");
    if (g < 0 || g > 64) return ctx->fail(GWL_EINVAL, "gwl_set_polynomial: g out of range [0, 64]");
    if (g == 0) {
        ctx->g = 0;
        ctx->cheb.clear();
        invalidate_run(ctx);
        return GWL_OK;
    }
    if (cheb == nullptr || !(hi > lo) || !std::isfinite(lo) || !std::isfinite(hi))
        return ctx->fail(GWL_EINVAL, "gwl_set_polynomial: need cheb != NULL and hi > lo");
    if (ctx->approx != GWL_RPA)
        return ctx->fail(GWL_ESTATE, "gwl_set_polynomial: the polynomial square root applies to C (RPA) only");
    ctx->g = g;
    ctx->cheb.assign(cheb, cheb + g + 1);
    ctx->lo = lo;
    ctx->hi = hi;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_set_approximation(gwl_ctx* ctx, int approximation) {
    if (ctx == nullptr || (approximation != GWL_RPA && approximation != GWL_TDA)) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) {  // GWL_TDA (default): Lanczos on A(q); GWL_RPA: pseudo-Hermitian Lanczos on C^RPA(q); Delta and s are shared
        ctx->approx = approximation;
        invalidate_run(ctx);
        return GWL_OK;
    }
    if (ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_set_approximation: symmetry-block (gwl_sym_create) contexts run the RPA operator C only");
    if (approximation == GWL_TDA && ctx->g > 0)
        return ctx->fail(GWL_ESTATE, "gwl_set_approximation: clear the polynomial first (it approximates sqrt(C), RPA only)");
    ctx->approx = approximation;
    invalidate_run(ctx);
    if (ctx->have_eps) {  // rebuild the diagonal term and the scaling for the new operator
        LaunchScope ls(ctx);
        cudaStream_t st = ctx->stream;
        CKL(4, launch_build_delta(ctx->eps_v.as<double>(), ctx->eps_c.as<double>(), ctx->n_v, ctx->n_c,
                              ctx->d2.as<double>(), ctx->s.as<double>(), ctx->approx, st));
        CK(cudaStreamSynchronize(st));
    }
    return GWL_OK;
}

gwl_status gwl_casida_matvec(gwl_ctx* ctx, const double* x, double* y, int64_t nvec) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_casida_matvec: real-orbital call on a complex (gwl_tdc_create) context");
    if (ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_casida_matvec: symmetry-block (gwl_sym_create) context: use gwl_sym_matvec");
    if (nvec < 0) return ctx->fail(GWL_EINVAL, "gwl_casida_matvec: nvec < 0");
    if (nvec == 0) return GWL_OK;
    if (x == nullptr || y == nullptr) return ctx->fail(GWL_EINVAL, "gwl_casida_matvec: NULL vector");
    if (!ready(ctx)) return ctx->fail(GWL_ESTATE, "gwl_casida_matvec: orbitals, energies and kernel must be set");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int chunk = (int)std::min<int64_t>(nvec, 256);
    gwl_status rs = ensure_workspace(ctx, chunk);
    if (rs != GWL_OK) return rs;
    const int64_t ldxs = (int64_t)ctx->n_v * ctx->n_cp;
    if (!ctx->device_ptrs) {
        CK(ctx->io_x.ensure((size_t)chunk * ctx->n_vc * 8, st));
        CK(ctx->io_y.ensure((size_t)chunk * ctx->n_vc * 8, st));
    }
    for (int64_t j0 = 0; j0 < nvec; j0 += chunk) {
        const int nb = (int)std::min<int64_t>(chunk, nvec - j0);
        const double* xd;
        double* yd;
        if (ctx->device_ptrs) {
            xd = x + j0 * ctx->n_vc;
            yd = y + j0 * ctx->n_vc;
        } else {
            CK(cudaMemcpyAsync(ctx->io_x.p, x + j0 * ctx->n_vc, (size_t)nb * ctx->n_vc * 8, cudaMemcpyHostToDevice, st));
            xd = ctx->io_x.as<double>();
            yd = ctx->io_y.as<double>();
        }
        CKL(4, launch_prescale(xd, ctx->n_vc, ctx->xs.as<double>(), ldxs, ctx->s.as<double>(), ctx->n_v, ctx->n_c,
                           ctx->n_cp, nb, st));
        rs = apply_casida_core(ctx, xd, ctx->n_vc, yd, ctx->n_vc, nb, nullptr, 0);
        if (rs != GWL_OK) return rs;
        if (!ctx->device_ptrs) {
            CK(cudaMemcpyAsync(y + j0 * ctx->n_vc, yd, (size_t)nb * ctx->n_vc * 8, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
        }
    }
    return GWL_OK;
}

gwl_status gwl_set_chains(gwl_ctx* ctx, int64_t n_chains, const int32_t* n_idx, const int32_t* m_idx) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_set_chains: real-orbital call on a complex (gwl_tdc_create) context");
    if (n_chains < 0 || (n_chains > 0 && (n_idx == nullptr || m_idx == nullptr)))
        return ctx->fail(GWL_EINVAL, "gwl_set_chains: bad arguments");
    if (!ctx->have_eps) return ctx->fail(GWL_ESTATE, "gwl_set_chains: energies must be set first");
    if (ctx->sym && ctx->sym_gamma < 0) return ctx->fail(GWL_ESTATE, "gwl_set_chains: select a symmetry block first (gwl_sym_select)");
    const int nv_orb = ctx->sym ? ctx->sym_nv_tot : ctx->n_v;
    const int n_orb = nv_orb + (ctx->sym ? ctx->sym_nc_tot : ctx->n_c);
    std::vector<double> eps(n_chains);
    std::vector<int32_t> sgn(n_chains), n_pos, m_pos;
    for (int64_t j = 0; j < n_chains; ++j) {
        if (n_idx[j] < 0 || n_idx[j] >= n_orb || m_idx[j] < 0 || m_idx[j] >= n_orb)
            return ctx->fail(GWL_EINVAL, "gwl_set_chains: orbital index out of range");
        const bool occ = n_idx[j] < nv_orb;
        eps[j] = occ ? ctx->h_eps_v[n_idx[j]] : ctx->h_eps_c[n_idx[j] - nv_orb];
        sgn[j] = occ ? 1 : -1;
    }
    if (ctx->sym) {  // |P_nm> lives in block Gamma_n ^ Gamma_m; conduction indices become rows of the padded Phi_c^T
        auto locate = [&](int idx, int& irrep, int& pos) {
            const bool occ = idx < nv_orb;
            const int loc = occ ? idx : idx - nv_orb;
            const int* off = occ ? ctx->sym_voff : ctx->sym_coff;
            const int* cnt = occ ? ctx->sym_nv : ctx->sym_nc;
            irrep = 0;
            while (irrep + 1 < ctx->sym_g && loc >= off[irrep] + cnt[irrep]) ++irrep;
            pos = occ ? idx : nv_orb + ctx->sym_cpoff[irrep] + (loc - off[irrep]);
        };
        n_pos.resize(n_chains);
        m_pos.resize(n_chains);
        for (int64_t j = 0; j < n_chains; ++j) {
            int gn, gm;
            locate(n_idx[j], gn, n_pos[j]);
            locate(m_idx[j], gm, m_pos[j]);
            if ((gn ^ gm) != ctx->sym_gamma)
                return ctx->fail(GWL_EINVAL, "gwl_set_chains: the pair (n, m) does not belong to the selected symmetry block");
        }
        n_idx = n_pos.data();
        m_idx = m_pos.data();
    }
    cudaStream_t st = ctx->stream;
    CK(ctx->d_nidx.ensure((size_t)n_chains * 4, st));
    CK(ctx->d_midx.ensure((size_t)n_chains * 4, st));
    CK(ctx->d_eps_n.ensure((size_t)n_chains * 8, st));
    CK(ctx->d_sgn_n.ensure((size_t)n_chains * 4, st));
    if (n_chains > 0) {
        CK(cudaMemcpyAsync(ctx->d_nidx.p, n_idx, (size_t)n_chains * 4, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_midx.p, m_idx, (size_t)n_chains * 4, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_eps_n.p, eps.data(), (size_t)n_chains * 8, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_sgn_n.p, sgn.data(), (size_t)n_chains * 4, cudaMemcpyHostToDevice, st));
    }
    CK(cudaStreamSynchronize(st));
    ctx->chain_mode = 1;
    ctx->n_chains_set = n_chains;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_set_start_vectors(gwl_ctx* ctx, int64_t n_chains, const double* p, const double* eps_n,
                                 const int32_t* sgn_n) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_set_start_vectors: real-orbital call on a complex (gwl_tdc_create) context");
    if (ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_set_start_vectors: symmetry-block (gwl_sym_create) context: chains are set by orbital indices");
    if (n_chains < 0 || (n_chains > 0 && (p == nullptr || eps_n == nullptr || sgn_n == nullptr)))
        return ctx->fail(GWL_EINVAL, "gwl_set_start_vectors: bad arguments");
    for (int64_t j = 0; j < n_chains; ++j)
        if (sgn_n[j] != 1 && sgn_n[j] != -1) return ctx->fail(GWL_EINVAL, "gwl_set_start_vectors: sgn_n must be +1/-1");
    cudaStream_t st = ctx->stream;
    CK(ctx->d_start.ensure((size_t)n_chains * ctx->n_vc * 8, st));
    CK(ctx->d_eps_n.ensure((size_t)n_chains * 8, st));
    CK(ctx->d_sgn_n.ensure((size_t)n_chains * 4, st));
    if (n_chains > 0) {
        CK(cudaMemcpyAsync(ctx->d_start.p, p, (size_t)n_chains * ctx->n_vc * 8,
                           ctx->device_ptrs ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_eps_n.p, eps_n, (size_t)n_chains * 8, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_sgn_n.p, sgn_n, (size_t)n_chains * 4, cudaMemcpyHostToDevice, st));
    }
    CK(cudaStreamSynchronize(st));
    ctx->chain_mode = 2;
    ctx->n_chains_set = n_chains;
    invalidate_run(ctx);
    return GWL_OK;
}

static gwl_status lanczos_impl(gwl_ctx* ctx, int64_t n_chains, int64_t steps, int64_t block, int reorth, double* alpha,
                               double* beta, double* norm2, int32_t* len, bool graph_active) {
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int L = (int)steps;
    // `block` is a batching hint: chains per launch are capped by grid.y of the vector kernels
    const int nbmax = (int)std::min<int64_t>(std::min<int64_t>(block, 65535), std::max<int64_t>(n_chains, 1));
    const int64_t n_vc = ctx->n_vc;
    const int64_t ldxs = (int64_t)ctx->n_v * ctx->n_cp;
    const int npart = vec_parts(n_vc);
    const int rparts = ctx->cplx ? reorth_parts(n_vc / 2) : reorth_parts(n_vc);
    const bool poly = ctx->g > 0;

    invalidate_run(ctx);  // stays invalid if this call fails part-way
    ctx->ev_used = 0;
    ctx->kev_used = 0;
    ctx->kev_class.clear();
    CK(ctx->alpha.ensure((size_t)std::max<int64_t>(n_chains, 1) * L * 8, st));
    CK(ctx->beta.ensure((size_t)std::max<int64_t>(n_chains, 1) * L * 8, st));
    CK(ctx->norm2.ensure((size_t)std::max<int64_t>(n_chains, 1) * 8, st));
    CK(ctx->len.ensure((size_t)std::max<int64_t>(n_chains, 1) * 4, st));
    CK(cudaMemsetAsync(ctx->alpha.p, 0, ctx->alpha.bytes, st));
    CK(cudaMemsetAsync(ctx->beta.p, 0, ctx->beta.bytes, st));
    if (prpa(ctx)) {
        if (ctx->chain_mode != 1) return ctx->fail(GWL_ESTATE, "gwl_lanczos: the complex RPA needs gwl_tdc_set_chains");
        if (n_chains > 0) {
            gwl_status rs = lanczos_prpa(ctx, n_chains, L, nbmax, reorth);
            if (rs != GWL_OK) return rs;
        }
        ctx->run_chains = n_chains;
        ctx->run_steps = L;
        ctx->run_poly = 3;
        if (n_chains > 0) {
            const cudaMemcpyKind kind = ctx->device_ptrs ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
            if (alpha) CK(cudaMemcpyAsync(alpha, ctx->alpha.p, (size_t)n_chains * L * 8, kind, st));
            if (beta) CK(cudaMemcpyAsync(beta, ctx->beta.p, (size_t)n_chains * L * 8, kind, st));
            if (norm2) CK(cudaMemcpyAsync(norm2, ctx->norm2.p, (size_t)n_chains * 8, kind, st));
            if (len) CK(cudaMemcpyAsync(len, ctx->len.p, (size_t)n_chains * 4, kind, st));
        }
        if (!ctx->device_ptrs) CK(cudaStreamSynchronize(st));
        return GWL_OK;
    }
    if (n_chains > 0) {
        gwl_status rs = ensure_workspace(ctx, nbmax);
        if (rs != GWL_OK) return rs;
        CK(ctx->scale.ensure((size_t)2 * nbmax * 8, st));
        CK(ctx->alive.ensure((size_t)2 * nbmax * 4, st));
        const int nslots = reorth ? L + 1 : 3;
        CK(ctx->basis.ensure((size_t)nslots * nbmax * n_vc * 8, st));
        if (reorth) CK(ctx->coefpart.ensure((size_t)nbmax * L * rparts * 8 * (ctx->cplx ? 2 : 1), st));
        if (poly) {
            CK(ctx->tA.ensure((size_t)nbmax * n_vc * 8, st));
            CK(ctx->tB.ensure((size_t)nbmax * n_vc * 8, st));
        }
    }
    // with more than one block of index chains, S1 of block i+1 (rho, V rho, K^T: 1.5 GEMMs) runs on a side
    // stream with its own GEMM scratch under the step loop of block i, into `pnext`; block i+1 then starts with a copy.
    const bool overlap = ctx->chain_mode == 1 && n_chains > nbmax;
    if (overlap) {
        if (ctx->stream2 == nullptr) {
            CK(cudaStreamCreateWithFlags(&ctx->stream2, cudaStreamNonBlocking));
            CK(cudaEventCreateWithFlags(&ctx->ev_consumed, cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&ctx->ev_s1, cudaEventDisableTiming));
        }
        ctx->cur = 1;
        gwl_status rs = ensure_workspace(ctx, nbmax);
        ctx->cur = 0;
        if (rs != GWL_OK) return rs;
        CK(ctx->pnext.ensure((size_t)nbmax * n_vc * 8, st));
        CK(ctx->pnext_part.ensure((size_t)nbmax * casida_ndot(ctx, nbmax) * 8, st));
    }

    for (int64_t j0 = 0; j0 < n_chains; j0 += nbmax) {
        const int nb = (int)std::min<int64_t>(nbmax, n_chains - j0);
        const int ndot_c = casida_ndot(ctx, nb);
        const int64_t slot_stride = (int64_t)nb * n_vc;
        double* basis = ctx->basis.as<double>();
        auto slot = [&](int k) -> double* { return basis + (int64_t)(reorth ? k : ((k % 3) + 3) % 3) * slot_stride; };
        LanczosState S;
        S.alpha = ctx->alpha.as<double>() + j0 * L;
        S.beta = ctx->beta.as<double>() + j0 * L;
        S.norm2 = ctx->norm2.as<double>() + j0;
        S.len = ctx->len.as<int32_t>() + j0;
        S.scale = ctx->scale.as<double>();
        S.alive = ctx->alive.as<int32_t>();
        S.steps = L;
        double* dotpart = ctx->dotpart.as<double>();
        double* normpart = ctx->normpart.as<double>();

        // ---- S1: start vectors into slot 0 ----
        if (ctx->chain_mode == 1) {
            if (overlap && j0 > 0) {  // built on the side stream while the previous block was stepping
                CK(cudaStreamWaitEvent(st, ctx->ev_s1, 0));
                CK(cudaMemcpyAsync(slot(0), ctx->pnext.p, (size_t)nb * n_vc * 8, cudaMemcpyDeviceToDevice, st));
                CK(cudaMemcpyAsync(dotpart, ctx->pnext_part.p, (size_t)nb * ndot_c * 8, cudaMemcpyDeviceToDevice, st));
            } else {
                gwl_status rs = build_start_vectors(ctx, j0, nb, slot(0), dotpart, ndot_c);
                if (rs != GWL_OK) return rs;
            }
            CKL(5, launch_lanczos_init(slot(0), n_vc, nb, dotpart, ndot_c, S, ctx->xs.as<double>(), ldxs,
                                   ctx->s.as<double>(), ctx->n_v, ctx->n_c, ctx->n_cp, st));
            if (overlap && j0 + nbmax < n_chains) {
                const int nb_next = (int)std::min<int64_t>(nbmax, n_chains - j0 - nbmax);
                CK(cudaEventRecord(ctx->ev_consumed, st));  // pnext / pnext_part of this block have been copied out
                CK(cudaStreamWaitEvent(ctx->stream2, ctx->ev_consumed, 0));
                ctx->cur = 1;
                gwl_status rs = build_start_vectors(ctx, j0 + nbmax, nb_next, ctx->pnext.as<double>(),
                                                    ctx->pnext_part.as<double>(), casida_ndot(ctx, nb_next));
                ctx->cur = 0;
                if (rs != GWL_OK) return rs;
                CK(cudaEventRecord(ctx->ev_s1, ctx->stream2));
            }
        } else {
            CK(cudaMemcpyAsync(slot(0), ctx->d_start.as<double>() + j0 * n_vc, (size_t)nb * n_vc * 8,
                               cudaMemcpyDeviceToDevice, st));
            CKL(4, launch_dot_partials(slot(0), slot(0), n_vc, n_vc, nb, normpart, npart, st));
            CKL(5, launch_lanczos_init(slot(0), n_vc, nb, normpart, npart, S, ctx->xs.as<double>(), ldxs,
                                   ctx->s.as<double>(), ctx->n_v, ctx->n_c, ctx->n_cp, st));
        }

        // ---- S2-S4: the step loop; nothing below touches the host ----
        // One Lanczos step.  k selects the vector slots (period 3) and the state parity (period 2); the fused update gets
        // k_arg and adds the device step counter Sk.kbase when that is set (graph replay, below).
        auto enqueue_step = [&](int k, int k_arg, const LanczosState& Sk) -> gwl_status {
            double* q = slot(k);
            double* w = slot(k + 1);
            const double* qp = k > 0 ? slot(k - 1) : nullptr;
            const bool tstep = ctx->prof_level >= 1;
            cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr;
            if (tstep) {
                e0 = ctx->next_event();
                e1 = ctx->next_event();
                e2 = ctx->next_event();
                CK(cudaEventRecord(e0, st));
            }
            int ndot, dstride;
            if (!poly) {
                gwl_status rs = apply_casida_core(ctx, q, n_vc, w, n_vc, nb, dotpart, ndot_c);
                if (rs != GWL_OK) return rs;
                ndot = ndot_c;
                dstride = ndot_c;
            } else {
                // w = p_g(C) q by the Chebyshev three-term recurrence on Ct = (2C - (hi+lo))/(hi-lo):
                //   t_1 = Ct q,  t_j = 2 Ct t_{j-1} - t_{j-2},  w = sum_j c_j t_j.
                // Every term is ONE Casida product whose K^T.W epilogue (EPI_CHEB) forms t_j from the accumulators, adds
                // c_j t_j to w, writes the scaled copy s o t_j that the next K.X reads and, on the last term, the
                // partial dots q.w of alpha: no streaming kernel between the GEMMs.
                const double hl = ctx->hi - ctx->lo, hs = ctx->hi + ctx->lo;
                double* tb[2] = {ctx->tA.as<double>(), ctx->tB.as<double>()};
                const double* x = q;         // t_{j-1}
                const double* t0 = nullptr;  // t_{j-2}
                for (int jj = 1; jj <= ctx->g; ++jj) {
                    const bool last = jj == ctx->g;
                    double* out = tb[(jj - 1) & 1];  // j >= 3: aliases t_{j-2} (read and written by the same thread)
                    ChebTerm ct;
                    ct.t0 = t0;
                    ct.w = w;
                    ct.q = last ? q : nullptr;
                    ct.xs_out = last ? nullptr : ctx->xs.as<double>();
                    ct.ca = (jj == 1 ? 2.0 : 4.0) / hl;
                    ct.cb = (jj == 1 ? -1.0 : -2.0) * hs / hl;
                    ct.cc = -1.0;
                    ct.cw = ctx->cheb[jj];
                    ct.c0 = ctx->cheb[0];
                    ct.first = jj == 1;
                    gwl_status rs = gemm_kx(ctx, nb);
                    if (rs == GWL_OK) rs = gemm_v(ctx, nb);
                    if (rs == GWL_OK) rs = gemm_ktw(ctx, x, n_vc, out, n_vc, nb, last ? dotpart : nullptr, ndot_c, &ct);
                    if (rs != GWL_OK) return rs;
                    t0 = x;
                    x = out;
                }
                ndot = ndot_c;
                dstride = ndot_c;
            }
            if (tstep) CK(cudaEventRecord(e1, st));
            if (!reorth && lanczos_fused_fits(n_vc)) {
                CKL(5, launch_lanczos_fused(w, q, qp, n_vc, nb, dotpart, ndot, dstride, Sk, k_arg, ctx->xs.as<double>(), ldxs,
                                        ctx->s.as<double>(), ctx->n_v, ctx->n_c, ctx->n_cp, st));
                if (tstep) CK(cudaEventRecord(e2, st));
                return GWL_OK;
            }
            CKL(5, launch_lanczos_update1(w, q, qp, n_vc, nb, dotpart, ndot, dstride, Sk, k, normpart, npart, st));
            if (reorth) {
                for (int pass = 0; pass < 2; ++pass) {
                    if (ctx->cplx) {  // complex projection coefficients <q_j, w>
                        CKL(6, launch_reorth_dots_c(basis, slot_stride, k + 1, w, n_vc, nb, ctx->coefpart.as<double>(), rparts,
                                                    st));
                        CKL(6, launch_reorth_apply_c(basis, slot_stride, k + 1, w, n_vc, nb, ctx->coefpart.as<double>(),
                                                     rparts, pass == 1 ? normpart : nullptr, st));
                        continue;
                    }
                    CKL(6, launch_reorth_dots(basis, slot_stride, k + 1, w, n_vc, nb, ctx->coefpart.as<double>(), rparts,
                                          st));
                    CKL(6, launch_reorth_apply(basis, slot_stride, k + 1, w, n_vc, nb, ctx->coefpart.as<double>(), rparts,
                                           pass == 1 ? normpart : nullptr, st));
                }
            }
            CKL(5, launch_lanczos_update2(w, n_vc, nb, normpart, reorth ? rparts : npart, Sk, k, ctx->xs.as<double>(), ldxs,
                                      ctx->s.as<double>(), ctx->n_v, ctx->n_c, ctx->n_cp, st));
            if (tstep) CK(cudaEventRecord(e2, st));
            return GWL_OK;
        };

        int k = 0;
        // Launch-bound sizes (fused-update path): after a few plain steps, which also size every workspace, the rest of the
        // chain is replayed from a CUDA graph of six steps.
        if (graph_active && !ctx->graph_off && ctx->prof_level == 0 && !reorth && !ctx->cplx && lanczos_fused_fits(n_vc) &&
            L >= 16) {
            const int pfx = ((L - 2) % 6) + 2;  // 2..7, (L - pfx) % 6 == 0
            for (; k < pfx; ++k) {
                gwl_status rs = enqueue_step(k, k, S);
                if (rs != GWL_OK) return rs;
            }
            // everything a replay depends on that is not reached through one of the hashed pointers
            uint64_t key = 1469598103934665603ull;
            auto mix = [&key](uint64_t v) {
                key ^= v;
                key *= 1099511628211ull;
            };
            const void* ptrs[] = {basis, ctx->xs.p, dotpart, S.alpha, S.beta, S.norm2, S.len, S.scale, S.alive, ctx->ws().T.p,
                                  ctx->ws().W.p, ctx->ws().part.p, ctx->ws().sk_ws.p, ctx->ws().sk_flags.p, ctx->phi_c.p,
                                  ctx->phi_cT.p, ctx->phi_vT.p, ctx->V.p, ctx->d2.p, ctx->s.p, ctx->tA.p, ctx->tB.p};
            for (const void* q : ptrs) mix((uint64_t)(uintptr_t)q);
            const int64_t ints[] = {nb, L, pfx, ctx->g, ctx->approx, n_vc, ctx->n_v, ctx->n_c, ctx->n_mu, ctx->v_sel,
                                    ctx->sym ? ctx->sym_gamma : -1};
            for (int64_t v : ints) mix((uint64_t)v);
            auto mixd = [&mix](double d) {
                uint64_t u;
                std::memcpy(&u, &d, 8);
                mix(u);
            };
            mixd(ctx->lo);
            mixd(ctx->hi);
            for (double c : ctx->cheb) mixd(c);
            gwl_ctx::StepGraph* sg = nullptr;
            for (gwl_ctx::StepGraph& g : ctx->graphs)
                if (g.key == key && g.exec != nullptr) sg = &g;
            if (sg == nullptr) {
                CK(ctx->kbase.ensure(4, st));
                gwl_ctx::StepGraph ng;
                ng.key = key;
                const unsigned epoch_saved = ctx->ws().sk_epoch;
                const int64_t launches_before = ctx->launches;
                cudaGraph_t graph = nullptr;
                bool ok = cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
                if (ok) {
                    // the stream-K hand-over flags start from zero in every replay, the epochs of the captured launches from 1
                    ok = cudaMemsetAsync(ctx->ws().sk_flags.p, 0, ctx->ws().sk_flags.bytes, st) == cudaSuccess;
                    ctx->ws().sk_epoch = 0;
                    LanczosState Sg = S;
                    Sg.kbase = ctx->kbase.as<int>();
                    for (int i = 0; i < 6 && ok; ++i) ok = enqueue_step(pfx + i, i, Sg) == GWL_OK;
                    if (ok) ok = launch_add_int(ctx->kbase.as<int>(), 6, st) == cudaSuccess;
                    const cudaError_t ee = cudaStreamEndCapture(st, &graph);
                    ok = ok && ee == cudaSuccess && graph != nullptr;
                    ng.max_epoch = ctx->ws().sk_epoch;
                    ctx->ws().sk_epoch = std::max(epoch_saved, ng.max_epoch);
                }
                if (ok) ok = cudaGraphInstantiate(&ng.exec, graph, 0) == cudaSuccess;
                if (graph != nullptr) cudaGraphDestroy(graph);
                ng.launches = (int)(ctx->launches - launches_before);
                ctx->launches = launches_before;  // captured, not launched
                if (!ok) {  // no graphs on this stream / driver: plain launches from here on
                    cudaGetLastError();
                    ctx->graph_off = true;
                } else {
                    if (ctx->graphs.size() >= 8) {  // evict the least recently used
                        size_t old = 0;
                        for (size_t i = 1; i < ctx->graphs.size(); ++i)
                            if (ctx->graphs[i].stamp < ctx->graphs[old].stamp) old = i;
                        cudaGraphExecDestroy(ctx->graphs[old].exec);
                        ctx->graphs.erase(ctx->graphs.begin() + old);
                    }
                    ctx->graphs.push_back(ng);
                    sg = &ctx->graphs.back();
                }
            }
            if (sg != nullptr) {
                sg->stamp = ++ctx->graph_stamp;
                ctx->ws().sk_epoch = std::max(ctx->ws().sk_epoch, sg->max_epoch);  // later plain launches: epochs the flags cannot hold
                CK(launch_set_int(ctx->kbase.as<int>(), pfx, st));
                for (; k < L; k += 6) {
                    CK(cudaGraphLaunch(sg->exec, st));
                    ctx->launches += sg->launches;
                }
            }
        }
        for (; k < L; ++k) {
            gwl_status rs = enqueue_step(k, k, S);
            if (rs != GWL_OK) return rs;
        }
    }
    ctx->run_chains = n_chains;
    ctx->run_steps = L;
    ctx->run_poly = poly ? 1 : (ctx->approx == GWL_TDA ? 2 : 0);
    if (n_chains > 0) {
        const cudaMemcpyKind kind = ctx->device_ptrs ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
        if (alpha) CK(cudaMemcpyAsync(alpha, ctx->alpha.p, (size_t)n_chains * L * 8, kind, st));
        if (beta) CK(cudaMemcpyAsync(beta, ctx->beta.p, (size_t)n_chains * L * 8, kind, st));
        if (norm2) CK(cudaMemcpyAsync(norm2, ctx->norm2.p, (size_t)n_chains * 8, kind, st));
        if (len) CK(cudaMemcpyAsync(len, ctx->len.p, (size_t)n_chains * 4, kind, st));
    }
    if (!ctx->device_ptrs) CK(cudaStreamSynchronize(st));
    return GWL_OK;
}

gwl_status gwl_lanczos(gwl_ctx* ctx, int64_t n_chains, int64_t steps, int64_t block, int reorth, double* alpha,
                       double* beta, double* norm2, int32_t* len) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (n_chains < 0 || steps < 1 || steps > 100000 || block < 1 || (reorth != 0 && reorth != 1))
        return ctx->fail(GWL_EINVAL, "gwl_lanczos: bad arguments");
    if (!ready(ctx)) return ctx->fail(GWL_ESTATE, "gwl_lanczos: orbitals, energies and kernel must be set");
    if (ctx->chain_mode == 0) return ctx->fail(GWL_ESTATE, "gwl_lanczos: no chains set");
    if (n_chains > ctx->n_chains_set) return ctx->fail(GWL_EINVAL, "gwl_lanczos: more chains than were set");
    // Step graphs (small problems, no profiling events, no reorthogonalisation): the whole call runs on an internal stream
    // fenced against the caller's stream on both sides, because the caller's stream may be the legacy default stream.
    static const bool graphs_allowed = std::getenv("GWL_NO_GRAPH") == nullptr;
    const bool want_graph = graphs_allowed && !ctx->graph_off && ctx->prof_level == 0 && reorth == 0 && !ctx->cplx && steps >= 16 &&
                            n_chains > 0 && lanczos_fused_fits(ctx->n_vc);
    if (!want_graph) return lanczos_impl(ctx, n_chains, steps, block, reorth, alpha, beta, norm2, len, false);
    if (ctx->gstream == nullptr) {
        CK(cudaStreamCreateWithFlags(&ctx->gstream, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&ctx->ev_gin, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ctx->ev_gout, cudaEventDisableTiming));
    }
    cudaStream_t user = ctx->stream;
    CK(cudaEventRecord(ctx->ev_gin, user));
    CK(cudaStreamWaitEvent(ctx->gstream, ctx->ev_gin, 0));
    ctx->stream = ctx->gstream;
    const gwl_status rs = lanczos_impl(ctx, n_chains, steps, block, reorth, alpha, beta, norm2, len, true);
    ctx->stream = user;
    if (cudaEventRecord(ctx->ev_gout, ctx->gstream) == cudaSuccess) cudaStreamWaitEvent(user, ctx->ev_gout, 0);
    return rs;
}

gwl_status gwl_resolvent(gwl_ctx* ctx, const double* zeta, int64_t n_zeta, double* r) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (n_zeta < 0 || (n_zeta > 0 && (zeta == nullptr || r == nullptr)))
        return ctx->fail(GWL_EINVAL, "gwl_resolvent: bad arguments");
    if (ctx->run_steps == 0) return ctx->fail(GWL_ESTATE, "gwl_resolvent: run gwl_lanczos first");
    if (n_zeta == 0 || ctx->run_chains == 0) return GWL_OK;
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const double* dz = zeta;
    double* dr = r;
    const size_t nr = (size_t)ctx->run_chains * n_zeta * 2 * 8;
    if (!ctx->device_ptrs) {
        CK(ctx->d_zeta.ensure((size_t)n_zeta * 16, st));
        CK(ctx->d_sigma.ensure(nr, st));
        CK(cudaMemcpyAsync(ctx->d_zeta.p, zeta, (size_t)n_zeta * 16, cudaMemcpyHostToDevice, st));
        dz = ctx->d_zeta.as<double>();
        dr = ctx->d_sigma.as<double>();
    }
    CKL(7, launch_contfrac(ctx->alpha.as<double>(), ctx->beta.as<double>(), ctx->norm2.as<double>(),
                       ctx->len.as<int32_t>(), ctx->run_steps, (int)ctx->run_chains, dz, (int)n_zeta, dr, st));
    if (!ctx->device_ptrs) {
        CK(cudaMemcpyAsync(r, dr, nr, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    return GWL_OK;
}

gwl_status gwl_selfenergy(gwl_ctx* ctx, const double* omega, int64_t n_omega, double eta, double* sigma,
                          double* sigma_sum) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (n_omega < 0 || (n_omega > 0 && omega == nullptr) || !(eta > 0.0))
        return ctx->fail(GWL_EINVAL, "gwl_selfenergy: bad arguments (eta must be > 0)");
    if (ctx->run_steps == 0) return ctx->fail(GWL_ESTATE, "gwl_selfenergy: run gwl_lanczos first");
    if (n_omega == 0) return GWL_OK;
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int nch = (int)ctx->run_chains, L = ctx->run_steps;
    // Only the sum is wanted (gwl_selfenergy_state): Sigma[chain][omega] is never materialised -- the chains go through a
    // small buffer in chunks and Eq. 10 is accumulated chunk by chunk on the device, in a fixed order.
    const bool sum_only = sigma == nullptr && sigma_sum != nullptr;
    const int chunk = sum_only ? std::min(std::max(nch, 1), 256) : std::max(nch, 1);
    const size_t nsig = (size_t)chunk * n_omega * 16;
    const double* dom = omega;
    double* dsig = sigma;
    double* dsum = sigma_sum;
    if (!ctx->device_ptrs) {
        CK(ctx->d_omega.ensure((size_t)n_omega * 8, st));
        CK(cudaMemcpyAsync(ctx->d_omega.p, omega, (size_t)n_omega * 8, cudaMemcpyHostToDevice, st));
        dom = ctx->d_omega.as<double>();
    }
    if (!ctx->device_ptrs || sigma == nullptr) {
        CK(ctx->d_sigma.ensure(nsig, st));
        dsig = ctx->d_sigma.as<double>();
    }
    if (sigma_sum != nullptr && !ctx->device_ptrs) {
        CK(ctx->d_sigsum.ensure((size_t)n_omega * 16, st));
        dsum = ctx->d_sigsum.as<double>();
    }
    if (nch > 0 && (ctx->run_poly == 0 || ctx->run_poly == 3)) {
        CK(ctx->theta.ensure((size_t)nch * L * 8, st));
        CK(ctx->wgt.ensure((size_t)nch * L * 8, st));
        CK(ctx->ritz_info.ensure((size_t)nch * 4, st));
        // divide and conquer (parallel) when T_L fits one CTA's shared memory, else the sequential QL kernel
        if (ritz_dc_fits(L))
            CKL(7, launch_ritz_dc(ctx->alpha.as<double>(), ctx->beta.as<double>(), ctx->len.as<int32_t>(), L, nch,
                              ctx->theta.as<double>(), ctx->wgt.as<double>(), ctx->ritz_info.as<int32_t>(), st));
        else
            CKL(7, launch_ritz(ctx->alpha.as<double>(), ctx->beta.as<double>(), ctx->len.as<int32_t>(), L, nch,
                           ctx->theta.as<double>(), ctx->wgt.as<double>(), nullptr, ctx->ritz_info.as<int32_t>(), st));
    }
    for (int c0 = 0; c0 < nch; c0 += chunk) {
        const int nc = std::min(chunk, nch - c0);
        double* out = sum_only ? dsig : dsig + (size_t)c0 * n_omega * 2;
        const double* al = ctx->alpha.as<double>() + (size_t)c0 * L;
        const double* be = ctx->beta.as<double>() + (size_t)c0 * L;
        const double* n2 = ctx->norm2.as<double>() + c0;
        const int32_t* ln = ctx->len.as<int32_t>() + c0;
        const double* en = ctx->d_eps_n.as<double>() + c0;
        const int32_t* sg = ctx->d_sgn_n.as<int32_t>() + c0;
        if (ctx->run_poly == 2)
            CKL(7, launch_sigma_tda(al, be, n2, ln, L, nc, en, sg, dom, (int)n_omega, eta,
                                    ctx->cplx ? 2.0 / ((double)ctx->n_q * ctx->n_k) : 1.0, out, st));
        else if (ctx->run_poly == 1)
            CKL(7, launch_sigma_poly(al, be, n2, ln, L, nc, en, sg, dom, (int)n_omega, eta, out, st));
        else if (ctx->run_poly == 3)  // complex RPA: positive Ritz branch of T, prefactor 2/(N_q N_k)
            CKL(7, launch_sigma_direct(ctx->theta.as<double>() + (size_t)c0 * L, ctx->wgt.as<double>() + (size_t)c0 * L, n2, ln,
                                       L, nc, en, sg, dom, (int)n_omega, eta, 1, 2.0 / ((double)ctx->n_q * ctx->n_k), out, st));
        else
            CKL(7, launch_sigma_direct(ctx->theta.as<double>() + (size_t)c0 * L, ctx->wgt.as<double>() + (size_t)c0 * L, n2, ln,
                                       L, nc, en, sg, dom, (int)n_omega, eta, 0, 1.0, out, st));
        if (sigma_sum != nullptr) CKL(7, launch_sigma_sum(out, nc, (int)n_omega, dsum, (c0 > 0 || ctx->sig_accumulate) ? 1 : 0, st));
    }
    if (sigma_sum != nullptr && nch == 0) CKL(7, launch_sigma_sum(dsig, 0, (int)n_omega, dsum, 0, st));
    if (!ctx->device_ptrs) {
        if (sigma != nullptr && nch > 0)
            CK(cudaMemcpyAsync(sigma, dsig, (size_t)nch * n_omega * 16, cudaMemcpyDeviceToHost, st));
        if (sigma_sum != nullptr)
            CK(cudaMemcpyAsync(sigma_sum, dsum, (size_t)n_omega * 16, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    return GWL_OK;
}

gwl_status gwl_selfenergy_state(gwl_ctx* ctx, int32_t m_idx, int64_t steps, int64_t block, int reorth,
                                const double* omega, int64_t n_omega, double eta, double* sigma_mm) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_selfenergy_state: real-orbital call on a complex (gwl_tdc_create) context");
    if (ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_selfenergy_state: symmetry-block (gwl_sym_create) context: use gwl_sym_selfenergy_state");
    if (sigma_mm == nullptr || omega == nullptr || n_omega < 1)
        return ctx->fail(GWL_EINVAL, "gwl_selfenergy_state: bad arguments");
    const int n_orb = ctx->n_v + ctx->n_c;
    std::vector<int32_t> n_idx(n_orb), m_rep(n_orb, m_idx);
    for (int i = 0; i < n_orb; ++i) n_idx[i] = i;
    gwl_status rs = gwl_set_chains(ctx, n_orb, n_idx.data(), m_rep.data());
    if (rs != GWL_OK) return rs;
    rs = gwl_lanczos(ctx, n_orb, steps, block, reorth, nullptr, nullptr, nullptr, nullptr);
    if (rs != GWL_OK) return rs;
    return gwl_selfenergy(ctx, omega, n_omega, eta, nullptr, sigma_mm);
}

gwl_status gwl_exchange(gwl_ctx* ctx, int64_t n_states, const int32_t* m_idx, double* sigma_x) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_exchange: real-orbital call on a complex (gwl_tdc_create) context");
    if (n_states < 0 || (n_states > 0 && (m_idx == nullptr || sigma_x == nullptr)))
        return ctx->fail(GWL_EINVAL, "gwl_exchange: bad arguments");
    if (!ctx->have_orb || !ctx->have_V) return ctx->fail(GWL_ESTATE, "gwl_exchange: orbitals and kernel must be set");
    if (n_states == 0) return GWL_OK;
    const int nv_orb = ctx->sym ? ctx->sym_nv_tot : ctx->n_v;
    const int n_orb = nv_orb + (ctx->sym ? ctx->sym_nc_tot : ctx->n_c);
    for (int64_t j = 0; j < n_states; ++j)
        if (m_idx[j] < 0 || m_idx[j] >= n_orb) return ctx->fail(GWL_EINVAL, "gwl_exchange: orbital index out of range");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int chunk = std::min(nv_orb, 256);
    const int64_t ldm = ctx->n_mup;
    const int npart = vec_parts(ctx->n_mu);
    // only what rho -> V rho -> dot touches: T, W and the V.T split-K partials (none of the N_vc-sized Casida buffers)
    CK(ctx->ws().T.ensure((size_t)chunk * ldm * 8, st));
    CK(ctx->ws().W.ensure((size_t)chunk * ldm * 8, st));
    gwl_status rs = GWL_OK;
    // Symmetry-block contexts (reading Q25): rho_vm transforms as gamma = irrep(v) ^ irrep(m), so (vm|vm) over all points is
    // rho_w^T V^gamma rho_w on the wedge; the occupied orbitals go irrep by irrep, each against its own reduced kernel.
    auto irrep_pos = [&](int idx, int& irrep, int& pos) {
        irrep = 0;
        pos = idx;
        if (!ctx->sym) return;
        const bool occ = idx < nv_orb;
        const int loc = occ ? idx : idx - nv_orb;
        const int* off = occ ? ctx->sym_voff : ctx->sym_coff;
        const int* cnt = occ ? ctx->sym_nv : ctx->sym_nc;
        while (irrep + 1 < ctx->sym_g && loc >= off[irrep] + cnt[irrep]) ++irrep;
        pos = occ ? idx : nv_orb + ctx->sym_cpoff[irrep] + (loc - off[irrep]);  // row of the padded Phi_c^T
    };
    // (v, m) index pairs of every rho_vm, state-major
    std::vector<int32_t> hv((size_t)n_states * nv_orb), hm((size_t)n_states * nv_orb), gm(n_states);
    for (int64_t j = 0; j < n_states; ++j) {
        int irr, pos;
        irrep_pos(m_idx[j], irr, pos);
        gm[j] = irr;
        for (int v = 0; v < nv_orb; ++v) {
            hv[(size_t)j * nv_orb + v] = v;
            hm[(size_t)j * nv_orb + v] = pos;
        }
    }
    CK(ctx->x_nidx.ensure(hv.size() * 4, st));
    CK(ctx->x_midx.ensure(hm.size() * 4, st));
    CK(ctx->x_part.ensure((size_t)chunk * npart * 8, st));
    CK(cudaMemcpyAsync(ctx->x_nidx.p, hv.data(), hv.size() * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->x_midx.p, hm.data(), hm.size() * 4, cudaMemcpyHostToDevice, st));
    double* dout = sigma_x;
    if (!ctx->device_ptrs) {
        CK(ctx->x_sig.ensure((size_t)n_states * 8, st));
        dout = ctx->x_sig.as<double>();
    }
    struct RestoreKernel {  // whatever path leaves this function, the V GEMM points at the selected block's kernel again
        gwl_ctx* c;
        int64_t saved;
        ~RestoreKernel() { c->v_sel = saved; }
    } restore_kernel{ctx, ctx->v_sel};
    const int n_seg = ctx->sym ? ctx->sym_g : 1;
    for (int64_t j = 0; j < n_states; ++j) {
        bool first = true;
        for (int a = 0; a < n_seg; ++a) {
            const int seg0 = ctx->sym ? ctx->sym_voff[a] : 0, seg1 = ctx->sym ? seg0 + ctx->sym_nv[a] : nv_orb;
            if (ctx->sym) ctx->v_sel = (int64_t)(a ^ gm[j]) * ctx->n_mu * ctx->n_mup;
            for (int v0 = seg0; v0 < seg1; v0 += chunk) {
                const int nb = std::min(chunk, seg1 - v0);
                const int64_t off = j * nv_orb + v0;
                // rho_vm -> T;  W = V T;  sum_v rho_vm . (V rho_vm)
                CKL(4, launch_rho(ctx->phi_vT.as<double>(), ctx->phi_cT.as<double>(), ldm, nv_orb, ctx->n_mu,
                                  ctx->x_nidx.as<int32_t>() + off, ctx->x_midx.as<int32_t>() + off, ctx->ws().T.as<double>(), ldm, nb,
                                  st));
                rs = gemm_v(ctx, nb);
                if (rs != GWL_OK) return rs;
                CKL(4, launch_dot_partials(ctx->ws().T.as<double>(), ctx->ws().W.as<double>(), ldm, ctx->n_mu, nb,
                                           ctx->x_part.as<double>(), npart, st));
                CKL(4, launch_accum_neg(ctx->x_part.as<double>(), nb * npart, dout + j, first ? 1 : 0, st));
                first = false;
            }
        }
    }
    if (!ctx->device_ptrs) {
        CK(cudaMemcpyAsync(sigma_x, dout, (size_t)n_states * 8, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    return GWL_OK;
}

gwl_status gwl_qp_solve(gwl_ctx* ctx, int64_t n_states, const double* eps_m, const double* vxc_m,
                        const double* sigma_x, const double* sigma_c, const double* omega, int64_t n_omega,
                        double* e_qp, double* z_qp, int32_t* iters) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (n_states < 0 || n_omega < 2 || n_omega > (1 << 28))
        return ctx->fail(GWL_EINVAL, "gwl_qp_solve: need n_states >= 0 and n_omega >= 2");
    if (n_states == 0) return GWL_OK;
    if (eps_m == nullptr || vxc_m == nullptr || sigma_x == nullptr || sigma_c == nullptr || omega == nullptr ||
        e_qp == nullptr || z_qp == nullptr)
        return ctx->fail(GWL_EINVAL, "gwl_qp_solve: NULL argument");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    CK(ctx->x_eps.ensure((size_t)n_states * 8, st));
    CK(ctx->x_vxc.ensure((size_t)n_states * 8, st));
    CK(cudaMemcpyAsync(ctx->x_eps.p, eps_m, (size_t)n_states * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->x_vxc.p, vxc_m, (size_t)n_states * 8, cudaMemcpyHostToDevice, st));
    const double *dsx = sigma_x, *dsc = sigma_c, *dom = omega;
    double *de = e_qp, *dz = z_qp;
    int32_t* dit = iters;
    if (!ctx->device_ptrs) {
        const size_t nsc = (size_t)n_states * n_omega * 16;
        CK(ctx->x_sig.ensure((size_t)n_states * 8, st));
        CK(ctx->x_sc.ensure(nsc, st));
        CK(ctx->d_omega.ensure((size_t)n_omega * 8, st));
        CK(ctx->x_e.ensure((size_t)n_states * 8, st));
        CK(ctx->x_z.ensure((size_t)n_states * 8, st));
        CK(ctx->x_it.ensure((size_t)n_states * 4, st));
        CK(cudaMemcpyAsync(ctx->x_sig.p, sigma_x, (size_t)n_states * 8, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->x_sc.p, sigma_c, nsc, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_omega.p, omega, (size_t)n_omega * 8, cudaMemcpyHostToDevice, st));
        dsx = ctx->x_sig.as<double>();
        dsc = ctx->x_sc.as<double>();
        dom = ctx->d_omega.as<double>();
        de = ctx->x_e.as<double>();
        dz = ctx->x_z.as<double>();
        dit = ctx->x_it.as<int32_t>();
    }
    CKL(7, launch_qp_solve((int)n_states, ctx->x_eps.as<double>(), ctx->x_vxc.as<double>(), dsx, dsc, dom, (int)n_omega,
                           de, dz, dit, st));
    if (!ctx->device_ptrs) {
        CK(cudaMemcpyAsync(e_qp, de, (size_t)n_states * 8, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(z_qp, dz, (size_t)n_states * 8, cudaMemcpyDeviceToHost, st));
        if (iters != nullptr) CK(cudaMemcpyAsync(iters, dit, (size_t)n_states * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    return GWL_OK;
}

gwl_status gwl_spectrum_bounds(gwl_ctx* ctx, int64_t steps, double* lam_min, double* lam_max) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_spectrum_bounds: real-orbital call on a complex (gwl_tdc_create) context");
    if (steps < 2 || steps > 512 || lam_min == nullptr || lam_max == nullptr)
        return ctx->fail(GWL_EINVAL, "gwl_spectrum_bounds: need 2 <= steps <= 512 and non-NULL outputs");
    if (!ready(ctx)) return ctx->fail(GWL_ESTATE, "gwl_spectrum_bounds: orbitals, energies and kernel must be set");
    if (ctx->sym && ctx->sym_gamma < 0) return ctx->fail(GWL_ESTATE, "gwl_spectrum_bounds: select a symmetry block first (gwl_sym_select)");
    cudaStream_t st = ctx->stream;
    const int L = (int)std::min<int64_t>(steps, ctx->sym ? ctx->sym_npairs : ctx->n_vc);
    // one chain from a generic (counter-based pseudo-random) start vector, on the operator itself (never p_g)
    {
        LaunchScope ls(ctx);
        CK(ctx->d_start.ensure((size_t)ctx->n_vc * 8, st));
        CK(ctx->d_eps_n.ensure(8, st));
        CK(ctx->d_sgn_n.ensure(4, st));
        CKL(4, launch_fill_hash(ctx->d_start.as<double>(), ctx->n_vc, 0x9E3779B97F4A7C15ull, st));
        if (ctx->sym)  // the padding pairs are not part of the block: keep the probe vector off them
            for (int a = 0; a < ctx->sym_g; ++a) {
                const int b = a ^ ctx->sym_gamma;
                CKL(4, launch_sym_zero_pad(ctx->d_start.as<double>() + ctx->sym_vecoff[a], ctx->n_vc, ctx->sym_nv[a], ctx->sym_nc[b],
                                           ctx->sym_ncp[b], 1, st));
            }
        const double e0 = 0.0;
        const int32_t s0 = 1;
        CK(cudaMemcpyAsync(ctx->d_eps_n.p, &e0, 8, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_sgn_n.p, &s0, 4, cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));
    }
    ctx->chain_mode = 2;
    ctx->n_chains_set = 1;
    const int g_saved = ctx->g, ptr_saved = ctx->device_ptrs;
    ctx->g = 0;
    ctx->device_ptrs = 0;
    std::vector<double> a(L), b(L);
    double n2 = 0.0;
    int32_t len = 0;
    gwl_status rs = gwl_lanczos(ctx, 1, L, 1, 0, a.data(), b.data(), &n2, &len);
    ctx->g = g_saved;
    ctx->device_ptrs = ptr_saved;
    ctx->chain_mode = 0;  // the probe chain is not the caller's chain list
    ctx->n_chains_set = 0;
    invalidate_run(ctx);
    if (rs != GWL_OK) return rs;
    if (len < 1) return ctx->fail(GWL_ECUDA, "gwl_spectrum_bounds: Lanczos broke down at the first step");
    // Ritz values of T_len and, for the residual bound beta_len |s_len,i|, the LAST eigenvector components:
    // those are the first components of the reversed tridiagonal (same QL kernel, second launch).
    const int n = len;
    std::vector<double> h(4 * (size_t)n, 0.0);  // a, b, reversed a, reversed b
    for (int i = 0; i < n; ++i) {
        h[i] = a[i];
        h[n + i] = (i + 1 < n) ? b[i] : 0.0;
        h[2 * n + i] = a[n - 1 - i];
        h[3 * n + i] = (i + 1 < n) ? b[n - 2 - i] : 0.0;
    }
    LaunchScope ls(ctx);
    CK(ctx->theta.ensure((size_t)4 * n * 8, st));
    CK(ctx->wgt.ensure((size_t)4 * n * 8, st));
    CK(ctx->ritz_info.ensure(16, st));
    double* dT = ctx->theta.as<double>();  // [a | b | ra | rb]
    double* dO = ctx->wgt.as<double>();    // [theta | w_first | theta_r | w_last]
    const int32_t lens[2] = {n, n};
    CK(cudaMemcpyAsync(dT, h.data(), (size_t)4 * n * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->ritz_info.as<int32_t>() + 2, lens, 8, cudaMemcpyHostToDevice, st));
    CKL(7, launch_ritz(dT, dT + n, ctx->ritz_info.as<int32_t>() + 2, n, 1, dO, dO + n, nullptr,
                       ctx->ritz_info.as<int32_t>(), st));
    CKL(7, launch_ritz(dT + 2 * n, dT + 3 * n, ctx->ritz_info.as<int32_t>() + 3, n, 1, dO + 2 * n, dO + 3 * n, nullptr,
                       ctx->ritz_info.as<int32_t>() + 1, st));
    std::vector<double> o(4 * (size_t)n);
    CK(cudaMemcpyAsync(o.data(), dO, (size_t)4 * n * 8, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    int imax = 0, imin = 0, rmax = 0, rmin = 0;
    for (int i = 1; i < n; ++i) {
        if (o[i] > o[imax]) imax = i;
        if (o[i] < o[imin]) imin = i;
        if (o[2 * n + i] > o[2 * n + rmax]) rmax = i;
        if (o[2 * n + i] < o[2 * n + rmin]) rmin = i;
    }
    const double b_last = (len == L) ? b[n - 1] : 0.0;  // after a breakdown the Krylov space is invariant: exact
    *lam_max = o[imax] + b_last * std::sqrt(std::max(o[3 * n + rmax], 0.0));
    *lam_min = o[imin] - b_last * std::sqrt(std::max(o[3 * n + rmin], 0.0));
    return GWL_OK;
}

// ---- complex orbitals, k-points, Tamm-Dancoff ---------------------------------
gwl_status gwl_tdc_set_orbitals(gwl_ctx* ctx, const double* psi_v, const double* psi_cq) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_tdc_set_orbitals: not a gwl_tdc_create context");
    if (psi_v == nullptr || psi_cq == nullptr) return ctx->fail(GWL_EINVAL, "gwl_tdc_set_orbitals: NULL input");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const size_t nv = (size_t)ctx->n_k * ctx->n_mu * ctx->nv_k, nc = (size_t)ctx->n_k * ctx->n_mu * ctx->n_c;
    const int64_t ldm = ctx->n_mup, lda = (int64_t)ctx->n_k * ctx->n_cp;
    DevBuf& tmp = ctx->stage;
    CK(tmp.ensure(std::max(nv, nc) * 16, st));
    CK(ctx->phi_c.ensure((size_t)2 * ctx->n_mu * lda * 8, st));                       // psi_cq planar [2][n_mu][n_k n_cp]
    CK(ctx->phi_cT.ensure((size_t)2 * ctx->n_k * ctx->n_c * ldm * 8, st));            // psi_cq^T planar [2][n_k n_c][n_mup]
    CK(ctx->phi_vT.ensure((size_t)2 * ctx->n_kv * ldm * 8, st));                      // psi_v^T planar [2][n_kv][n_mup]
    CK(cudaMemsetAsync(ctx->phi_c.p, 0, ctx->phi_c.bytes, st));
    CK(cudaMemsetAsync(ctx->phi_cT.p, 0, ctx->phi_cT.bytes, st));
    CK(cudaMemsetAsync(ctx->phi_vT.p, 0, ctx->phi_vT.bytes, st));
    CK(cudaMemcpyAsync(tmp.p, psi_cq, nc * 16, cudaMemcpyHostToDevice, st));
    CKL(4, launch_scatter_complex(tmp.as<double>(), ctx->n_k, ctx->n_mu, ctx->n_c, ctx->phi_c.as<double>(),
                                  ctx->phi_c.as<double>() + (int64_t)ctx->n_mu * lda, ctx->n_cp, lda, 1, st));
    CKL(4, launch_scatter_complex(tmp.as<double>(), ctx->n_k, ctx->n_mu, ctx->n_c, ctx->phi_cT.as<double>(),
                                  ctx->phi_cT.as<double>() + (int64_t)ctx->n_k * ctx->n_c * ldm, (int64_t)ctx->n_c * ldm, 1,
                                  ldm, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaMemcpyAsync(tmp.p, psi_v, nv * 16, cudaMemcpyHostToDevice, st));
    CKL(4, launch_scatter_complex(tmp.as<double>(), ctx->n_k, ctx->n_mu, ctx->nv_k, ctx->phi_vT.as<double>(),
                                  ctx->phi_vT.as<double>() + (int64_t)ctx->n_kv * ldm, (int64_t)ctx->nv_k * ldm, 1, ldm, st));
    CK(cudaStreamSynchronize(st));
    ctx->have_orb = true;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_tdc_set_energies(gwl_ctx* ctx, const double* eps_v, const double* eps_cq) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_tdc_set_energies: not a gwl_tdc_create context");
    if (eps_v == nullptr || eps_cq == nullptr) return ctx->fail(GWL_EINVAL, "gwl_tdc_set_energies: NULL input");
    const size_t nv = (size_t)ctx->n_kv, nc = (size_t)ctx->n_k * ctx->n_c;
    double vmax = -INFINITY, cmin = INFINITY;
    for (size_t i = 0; i < nv; ++i) {
        if (!std::isfinite(eps_v[i])) return ctx->fail(GWL_EINVAL, "gwl_tdc_set_energies: non-finite eps_v");
        vmax = std::max(vmax, eps_v[i]);
    }
    for (size_t i = 0; i < nc; ++i) {
        if (!std::isfinite(eps_cq[i])) return ctx->fail(GWL_EINVAL, "gwl_tdc_set_energies: non-finite eps_cq");
        cmin = std::min(cmin, eps_cq[i]);
    }
    if (!(cmin > vmax)) return ctx->fail(GWL_EINVAL, "gwl_tdc_set_energies: need min(eps_cq) > max(eps_v)");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    ctx->h_eps_v.assign(eps_v, eps_v + nv);
    ctx->h_eps_c.assign(eps_cq, eps_cq + nc);
    CK(ctx->eps_v.ensure(nv * 8, st));
    CK(ctx->eps_c.ensure(nc * 8, st));
    CK(ctx->d2.ensure((size_t)ctx->n_vc * 8, st));
    CK(ctx->s.ensure((size_t)ctx->n_vc * 8, st));
    CK(cudaMemcpyAsync(ctx->eps_v.p, eps_v, nv * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->eps_c.p, eps_cq, nc * 8, cudaMemcpyHostToDevice, st));
    CKL(4, launch_build_delta_c(ctx->eps_v.as<double>(), ctx->eps_c.as<double>(), ctx->n_k, ctx->nv_k, ctx->n_c,
                                ctx->d2.as<double>(), ctx->s.as<double>(), st));
    CK(cudaStreamSynchronize(st));
    ctx->have_eps = true;
    invalidate_run(ctx);
    ctx->chain_mode = 0;
    ctx->n_chains_set = 0;
    return GWL_OK;
}

gwl_status gwl_tdc_set_chains(gwl_ctx* ctx, int64_t n_chains, const int32_t* chains) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_tdc_set_chains: not a gwl_tdc_create context");
    if (n_chains < 0 || (n_chains > 0 && chains == nullptr)) return ctx->fail(GWL_EINVAL, "gwl_tdc_set_chains: bad arguments");
    if (!ctx->have_eps) return ctx->fail(GWL_ESTATE, "gwl_tdc_set_chains: energies must be set first");
    const int n_orb = ctx->nv_k + ctx->n_c;
    std::vector<double> eps(n_chains);
    std::vector<int32_t> sgn(n_chains);
    for (int64_t j = 0; j < n_chains; ++j) {
        const int32_t kn = chains[4 * j], n = chains[4 * j + 1], km = chains[4 * j + 2], m = chains[4 * j + 3];
        if (kn < 0 || kn >= ctx->n_k || km < 0 || km >= ctx->n_k || n < 0 || n >= n_orb || m < 0 || m >= n_orb)
            return ctx->fail(GWL_EINVAL, "gwl_tdc_set_chains: k slot or orbital index out of range");
        const bool occ = n < ctx->nv_k;
        eps[j] = occ ? ctx->h_eps_v[(size_t)kn * ctx->nv_k + n] : ctx->h_eps_c[(size_t)kn * ctx->n_c + (n - ctx->nv_k)];
        sgn[j] = occ ? 1 : -1;
    }
    cudaStream_t st = ctx->stream;
    CK(ctx->d_nidx.ensure((size_t)n_chains * 16, st));
    CK(ctx->d_eps_n.ensure((size_t)n_chains * 8, st));
    CK(ctx->d_sgn_n.ensure((size_t)n_chains * 4, st));
    if (n_chains > 0) {
        CK(cudaMemcpyAsync(ctx->d_nidx.p, chains, (size_t)n_chains * 16, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_eps_n.p, eps.data(), (size_t)n_chains * 8, cudaMemcpyHostToDevice, st));
        CK(cudaMemcpyAsync(ctx->d_sgn_n.p, sgn.data(), (size_t)n_chains * 4, cudaMemcpyHostToDevice, st));
    }
    CK(cudaStreamSynchronize(st));
    ctx->chain_mode = 1;
    ctx->n_chains_set = n_chains;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_tdc_matvec(gwl_ctx* ctx, const double* x, double* y, int64_t nvec) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_tdc_matvec: not a gwl_tdc_create context");
    if (nvec < 0) return ctx->fail(GWL_EINVAL, "gwl_tdc_matvec: nvec < 0");
    if (nvec == 0) return GWL_OK;
    if (x == nullptr || y == nullptr) return ctx->fail(GWL_EINVAL, "gwl_tdc_matvec: NULL vector");
    if (!ready(ctx)) return ctx->fail(GWL_ESTATE, "gwl_tdc_matvec: orbitals, energies and kernel must be set");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int chunk = (int)std::min<int64_t>(nvec, 128);
    gwl_status rs = ensure_workspace(ctx, chunk);
    if (rs != GWL_OK) return rs;
    const int64_t n_vc = ctx->n_vc, n_kvc = n_vc / 2;  // n_vc real entries = n_kvc complex ones
    const int64_t ldxs = (int64_t)ctx->n_v * ctx->n_cp;
    CK(ctx->io_x.ensure((size_t)chunk * n_vc * 8, st));  // planar copies
    CK(ctx->io_y.ensure((size_t)chunk * n_vc * 8, st));
    if (!ctx->device_ptrs) CK(ctx->stage.ensure((size_t)chunk * n_vc * 8, st));
    for (int64_t j0 = 0; j0 < nvec; j0 += chunk) {
        const int nb = (int)std::min<int64_t>(chunk, nvec - j0);
        const double* xin = x + j0 * n_vc;
        if (!ctx->device_ptrs) {
            CK(cudaMemcpyAsync(ctx->stage.p, xin, (size_t)nb * n_vc * 8, cudaMemcpyHostToDevice, st));
            xin = ctx->stage.as<double>();
        }
        CKL(4, launch_deinterleave(xin, n_kvc, nb, ctx->io_x.as<double>(), st));
        CKL(4, launch_prescale(ctx->io_x.as<double>(), n_vc, ctx->xs.as<double>(), ldxs, ctx->s.as<double>(), ctx->n_v,
                               ctx->n_c, ctx->n_cp, nb, st));
        rs = apply_casida_core(ctx, ctx->io_x.as<double>(), n_vc, ctx->io_y.as<double>(), n_vc, nb, nullptr, 0);
        if (rs != GWL_OK) return rs;
        if (ctx->device_ptrs) {
            CKL(4, launch_interleave(ctx->io_y.as<double>(), n_kvc, nb, y + j0 * n_vc, st));
        } else {
            CKL(4, launch_interleave(ctx->io_y.as<double>(), n_kvc, nb, ctx->stage.as<double>(), st));
            CK(cudaMemcpyAsync(y + j0 * n_vc, ctx->stage.p, (size_t)nb * n_vc * 8, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
        }
    }
    return GWL_OK;
}

gwl_status gwl_tdc_matvec_rpa(gwl_ctx* ctx, const double* x, const double* y, double* ox, double* oy, int64_t nvec) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_tdc_matvec_rpa: not a gwl_tdc_create context");
    if (nvec < 0) return ctx->fail(GWL_EINVAL, "gwl_tdc_matvec_rpa: nvec < 0");
    if (nvec == 0) return GWL_OK;
    if (x == nullptr || y == nullptr || ox == nullptr || oy == nullptr) return ctx->fail(GWL_EINVAL, "gwl_tdc_matvec_rpa: NULL vector");
    if (!ready(ctx)) return ctx->fail(GWL_ESTATE, "gwl_tdc_matvec_rpa: orbitals, energies and kernel must be set");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int chunk = (int)std::min<int64_t>(nvec, 64);
    gwl_status rs = prpa_workspace(ctx, chunk);
    if (rs != GWL_OK) return rs;
    const int64_t n_vc = ctx->n_vc, n_kvc = n_vc / 2, n4 = 2 * n_vc;
    const int64_t ldxs = (int64_t)ctx->n_v * ctx->n_cp;
    CK(ctx->io_x.ensure((size_t)chunk * n4 * 8, st));
    CK(ctx->io_y.ensure((size_t)chunk * n4 * 8, st));
    if (!ctx->device_ptrs) CK(ctx->stage.ensure((size_t)2 * chunk * n_vc * 8, st));
    for (int64_t j0 = 0; j0 < nvec; j0 += chunk) {
        const int nb = (int)std::min<int64_t>(chunk, nvec - j0);
        const double* xin = x + j0 * n_vc;
        const double* yin = y + j0 * n_vc;
        double* stage = ctx->stage.as<double>();
        if (!ctx->device_ptrs) {
            CK(cudaMemcpyAsync(stage, xin, (size_t)nb * n_vc * 8, cudaMemcpyHostToDevice, st));
            CK(cudaMemcpyAsync(stage + (int64_t)chunk * n_vc, yin, (size_t)nb * n_vc * 8, cudaMemcpyHostToDevice, st));
            xin = stage;
            yin = stage + (int64_t)chunk * n_vc;
        }
        CKL(4, launch_prpa_pack(xin, yin, n_kvc, nb, ctx->io_x.as<double>(), st));
        CKL(4, launch_prescale(ctx->io_x.as<double>(), n_vc, ctx->xs.as<double>(), ldxs, ctx->s.as<double>(), ctx->n_v, ctx->n_c,
                               ctx->n_cp, 2 * nb, st));
        rs = prpa_apply(ctx, ctx->io_x.as<double>(), ctx->io_y.as<double>(), nb);
        if (rs != GWL_OK) return rs;
        if (ctx->device_ptrs) {
            CKL(4, launch_prpa_unpack(ctx->io_y.as<double>(), n_kvc, nb, ox + j0 * n_vc, oy + j0 * n_vc, st));
        } else {
            CKL(4, launch_prpa_unpack(ctx->io_y.as<double>(), n_kvc, nb, stage, stage + (int64_t)chunk * n_vc, st));
            CK(cudaMemcpyAsync(ox + j0 * n_vc, stage, (size_t)nb * n_vc * 8, cudaMemcpyDeviceToHost, st));
            CK(cudaMemcpyAsync(oy + j0 * n_vc, stage + (int64_t)chunk * n_vc, (size_t)nb * n_vc * 8, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
        }
    }
    return GWL_OK;
}

// ---- SURVEY.md 8(f)-4, second part: point-group symmetry blocks of C (reading Q25) -----------------
gwl_status gwl_sym_create(gwl_ctx** out, int n_gen, const int32_t* nv_irrep, const int32_t* nc_irrep, int64_t n_mu_w) {
    if (out == nullptr) return GWL_EINVAL;
    *out = nullptr;
    if (n_gen < 0 || n_gen > 3 || nv_irrep == nullptr || nc_irrep == nullptr || n_mu_w < 1) return GWL_EINVAL;
    const int g = 1 << n_gen;
    int64_t nv = 0, nc = 0, ncp = 0;
    for (int a = 0; a < g; ++a) {
        if (nv_irrep[a] < 0 || nc_irrep[a] < 0) return GWL_EINVAL;
        nv += nv_irrep[a];
        nc += nc_irrep[a];
        ncp += round_up(nc_irrep[a], BK);
    }
    if (nv < 1 || nc < 1) return GWL_EINVAL;
    gwl_status rs = create_common(out, 1, nv, ncp, n_mu_w, false, 1);
    if (rs != GWL_OK) return rs;
    gwl_ctx* ctx = *out;
    ctx->sym = true;
    ctx->sym_g = g;
    ctx->sym_nv_tot = (int)nv;
    ctx->sym_nc_tot = (int)nc;
    ctx->sym_ncp_tot = (int)ncp;
    int vo = 0, co = 0, cpo = 0;
    for (int a = 0; a < g; ++a) {
        ctx->sym_nv[a] = nv_irrep[a];
        ctx->sym_nc[a] = nc_irrep[a];
        ctx->sym_ncp[a] = (int)round_up(nc_irrep[a], BK);
        ctx->sym_voff[a] = vo;
        ctx->sym_coff[a] = co;
        ctx->sym_cpoff[a] = cpo;
        vo += nv_irrep[a];
        co += nc_irrep[a];
        cpo += ctx->sym_ncp[a];
    }
    return GWL_OK;
}

gwl_status gwl_sym_set_orbitals(gwl_ctx* ctx, const double* phi_v_w, const double* phi_c_w) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_sym_set_orbitals: not a gwl_sym_create context");
    if (phi_v_w == nullptr || phi_c_w == nullptr) return ctx->fail(GWL_EINVAL, "gwl_sym_set_orbitals: NULL input");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int n_w = ctx->n_mu, nv = ctx->sym_nv_tot, nc = ctx->sym_nc_tot, ncp = ctx->sym_ncp_tot;
    const int64_t ldm = ctx->n_mup;
    DevBuf& tmp = ctx->stage;
    CK(tmp.ensure(((size_t)n_w * nv + (size_t)n_w * nc) * 8, st));
    double* dv = tmp.as<double>();
    double* dc = dv + (size_t)n_w * nv;
    CK(cudaMemcpyAsync(dv, phi_v_w, (size_t)n_w * nv * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(dc, phi_c_w, (size_t)n_w * nc * 8, cudaMemcpyHostToDevice, st));
    CK(ctx->phi_c.ensure((size_t)n_w * ncp * 8, st));    // [n_w][ncp_tot]: every irrep's columns padded to 16 with zero orbitals
    CK(ctx->phi_cT.ensure((size_t)ncp * ldm * 8, st));   // [ncp_tot][n_mup]
    CK(ctx->phi_vT.ensure((size_t)nv * ldm * 8, st));
    CK(cudaMemsetAsync(ctx->phi_c.p, 0, ctx->phi_c.bytes, st));
    CK(cudaMemsetAsync(ctx->phi_cT.p, 0, ctx->phi_cT.bytes, st));
    CK(cudaMemsetAsync(ctx->phi_vT.p, 0, ctx->phi_vT.bytes, st));
    for (int b = 0; b < ctx->sym_g; ++b) {
        if (ctx->sym_nc[b] == 0) continue;
        CK(cudaMemcpy2DAsync(ctx->phi_c.as<double>() + ctx->sym_cpoff[b], (size_t)ncp * 8, dc + ctx->sym_coff[b], (size_t)nc * 8,
                             (size_t)ctx->sym_nc[b] * 8, (size_t)n_w, cudaMemcpyDeviceToDevice, st));
    }
    CKL(4, launch_transpose(ctx->phi_c.as<double>(), n_w, ncp, ctx->phi_cT.as<double>(), ldm, st));
    CKL(4, launch_transpose(dv, n_w, nv, ctx->phi_vT.as<double>(), ldm, st));
    CK(cudaStreamSynchronize(st));
    ctx->have_orb = true;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_sym_set_kernel(gwl_ctx* ctx, const double* V_wf) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_sym_set_kernel: not a gwl_sym_create context");
    if (V_wf == nullptr) return ctx->fail(GWL_EINVAL, "gwl_sym_set_kernel: NULL input");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int n_w = ctx->n_mu, g = ctx->sym_g;
    const size_t n_in = (size_t)n_w * g * n_w;
    CK(ctx->stage.ensure(n_in * 8, st));
    CK(cudaMemcpyAsync(ctx->stage.p, V_wf, n_in * 8, cudaMemcpyHostToDevice, st));
    CK(ctx->V.ensure((size_t)g * n_w * ctx->n_mup * 8, st));
    CK(cudaMemsetAsync(ctx->V.p, 0, ctx->V.bytes, st));
    CKL(4, launch_sym_reduce_kernel(ctx->stage.as<double>(), n_w, g, ctx->V.as<double>(), ctx->n_mup, st));
    CK(cudaStreamSynchronize(st));
    ctx->have_V = true;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_sym_select(gwl_ctx* ctx, int gamma, int64_t* n_pairs) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_sym_select: not a gwl_sym_create context");
    if (gamma < 0 || gamma >= ctx->sym_g) return ctx->fail(GWL_EINVAL, "gwl_sym_select: no such irreducible representation");
    if (!ctx->have_eps) return ctx->fail(GWL_ESTATE, "gwl_sym_select: energies must be set first");
    int64_t npad = 0, napi = 0;
    int64_t vecoff[8], apioff[8];
    for (int a = 0; a < ctx->sym_g; ++a) {
        const int b = a ^ gamma;
        vecoff[a] = npad;
        apioff[a] = napi;
        npad += (int64_t)ctx->sym_nv[a] * ctx->sym_ncp[b];
        napi += (int64_t)ctx->sym_nv[a] * ctx->sym_nc[b];
    }
    if (n_pairs != nullptr) *n_pairs = napi;
    if (napi == 0) return ctx->fail(GWL_EINVAL, "gwl_sym_select: this block has no pairs");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    CK(cudaStreamSynchronize(st));
    ctx->sym_gamma = gamma;
    ctx->sym_npairs = napi;
    for (int a = 0; a < ctx->sym_g; ++a) {
        ctx->sym_vecoff[a] = vecoff[a];
        ctx->sym_apioff[a] = apioff[a];
    }
    ctx->n_c = ctx->n_cp = BK;  // the vector kernels see ONE padded block vector whose K.X copy has the same layout
    ctx->n_v = (int)(npad / BK);
    ctx->n_vc = npad;
    ctx->v_sel = (int64_t)gamma * ctx->n_mu * ctx->n_mup;
    CK(ctx->d2.ensure((size_t)npad * 8, st));
    CK(ctx->s.ensure((size_t)npad * 8, st));
    for (int a = 0; a < ctx->sym_g; ++a) {
        const int b = a ^ gamma;
        CKL(4, launch_sym_build_delta(ctx->eps_v.as<double>() + ctx->sym_voff[a], ctx->eps_c.as<double>() + ctx->sym_coff[b],
                                      ctx->sym_nv[a], ctx->sym_nc[b], ctx->sym_ncp[b], ctx->d2.as<double>() + vecoff[a],
                                      ctx->s.as<double>() + vecoff[a], st));
    }
    CK(cudaStreamSynchronize(st));
    invalidate_run(ctx);
    ctx->chain_mode = 0;
    ctx->n_chains_set = 0;
    return GWL_OK;
}

gwl_status gwl_sym_matvec(gwl_ctx* ctx, const double* x, double* y, int64_t nvec) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_sym_matvec: not a gwl_sym_create context");
    if (nvec < 0) return ctx->fail(GWL_EINVAL, "gwl_sym_matvec: nvec < 0");
    if (nvec == 0) return GWL_OK;
    if (x == nullptr || y == nullptr) return ctx->fail(GWL_EINVAL, "gwl_sym_matvec: NULL vector");
    if (!ready(ctx) || ctx->sym_gamma < 0) return ctx->fail(GWL_ESTATE, "gwl_sym_matvec: orbitals, energies, kernel and a selected block are needed");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int chunk = (int)std::min<int64_t>(nvec, 256);
    gwl_status rs = ensure_workspace(ctx, chunk);
    if (rs != GWL_OK) return rs;
    const int64_t npad = ctx->n_vc, napi = ctx->sym_npairs;
    CK(ctx->io_x.ensure((size_t)chunk * npad * 8, st));
    CK(ctx->io_y.ensure((size_t)chunk * npad * 8, st));
    if (!ctx->device_ptrs) CK(ctx->stage.ensure((size_t)chunk * napi * 8, st));
    for (int64_t j0 = 0; j0 < nvec; j0 += chunk) {
        const int nb = (int)std::min<int64_t>(chunk, nvec - j0);
        double* api = const_cast<double*>(x) + j0 * napi;
        if (!ctx->device_ptrs) {
            CK(cudaMemcpyAsync(ctx->stage.p, x + j0 * napi, (size_t)nb * napi * 8, cudaMemcpyHostToDevice, st));
            api = ctx->stage.as<double>();
        }
        for (int a = 0; a < ctx->sym_g; ++a) {
            const int b = a ^ ctx->sym_gamma;
            CKL(4, launch_sym_copy_rect(api + ctx->sym_apioff[a], napi, ctx->io_x.as<double>() + ctx->sym_vecoff[a], npad,
                                        ctx->sym_nv[a], ctx->sym_nc[b], ctx->sym_ncp[b], nb, 0, st));
        }
        CKL(4, launch_prescale(ctx->io_x.as<double>(), npad, ctx->xs.as<double>(), npad, ctx->s.as<double>(), ctx->n_v, ctx->n_c,
                               ctx->n_cp, nb, st));
        rs = apply_casida_core(ctx, ctx->io_x.as<double>(), npad, ctx->io_y.as<double>(), npad, nb, nullptr, 0);
        if (rs != GWL_OK) return rs;
        double* out = ctx->device_ptrs ? y + j0 * napi : ctx->stage.as<double>();
        for (int a = 0; a < ctx->sym_g; ++a) {
            const int b = a ^ ctx->sym_gamma;
            CKL(4, launch_sym_copy_rect(out + ctx->sym_apioff[a], napi, ctx->io_y.as<double>() + ctx->sym_vecoff[a], npad,
                                        ctx->sym_nv[a], ctx->sym_nc[b], ctx->sym_ncp[b], nb, 1, st));
        }
        if (!ctx->device_ptrs) {
            CK(cudaMemcpyAsync(y + j0 * napi, ctx->stage.p, (size_t)nb * napi * 8, cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
        }
    }
    return GWL_OK;
}

gwl_status gwl_sym_selfenergy_state(gwl_ctx* ctx, int32_t m_idx, int64_t steps, int64_t block, int reorth, const double* omega,
                                    int64_t n_omega, double eta, double* sigma_mm) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_sym_selfenergy_state: not a gwl_sym_create context");
    if (sigma_mm == nullptr || omega == nullptr || n_omega < 1) return ctx->fail(GWL_EINVAL, "gwl_sym_selfenergy_state: bad arguments");
    const int nv = ctx->sym_nv_tot, n_orb = nv + ctx->sym_nc_tot;
    if (m_idx < 0 || m_idx >= n_orb) return ctx->fail(GWL_EINVAL, "gwl_sym_selfenergy_state: orbital index out of range");
    auto irrep_of = [&](int idx) {
        const bool occ = idx < nv;
        const int loc = occ ? idx : idx - nv;
        const int* off = occ ? ctx->sym_voff : ctx->sym_coff;
        const int* cnt = occ ? ctx->sym_nv : ctx->sym_nc;
        int a = 0;
        while (a + 1 < ctx->sym_g && loc >= off[a] + cnt[a]) ++a;
        return a;
    };
    const int gm = irrep_of(m_idx);
    bool first = true;
    gwl_status rs = GWL_OK;
    for (int gamma = 0; gamma < ctx->sym_g && rs == GWL_OK; ++gamma) {
        std::vector<int32_t> n_idx;
        for (int n = 0; n < n_orb; ++n)
            if ((irrep_of(n) ^ gm) == gamma) n_idx.push_back(n);
        if (n_idx.empty()) continue;
        int64_t npairs = -1;
        rs = gwl_sym_select(ctx, gamma, &npairs);
        if (rs != GWL_OK) {
            if (npairs == 0) {  // no excitation carries this symmetry: these chains contribute nothing
                rs = GWL_OK;
                continue;
            }
            break;
        }
        std::vector<int32_t> m_rep(n_idx.size(), m_idx);
        rs = gwl_set_chains(ctx, (int64_t)n_idx.size(), n_idx.data(), m_rep.data());
        if (rs == GWL_OK) rs = gwl_lanczos(ctx, (int64_t)n_idx.size(), steps, block, reorth, nullptr, nullptr, nullptr, nullptr);
        if (rs != GWL_OK) break;
        ctx->sig_accumulate = !first;
        rs = gwl_selfenergy(ctx, omega, n_omega, eta, nullptr, sigma_mm);
        ctx->sig_accumulate = false;
        first = false;
    }
    if (rs == GWL_OK && first) return ctx->fail(GWL_EINVAL, "gwl_sym_selfenergy_state: no symmetry block has pairs");
    return rs;
}

// ---- ISDF front end (PAPER.md:115-128, Eq. 15-17; :319) ---------------------------------------------
gwl_status gwl_isdf_build(gwl_ctx* ctx, int64_t n_r, const double* phi_v_grid, const double* phi_c_grid, const double* r,
                          double weight, double soft, const int32_t* idx, double* zeta_t, double* V_out) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_isdf_build: real-orbital call on a complex (gwl_tdc_create) context");
    if (ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_isdf_build: symmetry-block (gwl_sym_create) context: not available on a symmetry-block context");
    if (phi_v_grid == nullptr || phi_c_grid == nullptr || r == nullptr || idx == nullptr)
        return ctx->fail(GWL_EINVAL, "gwl_isdf_build: NULL input");
    if (n_r < ctx->n_mu || n_r > 65535 || !(weight > 0.0) || !(soft > 0.0))
        return ctx->fail(GWL_EINVAL, "gwl_isdf_build: need n_mu <= n_r <= 65535, weight > 0, soft > 0");
    const int n_mu = ctx->n_mu, n_orb = ctx->n_v + ctx->n_c, nr = (int)n_r;
    {
        std::vector<char> seen((size_t)n_r, 0);
        for (int m = 0; m < n_mu; ++m) {
            if (idx[m] < 0 || idx[m] >= n_r || seen[idx[m]])
                return ctx->fail(GWL_EINVAL, "gwl_isdf_build: interpolation point index out of range or repeated");
            seen[idx[m]] = 1;
        }
    }
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int64_t nop = round_up(n_orb, BK), nrp = round_up(n_r, BK), ldm = ctx->n_mup;
    DevBuf &Phi = ctx->isdf_phi, &PhiMu = ctx->isdf_phimu, &Y = ctx->isdf_y, &S = ctx->isdf_s, &G = ctx->isdf_g, &U = ctx->isdf_u;
    CK(Phi.ensure((size_t)n_r * nop * 8, st));
    CK(PhiMu.ensure((size_t)n_mu * nop * 8 + (size_t)n_mu * n_orb * 8, st));
    CK(Y.ensure((size_t)n_mu * nrp * 8, st));
    CK(S.ensure((size_t)n_mu * ldm * 8 + (size_t)n_r * 24 + 8 + (size_t)n_mu * 4 + 16, st));
    CK(G.ensure((size_t)n_r * nrp * 8, st));
    CK(U.ensure((size_t)n_mu * nrp * 8, st));
    CK(ctx->V.ensure((size_t)n_mu * ldm * 8, st));
    CK(cudaMemsetAsync(Phi.p, 0, Phi.bytes, st));
    CK(cudaMemsetAsync(PhiMu.p, 0, PhiMu.bytes, st));
    CK(cudaMemsetAsync(Y.p, 0, Y.bytes, st));
    CK(cudaMemsetAsync(S.p, 0, S.bytes, st));
    CK(cudaMemsetAsync(G.p, 0, G.bytes, st));
    CK(cudaMemsetAsync(U.p, 0, U.bytes, st));
    CK(cudaMemsetAsync(ctx->V.p, 0, ctx->V.bytes, st));
    double* dS = S.as<double>();
    double* d_r = dS + (size_t)n_mu * ldm;
    double* d_scale = d_r + (size_t)n_r * 3;
    int32_t* d_idx = reinterpret_cast<int32_t*>(d_scale + 1);
    int* d_info = d_idx + n_mu;
    // all orbitals side by side, [n_r][v | c], zero-padded to a multiple of 16 columns
    CK(cudaMemcpy2DAsync(Phi.p, (size_t)nop * 8, phi_v_grid, (size_t)ctx->n_v * 8, (size_t)ctx->n_v * 8, (size_t)n_r,
                         cudaMemcpyHostToDevice, st));
    CK(cudaMemcpy2DAsync(Phi.as<double>() + ctx->n_v, (size_t)nop * 8, phi_c_grid, (size_t)ctx->n_c * 8, (size_t)ctx->n_c * 8,
                         (size_t)n_r, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(d_r, r, (size_t)n_r * 24, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(d_idx, idx, (size_t)n_mu * 4, cudaMemcpyHostToDevice, st));
    CKL(4, launch_gather_rows(Phi.as<double>(), nop, (int)nop, d_idx, n_mu, PhiMu.as<double>(), nop, st));
    // P[mu][r] = sum_n phi_n(r_mu) phi_n(r);  Z C^T = P o P (pairs of ALL orbitals);  C C^T = its columns at the points
    gwl_status rs = plain_gemm(ctx, Phi.as<double>(), nop, PhiMu.as<double>(), nop, nr, n_mu, (int)(nop / BK), Y.as<double>(),
                               nrp, 1);
    if (rs != GWL_OK) return rs;
    CKL(4, launch_hadamard(Y.as<double>(), Y.as<double>(), (int64_t)n_mu * nrp, st));
    CKL(4, launch_gather_cols(Y.as<double>(), nrp, d_idx, n_mu, dS, ldm, st));
    // zeta^T = (C C^T)^{-1} (Z C^T)^T by Cholesky
    CKL(4, launch_cholesky(dS, ldm, n_mu, d_scale, d_info, st));
    int h_info = 0;
    CK(cudaMemcpyAsync(&h_info, d_info, 4, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (h_info != 0)
        return ctx->fail(GWL_EINVAL, "gwl_isdf_build: C C^T is not positive definite (pivot " + std::to_string(h_info) +
                                         "): the interpolation points do not resolve the pair products");
    CKL(4, launch_cholesky_solve(dS, ldm, n_mu, Y.as<double>(), nrp, nr, st));
    // (alpha|beta) = zeta^T G zeta with the Coulomb quadrature matrix of the grid
    CKL(4, launch_coulomb_grid(d_r, nr, weight, soft, G.as<double>(), nrp, st));
    rs = plain_gemm(ctx, G.as<double>(), nrp, Y.as<double>(), nrp, nr, n_mu, (int)(nrp / BK), U.as<double>(), nrp, 1);
    if (rs != GWL_OK) return rs;
    rs = plain_gemm(ctx, Y.as<double>(), nrp, U.as<double>(), nrp, n_mu, n_mu, (int)(nrp / BK), ctx->V.as<double>(), ldm, 1);
    if (rs != GWL_OK) return rs;
    // the orbitals at the interpolation points become the context's orbitals
    double* compact = PhiMu.as<double>() + (size_t)n_mu * nop;  // [n_mu][n_v] then [n_mu][n_c]
    CK(cudaMemcpy2DAsync(compact, (size_t)ctx->n_v * 8, PhiMu.p, (size_t)nop * 8, (size_t)ctx->n_v * 8, (size_t)n_mu,
                         cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpy2DAsync(compact + (size_t)n_mu * ctx->n_v, (size_t)ctx->n_c * 8, PhiMu.as<double>() + ctx->n_v, (size_t)nop * 8,
                         (size_t)ctx->n_c * 8, (size_t)n_mu, cudaMemcpyDeviceToDevice, st));
    rs = install_orbitals(ctx, compact, compact + (size_t)n_mu * ctx->n_v);
    if (rs != GWL_OK) return rs;
    if (zeta_t != nullptr)
        CK(cudaMemcpy2DAsync(zeta_t, (size_t)n_r * 8, Y.p, (size_t)nrp * 8, (size_t)n_r * 8, (size_t)n_mu, cudaMemcpyDeviceToHost,
                             st));
    if (V_out != nullptr)
        CK(cudaMemcpy2DAsync(V_out, (size_t)n_mu * 8, ctx->V.p, (size_t)ldm * 8, (size_t)n_mu * 8, (size_t)n_mu,
                             cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    ctx->have_orb = true;
    ctx->have_V = true;
    invalidate_run(ctx);
    return GWL_OK;
}

gwl_status gwl_isdf_select_points(gwl_ctx* ctx, int64_t n_r, const double* r, const double* weight, const int32_t* init_idx,
                                  int64_t max_iters, int32_t* idx, int32_t* iters_done) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (r == nullptr || weight == nullptr || init_idx == nullptr || idx == nullptr)
        return ctx->fail(GWL_EINVAL, "gwl_isdf_select_points: NULL argument");
    const int n_mu = ctx->n_mu;
    if (n_r < n_mu || n_r > (1 << 30) || max_iters < 0 || max_iters > 100000)
        return ctx->fail(GWL_EINVAL, "gwl_isdf_select_points: need n_mu <= n_r and 0 <= max_iters <= 100000");
    for (int m = 0; m < n_mu; ++m)
        if (init_idx[m] < 0 || init_idx[m] >= n_r) return ctx->fail(GWL_EINVAL, "gwl_isdf_select_points: init_idx out of range");
    LaunchScope ls(ctx);
    cudaStream_t st = ctx->stream;
    const int nr = (int)n_r;
    // scratch in isdf_s: r [n_r][3], w [n_r], c [n_mu][3], assign [n_r], idx [n_mu], changed
    DevBuf& buf = ctx->isdf_s;
    CK(buf.ensure((size_t)n_r * 32 + (size_t)n_mu * 24 + (size_t)n_r * 4 + (size_t)n_mu * 4 + 16, st));
    double* d_r = buf.as<double>();
    double* d_w = d_r + (size_t)n_r * 3;
    double* d_c = d_w + n_r;
    int32_t* d_assign = reinterpret_cast<int32_t*>(d_c + (size_t)n_mu * 3);
    int32_t* d_idx = d_assign + n_r;
    int* d_changed = d_idx + n_mu;
    std::vector<double> c0((size_t)n_mu * 3);
    for (int m = 0; m < n_mu; ++m)
        for (int q = 0; q < 3; ++q) c0[3 * (size_t)m + q] = r[3 * (size_t)init_idx[m] + q];
    CK(cudaMemcpyAsync(d_r, r, (size_t)n_r * 24, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(d_w, weight, (size_t)n_r * 8, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(d_c, c0.data(), (size_t)n_mu * 24, cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(d_assign, 0xff, (size_t)n_r * 4, st));  // -1: the first assignment always counts as a change
    int done = 0;
    for (int it = 0; it < max_iters; ++it) {
        int changed = 0;
        CK(cudaMemsetAsync(d_changed, 0, 4, st));
        CKL(4, launch_cvt_assign(d_r, nr, d_c, n_mu, d_assign, d_changed, st));
        CK(cudaMemcpyAsync(&changed, d_changed, 4, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));  // a set-up step: the host decides whether Lloyd has converged
        if (!changed) break;
        CKL(4, launch_cvt_update(d_r, d_w, nr, d_assign, n_mu, d_c, st));
        done = it + 1;
    }
    CK(cudaMemsetAsync(d_changed, 0, 4, st));
    CKL(4, launch_cvt_assign(d_r, nr, d_c, n_mu, d_assign, d_changed, st));
    CKL(4, launch_cvt_snap(d_r, nr, d_assign, d_c, n_mu, d_idx, st));
    CK(cudaMemcpyAsync(idx, d_idx, (size_t)n_mu * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (iters_done != nullptr) *iters_done = done;
    return GWL_OK;
}

gwl_status gwl_get_timing(gwl_ctx* ctx, double* ms_matvec, double* ms_vecops, double* ms_total) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    double tm = 0.0, tv = 0.0;
    for (size_t i = 0; i + 2 < ctx->ev_used; i += 3) {
        float a = 0.f, b = 0.f;
        CK(cudaEventElapsedTime(&a, ctx->ev[i], ctx->ev[i + 1]));
        CK(cudaEventElapsedTime(&b, ctx->ev[i + 1], ctx->ev[i + 2]));
        tm += a;
        tv += b;
    }
    if (ms_matvec) *ms_matvec = tm;
    if (ms_vecops) *ms_vecops = tv;
    if (ms_total) *ms_total = tm + tv;
    return GWL_OK;
}

gwl_status gwl_set_profiling(gwl_ctx* ctx, int level) {
    if (ctx == nullptr || level < 0 || level > 2) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    ctx->prof_level = level;
    return GWL_OK;
}

gwl_status gwl_get_kernel_times(gwl_ctx* ctx, double* ms, int64_t* count) {
    if (ctx == nullptr || ms == nullptr || count == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < GWL_N_KERNEL_CLASSES; ++i) {
        ms[i] = 0.0;
        count[i] = 0;
    }
    for (size_t i = 0; i < ctx->kev_class.size() && 2 * i + 1 < ctx->kev_used; ++i) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, ctx->kev[2 * i], ctx->kev[2 * i + 1]));
        ms[ctx->kev_class[i]] += t;
        count[ctx->kev_class[i]] += 1;
    }
    return GWL_OK;
}

gwl_status gwl_get_launch_count(gwl_ctx* ctx, int64_t* n_launches) {
    if (ctx == nullptr || n_launches == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    *n_launches = ctx->launches;
    return GWL_OK;
}

gwl_status gwl_probe_fp64_peak(int kind, double* tflops) {
    if (tflops == nullptr || (kind != 0 && kind != 1)) return GWL_EINVAL;
    cudaError_t e = probe_fp64_peak(kind, tflops);
    return e == cudaSuccess ? GWL_OK : GWL_ECUDA;
}

}  // extern "C"
