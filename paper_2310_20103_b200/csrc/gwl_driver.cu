// Host driver of libgwl: the three contractions of the Casida product for real, complex and symmetry-block contexts (each with
// its split-K reduction where the planner asks for one), the start vectors, and the pseudo-Hermitian RPA Lanczos driver.
#include "gwl_ctx.h"

namespace gwl {

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
                    int dot_stride, const ChebTerm* cheb) {
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

gwl_status create_common(gwl_ctx** out, int64_t n_k, int64_t n_v, int64_t n_c, int64_t n_mu, bool cplx, int64_t n_q) {
    if (out == nullptr) return GWL_EINVAL;
    *out = nullptr;
    if (n_v < 1 || n_c < 1 || n_mu < 1 || n_k < 1 || n_q < 1 || n_k > 4096 || n_k * n_v > (1 << 20) || n_c > (1 << 20) ||
        n_mu > (1 << 24))
        return GWL_EINVAL;
    // the complex Khatri-Rao GEMMs index the (k, v) planes through grid.z (kr_gemm_c.cu): reject here, where the caller can
    // see why, instead of failing every later product with an opaque CUDA error (include/gwl.h states the limit)
    if (cplx && n_k * n_v > GWL_TDC_MAX_KV) return GWL_EINVAL;
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

// Orbitals at the fitting points from compact DEVICE arrays d_phi_v [n_mu][n_v], d_phi_c [n_mu][n_c]: the padded and
// transposed copies the GEMMs read
gwl_status install_orbitals(gwl_ctx* ctx, const double* d_phi_v, const double* d_phi_c) {
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

}  // namespace gwl
