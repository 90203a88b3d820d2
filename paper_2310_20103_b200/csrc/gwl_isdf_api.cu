// C ABI, ISDF front end (gwl_isdf_*): host driver around the kernels of isdf.cu.
#include "gwl_ctx.h"

using namespace gwl;

extern "C" {

// ---- ISDF front end (PAPER.md:115-128, Eq. 15-17; :319) ---------------------------------------------
gwl_status gwl_isdf_build(gwl_ctx* ctx, int64_t n_r, const double* phi_v_grid, const double* phi_c_grid, const double* r,
                          double weight, double soft, const int32_t* idx, double* zeta_t, double* V_out) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_isdf_build: real-orbital call on a complex (gwl_tdc_create) context");
    if (ctx->sym) return ctx->fail(GWL_ESTATE, "gwl_isdf_build: symmetry-block (gwl_sym_create) context: not available on a symmetry-block context");
    if (phi_v_grid == nullptr || phi_c_grid == nullptr || r == nullptr || idx == nullptr)
        return ctx->fail(GWL_EINVAL, "gwl_isdf_build: NULL input");
    if (n_r < ctx->n_mu || n_r > GWL_ISDF_MAX_NR || !(weight > 0.0) || !(soft > 0.0))
        return ctx->fail(GWL_EINVAL, "gwl_isdf_build: need n_mu <= n_r <= GWL_ISDF_MAX_NR (4 194 304), weight > 0, soft > 0");
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
    // G also stages the finished (alpha|beta): the context's own V and orbitals are only touched once every step that can
    // fail on the inputs (a singular C C^T) has passed, so a failed build leaves a ready context exactly as it was.
    const size_t v_bytes = (size_t)n_mu * ldm * 8;
    // The Coulomb quadrature matrix is walked in row panels of G_PANEL rows: memory scales as N_r N_mu, not N_r^2.
    constexpr int G_PANEL = 8192;
    const int g_rows = std::min(nr, G_PANEL);
    CK(G.ensure(std::max((size_t)g_rows * nrp * 8, v_bytes), st));
    CK(U.ensure((size_t)n_mu * nrp * 8, st));
    CK(cudaMemsetAsync(Phi.p, 0, Phi.bytes, st));
    CK(cudaMemsetAsync(PhiMu.p, 0, PhiMu.bytes, st));
    CK(cudaMemsetAsync(Y.p, 0, Y.bytes, st));
    CK(cudaMemsetAsync(S.p, 0, S.bytes, st));
    CK(cudaMemsetAsync(G.p, 0, G.bytes, st));
    CK(cudaMemsetAsync(U.p, 0, U.bytes, st));
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
    // U[mu][i] = sum_j G[i][j] zeta_mu(r_j), panel of rows i by panel (G is symmetric; each panel is generated, used, dropped;
    // the padding columns n_r .. nrp of a panel stay zero from the memset above, no kernel writes them)
    for (int i0 = 0; i0 < nr; i0 += G_PANEL) {
        const int rows = std::min(G_PANEL, nr - i0);
        CKL(4, launch_coulomb_grid(d_r, nr, i0, rows, weight, soft, G.as<double>(), nrp, st));
        rs = plain_gemm(ctx, G.as<double>(), nrp, Y.as<double>(), nrp, rows, n_mu, (int)(nrp / BK), U.as<double>() + i0, nrp, 1);
        if (rs != GWL_OK) return rs;
    }
    CK(cudaMemsetAsync(G.p, 0, v_bytes, st));  // G itself is consumed; its head becomes the staging copy of V (zero padding)
    rs = plain_gemm(ctx, Y.as<double>(), nrp, U.as<double>(), nrp, n_mu, n_mu, (int)(nrp / BK), G.as<double>(), ldm, 1);
    if (rs != GWL_OK) return rs;
    // Commit.  From here on only a CUDA failure can stop the call; if one does, the context is left "not ready"
    // (GWL_ESTATE from the next product) instead of holding a kernel and orbitals that do not belong together.
    struct CommitGuard {
        gwl_ctx* c;
        bool done = false;
        ~CommitGuard() {
            if (!done) {
                c->have_V = false;
                c->have_orb = false;
                invalidate_run(c);
            }
        }
    } commit{ctx};
    CK(ctx->V.ensure(v_bytes, st));
    CK(cudaMemcpyAsync(ctx->V.p, G.p, v_bytes, cudaMemcpyDeviceToDevice, st));
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
    commit.done = true;
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

}  // extern "C"
