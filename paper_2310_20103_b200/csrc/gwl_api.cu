// C ABI of libgwl (include/gwl.h): context, input staging, and the host driver that strings the kernels
// together.  There is no host<->device traffic and no host synchronisation inside the Lanczos step loop:
// alpha/beta/len live on the device and are copied out once at the end.
#include "gwl_ctx.h"

using namespace gwl;

extern "C" {

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

// Least-squares fit of sqrt(x) at the M = 4 (g + 1) first-kind Chebyshev nodes of [lo, hi] (
// DESIGN.md Q13).  In the Chebyshev basis the normal equations are diagonal -- sum_k T_i(t_k) T_j(t_k) = (M/2) delta_ij
// (M for i = j = 0) on the nodes t_k = cos(pi (k + 1/2) / M) -- so c_j = (2/M) sum_k sqrt(x_k) cos(j theta_k), c_0 halved.
// Host arithmetic only: no context, no device.
gwl_status gwl_fit_sqrt_polynomial(int g, double lo, double hi, double* cheb) {
    if (cheb == nullptr || g < 1 || g > 64 || !(lo > 0.0) || !(hi > lo) || !std::isfinite(hi)) return GWL_EINVAL;
    const int M = 4 * (g + 1);
    const double pi = 3.14159265358979323846;
    std::vector<double> f((size_t)M), th((size_t)M);
    for (int k = 0; k < M; ++k) {
        th[k] = pi * (k + 0.5) / M;
        f[k] = std::sqrt(0.5 * (hi + lo) + 0.5 * (hi - lo) * std::cos(th[k]));
    }
    for (int j = 0; j <= g; ++j) {
        double acc = 0.0;
        for (int k = 0; k < M; ++k) acc += f[k] * std::cos(j * th[k]);
        cheb[j] = (j == 0 ? 1.0 : 2.0) * acc / M;
    }
    return GWL_OK;
}

// Fitting range of p_g.  steps = 0: the paper's heuristic [0.8 min Delta^2, 1.25 max Delta^2] (reading Q12).
// steps >= 2: lo as before (a true lower bound of C when V is positive semidefinite), hi = (1 + margin) max(Lanczos
// estimate of gwl_spectrum_bounds, max Delta^2) (reading Q23: the heuristic upper end is not a bound once the coupling is
// strong).  The margin is a cushion for an unconverged top Ritz value, not a guarantee.
gwl_status gwl_sqrt_fit_range(gwl_ctx* ctx, int64_t steps, double margin, double* lo, double* hi) {
    if (ctx == nullptr) return GWL_EINVAL;
    if (lo == nullptr || hi == nullptr || !(margin >= 0.0) || steps < 0 || steps == 1)
        return ctx->fail(GWL_EINVAL, "gwl_sqrt_fit_range: need lo, hi != NULL, margin >= 0 and steps = 0 or >= 2");
    if (ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_sqrt_fit_range: the polynomial square root applies to real-orbital contexts");
    if (!ctx->have_eps || ctx->h_eps_v.empty() || ctx->h_eps_c.empty())
        return ctx->fail(GWL_ESTATE, "gwl_sqrt_fit_range: energies must be set");
    const double v_min = *std::min_element(ctx->h_eps_v.begin(), ctx->h_eps_v.end());
    const double v_max = *std::max_element(ctx->h_eps_v.begin(), ctx->h_eps_v.end());
    const double c_min = *std::min_element(ctx->h_eps_c.begin(), ctx->h_eps_c.end());
    const double c_max = *std::max_element(ctx->h_eps_c.begin(), ctx->h_eps_c.end());
    const double d_min = c_min - v_max, d_max = c_max - v_min;
    *lo = 0.8 * d_min * d_min;
    if (steps == 0) {
        *hi = 1.25 * d_max * d_max;
        return GWL_OK;
    }
    double lam_min = 0.0, lam_max = 0.0;
    const gwl_status rs = gwl_spectrum_bounds(ctx, steps, &lam_min, &lam_max);
    if (rs != GWL_OK) return rs;
    *hi = (1.0 + margin) * std::max(lam_max, d_max * d_max);
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
    if (reorth == 1 && steps > GWL_MAX_REORTH_STEPS)
        return ctx->fail(GWL_EINVAL, "gwl_lanczos: reorth = 1 needs steps <= GWL_MAX_REORTH_STEPS = " + std::to_string(GWL_MAX_REORTH_STEPS) +
                                         " (the projection coefficients of all earlier vectors sit in shared memory)");
    if (!ready(ctx)) return ctx->fail(GWL_ESTATE, "gwl_lanczos: orbitals, energies and kernel must be set");
    if (ctx->chain_mode == 0) return ctx->fail(GWL_ESTATE, "gwl_lanczos: no chains set");
    if (n_chains > ctx->n_chains_set) return ctx->fail(GWL_EINVAL, "gwl_lanczos: more chains than were set");
    // Step graphs (small problems, no profiling events, no reorthogonalisation): the whole call runs on an internal stream
    // fenced against the caller's stream on both sides, because the caller's stream may be the legacy default stream.
    // A captured graph is tied to its chain block (the alpha/beta bases of the block are baked into the kernel arguments),
    // and the context caches eight of them: with more blocks than that every block would re-capture on every call, which
    // costs more than the replay saves, so such calls use plain launches.  Switch: gwl_set_profiling(ctx, 0) enables the
    // replay, any other level (the default is 1) disables it.
    const int64_t n_blocks = (n_chains + block - 1) / block;
    const bool want_graph = !ctx->graph_off && ctx->prof_level == 0 && reorth == 0 && !ctx->cplx && steps >= 16 &&
                            n_chains > 0 && n_blocks <= 8 && lanczos_fused_fits(ctx->n_vc);
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
