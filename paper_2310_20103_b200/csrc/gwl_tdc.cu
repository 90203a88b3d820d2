// C ABI, complex orbitals and k-points (gwl_tdc_*): Tamm-Dancoff and pseudo-Hermitian RPA products, inputs, chains.
#include "gwl_ctx.h"

using namespace gwl;

extern "C" {

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

gwl_status gwl_tdc_selfenergy_state(gwl_ctx* ctx, int32_t kn, int32_t km, int32_t m_idx, int64_t steps, int64_t block, int reorth,
                                    const double* omega, int64_t n_omega, double eta, double* sigma_mm) {
    if (ctx == nullptr) return GWL_EINVAL;
    DeviceGuard dg(ctx);
    if (!ctx->cplx) return ctx->fail(GWL_ESTATE, "gwl_tdc_selfenergy_state: not a gwl_tdc_create context");
    if (sigma_mm == nullptr || omega == nullptr || n_omega < 1)
        return ctx->fail(GWL_EINVAL, "gwl_tdc_selfenergy_state: bad arguments");
    const int n_orb = ctx->nv_k + ctx->n_c;
    std::vector<int32_t> chains((size_t)4 * n_orb);
    for (int n = 0; n < n_orb; ++n) {
        chains[4 * n] = kn;
        chains[4 * n + 1] = n;
        chains[4 * n + 2] = km;
        chains[4 * n + 3] = m_idx;
    }
    gwl_status rs = gwl_tdc_set_chains(ctx, n_orb, chains.data());
    if (rs != GWL_OK) return rs;
    rs = gwl_lanczos(ctx, n_orb, steps, block, reorth, nullptr, nullptr, nullptr, nullptr);
    if (rs != GWL_OK) return rs;
    return gwl_selfenergy(ctx, omega, n_omega, eta, nullptr, sigma_mm);
}

}  // extern "C"
