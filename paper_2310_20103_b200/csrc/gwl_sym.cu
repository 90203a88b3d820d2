// C ABI, point-group symmetry blocks of the Casida matrix (gwl_sym_*, reading Q25).
#include "gwl_ctx.h"

using namespace gwl;

extern "C" {

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

}  // extern "C"
