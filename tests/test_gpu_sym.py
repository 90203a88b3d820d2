"""GPU parity of the point-group symmetry blocks (gwl_sym_*, reading Q25) against
oracle/symmetry.py AND against the unreduced method (gw_oracle on the unfolded problem; the plain gwl context on the GPU) on the
same seeded inputs.  Tolerances of the protocol: product 1e-12 relative, alpha/beta 1e-9, Sigma 1e-6 eV."""
import numpy as np
import pytest

from oracle import gw_oracle as orc
from oracle import symmetry as sym
from paper_2310_20103_b200 import gwl, polyfit, synth

pytestmark = pytest.mark.gpu

DLT = 0.1


def _ctx(p):
    ctx = gwl.SymContext(p.n_refl, p.nv_irrep, p.nc_irrep, p.n_w)
    ctx.set_orbitals(p.phi_v_w, p.phi_c_w)
    ctx.set_energies(p.eps_v, p.eps_c)
    ctx.set_kernel(p.V_wf)
    return ctx


def _chains_of_block(p, gamma, m, count):
    """The first `count` orbitals n (alternating occupied / empty) with irrep(n) ^ irrep(m) = gamma."""
    irr = np.concatenate([p.irrep_v, p.irrep_c])
    n_v = len(p.irrep_v)
    occ = [n for n in range(n_v) if irr[n] ^ irr[m] == gamma]
    emp = [n for n in range(n_v, len(irr)) if irr[n] ^ irr[m] == gamma]
    out = []
    for i in range(max(len(occ), len(emp))):
        out += occ[i:i + 1] + emp[i:i + 1]
    return np.array(out[:count], dtype=np.int32)


@pytest.mark.parametrize("n_refl,nv,nc,n_w,nvec", [(0, [3], [5], 20, 2), (1, [2, 3], [5, 17], 37, 3),
                                                  (2, [3, 2, 4, 1], [16, 9, 33, 20], 130, 70),
                                                  (3, [1, 0, 2, 1, 1, 2, 0, 1], [4, 3, 0, 7, 18, 2, 5, 1], 65, 4)])
def test_block_matvec_ragged(n_refl, nv, nc, n_w, nvec):
    """Every block gamma of ragged problems (empty irreps, conduction counts off the 16-column padding, more vectors than
    one N tile) against the oracle's block product."""
    p = synth.make_symmetric(n_refl, nv, nc, n_w, seed=50 + n_refl)
    with _ctx(p) as ctx:
        for gamma in range(p.g):
            vs, cs = sym.pair_block(p.irrep_v, p.irrep_c, gamma)
            if vs.size == 0:
                with pytest.raises(gwl.GwlError) as e:
                    ctx.select(gamma)
                assert e.value.status == gwl.GWL_EINVAL
                continue
            assert ctx.select(gamma) == vs.size
            X = np.random.default_rng(gamma).standard_normal((nvec, vs.size))
            Y = ctx.matvec(X)
            ref = sym.block_matvec(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, gamma, X)
            assert np.abs(Y - ref).max() <= 1e-12 * np.abs(ref).max()


def test_block_equals_the_unreduced_product_on_the_gpu():
    """The SAME system through the plain context (all g n_w points, all pairs): a vector supported on block gamma gives the
    block product inside the block and zero outside."""
    p = synth.make_symmetric(2, [3, 2, 2, 1], [6, 5, 9, 4], 40, seed=61)
    phi_v = sym.unfold_orbitals(p.phi_v_w, p.irrep_v, p.g)
    phi_c = sym.unfold_orbitals(p.phi_c_w, p.irrep_c, p.g)
    n_v, n_c = phi_v.shape[1], phi_c.shape[1]
    with gwl.Context(n_v, n_c, p.g * p.n_w) as full, _ctx(p) as ctx:
        full.set_orbitals(phi_v, phi_c)
        full.set_energies(p.eps_v, p.eps_c)
        full.set_kernel(p.V_full)
        for gamma in range(p.g):
            vs, cs = sym.pair_block(p.irrep_v, p.irrep_c, gamma)
            ctx.select(gamma)
            X = np.random.default_rng(7 + gamma).standard_normal((2, vs.size))
            Xf = np.zeros((2, n_v * n_c))
            Xf[:, vs * n_c + cs] = X
            Yf = full.casida_matvec(Xf).reshape(2, -1)
            Y = ctx.matvec(X)
            assert np.abs(Y - Yf[:, vs * n_c + cs]).max() <= 1e-12 * np.abs(Yf).max()
            rest = np.setdiff1d(np.arange(n_v * n_c), vs * n_c + cs)
            assert np.abs(Yf[:, rest]).max() <= 1e-12 * np.abs(Yf).max()


def test_sym_lanczos_and_sigma_against_oracle_and_unreduced_oracle():
    p = synth.make_symmetric(2, [3, 2, 2, 1], [10, 7, 12, 9], 48, seed=62, n_omega=201)
    m = 2                                                   # an occupied orbital of irrep 0
    L = 30
    phi_v = sym.unfold_orbitals(p.phi_v_w, p.irrep_v, p.g)
    phi_c = sym.unfold_orbitals(p.phi_c_w, p.irrep_c, p.g)
    with _ctx(p) as ctx:
        for gamma in range(p.g):
            n_idx = _chains_of_block(p, gamma, m, 5)
            m_idx = np.full(n_idx.size, m, dtype=np.int32)
            ctx.select(gamma)
            ctx.set_chains(n_idx, m_idx)
            a, b, n2, ln = ctx.lanczos(n_idx.size, L, 3, 1)              # blocks of 3 + 2
            sig, ssum = ctx.selfenergy(p.omega, DLT, n_idx.size)
            a0, b0, _, _ = ctx.lanczos(n_idx.size, 20, 8, 0)
            ref = sym.run_chains_sym(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, n_idx, m_idx, L,
                                     p.omega, DLT, reorth=True)
            assert (ref["gamma"] == gamma).all() and (ln == ref["len"]).all()
            assert (np.abs(n2 - ref["norm2"]) <= 1e-12 * ref["norm2"]).all()
            assert (np.abs(a - ref["alpha"]) <= 1e-9 * np.abs(ref["alpha"])).all()
            assert (np.abs(b - ref["beta"]) <= 1e-9 * np.abs(ref["beta"])).all()
            assert np.abs(sig - ref["sigma"]).max() <= 1e-6 and np.abs(ssum - ref["sigma_sum"]).max() <= 1e-6
            ref0 = sym.run_chains_sym(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, n_idx, m_idx, 20,
                                      p.omega, DLT, reorth=False)
            assert (np.abs(a0 - ref0["alpha"]) <= 1e-9 * np.abs(ref0["alpha"])).all()
            assert (np.abs(b0 - ref0["beta"]) <= 1e-9 * np.abs(ref0["beta"])).all()
            # the unreduced oracle (no symmetry used anywhere)
            full = orc.run_chains(phi_v, phi_c, p.eps_v, p.eps_c, p.V_full, n_idx, m_idx, L, p.omega, DLT, reorth=True)
            assert np.abs(sig - full["sigma"]).max() <= 1e-6
            with pytest.raises(gwl.GwlError) as e:                       # a pair of another block
                wrong = _chains_of_block(p, gamma ^ 1, m, 1)
                ctx.set_chains(wrong, np.array([m], dtype=np.int32))
            assert e.value.status == gwl.GWL_EINVAL


def test_sym_selfenergy_state_equals_the_unreduced_state():
    """Sigma_mm summed over ALL n, walked block by block (gwl_sym_selfenergy_state), against the plain context's
    gwl_selfenergy_state on the unfolded problem and against the unreduced oracle."""
    p = synth.make_symmetric(2, [2, 2, 1, 2], [5, 4, 6, 3], 36, seed=63, n_omega=101)
    phi_v = sym.unfold_orbitals(p.phi_v_w, p.irrep_v, p.g)
    phi_c = sym.unfold_orbitals(p.phi_c_w, p.irrep_c, p.g)
    n_v, n_c = phi_v.shape[1], phi_c.shape[1]
    L = 12
    for m in (n_v - 1, n_v + 3):
        with _ctx(p) as ctx:
            s_sym = ctx.selfenergy_state(m, L, 8, 1, p.omega, DLT)
        with gwl.Context(n_v, n_c, p.g * p.n_w) as full:
            full.set_orbitals(phi_v, phi_c)
            full.set_energies(p.eps_v, p.eps_c)
            full.set_kernel(p.V_full)
            s_full = full.selfenergy_state(m, L, 8, 1, p.omega, DLT)
        ref = orc.sigma_state(phi_v, phi_c, p.eps_v, p.eps_c, p.V_full, m, L, p.omega, DLT, reorth=True)
        assert np.abs(s_sym - ref).max() <= 1e-6
        assert np.abs(s_sym - s_full).max() <= 1e-6


def test_sym_poly_mode_and_state_errors():
    """The paper's route (Lanczos on p_g(C), fused Chebyshev epilogue) inside a block against the same polynomial applied to
    the block operator by the oracle; out-of-order and wrong-context calls."""
    p = synth.make_symmetric(1, [3, 2], [9, 20], 40, seed=64, n_omega=101)
    gamma, m = 1, 0
    vs, cs = sym.pair_block(p.irrep_v, p.irrep_c, gamma)
    Cg = sym.casida_block_dense(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, gamma)
    lam = np.linalg.eigvalsh(Cg)
    lo, hi = 0.9 * lam[0], 1.05 * lam[-1]
    g = 8
    c = polyfit.sqrt_chebyshev(g, lo, hi)
    n_idx = _chains_of_block(p, gamma, m, 4)
    m_idx = np.full(n_idx.size, m, dtype=np.int32)
    with _ctx(p) as ctx:
        with pytest.raises(gwl.GwlError) as e:
            ctx.set_chains(n_idx, m_idx)                                  # no block selected yet
        assert e.value.status == gwl.GWL_ESTATE
        ctx.select(gamma)
        ctx.set_polynomial(g, c, lo, hi)
        ctx.set_chains(n_idx, m_idx)
        a, b, n2, ln = ctx.lanczos(n_idx.size, 10, 4, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, n_idx.size)
        for bad in (lambda: ctx.casida_matvec(np.zeros((1, vs.size))), lambda: ctx.set_approximation(gwl.GWL_TDA),
                    lambda: gwl.Context.selfenergy_state(ctx, 0, 4, 4, 0, p.omega, DLT),     # the plain-context entry point
                    lambda: gwl.Context.set_kernel(ctx, np.zeros((p.n_w, p.n_w)))):
            with pytest.raises(gwl.GwlError) as e:
                bad()
            assert e.value.status == gwl.GWL_ESTATE

    def op_C(x):
        return Cg @ x

    for j in range(n_idx.size):
        _, P = sym.start_vector_block(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, int(n_idx[j]), m)
        ar, br, n2r, lnr = orc.lanczos(lambda x: orc.poly_apply(op_C, c, lo, hi, x), P, 10, reorth=True)
        e_n, sg = orc.orbital_energy_sign(p.eps_v, p.eps_c, int(n_idx[j]))
        ref = orc.sigma_poly(ar, br, n2r, lnr, p.omega, e_n, sg, DLT)
        assert (np.abs(a[j] - ar) <= 1e-9 * np.abs(ar)).all() and (np.abs(b[j] - br) <= 1e-9 * np.abs(br)).all()
        assert np.abs(sig[j] - ref).max() <= 1e-6


def test_sym_cluster_scale_sampled():
    """D2h-like group (g = 8) on a config-1-sized system: 64 occupied x 256 empty orbitals (8 + 32 per irrep), 192 wedge points =
    1536 fitting points.  One block of 64 chains in block gamma = 3 on the GPU (2048 pairs instead of 16 384); the oracle
    follows sampled columns and chains, the unreduced oracle one chain."""
    p = synth.make_symmetric(3, [8] * 8, [32] * 8, 192, box=15.0, seed=65, n_omega=401)
    gamma, m = 3, 0
    vs, cs = sym.pair_block(p.irrep_v, p.irrep_c, gamma)
    n_idx = _chains_of_block(p, gamma, m, 40)
    m_idx = np.full(n_idx.size, m, dtype=np.int32)
    idx = np.array([0, 17, 39])
    X = np.random.default_rng(3).standard_normal((64, vs.size))
    with _ctx(p) as ctx:
        assert ctx.select(gamma) == 8 * 8 * 32
        Y = ctx.matvec(X)
        ctx.set_chains(n_idx, m_idx)
        a, b, n2, ln = ctx.lanczos(n_idx.size, 25, 64, 0)
        ctx.set_chains(n_idx[idx], m_idx[idx])
        ar, br, _, _ = ctx.lanczos(3, 60, 3, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, 3)
        ctx.lanczos(1, 10, 1, 1)
        sig10, _ = ctx.selfenergy(p.omega, DLT, 1)
    ref = sym.block_matvec(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, gamma, X[idx])
    assert np.abs(Y[idx] - ref).max() <= 1e-12 * np.abs(ref).max()
    r0 = sym.run_chains_sym(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, n_idx[idx], m_idx[idx], 25,
                            p.omega, DLT, reorth=False)
    assert (np.abs(a[idx] - r0["alpha"]) <= 1e-9 * np.abs(r0["alpha"])).all()
    assert (np.abs(b[idx] - r0["beta"]) <= 1e-9 * np.abs(r0["beta"])).all()
    r1 = sym.run_chains_sym(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, n_idx[idx], m_idx[idx], 60,
                            p.omega, DLT, reorth=True)
    assert (np.abs(ar - r1["alpha"]) <= 1e-9 * np.abs(r1["alpha"])).all()
    assert (np.abs(br - r1["beta"]) <= 1e-9 * np.abs(r1["beta"])).all()
    assert np.abs(sig - r1["sigma"]).max() <= 1e-6
    phi_v = sym.unfold_orbitals(p.phi_v_w, p.irrep_v, p.g)
    phi_c = sym.unfold_orbitals(p.phi_c_w, p.irrep_c, p.g)
    # The unreduced run is compared over 10 steps only: in the full space rounding noise of the OTHER blocks (1e-16 in q_0) is
    # orthogonal to the basis, so reorthogonalisation does not remove it, and it grows like a power iteration towards the
    # well-separated top of those blocks' spectra (1.4e-3 eV of Sigma at L = 60); inside a block it cannot arise.
    full = orc.run_chains(phi_v, phi_c, p.eps_v, p.eps_c, p.V_full, n_idx[idx[:1]], m_idx[idx[:1]], 10, p.omega, DLT, reorth=True)
    assert np.abs(sig10[0] - full["sigma"][0]).max() <= 1e-6


def test_sym_exchange_spectrum_bounds_and_quasiparticle_state():
    """Sigma^x (Eq. 6) through the reduced kernels against gw_oracle.exchange_eq6 on the unfolded problem; the Lanczos bounds
    of every block against its dense spectrum (the probe vector stays off the padding pairs); then one whole quasiparticle
    state the paper's way inside the blocks (fitting range over all blocks, p_g(C), Eq. 10 over all n, Sigma^x, E(omega) = omega)
    against the unreduced oracle."""
    p = synth.make_symmetric(2, [2, 2, 1, 2], [5, 4, 6, 3], 36, seed=66, n_omega=161)
    phi_v = sym.unfold_orbitals(p.phi_v_w, p.irrep_v, p.g)
    phi_c = sym.unfold_orbitals(p.phi_c_w, p.irrep_c, p.g)
    n_v = phi_v.shape[1]
    ms = np.array([0, n_v - 1, n_v + 2, n_v + 9], dtype=np.int32)
    g_poly, L = 8, 10
    m = n_v - 1
    with _ctx(p) as ctx:
        sx = ctx.exchange(ms)
        lam_hi = 0.0
        for gamma in range(p.g):
            ctx.select(gamma)
            lo_g, hi_g = ctx.spectrum_bounds(40)
            lam = np.linalg.eigvalsh(sym.casida_block_dense(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf,
                                                            gamma))
            assert lam[-1] * (1 - 1e-10) <= hi_g <= 1.02 * lam[-1]
            assert lo_g <= lam[0] * (1 + 1e-10) and lo_g >= 0.5 * lam[0]
            lam_hi = max(lam_hi, hi_g)
        d_min = p.eps_c.min() - p.eps_v.max()
        lo, hi = 0.8 * d_min * d_min, 1.02 * lam_hi
        c = polyfit.sqrt_chebyshev(g_poly, lo, hi)
        ctx.set_polynomial(g_poly, c, lo, hi)
        sc = ctx.selfenergy_state(m, L, 8, 1, p.omega, 0.68)
        sxm = ctx.exchange([m])
        e_qp, z_qp, it = ctx.qp_solve([p.eps_v[m]], [-9.0], sxm, sc[None, :], p.omega)
    for j, mm in enumerate(ms):
        ref = orc.exchange_eq6(phi_v, phi_c, p.V_full, int(mm))
        assert abs(sx[j] - ref) <= 1e-12 * abs(ref)
    ref_c = orc.sigma_state(phi_v, phi_c, p.eps_v, p.eps_c, p.V_full, m, L, p.omega, 0.68, reorth=True, poly=(c, lo, hi))
    assert np.abs(sc - ref_c).max() <= 1e-6
    e_ref, z_ref, _ = orc.qp_solve(p.eps_v[m], -9.0, orc.exchange_eq6(phi_v, phi_c, p.V_full, m), ref_c, p.omega)
    assert abs(e_qp[0] - e_ref) <= 1e-6 and abs(z_qp[0] - z_ref) <= 1e-6


def test_sym_config4_scale_sampled():
    """The sizes of BASELINE.json:configs[4] with a group of order 8 (the shape of `bench.py --sym 3`: N_v = 1024, N_c = 4096,
    wedge of 2560 of the 20 480 points, 524 288 pairs per block), one block of 128 chains on the GPU in the launch configuration
    that arm times; the oracle follows sampled columns of the block product and one sampled chain (no reorthogonalisation:
    inside a block two correct FP64 runs stay together)."""
    p = synth.make_symmetric(3, [128] * 8, [512] * 8, 2560, box=40.0, seed=0, n_omega=101)
    gamma, m = 1, 0
    irr = np.concatenate([p.irrep_v, p.irrep_c])
    n_idx = np.array([n for n in range(irr.size) if irr[n] ^ irr[m] == gamma][:128], dtype=np.int32)
    m_idx = np.full(128, m, dtype=np.int32)
    cols = np.array([5, 127])
    j = np.array([77])
    L = 10
    with _ctx(p) as ctx:
        n_pairs = ctx.select(gamma)
        assert n_pairs == 8 * 128 * 512
        X = np.random.default_rng(9).standard_normal((128, n_pairs))
        Y = ctx.matvec(X)
        ctx.set_chains(n_idx, m_idx)
        a, b, n2, ln = ctx.lanczos(128, L, 128, 0)
        sig, _ = ctx.selfenergy(p.omega, DLT, 128)
    V_wf = p.V_wf
    ref = sym.block_matvec(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, V_wf, gamma, X[cols])
    assert np.abs(Y[cols] - ref).max() <= 1e-12 * np.abs(ref).max()
    r0 = sym.run_chains_sym(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, V_wf, n_idx[j], m_idx[j], L, p.omega, DLT,
                            reorth=False)
    assert abs(n2[j[0]] - r0["norm2"][0]) <= 1e-12 * r0["norm2"][0]
    assert (np.abs(a[j] - r0["alpha"]) <= 1e-9 * np.abs(r0["alpha"])).all()
    assert (np.abs(b[j] - r0["beta"]) <= 1e-9 * np.abs(r0["beta"])).all()
    assert np.abs(sig[j] - r0["sigma"]).max() <= 1e-6


def test_sym_device_pointer_mode_and_empty_chain_list():
    """Device-pointer mode of gwl_sym_matvec and gwl_sym_selfenergy_state (what bench.py uses) gives the bits of the host-pointer
    calls; an empty chain list is accepted."""
    import torch
    p = synth.make_symmetric(2, [3, 2, 2, 1], [6, 5, 9, 4], 40, seed=67, n_omega=61)
    gamma, m = 2, 1
    with _ctx(p) as ctx:
        n_pairs = ctx.select(gamma)
        X = np.random.default_rng(1).standard_normal((3, n_pairs))
        Y = ctx.matvec(X)
        s_host = ctx.selfenergy_state(m, 10, 4, 0, p.omega, DLT)
        ctx.select(gamma)
        ctx.set_chains(np.zeros(0, dtype=np.int32), np.zeros(0, dtype=np.int32))
        a, b, n2, ln = ctx.lanczos(0, 5, 4, 0)
        assert a.shape == (0, 5)
        ctx.set_pointer_mode(1)
        ctx.set_stream(torch.cuda.current_stream().cuda_stream)
        xd = torch.from_numpy(X).cuda()
        yd = torch.empty_like(xd)
        ctx.matvec(xd, yd)
        om = torch.from_numpy(p.omega).cuda()
        sd = torch.empty(len(p.omega), 2, dtype=torch.float64, device="cuda")
        ctx.selfenergy_state(m, 10, 4, 0, om, DLT, out=sd)
        torch.cuda.synchronize()
    assert np.array_equal(yd.cpu().numpy(), Y)
    sdev = sd.cpu().numpy()
    assert np.array_equal(sdev[:, 0] + 1j * sdev[:, 1], s_host)
