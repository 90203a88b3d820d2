"""GPU parity of the complex-orbital Tamm-Dancoff variant (gwl_tdc_*) against
oracle/tda_periodic.py on the same seeded inputs.  Tolerances as for the real path: mat-vec 1e-12 relative (max-norm),
alpha/beta 1e-9 relative, Sigma 1e-6 eV with reorthogonalisation on both sides."""
import numpy as np
import pytest

from oracle import tda_periodic as tdp
from paper_2310_20103_b200 import gwl, synth

pytestmark = pytest.mark.gpu

DLT = 0.1


def _ctx(p, n_q=1, chains=True):
    ctx = gwl.TdcContext(p.n_k, p.n_v, p.n_c, p.n_mu, n_q)
    ctx.set_orbitals(p.psi_v, p.psi_cq)
    ctx.set_energies(p.eps_v, p.eps_cq)
    ctx.set_kernel(p.V)
    if chains:
        ctx.set_chains(p.chains)
    return ctx


def _relmax(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.parametrize("n_k,n_v,n_c,n_mu,nvec", [(1, 1, 1, 1, 1), (2, 3, 5, 37, 3), (3, 4, 19, 130, 70), (1, 2, 33, 257, 130),
                                                  (2, 8, 40, 200, 5)])
def test_tdc_matvec_ragged_sizes(n_k, n_v, n_c, n_mu, nvec):
    """Odd N_c, N_mu and N_c off the tile sizes, several k-points (the conduction block changes with k inside one
    reduction), blocks wider than one N tile and more than one chunk of 128 vectors."""
    p = synth.make_periodic(n_k, n_v, n_c, n_mu, seed=n_mu)
    X = synth.random_complex_block(p.n_kvc, nvec, seed=2)
    with _ctx(p, chains=False) as ctx:
        Y = ctx.matvec(X)
    ref = tdp.tda_matvec_factored(p.psi_v, p.psi_cq, p.V, tdp.delta_kvc(p.eps_v, p.eps_cq), X)
    assert _relmax(Y, ref) <= 1e-12


def test_tdc_matvec_hermitian_and_device_pointers():
    import torch
    p = synth.make_periodic(2, 6, 24, 160, seed=3)
    X = synth.random_complex_block(p.n_kvc, 4, seed=5)
    with _ctx(p, chains=False) as ctx:
        Y = ctx.matvec(X)
        ctx.set_pointer_mode(1)
        ctx.set_stream(torch.cuda.current_stream().cuda_stream)
        xd = torch.from_numpy(X).cuda()
        yd = torch.empty_like(xd)
        ctx.matvec(xd, yd)
        torch.cuda.synchronize()
    assert np.array_equal(yd.cpu().numpy(), Y)
    # <x0, A x1> = conj(<x1, A x0>) through the GPU path
    a, b = np.vdot(X[0], Y[1]), np.vdot(X[1], Y[0])
    assert abs(a - np.conj(b)) <= 1e-11 * abs(a)


def test_tdc_lanczos_and_sigma_against_oracle():
    """Start vectors (reading Q20), Hermitian Lanczos, Eq. 14, prefactor 2/(N_q N_k): all chains, reorth on both sides."""
    p = synth.make_periodic(2, 4, 12, 96, seed=4, n_chains=6, n_omega=201)
    L, n_q = 40, 3
    with _ctx(p, n_q=n_q) as ctx:
        a, b, n2, ln = ctx.lanczos(6, L, 4, 1)                       # blocks of 4 + 2
        sig, ssum = ctx.selfenergy(p.omega, DLT, 6)
        a0, b0, _, _ = ctx.lanczos(6, 20, 6, 0)
    ref = tdp.run_chains(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, L, p.omega, DLT, n_q=n_q, reorth=True)
    assert (ln == ref["len"]).all()
    assert (np.abs(n2 - ref["norm2"]) <= 1e-12 * ref["norm2"]).all()
    assert (np.abs(a - ref["alpha"]) <= 1e-9 * np.abs(ref["alpha"])).all()
    assert (np.abs(b - ref["beta"]) <= 1e-9 * np.abs(ref["beta"])).all()
    assert np.abs(sig - ref["sigma"]).max() <= 1e-6
    assert np.abs(ssum - ref["sigma_sum"]).max() <= 1e-6
    ref0 = tdp.run_chains(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, 20, p.omega, DLT, n_q=n_q, reorth=False)
    assert (np.abs(a0 - ref0["alpha"]) <= 1e-9 * np.abs(ref0["alpha"])).all()
    assert (np.abs(b0 - ref0["beta"]) <= 1e-9 * np.abs(ref0["beta"])).all()
    # sign of Im Sigma per eta_n (Herglotz)
    occ = p.chains[:, 1] < p.n_v
    assert (sig[occ].imag > 0).all() and (sig[~occ].imag < 0).all()


def test_tdc_full_length_against_exact_pole_sum():
    """L = N_k N_v N_c with reorthogonalisation: the Lanczos resolvent equals the printed pole sum (PAPER.md:288-290 in the
    TDA) by full diagonalisation of A(q)."""
    p = synth.make_periodic(2, 2, 6, 24, seed=6, n_chains=4)
    delta = tdp.delta_kvc(p.eps_v, p.eps_cq)
    A = tdp.tda_dense(delta, tdp.pair_matrix(p.psi_v, p.psi_cq), p.V)
    lam, X = tdp.eig_tda(A)
    with _ctx(p) as ctx:
        a, b, n2, ln = ctx.lanczos(4, p.n_kvc, 4, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, 4)
    for j, (kn, n_idx, km, m_idx) in enumerate(p.chains):
        Pp = tdp.start_vector_printed(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
        e_n, sg = tdp.orbital_energy_sign(p.eps_v, p.eps_cq, kn, n_idx)
        exact = tdp.sigma_chain_exact(lam, X, Pp, p.omega, e_n, sg, DLT, tdp.prefactor(1, p.n_k))
        assert np.abs(sig[j] - exact).max() <= 1e-8 * max(1.0, np.abs(exact).max())


def test_tdc_real_orbitals_equal_the_real_tda_path():
    """Real orbitals, one k-point: the complex kernels give what gwl_set_approximation(GWL_TDA) gives on the real path
    (times the prefactor 2/(N_q N_k) = 2)."""
    p = synth.make_periodic(1, 5, 17, 80, seed=7, n_chains=4, real_orbitals=True)
    with _ctx(p) as ctx:
        a, b, n2, ln = ctx.lanczos(4, 25, 4, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, 4)
    with gwl.Context(p.n_v, p.n_c, p.n_mu) as ctx:
        ctx.set_orbitals(p.psi_v[0].real, p.psi_cq[0].real)
        ctx.set_energies(p.eps_v[0], p.eps_cq[0])
        ctx.set_kernel(p.V)
        ctx.set_approximation(gwl.GWL_TDA)
        ctx.set_chains(p.chains[:, 1], p.chains[:, 3])
        ar, br, n2r, lnr = ctx.lanczos(4, 25, 4, 1)
        sigr, _ = ctx.selfenergy(p.omega, DLT, 4)
    assert (np.abs(a - ar) <= 1e-10 * np.abs(ar)).all() and (np.abs(b - br) <= 1e-10 * np.abs(br)).all()
    assert (np.abs(n2 - n2r) <= 1e-12 * n2r).all()
    assert np.abs(sig - 2.0 * sigr).max() <= 1e-8


def test_tdc_block_invariance_repeatability_and_errors():
    p = synth.make_periodic(2, 4, 12, 96, seed=8, n_chains=6)
    with _ctx(p) as ctx:
        a6, b6, n6, _ = ctx.lanczos(6, 15, 6, 0)
        a6b, b6b, _, _ = ctx.lanczos(6, 15, 6, 0)
        a1, b1, n1, _ = ctx.lanczos(6, 15, 1, 0)
        with pytest.raises(gwl.GwlError) as e:
            ctx._ck(ctx._lib.gwl_set_polynomial(ctx._h, 2, None, 1.0, 2.0))
        assert e.value.status == gwl.GWL_ESTATE
        with pytest.raises(gwl.GwlError):
            ctx.set_chains(np.array([[2, 0, 0, 0]]))                 # k slot out of range
        with pytest.raises(gwl.GwlError):
            ctx.set_energies(p.eps_v, p.eps_cq - 100.0)
    assert np.array_equal(a6, a6b) and np.array_equal(b6, b6b)
    assert (np.abs(a1 - a6) <= 1e-10 * np.abs(a6)).all() and (np.abs(b1 - b6) <= 1e-10 * np.abs(b6)).all()
    with gwl.Context(2, 2, 8) as ctx:
        with pytest.raises(gwl.GwlError) as e:
            ctx._ck(ctx._lib.gwl_tdc_set_chains(ctx._h, 0, None))
        assert e.value.status == gwl.GWL_ESTATE


def test_tdc_cluster_scale_sampled():
    """A ~config-1-sized periodic problem (N_k = 4, N_v = 16, N_c = 256: 16 384 complex pairs, N_mu = 1536), one block
    of 64 chains on the GPU; the oracle follows sampled columns of the product and sampled chains."""
    p = synth.make_periodic(4, 16, 256, 1536, box=15.0, seed=9, n_chains=64, n_omega=401)
    X = synth.random_complex_block(p.n_kvc, 64, seed=3)
    delta = tdp.delta_kvc(p.eps_v, p.eps_cq)
    idx = np.array([0, 21, 63])
    with _ctx(p) as ctx:
        Y = ctx.matvec(X)
        a, b, n2, ln = ctx.lanczos(64, 20, 64, 0)
        ctx.set_chains(p.chains[idx])
        ar, br, _, _ = ctx.lanczos(3, 40, 3, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, 3)
    ref = tdp.tda_matvec_factored(p.psi_v, p.psi_cq, p.V, delta, X[idx])
    assert _relmax(Y[idx], ref) <= 1e-12
    # reorthogonalisation off: as at config 2 of the real path, the top of the spectrum converges within a few steps and two
    # correct FP64 runs drift apart afterwards; the leading 8 steps are compared
    r0 = tdp.run_chains(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains[idx], 8, p.omega, DLT, reorth=False)
    assert (np.abs(a[idx, :8] - r0["alpha"]) <= 1e-9 * np.abs(r0["alpha"])).all()
    assert (np.abs(b[idx, :8] - r0["beta"]) <= 1e-9 * np.abs(r0["beta"])).all()
    r1 = tdp.run_chains(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains[idx], 40, p.omega, DLT, reorth=True)
    assert (np.abs(ar - r1["alpha"]) <= 1e-9 * np.abs(r1["alpha"])).all()
    assert (np.abs(br - r1["beta"]) <= 1e-9 * np.abs(r1["beta"])).all()
    assert np.abs(sig - r1["sigma"]).max() <= 1e-6
