"""GPU parity of the complex-orbital RPA variant (gwl_set_approximation(GWL_RPA) on a gwl_tdc_create context: the
pseudo-Hermitian Lanczos of PAPER.md:159 for the pole sum of PAPER.md:286-304, reading Q24) against
oracle/rpa_periodic.py on the same seeded inputs.  Tolerances as for the other paths: product with Omega^ 1e-12 relative
(max-norm), alpha/beta 1e-9 relative, Sigma 1e-6 eV with reorthogonalisation on both sides."""
import numpy as np
import pytest

from oracle import rpa_periodic as rpa
from oracle import tda_periodic as tdp
from paper_2310_20103_b200 import gwl, synth

pytestmark = pytest.mark.gpu

DLT = 0.1


def _ctx(p, n_q=1, chains=True):
    ctx = gwl.TdcContext(p.n_k, p.n_v, p.n_c, p.n_mu, n_q)
    ctx.set_orbitals(p.psi_v, p.psi_cq)
    ctx.set_energies(p.eps_v, p.eps_cq)
    ctx.set_kernel(p.V)
    ctx.set_approximation(gwl.GWL_RPA)
    if chains:
        ctx.set_chains(p.chains)
    return ctx


def _relmax(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.parametrize("n_k,n_v,n_c,n_mu,nvec", [(1, 1, 1, 1, 1), (2, 3, 5, 37, 3), (3, 4, 19, 130, 70), (1, 2, 33, 257, 130),
                                                  (2, 8, 40, 200, 5)])
def test_omega_hat_product_ragged_sizes(n_k, n_v, n_c, n_mu, nvec):
    """[ox; oy] = [[A, B], [B^*, A^*]] [x; y]: odd sizes off the tile shapes, several k-points, more pairs than one chunk."""
    p = synth.make_periodic(n_k, n_v, n_c, n_mu, seed=n_mu)
    X = synth.random_complex_block(p.n_kvc, nvec, seed=2)
    Y = synth.random_complex_block(p.n_kvc, nvec, seed=3)
    with _ctx(p, chains=False) as ctx:
        ox, oy = ctx.matvec_rpa(X, Y)
    rx, ry = rpa.omega_hat_factored(p.psi_v, p.psi_cq, p.V, tdp.delta_kvc(p.eps_v, p.eps_cq), X, Y)
    scale = max(np.abs(rx).max(), np.abs(ry).max())
    assert np.abs(ox - rx).max() <= 1e-12 * scale and np.abs(oy - ry).max() <= 1e-12 * scale


def test_omega_hat_product_is_hermitian_and_reduces_to_A_for_y_zero():
    import torch
    p = synth.make_periodic(2, 6, 24, 160, seed=3)
    X = synth.random_complex_block(p.n_kvc, 4, seed=5)
    Y = synth.random_complex_block(p.n_kvc, 4, seed=6)
    with _ctx(p, chains=False) as ctx:
        ox, oy = ctx.matvec_rpa(X, Y)
        ax, _ = ctx.matvec_rpa(X, np.zeros_like(X))
        ctx.set_approximation(gwl.GWL_TDA)
        A_x = ctx.matvec(X)
        ctx.set_approximation(gwl.GWL_RPA)
        ctx.set_pointer_mode(1)
        ctx.set_stream(torch.cuda.current_stream().cuda_stream)
        xd, yd = torch.from_numpy(X).cuda(), torch.from_numpy(Y).cuda()
        oxd, oyd = torch.empty_like(xd), torch.empty_like(yd)
        ctx.matvec_rpa(xd, yd, oxd, oyd)
        torch.cuda.synchronize()
    assert np.array_equal(oxd.cpu().numpy(), ox) and np.array_equal(oyd.cpu().numpy(), oy)
    assert _relmax(ax, A_x) <= 1e-13                                     # upper-left block of Omega^ is A(q)
    # <p0, Omega^ p1> = conj(<p1, Omega^ p0>) for the pairs p = [x; y]
    a = np.vdot(X[0], ox[1]) + np.vdot(Y[0], oy[1])
    b = np.vdot(X[1], ox[0]) + np.vdot(Y[1], oy[0])
    assert abs(a - np.conj(b)) <= 1e-11 * abs(a)


def test_prpa_lanczos_and_sigma_against_oracle():
    """Start vectors u = F conj([P1; P2]), Lanczos in the Omega^ inner product, positive Ritz branch, prefactor 2/(N_q N_k):
    all chains, reorthogonalisation on both sides; then the leading steps with reorthogonalisation off."""
    p = synth.make_periodic(2, 4, 12, 96, seed=4, n_chains=6, n_omega=201)
    L, n_q = 40, 3
    with _ctx(p, n_q=n_q) as ctx:
        a, b, n2, ln = ctx.lanczos(6, L, 4, 1)                       # blocks of 4 + 2
        sig, ssum = ctx.selfenergy(p.omega, DLT, 6)
        a0, b0, _, _ = ctx.lanczos(6, 20, 6, 0)
    ref = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, L, p.omega, DLT, n_q=n_q, reorth=True)
    assert (ln == ref["len"]).all()
    assert (np.abs(n2 - ref["norm2"]) <= 1e-12 * ref["norm2"]).all()
    scale = np.abs(ref["beta"]).max()                                # alpha of H = F Omega^ can pass through zero: absolute scale
    assert np.abs(a - ref["alpha"]).max() <= 1e-9 * scale
    assert (np.abs(b - ref["beta"]) <= 1e-9 * np.abs(ref["beta"])).all()
    assert np.abs(sig - ref["sigma"]).max() <= 1e-6
    assert np.abs(ssum - ref["sigma_sum"]).max() <= 1e-6
    ref0 = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, 20, p.omega, DLT, n_q=n_q, reorth=False)
    assert np.abs(a0 - ref0["alpha"]).max() <= 1e-9 * scale
    assert (np.abs(b0 - ref0["beta"]) <= 1e-9 * np.abs(ref0["beta"])).all()
    occ = p.chains[:, 1] < p.n_v
    assert (sig[occ].imag > 0).all() and (sig[~occ].imag < 0).all()   # Herglotz sign per eta_n


def test_prpa_full_length_against_exact_pole_sum():
    """L = 2 N_k N_v N_c with reorthogonalisation: the GPU result equals the printed pole sum by full
    diagonalisation of C^RPA(q)."""
    p = synth.make_periodic(2, 2, 6, 24, seed=6, n_chains=4)
    delta = tdp.delta_kvc(p.eps_v, p.eps_cq)
    K = tdp.pair_matrix(p.psi_v, p.psi_cq)
    om, X, Y = rpa.rpa_eig(tdp.tda_dense(delta, K, p.V), tdp.coupling_B(K, p.V))
    with _ctx(p) as ctx:
        a, b, n2, ln = ctx.lanczos(4, 2 * p.n_kvc, 4, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, 4)
    for j, (kn, n_idx, km, m_idx) in enumerate(p.chains):
        P1, P2 = rpa.printed_elements(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx)
        e_n, sg = tdp.orbital_energy_sign(p.eps_v, p.eps_cq, kn, n_idx)
        exact = rpa.sigma_chain_exact_rpa(om, X, Y, P1, P2, p.omega, e_n, sg, DLT, tdp.prefactor(1, p.n_k))
        # the oracle's own full-length Lanczos sits 3e-7 eV from this sum on this problem (general eigensolver of the
        # non-normal 2N x 2N matrix, poles 0.1 eV off the axis): the bar is the Sigma tolerance of the protocol
        assert np.abs(sig[j] - exact).max() <= 1e-6


def test_prpa_real_orbitals_equal_the_real_rpa_path():
    """Real orbitals, one k-point: the pseudo-Hermitian route at full length gives what the real path (Lanczos on
    C = (A-B)^{1/2}(A+B)(A-B)^{1/2}, direct mode) gives, times the prefactor 2/(N_q N_k) = 2."""
    p = synth.make_periodic(1, 3, 7, 40, seed=7, n_chains=4, real_orbitals=True)
    n = p.n_kvc
    with _ctx(p) as ctx:
        ctx.lanczos(4, 2 * n, 4, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, 4)
    with gwl.Context(p.n_v, p.n_c, p.n_mu) as ctx:
        ctx.set_orbitals(p.psi_v[0].real, p.psi_cq[0].real)
        ctx.set_energies(p.eps_v[0], p.eps_cq[0])
        ctx.set_kernel(p.V)
        ctx.set_chains(p.chains[:, 1], p.chains[:, 3])
        ctx.lanczos(4, n, 4, 1)
        sigr, _ = ctx.selfenergy(p.omega, DLT, 4)
    assert np.abs(sig - 2.0 * sigr).max() <= 1e-7


def test_prpa_block_invariance_repeatability_and_state():
    p = synth.make_periodic(2, 4, 12, 96, seed=8, n_chains=6)
    with _ctx(p) as ctx:
        a6, b6, n6, _ = ctx.lanczos(6, 15, 6, 0)
        a6b, b6b, _, _ = ctx.lanczos(6, 15, 6, 0)
        a1, b1, n1, _ = ctx.lanczos(6, 15, 1, 0)
        ctx.set_approximation(gwl.GWL_TDA)                            # switching invalidates the tridiagonals
        with pytest.raises(gwl.GwlError) as e:
            ctx.selfenergy(p.omega, DLT, 6)
        assert e.value.status == gwl.GWL_ESTATE
        at, bt, _, _ = ctx.lanczos(6, 15, 6, 0)
    assert np.array_equal(a6, a6b) and np.array_equal(b6, b6b)
    scale = np.abs(b6).max()
    assert np.abs(a1 - a6).max() <= 1e-10 * scale and (np.abs(b1 - b6) <= 1e-10 * np.abs(b6)).all()
    assert np.array_equal(n1, n6)
    assert np.abs(at - a6).max() > 1e-3 * scale                       # the TDA chain is a different operator


def test_prpa_cluster_scale_sampled():
    """16 384 complex pairs (N_k = 4, N_v = 16, N_c = 256, N_mu = 1536), one block of 32 chains = 64 GEMM columns on the GPU;
    the oracle follows sampled pairs of the product and sampled chains."""
    p = synth.make_periodic(4, 16, 256, 1536, box=15.0, seed=9, n_chains=32, n_omega=401)
    X = synth.random_complex_block(p.n_kvc, 32, seed=3)
    Y = synth.random_complex_block(p.n_kvc, 32, seed=4)
    delta = tdp.delta_kvc(p.eps_v, p.eps_cq)
    idx = np.array([0, 13, 31])
    with _ctx(p) as ctx:
        ox, oy = ctx.matvec_rpa(X, Y)
        a, b, n2, ln = ctx.lanczos(32, 12, 32, 0)
        ctx.set_chains(p.chains[idx])
        ar, br, _, _ = ctx.lanczos(3, 30, 3, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, 3)
    rx, ry = rpa.omega_hat_factored(p.psi_v, p.psi_cq, p.V, delta, X[idx], Y[idx])
    scale = max(np.abs(rx).max(), np.abs(ry).max())
    assert np.abs(ox[idx] - rx).max() <= 1e-12 * scale and np.abs(oy[idx] - ry).max() <= 1e-12 * scale
    r0 = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains[idx], 6, p.omega, DLT, reorth=False)
    bs = np.abs(r0["beta"]).max()
    assert np.abs(a[idx, :6] - r0["alpha"]).max() <= 1e-9 * bs
    assert (np.abs(b[idx, :6] - r0["beta"]) <= 1e-9 * np.abs(r0["beta"])).all()
    r1 = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains[idx], 30, p.omega, DLT, reorth=True)
    assert np.abs(ar - r1["alpha"]).max() <= 1e-9 * bs
    assert (np.abs(br - r1["beta"]) <= 1e-9 * np.abs(r1["beta"])).all()
    assert np.abs(sig - r1["sigma"]).max() <= 1e-6


def test_prpa_resolvent_against_oracle_and_dense_solve():
    """gwl_resolvent on a complex-RPA run: <u|(zeta - C^RPA)^-1|u>_O by Eq. 14, against the oracle's continued fraction at the
    same length and, at full length, against the dense solve u^H Omega^ (zeta - F Omega^)^-1 u."""
    p = synth.make_periodic(2, 2, 5, 20, seed=12, n_chains=3)
    zeta = np.array([3.0 + 0.5j, -7.0 + 0.2j, 0.1j, 25.0 - 1.0j])
    delta = tdp.delta_kvc(p.eps_v, p.eps_cq)
    K = tdp.pair_matrix(p.psi_v, p.psi_cq)
    A, B = tdp.tda_dense(delta, K, p.V), tdp.coupling_B(K, p.V)
    with _ctx(p) as ctx:
        ctx.lanczos(3, 12, 3, 1)
        r12 = ctx.resolvent(zeta, 3)
        ctx.lanczos(3, 2 * p.n_kvc, 3, 1)
        rfull = ctx.resolvent(zeta, 3)
    ref = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains, 12, p.omega, DLT, reorth=True)
    for j, (kn, n_idx, km, m_idx) in enumerate(p.chains):
        cf = rpa.resolvent_chain(ref["alpha"][j], ref["beta"][j], ref["norm2"][j], ref["len"][j], zeta)
        assert np.abs(r12[j] - cf).max() <= 1e-9 * np.abs(cf).max()
        u1, u2 = rpa.start_vector_rpa(*rpa.printed_elements(p.psi_v, p.psi_cq, p.V, kn, n_idx, km, m_idx))
        ex = rpa.resolvent_exact_rpa(A, B, u1, u2, zeta)
        assert np.abs(rfull[j] - ex).max() <= 1e-8 * np.abs(ex).max()


def test_complex_config2_scale_sampled():
    """262 144 complex pairs (N_k = 4, N_v = 64, N_c = 1024, N_mu = 6144: the shape of `bench.py --tdc 4,64,1024,6144`), 64 chain
    pairs = 128 GEMM columns on the GPU in the launch configuration that arm times; the oracle (about 15 s per product with
    Omega^ at this size) follows one sampled pair of the product, of A(q) x in the Tamm-Dancoff operator, and the leading steps of
    one sampled chain of the pseudo-Hermitian Lanczos."""
    p = synth.make_periodic(4, 64, 1024, 6144, box=20.0, seed=0, n_chains=64, n_omega=101)
    delta = tdp.delta_kvc(p.eps_v, p.eps_cq)
    X = synth.random_complex_block(p.n_kvc, 64, seed=3)
    Y = synth.random_complex_block(p.n_kvc, 64, seed=4)
    idx = np.array([37])
    j = np.array([21])
    L = 3
    with _ctx(p) as ctx:
        ox, oy = ctx.matvec_rpa(X, Y)
        a, b, n2, ln = ctx.lanczos(64, L, 64, 0)
        sig, _ = ctx.selfenergy(p.omega, DLT, 64)
        ctx.set_approximation(gwl.GWL_TDA)
        Ax = ctx.matvec(X)
    rx, ry = rpa.omega_hat_factored(p.psi_v, p.psi_cq, p.V, delta, X[idx], Y[idx])
    scale = max(np.abs(rx).max(), np.abs(ry).max())
    assert np.abs(ox[idx] - rx).max() <= 1e-12 * scale and np.abs(oy[idx] - ry).max() <= 1e-12 * scale
    # A x is the upper half of Omega^ [x; 0]: by linearity rx = A x + B y, so compare A x with rx - B y through a second product
    zx, _ = rpa.omega_hat_factored(p.psi_v, p.psi_cq, p.V, delta, X[idx], np.zeros_like(Y[idx]))
    assert _relmax(Ax[idx], zx) <= 1e-12
    r0 = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, p.chains[j], L, p.omega, DLT, reorth=False)
    bs = np.abs(r0["beta"]).max()
    assert abs(n2[j[0]] - r0["norm2"][0]) <= 1e-12 * r0["norm2"][0]
    assert np.abs(a[j] - r0["alpha"]).max() <= 1e-9 * bs
    assert (np.abs(b[j] - r0["beta"]) <= 1e-9 * np.abs(r0["beta"])).all()
    assert np.abs(sig[j] - r0["sigma"]).max() <= 1e-6


def test_tdc_selfenergy_state_both_approximations():
    """gwl_tdc_selfenergy_state: all n of one slot, Eq. 10-like sum on the device, Tamm-Dancoff and RPA, against the oracles."""
    p = synth.make_periodic(2, 3, 7, 48, seed=13, n_omega=81)
    n_orb = p.n_v + p.n_c
    kn, km, m, L = 1, 0, p.n_v - 1, 14
    chains = np.array([(kn, n, km, m) for n in range(n_orb)], dtype=np.int32)
    with _ctx(p, n_q=2, chains=False) as ctx:
        s_rpa = ctx.selfenergy_state(kn, km, m, L, 4, 1, p.omega, DLT)          # blocks of 4, 4, 2
        ctx.set_approximation(gwl.GWL_TDA)
        s_tda = ctx.selfenergy_state(kn, km, m, L, 16, 1, p.omega, DLT)
    r_rpa = rpa.run_chains_rpa(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, chains, L, p.omega, DLT, n_q=2, reorth=True)
    r_tda = tdp.run_chains(p.psi_v, p.psi_cq, p.eps_v, p.eps_cq, p.V, chains, L, p.omega, DLT, n_q=2, reorth=True)
    assert np.abs(s_rpa - r_rpa["sigma_sum"]).max() <= 1e-6
    assert np.abs(s_tda - r_tda["sigma_sum"]).max() <= 1e-6
    assert np.abs(s_rpa - s_tda).max() > 1e-4                                     # the two approximations differ
