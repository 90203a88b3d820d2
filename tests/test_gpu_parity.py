"""GPU parity: the CUDA path (through the C ABI of libgwl.so) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json:north_star, protocol of SURVEY.md §8(c)):
  matvec            max|y_gpu - y_cpu| / max|y_cpu| <= 1e-12
  alpha/beta[:30]   element-wise relative <= 1e-9, reorthogonalisation off
  Sigma^c(omega)    absolute <= 1e-6 eV over the whole grid, reorthogonalisation on, on both sides
"""
import numpy as np
import pytest

from oracle import gw_oracle as orc
from paper_2310_20103_b200 import gwl, synth

pytestmark = pytest.mark.gpu

TOL_MATVEC = 1e-12
TOL_AB = 1e-9
TOL_SIGMA = 1e-6
DLT = 0.1


def _ctx(p, chains=True):
    ctx = gwl.Context(p.cfg.n_v, p.cfg.n_c, p.cfg.n_mu)
    ctx.set_orbitals(p.phi_v, p.phi_c)
    ctx.set_energies(p.eps_v, p.eps_c)
    ctx.set_kernel(p.V)
    if chains:
        ctx.set_chains(p.n_idx, p.m_idx)
    return ctx


def _relmax(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def _oracle_matvec(p, X):
    return orc.casida_matvec_factored(p.phi_v, p.phi_c, p.V, orc.delta_vc(p.eps_v, p.eps_c), X)


@pytest.fixture(scope="module")
def p0():
    p = synth.make_problem(0)
    _ = p.V
    return p


@pytest.fixture(scope="module")
def p1():
    p = synth.make_problem(1)
    _ = p.V
    return p


# ---- S2: Casida block product ------------------------------------------------------------------
@pytest.mark.parametrize("nvec", [1, 4, 7])
def test_matvec_config0(p0, nvec):
    X = synth.random_block(p0.cfg, nvec)
    with _ctx(p0, chains=False) as ctx:
        Y = ctx.casida_matvec(X)
    assert Y.shape == X.shape
    assert _relmax(Y, _oracle_matvec(p0, X)) <= TOL_MATVEC


@pytest.mark.parametrize("n_v,n_c,n_mu,nvec", [(1, 1, 1, 1), (3, 5, 37, 3), (5, 19, 130, 70), (2, 33, 257, 130),
                                                (7, 16, 48, 300)])
def test_matvec_ragged_sizes(n_v, n_c, n_mu, nvec):
    """Odd N_c (unaligned rows), N_mu and N_c not multiples of the tiles, block wider than one N tile,
    and nvec > 256 (two chunks)."""
    p = synth.make_custom(n_v, n_c, n_mu, seed=n_mu)
    X = synth.random_block(p.cfg, nvec, seed=2)
    with _ctx(p, chains=False) as ctx:
        Y = ctx.casida_matvec(X)
    assert _relmax(Y, _oracle_matvec(p, X)) <= TOL_MATVEC


def test_matvec_zero_kernel_is_exact(p0):
    X = synth.random_block(p0.cfg, 3)
    with gwl.Context(p0.cfg.n_v, p0.cfg.n_c, p0.cfg.n_mu) as ctx:
        ctx.set_orbitals(p0.phi_v, p0.phi_c)
        ctx.set_energies(p0.eps_v, p0.eps_c)
        ctx.set_kernel(np.zeros_like(p0.V))
        Y = ctx.casida_matvec(X)
    d = orc.delta_vc(p0.eps_v, p0.eps_c).reshape(p0.cfg.n_v, p0.cfg.n_c)
    assert np.array_equal(Y, d * d * X)


def test_matvec_config1_full_block(p1):
    X = synth.random_block(p1.cfg, p1.cfg.block)
    with _ctx(p1, chains=False) as ctx:
        Y = ctx.casida_matvec(X)
        # columns do not depend on what else is in the block
        Y1 = ctx.casida_matvec(X[5:6])
    ref = _oracle_matvec(p1, X)
    assert _relmax(Y, ref) <= TOL_MATVEC
    assert _relmax(Y1, ref[5:6]) <= TOL_MATVEC
    assert _relmax(Y1, Y[5:6]) <= 1e-13
    # symmetry of C through the GPU path: x^T (C y) = y^T (C x)
    a, b = X[0].ravel(), X[1].ravel()
    assert abs(a @ Y[1].ravel() - b @ Y[0].ravel()) <= 1e-11 * abs(a @ Y[1].ravel())


def test_matvec_device_pointer_mode(p0):
    import torch
    X = synth.random_block(p0.cfg, 4)
    with _ctx(p0, chains=False) as ctx:
        ctx.set_pointer_mode(1)
        ctx.set_stream(torch.cuda.current_stream().cuda_stream)
        xd = torch.from_numpy(X).cuda()
        yd = torch.empty_like(xd)
        ctx.casida_matvec(xd, yd)
        torch.cuda.synchronize()
        Y = yd.cpu().numpy()
    assert _relmax(Y, _oracle_matvec(p0, X)) <= TOL_MATVEC


# ---- S1 + S4: start vectors and Lanczos --------------------------------------------------------------
def _oracle_chains(p, idx, steps, reorth, poly=None):
    return orc.run_chains(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, p.n_idx[idx], p.m_idx[idx], steps,
                          p.omega, DLT, reorth=reorth, poly=poly)


def _check_ab(a, b, ra, rb, upto):
    assert np.abs(a[:, :upto] - ra[:, :upto]).max() <= TOL_AB * np.abs(ra[:, :upto]).max()
    assert (np.abs(a[:, :upto] - ra[:, :upto]) <= TOL_AB * np.abs(ra[:, :upto])).all()
    assert (np.abs(b[:, :upto] - rb[:, :upto]) <= TOL_AB * np.abs(rb[:, :upto])).all()


def test_lanczos_config0_first30_no_reorth(p0):
    cfg = p0.cfg
    with _ctx(p0) as ctx:
        a, b, n2, ln = ctx.lanczos(cfg.n_chains, cfg.steps, cfg.block, reorth=0)
    ref = _oracle_chains(p0, slice(None), cfg.steps, False)
    assert (np.abs(n2 - ref["norm2"]) <= 1e-12 * ref["norm2"]).all()
    assert (ln == cfg.steps).all()
    _check_ab(a, b, ref["alpha"], ref["beta"], 30)


def test_lanczos_and_sigma_config0_reorth(p0):
    cfg = p0.cfg
    with _ctx(p0) as ctx:
        a, b, n2, ln = ctx.lanczos(cfg.n_chains, cfg.steps, cfg.block, reorth=1)
        sig, ssum = ctx.selfenergy(p0.omega, DLT, cfg.n_chains)
    ref = _oracle_chains(p0, slice(None), cfg.steps, True)
    _check_ab(a, b, ref["alpha"], ref["beta"], cfg.steps)
    assert np.abs(sig - ref["sigma"]).max() <= TOL_SIGMA
    assert np.abs(ssum - ref["sigma_sum"]).max() <= TOL_SIGMA


def test_sigma_config0_30_steps_no_reorth(p0):
    cfg = p0.cfg
    with _ctx(p0) as ctx:
        ctx.lanczos(cfg.n_chains, 30, cfg.block, reorth=0)
        sig, _ = ctx.selfenergy(p0.omega, DLT, cfg.n_chains)
    ref = _oracle_chains(p0, slice(None), 30, False)
    assert np.abs(sig - ref["sigma"]).max() <= TOL_SIGMA


def test_short_last_block_and_block_invariance(p0):
    """n_chains not a multiple of block; chain j gives the same tridiagonal whatever block it runs in (Q10)."""
    with _ctx(p0) as ctx:
        a4, b4, n4, _ = ctx.lanczos(4, 25, 4, reorth=0)
        a3, b3, n3, _ = ctx.lanczos(4, 25, 3, reorth=0)      # blocks of 3 + 1
        a1, b1, n1, _ = ctx.lanczos(4, 25, 1, reorth=0)
        a2, _, _, _ = ctx.lanczos(2, 25, 4, reorth=0)        # fewer chains than were set
    for x, y in [(a3, a4), (b3, b4), (a1, a4), (b1, b4), (n3, n4), (n1, n4), (a2, a4[:2])]:
        assert (np.abs(x - y) <= 1e-10 * np.abs(y)).all()


def test_negative_sign_chains_and_eq10_sum(p0):
    """m = highest valence, n over all N_v + N_c orbitals: exercises eta_n = -1 and the Eq. 10 sum."""
    cfg = p0.cfg
    n_idx = np.arange(cfg.n_v + cfg.n_c, dtype=np.int32)
    m_idx = np.full_like(n_idx, cfg.n_v - 1)
    L = 40
    with _ctx(p0, chains=False) as ctx:
        ctx.set_chains(n_idx, m_idx)
        a, b, n2, ln = ctx.lanczos(len(n_idx), L, 12, reorth=1)
        sig, ssum = ctx.selfenergy(p0.omega, DLT, len(n_idx))
    ref = orc.run_chains(p0.phi_v, p0.phi_c, p0.eps_v, p0.eps_c, p0.V, n_idx, m_idx, L, p0.omega, DLT, reorth=True)
    _check_ab(a, b, ref["alpha"], ref["beta"], L)
    assert np.abs(sig - ref["sigma"]).max() <= TOL_SIGMA
    assert np.abs(ssum - ref["sigma_sum"]).max() <= TOL_SIGMA
    assert (sig[: cfg.n_v].imag > 0).all() and (sig[cfg.n_v:].imag < 0).all()        # Herglotz sign per eta_n


def test_explicit_start_vectors_equal_index_chains(p0):
    cfg = p0.cfg
    delta = orc.delta_vc(p0.eps_v, p0.eps_c)
    P = np.array([orc.start_vector(p0.phi_v, p0.phi_c, p0.V, delta, int(n), int(m))
                  for n, m in zip(p0.n_idx, p0.m_idx)])
    es = [orc.orbital_energy_sign(p0.eps_v, p0.eps_c, int(n)) for n in p0.n_idx]
    with _ctx(p0) as ctx:
        a, b, n2, _ = ctx.lanczos(4, 20, 4, 0)
        s_idx, _ = ctx.selfenergy(p0.omega, DLT, 4)
        ctx.set_start_vectors(P, [e for e, _ in es], [s for _, s in es])
        a2, b2, n22, _ = ctx.lanczos(4, 20, 4, 0)
        s_vec, _ = ctx.selfenergy(p0.omega, DLT, 4)
    assert (np.abs(n2 - (P * P).sum(axis=1)) <= 1e-12 * n2).all()
    assert (np.abs(a - a2) <= 1e-10 * np.abs(a)).all() and (np.abs(b - b2) <= 1e-10 * np.abs(b)).all()
    assert np.abs(s_idx - s_vec).max() <= 1e-9


def test_breakdown_and_zero_start_vector():
    """Q9: with V = 0 the operator is diagonal; a start vector with 3 nonzeros spans a 3-dimensional invariant
    subspace -> len = 3, zero-filled tail; a zero start vector gives len = 0 and Sigma = 0."""
    p = synth.make_custom(2, 3, 16, seed=9)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    P = np.zeros((3, 6))
    P[0, [0, 2, 5]] = [1.0, 2.0, -1.0]
    P[2] = np.arange(1, 7)
    with gwl.Context(2, 3, 16) as ctx:
        ctx.set_orbitals(p.phi_v, p.phi_c)
        ctx.set_energies(p.eps_v, p.eps_c)
        ctx.set_kernel(np.zeros((16, 16)))
        ctx.set_start_vectors(P, [-6.0, -6.0, 1.0], [1, 1, -1])
        a, b, n2, ln = ctx.lanczos(3, 6, 3, 0)
        sig, _ = ctx.selfenergy(p.omega, DLT, 3)
        r = ctx.resolvent(np.array([1.0 + 1.0j, -5.0 + 0.2j]), 3)
    assert list(ln) == [3, 0, 6]
    assert (a[0, 3:] == 0).all() and (b[0, 2:] == 0).all() and (a[1] == 0).all() and n2[1] == 0
    ra, rb, rn2, rl = orc.lanczos(lambda x: delta ** 2 * x, P[0], 6)
    assert rl == 3 and np.abs(a[0] - ra).max() <= 1e-9 * np.abs(ra).max() and np.abs(b[0] - rb).max() <= 1e-9 * np.abs(ra).max()
    assert (sig[1] == 0).all() and (r[1] == 0).all()
    ref = orc.sigma_direct(ra, rb, rn2, rl, p.omega, -6.0, 1, DLT)
    assert np.abs(sig[0] - ref).max() <= TOL_SIGMA
    z = np.array([1.0 + 1.0j, -5.0 + 0.2j])
    exact = (P[0] ** 2 / (z[:, None] - delta[None, :] ** 2)).sum(axis=1)        # P11 closed form
    assert np.abs(r[0] - exact).max() <= 1e-10 * np.abs(exact).max()


def test_resolvent_matches_oracle_continued_fraction(p0):
    cfg = p0.cfg
    zeta = (p0.omega[::10] + 1j * DLT) ** 2
    with _ctx(p0) as ctx:
        a, b, n2, ln = ctx.lanczos(4, 30, 4, 0)
        r = ctx.resolvent(zeta, 4)
    for j in range(4):
        ref = orc.continued_fraction(a[j], b[j], n2[j], zeta, ln[j])
        assert np.abs(r[j] - ref).max() <= 1e-11 * np.abs(ref).max()


def test_poly_mode_config0(p0):
    """The paper's route: Lanczos on p_g(C), Sigma by Eq. 12 + Eq. 14; g = 7 and 8, N_iter = 8."""
    delta = orc.delta_vc(p0.eps_v, p0.eps_c)
    lo, hi = 0.8 * (delta ** 2).min(), 1.25 * (delta ** 2).max()
    for g in (7, 8):
        c = orc.fit_sqrt_chebyshev(g, lo, hi)
        with _ctx(p0) as ctx:
            ctx.set_polynomial(g, c, lo, hi)
            a, b, n2, ln = ctx.lanczos(4, 8, 4, 0)
            sig, ssum = ctx.selfenergy(p0.omega, DLT, 4)
            ctx.set_polynomial(0)
            a_dir, _, _, _ = ctx.lanczos(4, 8, 4, 0)
        ref = _oracle_chains(p0, slice(None), 8, False, poly=(c, lo, hi))
        _check_ab(a, b, ref["alpha"], ref["beta"], 8)
        assert np.abs(sig - ref["sigma"]).max() <= TOL_SIGMA
        assert np.abs(ssum - ref["sigma_sum"]).max() <= TOL_SIGMA
        assert np.abs(a_dir - a).max() > 1.0          # clearing the polynomial really switches back to Op = C


def test_lanczos_config1_first30_all_chains_no_reorth(p1):
    """Protocol item 2 at config 1: ALL 64 chains in the block of 64 bench.py times, reorthogonalisation off: the first
    30 alpha/beta of every chain to 1e-9, and Sigma of the 30-step tridiagonals to 1e-6 eV."""
    cfg = p1.cfg
    with _ctx(p1) as ctx:
        a, b, n2, ln = ctx.lanczos(cfg.n_chains, 30, cfg.block, 0)
        sig30, ssum = ctx.selfenergy(p1.omega, DLT, cfg.n_chains)
    ref = _oracle_chains(p1, slice(None), 30, False)
    assert (np.abs(n2 - ref["norm2"]) <= 1e-12 * ref["norm2"]).all()
    _check_ab(a, b, ref["alpha"], ref["beta"], 30)
    assert np.abs(sig30 - ref["sigma"]).max() <= TOL_SIGMA
    assert np.abs(ssum - ref["sigma_sum"]).max() <= TOL_SIGMA * cfg.n_chains


def test_sigma_config1_all_chains_full_length_reorth(p1):
    """Protocol item 3 at full strength: Sigma^c <= 1e-6 eV with two-pass reorthogonalisation on BOTH sides on ALL 64
    chains of config 1 at its FULL L = 200 (and alpha/beta to 1e-9 over all 200 steps)."""
    cfg = p1.cfg
    with _ctx(p1) as ctx:
        a, b, n2, ln = ctx.lanczos(cfg.n_chains, cfg.steps, cfg.block, 1)
        sig, ssum = ctx.selfenergy(p1.omega, DLT, cfg.n_chains)
    ref = _oracle_chains(p1, slice(None), cfg.steps, True)
    assert (ln == ref["len"]).all()
    _check_ab(a, b, ref["alpha"], ref["beta"], cfg.steps)
    assert np.abs(sig - ref["sigma"]).max() <= TOL_SIGMA
    assert np.abs(ssum - ref["sigma_sum"]).max() <= TOL_SIGMA * cfg.n_chains


def test_block_invariance_config1(p1):
    """Reading Q10 at config 1: chain j inside the block of 64 (fused cluster update, stream-K K^T.W) equals chain j run
    alone and in a block of 5 (other tile counts and split-K plans), reorthogonalisation off, 25 steps."""
    cfg = p1.cfg
    js = np.array([0, 21, 40, 62, 63])
    with _ctx(p1) as ctx:
        a64, b64, n64, _ = ctx.lanczos(cfg.n_chains, 25, cfg.block, 0)
        ctx.set_chains(p1.n_idx[js], p1.m_idx[js])
        a5, b5, n5, _ = ctx.lanczos(5, 25, 5, 0)
        a1, b1, n1, _ = ctx.lanczos(5, 25, 1, 0)
    for x, y in [(a5, a64[js]), (b5, b64[js]), (n5, n64[js]), (a1, a64[js]), (b1, b64[js]), (n1, n64[js])]:
        assert (np.abs(x - y) <= 1e-10 * np.abs(y)).all()


# ---- API behaviour -------------------------------------------------------------------------------------
def test_state_and_argument_errors(p0):
    cfg = p0.cfg
    with gwl.Context(cfg.n_v, cfg.n_c, cfg.n_mu) as ctx:
        with pytest.raises(gwl.GwlError) as e:
            ctx.casida_matvec(np.zeros((1, cfg.n_v, cfg.n_c)))
        assert e.value.status == gwl.GWL_ESTATE
        with pytest.raises(gwl.GwlError) as e:
            ctx.set_energies(p0.eps_v, p0.eps_c - 100.0)              # eps_c below eps_v
        assert e.value.status == gwl.GWL_EINVAL and "eps" in str(e.value)
        ctx.set_orbitals(p0.phi_v, p0.phi_c)
        ctx.set_energies(p0.eps_v, p0.eps_c)
        ctx.set_kernel(p0.V)
        with pytest.raises(gwl.GwlError) as e:
            ctx.lanczos(1, 5, 1, 0)                                   # no chains set
        assert e.value.status == gwl.GWL_ESTATE
        with pytest.raises(gwl.GwlError) as e:
            ctx.selfenergy(p0.omega, DLT, 1)                          # before lanczos
        assert e.value.status == gwl.GWL_ESTATE
        with pytest.raises(gwl.GwlError):
            ctx.set_chains([0], [cfg.n_v + cfg.n_c])                  # index out of range
        ctx.set_chains(p0.n_idx, p0.m_idx)
        with pytest.raises(gwl.GwlError):
            ctx.lanczos(5, 5, 1, 0)                                   # more chains than set
        with pytest.raises(gwl.GwlError):
            ctx.lanczos(1, 0, 1, 0)                                   # steps < 1
        with pytest.raises(gwl.GwlError) as e:
            ctx.lanczos(1, 8193, 1, 1)                                # reorth beyond GWL_MAX_REORTH_STEPS: named, not ECUDA
        assert e.value.status == gwl.GWL_EINVAL and "GWL_MAX_REORTH_STEPS" in str(e.value)
        a, b, n2, ln = ctx.lanczos(0, 5, 4, 0)                        # empty run is fine
        assert a.shape == (0, 5)
        assert ctx.casida_matvec(np.zeros((0, cfg.n_v, cfg.n_c))).shape == (0, cfg.n_v, cfg.n_c)
        assert ctx.get_launch_count() > 0


def test_sqrt_fit_range_heuristic_and_lanczos(p0):
    """gwl_sqrt_fit_range: steps = 0 is the paper's heuristic [0.8 min Delta^2, 1.25 max Delta^2] (Q12);
    steps > 0 takes hi from the Lanczos estimate, against the oracle's own bound on the oracle's product."""
    delta = orc.delta_vc(p0.eps_v, p0.eps_c)
    with _ctx(p0, chains=False) as ctx:
        lo, hi = ctx.sqrt_fit_range(0)
        assert abs(lo - 0.8 * (delta ** 2).min()) <= 1e-12 * lo and abs(hi - 1.25 * (delta ** 2).max()) <= 1e-12 * hi
        lo2, hi2 = ctx.sqrt_fit_range(40, 0.02)
    _, top = orc.spectrum_bounds_lanczos(
        lambda x: orc.casida_matvec_factored(p0.phi_v, p0.phi_c, p0.V, delta, x[None])[0], delta.size, 40)
    assert lo2 == lo and abs(hi2 - 1.02 * max(top, (delta ** 2).max())) <= 1e-6 * hi2


def test_spectrum_bounds_after_breakdown_match_the_oracle():
    """Breakdown inside the range probe: with V = 0 and only three distinct Delta the Krylov space of any start vector is
    three-dimensional, the fourth beta vanishes, and the bounds are the exact extreme eigenvalues min / max Delta^2 with a
    zero residual term -- on the GPU (b_last = 0 when len < steps) and in the oracle (beta[len-1] stored as 0) alike."""
    p = synth.make_custom(4, 6, 16, seed=2)
    eps_v = np.full(4, -7.0)
    eps_c = np.array([1.0, 1.0, 2.5, 2.5, 6.0, 6.0])
    delta = orc.delta_vc(eps_v, eps_c)
    with gwl.Context(4, 6, 16) as ctx:
        ctx.set_orbitals(p.phi_v, p.phi_c)
        ctx.set_energies(eps_v, eps_c)
        ctx.set_kernel(np.zeros((16, 16)))
        lo, hi = ctx.spectrum_bounds(10)
    olo, ohi = orc.spectrum_bounds_lanczos(lambda x: delta ** 2 * x, delta.size, 10)
    for got in ((lo, hi), (olo, ohi)):
        assert abs(got[0] - 64.0) <= 1e-10 * 64.0 and abs(got[1] - 169.0) <= 1e-10 * 169.0


def test_launches_and_timing_reported(p0):
    with _ctx(p0) as ctx:
        n0 = ctx.get_launch_count()
        ctx.lanczos(4, 10, 4, 0)
        assert ctx.get_launch_count() - n0 >= 10 * 5
        tm, tv, tt = ctx.get_timing()
        assert tm > 0 and tv > 0 and abs(tt - tm - tv) < 1e-9


# ---- one whole quasiparticle state ---------------------------------------------------
def test_state_selfenergy_exchange_and_qp_solve_config0(p0):
    """Sigma^corr_mm over all 32 chains (Eq. 10), Sigma^ex (Eq. 6) and the Newton-Raphson solve of
    E(omega) = omega for the HOMO and the LUMO, reorthogonalisation on both sides."""
    cfg = p0.cfg
    L = 40
    states = [cfg.n_v - 1, cfg.n_v]
    vxc = np.array([-9.0, -7.5])
    with _ctx(p0, chains=False) as ctx:
        sx = ctx.exchange(states)
        sc = np.array([ctx.selfenergy_state(m, L, 12, 1, p0.omega, DLT) for m in states])
        eps_m = np.array([p0.eps_v[-1], p0.eps_c[0]])
        eq, zq, it = ctx.qp_solve(eps_m, vxc, sx, sc, p0.omega)
    for k, m in enumerate(states):
        rx = orc.exchange_eq6(p0.phi_v, p0.phi_c, p0.V, m)
        rc = orc.sigma_state(p0.phi_v, p0.phi_c, p0.eps_v, p0.eps_c, p0.V, m, L, p0.omega, DLT, reorth=True)
        assert abs(sx[k] - rx) <= 1e-12 * abs(rx)
        assert np.abs(sc[k] - rc).max() <= TOL_SIGMA
        re, rz, rit = orc.qp_solve(eps_m[k], vxc[k], rx, rc, p0.omega)
        assert abs(eq[k] - re) <= TOL_SIGMA and abs(zq[k] - rz) <= 1e-6 and it[k] == rit
        # and on identical inputs (the oracle's Sigma) the solver agrees to rounding
    with _ctx(p0, chains=False) as ctx:
        rc = np.array([orc.sigma_state(p0.phi_v, p0.phi_c, p0.eps_v, p0.eps_c, p0.V, m, 10, p0.omega, DLT) for m in states])
        rx = np.array([orc.exchange_eq6(p0.phi_v, p0.phi_c, p0.V, m) for m in states])
        eq, zq, it = ctx.qp_solve(eps_m, vxc, rx, rc, p0.omega)
    for k in range(2):
        re, rz, rit = orc.qp_solve(eps_m[k], vxc[k], rx[k], rc[k], p0.omega)
        assert abs(eq[k] - re) <= 1e-12 and abs(zq[k] - rz) <= 1e-12 and it[k] == rit


def test_exchange_many_occupied_orbitals_two_chunks():
    """N_v > 256: the sum over v runs in two GEMM chunks; N_mu not a multiple of the tile."""
    p = synth.make_custom(300, 2, 70, seed=4)
    m = [0, 299, 301]
    with _ctx(p, chains=False) as ctx:
        sx = ctx.exchange(m)
    ref = np.array([orc.exchange_eq6(p.phi_v, p.phi_c, p.V, k) for k in m])
    assert (np.abs(sx - ref) <= 1e-12 * np.abs(ref)).all()


def test_qp_solve_device_pointer_mode_and_clamp(p0):
    import torch
    om = torch.linspace(-20, 20, 101, dtype=torch.float64, device="cuda")
    sc = torch.zeros(2, 101, 2, dtype=torch.float64, device="cuda")
    sc[0, :, 0] = -0.5 - 0.25 * om
    sx = torch.tensor([-4.0, 0.0], dtype=torch.float64, device="cuda")
    eq = torch.zeros(2, dtype=torch.float64, device="cuda")
    zq = torch.zeros_like(eq)
    it = torch.zeros(2, dtype=torch.int32, device="cuda")
    with gwl.Context(2, 2, 8) as ctx:
        ctx.set_pointer_mode(1)
        ctx.set_stream(torch.cuda.current_stream().cuda_stream)
        ctx.qp_solve([-6.0, 500.0], [-5.0, 0.0], sx, sc, om, out=(eq, zq, it))
        torch.cuda.synchronize()
    assert abs(eq[0].item() - (-6.0 - 4.0 - 0.5 + 5.0) / 1.25) <= 1e-12 and abs(zq[0].item() - 0.8) <= 1e-12
    assert eq[1].item() == 20.0                                   # root outside the grid: clamped


# ---- Ritz kernel (divide and conquer) on tridiagonals with ghost clusters ----------------------------------
@pytest.mark.parametrize("L", [1, 2, 3, 37, 192, 300])
def test_ritz_quadrature_on_gpu_tridiagonals(p0, L):
    """Direct-mode Sigma from the GPU's own alpha/beta against the oracle's Ritz evaluation (LAPACK) of the SAME
    tridiagonal: isolates S6.  L = 192, 300 without reorthogonalisation: T_L is full of ghost copies (tight clusters,
    heavy deflation); L = 300 > 256 threads; L = 1, 2, 3: degenerate trees."""
    cfg = p0.cfg
    with _ctx(p0) as ctx:
        a, b, n2, ln = ctx.lanczos(cfg.n_chains, L, cfg.block, 0)
        sig, _ = ctx.selfenergy(p0.omega, DLT, cfg.n_chains)
    for j in range(cfg.n_chains):
        e_n, sg = orc.orbital_energy_sign(p0.eps_v, p0.eps_c, int(p0.n_idx[j]))
        ref = orc.sigma_direct(a[j], b[j], n2[j], int(ln[j]), p0.omega, e_n, sg, DLT)
        assert np.abs(sig[j] - ref).max() <= 1e-9


def test_ritz_ql_fallback_above_dc_limit(p0):
    """L above the divide-and-conquer kernel's shared-memory limit (about 1500): gwl_selfenergy falls back to the
    sequential implicit-QL kernel (k_ritz).  Config 0 without reorthogonalisation at L = 1700 (N_vc = 192: the
    tridiagonal is almost all ghost copies), Sigma against LAPACK on the GPU's own tridiagonal."""
    cfg = p0.cfg
    L = 1700
    with _ctx(p0) as ctx:
        a, b, n2, ln = ctx.lanczos(2, L, 2, 0)
        sig, _ = ctx.selfenergy(p0.omega, DLT, 2)
    assert (ln == L).all()
    for j in range(2):
        e_n, sg = orc.orbital_energy_sign(p0.eps_v, p0.eps_c, int(p0.n_idx[j]))
        ref = orc.sigma_direct(a[j], b[j], n2[j], int(ln[j]), p0.omega, e_n, sg, DLT)
        assert np.abs(sig[j] - ref).max() <= 1e-9


# ---- fitting range of p_g from the spectrum of C ------------------------------------------------
def _strongly_coupled():
    """N_vc / N_mu = 12 in a 6 A box: lambda_max(C) ~ 2555 eV^2, far above the heuristic 1.25 max Delta^2 ~ 1054."""
    p = synth.make_custom(16, 48, 64, box=6.0, seed=3, chains_a=2, chains_b=2)
    _ = p.V
    return p


def test_spectrum_bounds_against_full_diagonalisation():
    p = _strongly_coupled()
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    lam = np.linalg.eigvalsh(orc.casida_dense(delta, orc.coupling_dense(orc.khatri_rao(p.phi_v, p.phi_c), p.V)))
    assert lam[-1] > 2.0 * 1.25 * (delta ** 2).max()                 # the heuristic range does not hold this spectrum
    with _ctx(p, chains=False) as ctx:
        lo40, hi40 = ctx.spectrum_bounds(40)
        lo2, hi2 = ctx.spectrum_bounds(2)
        with pytest.raises(gwl.GwlError):
            ctx.lanczos(1, 5, 1, 0)                                   # the probe chain is not left behind
        ra = orc.spectrum_bounds_lanczos(lambda x: orc.casida_matvec_factored(p.phi_v, p.phi_c, p.V, delta, x[None])[0],
                                         delta.size, 40)
    # the separated top eigenvalue has converged after 40 steps: upper bound tight from above
    assert lam[-1] * (1 - 1e-10) <= hi40 <= lam[-1] * (1 + 1e-6)
    assert abs(hi40 - ra[1]) <= 1e-6 * lam[-1]                        # the oracle's own 40-step estimate agrees
    span = lam[-1] - lam[0]
    assert lam[0] - span <= lo40 <= lam[0] + 0.1 * span               # lower end: an estimate only (dense edge)
    assert lam[0] <= hi2 <= lam[-1] + span and lo2 <= lam[-1]         # two steps: a wide but sane interval


def test_poly_mode_strongly_coupled_range_from_spectrum():
    """The paper's route where the heuristic fitting range fails (N_vc = 96, lambda_max(C) ~ 2138 eV^2 against
    1.25 max Delta^2 ~ 779): range from gwl_spectrum_bounds (polyfit.range_from_spectrum), g = 12, full-length Lanczos
    with reorthogonalisation.  GPU against the oracle on the ORACLE's fit over the same range, and against the exact
    Eq. 7 (full diagonalisation) within the bound the fit error eps = max_s |p_g(Omega_s^2) - Omega_s| allows:
    |dSigma| <= <P|P> eps (1/(Omega_min (Omega_min - eps)) + 1/delta^2) / delta."""
    from paper_2310_20103_b200 import polyfit
    p = synth.make_custom(6, 16, 16, box=3.0, seed=3, chains_a=2, chains_b=2)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    C = orc.casida_dense(delta, orc.coupling_dense(orc.khatri_rao(p.phi_v, p.phi_c), p.V))
    lam, Z = orc.eig_casida(C)
    assert lam[-1] > 2.0 * 1.25 * (delta ** 2).max()
    g, L, dl = 12, delta.size, 0.68
    with _ctx(p, chains=False) as ctx:
        lo, hi = polyfit.range_from_spectrum(ctx, p.eps_v, p.eps_c, steps=40)
        ctx.set_polynomial(g, polyfit.sqrt_chebyshev(g, lo, hi), lo, hi)
        ctx.set_chains(p.n_idx, p.m_idx)
        a, b, n2, ln = ctx.lanczos(4, L, 4, 1)
        sig, _ = ctx.selfenergy(p.omega, dl, 4)
    assert lo <= lam[0] and lam[-1] <= hi <= 1.03 * lam[-1]
    c = orc.fit_sqrt_chebyshev(g, lo, hi)
    ref = orc.run_chains(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, p.n_idx, p.m_idx, L, p.omega, dl, reorth=True,
                         poly=(c, lo, hi))
    _check_ab(a, b, ref["alpha"], ref["beta"], 60)
    assert np.abs(sig - ref["sigma"]).max() <= TOL_SIGMA
    eps = np.abs(orc.poly_eval_scalar(c, lo, hi, lam) - np.sqrt(lam)).max()
    o_min = np.sqrt(lam[0])
    for j in range(4):
        P = orc.start_vector(p.phi_v, p.phi_c, p.V, delta, int(p.n_idx[j]), int(p.m_idx[j]))
        e_n, sg = orc.orbital_energy_sign(p.eps_v, p.eps_c, int(p.n_idx[j]))
        exact = orc.sigma_exact_eq7(lam, Z, P, p.omega, e_n, sg, dl)
        bound = (P @ P) * eps * (1.0 / (o_min * (o_min - eps)) + 1.0 / dl ** 2) / dl
        assert np.abs(sig[j] - exact).max() <= bound
    # with the heuristic range the polynomial is evaluated far outside [-1, 1] at the top of the spectrum and diverges
    hlo, hhi = polyfit.default_range(p.eps_v, p.eps_c)
    assert abs(orc.poly_eval_scalar(orc.fit_sqrt_chebyshev(g, hlo, hhi), hlo, hhi, lam[-1])) > 100.0 * np.sqrt(lam[-1])


# ---- SURVEY.md §8(f)-3, first step: Tamm-Dancoff approximation (operator A) ------------------------------
def test_tda_mode_config0(p0):
    cfg = p0.cfg
    delta = orc.delta_vc(p0.eps_v, p0.eps_c)
    X = synth.random_block(cfg, 5)
    n_idx = np.array([0, 3, cfg.n_v, cfg.n_v + 5], dtype=np.int32)      # two occupied, two empty n
    m_idx = np.full_like(n_idx, cfg.n_v - 1)
    with _ctx(p0, chains=False) as ctx:
        y_rpa = ctx.casida_matvec(X)
        ctx.set_approximation(gwl.GWL_TDA)
        y = ctx.casida_matvec(X)
        ctx.set_chains(n_idx, m_idx)
        a, b, n2, ln = ctx.lanczos(4, 50, 3, 1)
        sig, ssum = ctx.selfenergy(p0.omega, DLT, 4)
        r = ctx.resolvent(np.array([3.0 + 0.5j]), 4)
        with pytest.raises(gwl.GwlError):
            ctx.set_polynomial(2, np.ones(3), 1.0, 2.0)               # sqrt(C) fit has no meaning for A
        ctx.set_approximation(gwl.GWL_RPA)
        with pytest.raises(gwl.GwlError):
            ctx.selfenergy(p0.omega, DLT, 4)                          # switching invalidates the last run
        y_back = ctx.casida_matvec(X)
    ref_y = orc.tda_matvec_factored(p0.phi_v, p0.phi_c, p0.V, delta, X.reshape(5, -1)).reshape(X.shape)
    assert _relmax(y, ref_y) <= TOL_MATVEC
    assert np.array_equal(y_back, y_rpa) and _relmax(y, y_rpa) > 1e-2
    ref = orc.run_chains_tda(p0.phi_v, p0.phi_c, p0.eps_v, p0.eps_c, p0.V, n_idx, m_idx, 50, p0.omega, DLT, reorth=True)
    assert (np.abs(n2 - ref["norm2"]) <= 1e-12 * ref["norm2"]).all()
    _check_ab(a, b, ref["alpha"], ref["beta"], 50)
    assert np.abs(sig - ref["sigma"]).max() <= TOL_SIGMA
    assert np.abs(ssum - ref["sigma_sum"]).max() <= TOL_SIGMA
    for j in range(4):
        rr = orc.continued_fraction(a[j], b[j], n2[j], np.array([3.0 + 0.5j]), ln[j])
        assert abs(r[j, 0] - rr[0]) <= 1e-11 * abs(rr[0])


def test_runs_are_bitwise_repeatable(p1):
    """Every reduction has a fixed order (split-K, stream-K hand-over, cluster norm, dot partials): two runs of the
    same problem give identical bits -- also a cheap detector of races in the flag/workspace hand-over."""
    cfg = p1.cfg
    outs = []
    with _ctx(p1) as ctx:
        for _ in range(3):
            a, b, n2, ln = ctx.lanczos(cfg.n_chains, 25, cfg.block, 0)
            sig, _ = ctx.selfenergy(p1.omega, DLT, cfg.n_chains)
            outs.append((a, b, n2, sig))
    X = synth.random_block(cfg, cfg.block)
    with _ctx(p1, chains=False) as ctx:
        ys = [ctx.casida_matvec(X) for _ in range(3)]
    for o in outs[1:]:
        assert all(np.array_equal(x, y) for x, y in zip(o, outs[0]))
    assert np.array_equal(ys[0], ys[1]) and np.array_equal(ys[0], ys[2])


def test_step_graph_replay_is_bitwise_identical(p0, p1):
    """Small problems (fused-update path) replay the step loop from a CUDA graph of six steps when no per-step events are
    recorded (profiling level 0): same kernels, same order, same arguments apart from the device-resident step counter, so
    alpha, beta, <P|P>, len and Sigma are IDENTICAL to the plain launches -- in direct mode, in poly mode, for several
    blocks, for chain lengths with every remainder mod 6, on a cache hit and after switching back to plain launches
    (the stream-K epochs of captured launches restart in every replay).  The launch count shows that the graph ran."""
    from paper_2310_20103_b200 import polyfit
    for prob, L0 in ((p0, 60), (p1, 40)):
        cfg = prob.cfg
        nch = cfg.n_chains
        with _ctx(prob) as ctx:
            for (L, blk, poly) in ((L0, cfg.block, False), (L0 + 1, cfg.block, False), (L0 + 3, max(2, cfg.block // 2), False),
                                   (18, cfg.block, True)):
                if poly:
                    lo, hi = polyfit.range_from_spectrum(ctx, prob.eps_v, prob.eps_c, steps=20)
                    ctx.set_polynomial(6, polyfit.sqrt_chebyshev(6, lo, hi), lo, hi)
                    ctx.set_chains(prob.n_idx, prob.m_idx)
                ctx.set_profiling(1)
                n0 = ctx.get_launch_count()
                ref = ctx.lanczos(nch, L, blk, 0)
                sig_ref, _ = ctx.selfenergy(prob.omega, DLT, nch)
                n_plain = ctx.get_launch_count() - n0
                ctx.set_profiling(0)
                for rep in range(2):                                      # capture, then cache hit
                    n0 = ctx.get_launch_count()
                    out = ctx.lanczos(nch, L, blk, 0)
                    sig, _ = ctx.selfenergy(prob.omega, DLT, nch)
                    n_graph = ctx.get_launch_count() - n0
                    assert all(np.array_equal(x, y) for x, y in zip(out, ref)), (cfg.name, L, blk, poly, rep)
                    assert np.array_equal(sig, sig_ref)
                    pfx = (L - 2) % 6 + 2
                    n_blocks = -(-nch // blk)
                    assert n_graph == n_plain + n_blocks * (1 + (L - pfx) // 6)   # set_int + one add_int per replay
                ctx.set_profiling(1)
                again = ctx.lanczos(nch, L, blk, 0)                       # plain launches after the replays
                assert all(np.array_equal(x, y) for x, y in zip(again, ref))


def test_chain_sharded_state_on_one_gpu(p0):
    """SURVEY.md §8(f)-2 on the GPU path: the slices two ranks would take (runtime.shard_range), run one after the
    other on this GPU through runtime.gwl_local_sigma_sum, add up to gwl_selfenergy_state; a single process
    (no process group) passes through."""
    import torch
    from paper_2310_20103_b200 import runtime
    cfg = p0.cfg
    n_orb, m, L = cfg.n_v + cfg.n_c, cfg.n_v - 1, 20
    with _ctx(p0, chains=False) as ctx:
        full_host = ctx.selfenergy_state(m, L, 12, 0, p0.omega, DLT)
        ctx.set_pointer_mode(1)
        ctx.set_stream(torch.cuda.current_stream().cuda_stream)
        om = torch.from_numpy(p0.omega).cuda()
        local = runtime.gwl_local_sigma_sum(ctx, m, L, 12, 0, om, DLT)
        parts = [local(*runtime.shard_range(n_orb, r, 2)) for r in range(2)]
        single = runtime.sharded_sigma_state(local, n_orb)
        torch.cuda.synchronize()
    tot = (parts[0] + parts[1]).cpu().numpy()
    assert np.abs(tot[:, 0] + 1j * tot[:, 1] - full_host).max() <= 1e-11 * np.abs(full_host).max()
    one = single.cpu().numpy()
    assert np.abs(one[:, 0] + 1j * one[:, 1] - full_host).max() <= 1e-11 * np.abs(full_host).max()
    ref = orc.sigma_state(p0.phi_v, p0.phi_c, p0.eps_v, p0.eps_c, p0.V, m, L, p0.omega, DLT)
    assert np.abs(full_host - ref).max() <= TOL_SIGMA


@pytest.mark.parametrize("n_v,n_c,n_mu,L", [(3, 5, 37, 12), (7, 331, 64, 25), (4, 600, 48, 30), (16, 8200, 32, 8)])
def test_reorthogonalised_lanczos_ragged_sizes(n_v, n_c, n_mu, L):
    """Full reorthogonalisation kernels on odd N_vc (scalar loads), on N_vc spanning several 2048-element slices with a
    ragged last slice, on an even N_vc (16-byte loads), and on N_vc = 131 200 > 64 x 2048 (slices longer than the
    shared-memory chunk, as at configs 3-4): alpha/beta and Sigma against the oracle, both sides reorthogonalised."""
    p = synth.make_custom(n_v, n_c, n_mu, seed=n_c, chains_a=2, chains_b=3)
    with _ctx(p) as ctx:
        a, b, n2, ln = ctx.lanczos(6, L, 4, 1)
        sig, _ = ctx.selfenergy(p.omega, DLT, 6)
    ref = orc.run_chains(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, p.n_idx, p.m_idx, L, p.omega, DLT, reorth=True)
    assert (ln == ref["len"]).all()
    _check_ab(a, b, ref["alpha"], ref["beta"], L)
    assert np.abs(sig - ref["sigma"]).max() <= TOL_SIGMA


def test_poly_mode_config1_paper_parameters(p1):
    """The paper's own parameters (g = 7, N_iter = 8) at config 1: full block of 64 chains on the GPU.  The
    fitting range comes from the spectrum: the ORACLE's 40-step Lanczos bound fixes [lo, hi] for both
    sides (inputs flow oracle -> GPU only), the GPU's own gwl_spectrum_bounds must agree with it, and each side fits
    its own Chebyshev coefficients (polyfit.py closed form / oracle lstsq)."""
    from paper_2310_20103_b200 import polyfit
    cfg = p1.cfg
    delta = orc.delta_vc(p1.eps_v, p1.eps_c)
    _, top = orc.spectrum_bounds_lanczos(
        lambda x: orc.casida_matvec_factored(p1.phi_v, p1.phi_c, p1.V, delta, x[None])[0], delta.size, 40)
    lo, hi = 0.8 * (delta ** 2).min(), 1.02 * top
    idx = np.array([0, 37, 63])
    with _ctx(p1, chains=False) as ctx:
        glo, ghi = polyfit.range_from_spectrum(ctx, p1.eps_v, p1.eps_c, steps=40)
        assert abs(glo - lo) <= 1e-12 * lo and abs(ghi - hi) <= 1e-6 * hi
        ctx.set_polynomial(7, polyfit.sqrt_chebyshev(7, lo, hi), lo, hi)
        ctx.set_chains(p1.n_idx, p1.m_idx)
        a, b, n2, ln = ctx.lanczos(cfg.n_chains, 8, cfg.block, 0)
        sig, _ = ctx.selfenergy(p1.omega, DLT, cfg.n_chains)
    ref = _oracle_chains(p1, idx, 8, False, poly=(orc.fit_sqrt_chebyshev(7, lo, hi), lo, hi))
    _check_ab(a[idx], b[idx], ref["alpha"], ref["beta"], 8)
    assert np.abs(sig[idx] - ref["sigma"]).max() <= TOL_SIGMA


def test_state_selfenergy_exchange_and_qp_solve_config1(p1):
    """SURVEY.md §8(f)-1 at a config-1-sized state: all N_v + N_c = 320 chains of the HOMO streamed through blocks of
    64 (L = 24, reorthogonalisation off, inside the window where two FP64 runs agree), Sigma^ex and the
    Newton-Raphson solve against the oracle."""
    cfg = p1.cfg
    m, L = cfg.n_v - 1, 24
    with _ctx(p1, chains=False) as ctx:
        sx = ctx.exchange([m])
        sc = ctx.selfenergy_state(m, L, cfg.block, 0, p1.omega, DLT)
        eq, zq, it = ctx.qp_solve([p1.eps_v[m]], [-9.0], sx, sc[None], p1.omega)
    rx = orc.exchange_eq6(p1.phi_v, p1.phi_c, p1.V, m)
    rc = orc.sigma_state(p1.phi_v, p1.phi_c, p1.eps_v, p1.eps_c, p1.V, m, L, p1.omega, DLT)
    assert abs(sx[0] - rx) <= 1e-12 * abs(rx)
    assert np.abs(sc - rc).max() <= TOL_SIGMA * 10          # a sum of 320 chains, each within 1e-6 eV (observed: far inside)
    re, rz, rit = orc.qp_solve(p1.eps_v[m], -9.0, rx, rc, p1.omega)
    assert abs(eq[0] - re) <= TOL_SIGMA * 10 and abs(zq[0] - rz) <= 1e-5


def test_out_of_memory_is_reported_and_context_survives():
    """A reorthogonalised run whose basis (8192 + 1 vectors x 64 chains x 65 536 doubles = 275 GB, at the largest step count
    reorth = 1 accepts, GWL_MAX_REORTH_STEPS) cannot be allocated returns GWL_ENOMEM from a single failed cudaMalloc; the
    context keeps working afterwards."""
    p = synth.make_custom(8, 8192, 32, seed=2)
    with _ctx(p) as ctx:
        ctx.set_chains(np.arange(64, dtype=np.int32), np.full(64, 7, dtype=np.int32))
        with pytest.raises(gwl.GwlError) as e:
            ctx._ck(ctx._lib.gwl_lanczos(ctx._h, 64, 8192, 64, 1, None, None, None, None))
        assert e.value.status == gwl.GWL_ENOMEM
        ctx.set_chains(p.n_idx, p.m_idx)
        a, b, n2, ln = ctx.lanczos(4, 10, 4, 1)
        assert (ln == 10).all() and np.isfinite(a).all() and (b > 0).all()
