"""Pins of oracle/symmetry.py (point-group symmetry blocks of C, reading Q25) against the UNREDUCED method:
the full Casida matrix of gw_oracle on the unfolded problem (all g n_w points, all N_v N_c pairs) is block diagonal in the pair
irreps, every block equals the reduced operator, start vectors and Sigma agree with the unreduced run; plus the group
facts the reduction rests on."""
import numpy as np
import pytest

from oracle import gw_oracle as orc
from oracle import symmetry as sym
from paper_2310_20103_b200 import synth

DLT = 0.1


def _full(p):
    """The same system without using its symmetry: orbitals at all points, full kernel, all pairs."""
    phi_v = sym.unfold_orbitals(p.phi_v_w, p.irrep_v, p.g)
    phi_c = sym.unfold_orbitals(p.phi_c_w, p.irrep_c, p.g)
    return phi_v, phi_c, p.V_full


@pytest.mark.parametrize("n_refl,nv,nc", [(1, [2, 1], [3, 2]), (2, [1, 2, 1, 1], [2, 1, 3, 2]),
                                          (3, [1, 0, 1, 1, 0, 1, 1, 1], [1, 2, 0, 1, 1, 1, 2, 1])])
def test_full_casida_matrix_is_block_diagonal_and_blocks_equal_the_reduced_operator(n_refl, nv, nc):
    p = synth.make_symmetric(n_refl, nv, nc, 7, seed=40 + n_refl)
    phi_v, phi_c, V = _full(p)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    C = orc.casida_dense(delta, orc.coupling_dense(orc.khatri_rao(phi_v, phi_c), V))
    n_c = len(p.eps_c)
    pair_gamma = (p.irrep_v[:, None] ^ p.irrep_c[None, :]).reshape(-1)
    scale = np.abs(C).max()
    seen = 0
    for gamma in range(p.g):
        vs, cs = sym.pair_block(p.irrep_v, p.irrep_c, gamma)
        flat = vs * n_c + cs
        assert (pair_gamma[flat] == gamma).all()
        seen += flat.size
        other = np.nonzero(pair_gamma != gamma)[0]
        assert np.abs(C[np.ix_(flat, other)]).max(initial=0.0) <= 1e-13 * scale           # no coupling between blocks
        Cg = sym.casida_block_dense(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, gamma)
        assert np.abs(Cg - C[np.ix_(flat, flat)]).max(initial=0.0) <= 1e-12 * scale        # block = reduced operator
        if flat.size:
            X = np.random.default_rng(gamma).standard_normal((3, flat.size))
            Y = sym.block_matvec(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, gamma, X)
            assert np.abs(Y - X @ Cg.T).max() <= 1e-12 * np.abs(Y).max()
    assert seen == pair_gamma.size                                                         # the blocks tile all pairs


def test_group_facts():
    """Characters: rows orthogonal, chi_a chi_b = chi_{a^b}; orbital unfolding has the stated parity; the kernel of the
    unfolded points is invariant; Vg is symmetric and Vg of the trivial irrep at g = 1 is V itself."""
    g = 8
    chi = np.array([[sym.character(a, h) for h in range(g)] for a in range(g)])
    assert np.array_equal(chi @ chi.T, g * np.eye(g))
    for a in range(g):
        for b in range(g):
            assert np.array_equal(chi[a] * chi[b], chi[a ^ b])
    p = synth.make_symmetric(2, [1, 1, 1, 1], [1, 1, 1, 1], 5, seed=44)
    phi = sym.unfold_orbitals(p.phi_v_w, p.irrep_v, p.g)
    n_w = p.n_w
    for h in range(p.g):
        sign = np.array([-1.0 if (h >> ax) & 1 else 1.0 for ax in range(3)])
        assert np.array_equal(p.r_full[h * n_w:(h + 1) * n_w], p.r_w * sign)
        for j, irr in enumerate(p.irrep_v):
            par = (-1.0) ** bin(int(irr) & h).count("1")
            assert np.array_equal(phi[h * n_w:(h + 1) * n_w, j], par * p.phi_v_w[:, j])
    V = p.V_full
    for h in range(p.g):                                  # V(h mu, h nu) = V(mu, nu): image index of (h', mu) under h is (h ^ h', mu)
        perm = np.concatenate([np.arange(n_w) + (h ^ h2) * n_w for h2 in range(p.g)])
        assert np.abs(V[np.ix_(perm, perm)] - V).max() <= 1e-13
    for gamma in range(p.g):
        Vg = sym.reduced_kernel(p.V_wf, gamma)
        assert np.abs(Vg - Vg.T).max() <= 1e-12 * np.abs(Vg).max()
    p2 = synth.make_symmetric(2, [1, 1, 1, 1], [1, 1, 1, 1], 5, seed=44)          # wedge rows computed without the full matrix
    assert np.array_equal(p2.V_wf, p.V_full[:n_w].reshape(n_w, p.g, n_w))
    p1 = synth.make_symmetric(0, [2], [3], 6, seed=45)
    assert np.array_equal(sym.reduced_kernel(p1.V_wf, 0), p1.V_full)


def test_start_vectors_and_sigma_equal_the_unreduced_run():
    """|P_nm> of the unreduced oracle is zero outside block Gamma_n ^ Gamma_m and equals the reduced start vector inside;
    alpha, beta, <P|P> and Sigma of the reduced chains equal those of gw_oracle.run_chains on the unfolded problem (valence and
    conduction n, reorthogonalisation on both sides)."""
    p = synth.make_symmetric(2, [2, 1, 1, 1], [2, 2, 1, 2], 9, seed=46, n_omega=81)
    phi_v, phi_c, V = _full(p)
    n_v, n_c = len(p.eps_v), len(p.eps_c)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    n_idx = np.array([0, 2, 4, n_v + 1, n_v + 6, 3], dtype=np.int32)
    m_idx = np.array([4, 4, 4, 4, 4, n_v + 2], dtype=np.int32)
    for n, m in zip(n_idx, m_idx):
        gamma, P = sym.start_vector_block(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, int(n), int(m))
        Pf = orc.start_vector(phi_v, phi_c, V, delta, int(n), int(m))
        vs, cs = sym.pair_block(p.irrep_v, p.irrep_c, gamma)
        flat = vs * n_c + cs
        assert np.abs(Pf[flat] - P).max() <= 1e-12 * np.abs(Pf).max()
        rest = np.setdiff1d(np.arange(Pf.size), flat)
        assert np.abs(Pf[rest]).max() <= 1e-13 * np.abs(Pf).max()
    L = 6
    rs = sym.run_chains_sym(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, n_idx, m_idx, L, p.omega, DLT,
                            reorth=True)
    rf = orc.run_chains(phi_v, phi_c, p.eps_v, p.eps_c, V, n_idx, m_idx, L, p.omega, DLT, reorth=True)
    ok = rs["len"] == L
    assert ok.all() and (rf["len"] == L).all()            # every block has more than L pairs
    assert np.abs(rs["norm2"] - rf["norm2"]).max() <= 1e-12 * rf["norm2"].max()
    assert np.abs(rs["alpha"][ok] - rf["alpha"][ok]).max() <= 1e-9 * np.abs(rf["alpha"]).max()
    assert np.abs(rs["beta"][ok, :L - 1] - rf["beta"][ok, :L - 1]).max() <= 1e-9 * np.abs(rf["alpha"]).max()
    assert np.abs(rs["sigma"][ok] - rf["sigma"][ok]).max() <= 1e-9 * max(1.0, np.abs(rf["sigma"]).max())


def test_block_sigma_against_exact_eq7_of_the_full_matrix():
    """Full-length reorthogonalised Lanczos inside the block against Eq. 7 evaluated with the eigenpairs of the FULL,
    unreduced C (gw_oracle.sigma_exact_eq7): the reduction loses nothing."""
    p = synth.make_symmetric(1, [2, 2], [3, 2], 8, seed=47, n_omega=61)
    phi_v, phi_c, V = _full(p)
    delta = orc.delta_vc(p.eps_v, p.eps_c)
    C = orc.casida_dense(delta, orc.coupling_dense(orc.khatri_rao(phi_v, phi_c), V))
    lam, Z = orc.eig_casida(C)
    n_idx = np.array([1, 2, 5], dtype=np.int32)
    m_idx = np.array([3, 3, 3], dtype=np.int32)
    rs = sym.run_chains_sym(p.phi_v_w, p.phi_c_w, p.eps_v, p.eps_c, p.irrep_v, p.irrep_c, p.V_wf, n_idx, m_idx, 10, p.omega, DLT,
                            reorth=True)
    for j, (n, m) in enumerate(zip(n_idx, m_idx)):
        Pf = orc.start_vector(phi_v, phi_c, V, delta, int(n), int(m))
        e_n, sg = orc.orbital_energy_sign(p.eps_v, p.eps_c, int(n))
        ex = orc.sigma_exact_eq7(lam, Z, Pf, p.omega, e_n, sg, DLT)
        assert np.abs(rs["sigma"][j] - ex).max() <= 1e-9 * max(1.0, np.abs(ex).max())
