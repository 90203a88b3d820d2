"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is INPUT GENERATION ONLY.  It holds none of the method's arithmetic
(no Casida product, no Lanczos, no continued fraction) and imports neither the
oracle nor the CUDA binding; the tests, bench.py and smoke() hand the very same
host arrays to both sides.

Recipe (BASELINE.json:configs): numpy.random.default_rng(seed),
draw order r, Phi_v, Phi_c, eps_v, eps_c.
  r_mu      uniform in a cube of side `box` (configs 0-3) or in a sphere of
            DIAMETER `box` (config 4, reading Q16)
  Phi_v/c   i.i.d. N(0,1)/sqrt(N_mu)       -- stand-ins for the orbitals at the
            ISDF points; real orbitals are not in the container
  eps_v     U[ev_lo, ev_hi], eps_c U[ec_lo, ec_hi], both sorted ascending (eV)
  V         14.4 / sqrt(|r_mu - r_nu|^2 + 0.25) eV, stand-in for (alpha|beta),
            PAPER.md:125 (Eq. 17); inverse multiquadric, positive definite
  omega     uniform grid on [-20, 20] eV, broadening 0.1 eV (the paper's delta)
  chains    (n, m) = {first a valence} x {first b conduction}, row-major (Q11);
            orbital index in [0, N_v + N_c): < N_v valence, else conduction
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    n_v: int
    n_c: int
    n_mu: int
    box: float            # cube side or sphere diameter, Angstrom
    sphere: bool
    ev: tuple             # (lo, hi) of eps_v
    ec: tuple             # (lo, hi) of eps_c
    chains_a: int         # number of valence n
    chains_b: int         # number of conduction m
    block: int
    steps: int
    n_omega: int
    omega_lo: float = -20.0
    omega_hi: float = 20.0
    eta: float = 0.1      # BASELINE's eta = the paper's delta (eV)

    @property
    def n_vc(self) -> int:
        return self.n_v * self.n_c

    @property
    def n_chains(self) -> int:
        return self.chains_a * self.chains_b

    def flop_per_vector(self) -> float:
        """F/B = 4 N_mu N_vc + 2 N_mu^2."""
        return 4.0 * self.n_mu * self.n_vc + 2.0 * self.n_mu * self.n_mu


CONFIGS = (
    Config("cfg0_tiny", 8, 24, 192, 10.0, False, (-10.0, -5.0), (-3.0, 20.0), 2, 2, 4, 60, 201),
    Config("cfg1_small_molecule", 64, 256, 1536, 15.0, False, (-10.0, -5.0), (-3.0, 20.0), 8, 8, 64, 200, 401),
    Config("cfg2_100_atom_cluster", 256, 1024, 6144, 20.0, False, (-10.0, -5.0), (-3.0, 20.0), 16, 16, 256, 300, 401),
    Config("cfg3_defect_cell", 512, 2048, 12288, 25.0, False, (-10.0, -5.0), (-3.0, 20.0), 16, 32, 256, 300, 401),
    Config("cfg4_si_quantum_dot", 1024, 4096, 20480, 40.0, True, (-12.0, -4.0), (-2.0, 25.0), 16, 16, 128, 200, 801),
)


@dataclass
class Problem:
    cfg: Config
    r: np.ndarray          # [n_mu, 3]
    phi_v: np.ndarray      # [n_mu, n_v]
    phi_c: np.ndarray      # [n_mu, n_c]
    eps_v: np.ndarray      # [n_v]
    eps_c: np.ndarray      # [n_c]
    omega: np.ndarray      # [n_omega]
    n_idx: np.ndarray      # [n_chains] int32
    m_idx: np.ndarray      # [n_chains] int32
    _V: np.ndarray | None = field(default=None, repr=False)

    @property
    def V(self) -> np.ndarray:
        if self._V is None:
            self._V = coulomb_kernel(self.r)
        return self._V


def coulomb_kernel(r: np.ndarray, row_chunk: int = 1024) -> np.ndarray:
    """V[mu,nu] = 14.4 / sqrt(|r_mu - r_nu|^2 + 0.25), built in row chunks."""
    n = r.shape[0]
    V = np.empty((n, n), dtype=np.float64)
    for i in range(0, n, row_chunk):
        d = r[i:i + row_chunk, None, :] - r[None, :, :]
        V[i:i + row_chunk] = 14.4 / np.sqrt(np.einsum("ijk,ijk->ij", d, d) + 0.25)
    return V


def chain_list(cfg: Config):
    """(n, m) pairs of Q11: n over the first `a` valence, m over the first `b` conduction."""
    n = np.repeat(np.arange(cfg.chains_a, dtype=np.int32), cfg.chains_b)
    m = np.tile(np.arange(cfg.chains_b, dtype=np.int32), cfg.chains_a) + np.int32(cfg.n_v)
    return n, m


def make_problem(cfg: Config | int, seed: int = 0) -> Problem:
    if isinstance(cfg, int):
        cfg = CONFIGS[cfg]
    rng = np.random.default_rng(seed)
    if cfg.sphere:
        # uniform in a ball of diameter `box`: R u^(1/3) times a unit vector
        u = rng.random(cfg.n_mu)
        g = rng.standard_normal((cfg.n_mu, 3))
        g /= np.linalg.norm(g, axis=1, keepdims=True)
        r = (0.5 * cfg.box) * np.cbrt(u)[:, None] * g
    else:
        r = rng.random((cfg.n_mu, 3)) * cfg.box
    phi_v = rng.standard_normal((cfg.n_mu, cfg.n_v)) / np.sqrt(cfg.n_mu)
    phi_c = rng.standard_normal((cfg.n_mu, cfg.n_c)) / np.sqrt(cfg.n_mu)
    eps_v = np.sort(rng.uniform(cfg.ev[0], cfg.ev[1], cfg.n_v))
    eps_c = np.sort(rng.uniform(cfg.ec[0], cfg.ec[1], cfg.n_c))
    omega = np.linspace(cfg.omega_lo, cfg.omega_hi, cfg.n_omega)
    n_idx, m_idx = chain_list(cfg)
    return Problem(cfg, r, phi_v, phi_c, eps_v, eps_c, omega, n_idx, m_idx)


def make_custom(n_v: int, n_c: int, n_mu: int, box: float = 10.0, seed: int = 0,
                n_omega: int = 101, chains_a: int = 2, chains_b: int = 2,
                steps: int = 20, block: int = 4) -> Problem:
    """Same generators at arbitrary (ragged) sizes, for edge-case tests."""
    cfg = Config(f"custom_{n_v}_{n_c}_{n_mu}", n_v, n_c, n_mu, box, False,
                 (-10.0, -5.0), (-3.0, 20.0), chains_a, chains_b, block, steps, n_omega)
    return make_problem(cfg, seed)


def random_block(cfg: Config, nvec: int, seed: int = 1) -> np.ndarray:
    """A seeded block of test vectors X[nvec][n_v][n_c] ~ N(0,1)."""
    rng = np.random.default_rng(seed)
    return rng.standard_normal((nvec, cfg.n_v, cfg.n_c))


# ---------------------------------------------------------------------------------------------
# complex-orbital (periodic) Tamm-Dancoff variant.
# Stand-ins for Bloch orbitals at N_k k-points and ONE transferred momentum q: complex Gaussians of the same
# normalisation as the real configs; the conduction set is the one already shifted by q (psi_{c k+q}).
# ---------------------------------------------------------------------------------------------
@dataclass
class PeriodicProblem:
    n_k: int
    n_v: int
    n_c: int
    n_mu: int
    r: np.ndarray          # [n_mu, 3]
    psi_v: np.ndarray      # [n_k, n_mu, n_v] complex128   psi_{v k}(r_mu)
    psi_cq: np.ndarray     # [n_k, n_mu, n_c] complex128   psi_{c k+q}(r_mu)
    eps_v: np.ndarray      # [n_k, n_v]
    eps_cq: np.ndarray     # [n_k, n_c]
    omega: np.ndarray      # [n_omega]
    chains: np.ndarray     # [n_chains, 4] int32: (k slot of n, n index, k slot of m, m index)
    eta: float = 0.1
    _V: np.ndarray | None = field(default=None, repr=False)

    @property
    def V(self) -> np.ndarray:
        if self._V is None:
            self._V = coulomb_kernel(self.r)
        return self._V

    @property
    def n_kvc(self) -> int:
        return self.n_k * self.n_v * self.n_c


def make_periodic(n_k: int, n_v: int, n_c: int, n_mu: int, box: float = 10.0, seed: int = 0, n_omega: int = 101,
                  n_chains: int = 4, real_orbitals: bool = False) -> PeriodicProblem:
    """Draw order r, Re/Im psi_v, Re/Im psi_cq, eps_v, eps_cq.  Chains: n runs over the first orbitals of slot
    (j mod n_k), alternating occupied / empty, m = the highest occupied orbital of slot 0."""
    rng = np.random.default_rng(seed)
    r = rng.random((n_mu, 3)) * box

    def orbitals(n):
        re = rng.standard_normal((n_k, n_mu, n))
        im = rng.standard_normal((n_k, n_mu, n))
        if real_orbitals:
            return (re / np.sqrt(n_mu)).astype(np.complex128)
        return (re + 1j * im) / np.sqrt(2.0 * n_mu)

    psi_v = orbitals(n_v)
    psi_cq = orbitals(n_c)
    eps_v = np.sort(rng.uniform(-10.0, -5.0, (n_k, n_v)), axis=1)
    eps_cq = np.sort(rng.uniform(-3.0, 20.0, (n_k, n_c)), axis=1)
    omega = np.linspace(-20.0, 20.0, n_omega)
    n_orb = n_v + n_c
    chains = np.zeros((n_chains, 4), dtype=np.int32)
    for j in range(n_chains):
        idx = (j // 2) % n_v if j % 2 == 0 else n_v + (j // 2) % n_c
        chains[j] = (j % n_k, min(idx, n_orb - 1), 0, n_v - 1)
    return PeriodicProblem(n_k, n_v, n_c, n_mu, r, psi_v, psi_cq, eps_v, eps_cq, omega, chains)


def random_complex_block(n: int, nvec: int, seed: int = 1) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.standard_normal((nvec, n)) + 1j * rng.standard_normal((nvec, n))


# ---------------------------------------------------------------------------------------------
# smooth synthetic orbitals on a real-space grid for the ISDF front end.
# Particle-in-a-box eigenfunctions on a uniform n^3 grid (the paper's orbitals live on a uniform real-space grid,
# PAPER.md:317): smooth, orthonormal under the grid quadrature, and their pair products have low numerical rank.
# ---------------------------------------------------------------------------------------------
def box_orbitals(n_grid: int, n_orb: int, box: float = 8.0):
    """Returns (r [n^3, 3], phi [n^3, n_orb], weight h^3): the n_orb lowest states sin(a pi x / L) sin(b pi y / L)
    sin(c pi z / L), (a, b, c) ordered by a^2 + b^2 + c^2 then lexicographically, on the interior points of a cube."""
    h = box / (n_grid + 1)
    x = h * np.arange(1, n_grid + 1)
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")
    r = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    q = [(a * a + b * b + c * c, a, b, c) for a in range(1, 12) for b in range(1, 12) for c in range(1, 12)]
    q.sort()
    s = {k: np.sqrt(2.0 / box) * np.sin(k * np.pi * x / box) for k in range(1, 12)}
    phi = np.empty((n_grid ** 3, n_orb))
    for j, (_, a, b, c) in enumerate(q[:n_orb]):
        phi[:, j] = (s[a][:, None, None] * s[b][None, :, None] * s[c][None, None, :]).ravel()
    return r, phi, h ** 3


def stride_points(n_r: int, n_mu: int, seed: int = 0) -> np.ndarray:
    """n_mu distinct grid indices, seeded: the interpolation points handed to both sides (their selection, by pivoted QR
    or k-means in the ISDF literature, is not part of the parity tests)."""
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(n_r, size=n_mu, replace=False)).astype(np.int32)


# ---------------------------------------------------------------------------------------------
# SURVEY.md §8(f)-4, second part: inputs with an abelian point group for the symmetry blocks of C.
# The group is generated by n_refl mirror planes (x -> -x, y -> -y, z -> -z: C_s, C_2v-like, D_2h-like; order g = 2^n_refl);
# element h in [0, g) reflects the axes whose bit is set in h.  Only the data are made here: fitting points in the
# irreducible wedge and all their images, orbital values on the wedge, an irreducible-representation label per orbital
# (a bit mask: bit i set = odd under mirror i).  What the labels MEAN (characters, unfolding, block structure) is the
# method's arithmetic and lives in oracle/symmetry.py and in the library separately.
# ---------------------------------------------------------------------------------------------
@dataclass
class SymmetricProblem:
    n_refl: int
    nv_irrep: np.ndarray   # [g] occupied orbitals per irrep (orbitals are sorted by irrep)
    nc_irrep: np.ndarray   # [g] empty orbitals per irrep
    r_w: np.ndarray        # [n_w, 3] fitting points of the wedge
    r_full: np.ndarray     # [g * n_w, 3]: r_full[h * n_w + mu] = image of r_w[mu] under element h
    phi_v_w: np.ndarray    # [n_w, N_v] orbital values on the wedge
    phi_c_w: np.ndarray    # [n_w, N_c]
    irrep_v: np.ndarray    # [N_v] int32 labels, ascending
    irrep_c: np.ndarray    # [N_c]
    eps_v: np.ndarray      # [N_v]
    eps_c: np.ndarray      # [N_c]
    omega: np.ndarray
    eta: float = 0.1
    _V: np.ndarray | None = field(default=None, repr=False)

    @property
    def g(self) -> int:
        return 1 << self.n_refl

    @property
    def n_w(self) -> int:
        return self.r_w.shape[0]

    @property
    def V_full(self) -> np.ndarray:
        """Coulomb kernel of ALL points (invariant under the group because reflections are isometries)."""
        if self._V is None:
            self._V = coulomb_kernel(self.r_full)
        return self._V

    @property
    def V_wf(self) -> np.ndarray:
        """[n_w][g][n_w]: rows of V_full for the wedge points against every image, V(r_mu, h r_nu): the same kernel formula
        evaluated for those rows only (the full g n_w x g n_w matrix is not needed to feed the library)."""
        if self._V is not None:
            rows = self._V[:self.n_w]
        else:
            rows = np.empty((self.n_w, self.g * self.n_w))
            for i in range(0, self.n_w, 1024):
                d = self.r_w[i:i + 1024, None, :] - self.r_full[None, :, :]
                rows[i:i + 1024] = 14.4 / np.sqrt(np.einsum("ijk,ijk->ij", d, d) + 0.25)
        return np.ascontiguousarray(rows.reshape(self.n_w, self.g, self.n_w))


def make_symmetric(n_refl: int, nv_irrep, nc_irrep, n_w: int, box: float = 12.0, seed: int = 0,
                   n_omega: int = 101) -> SymmetricProblem:
    """Draw order r_w, Phi_v, Phi_c, eps_v, eps_c.  Wedge points: coordinates along mirrored axes uniform in
    [0.3, box/2] (off the mirror planes, so the g images are distinct), the others uniform in [-box/2, box/2]."""
    g = 1 << n_refl
    nv_irrep = np.asarray(nv_irrep, dtype=np.int32)
    nc_irrep = np.asarray(nc_irrep, dtype=np.int32)
    if nv_irrep.shape != (g,) or nc_irrep.shape != (g,):
        raise ValueError("nv_irrep and nc_irrep need one entry per irrep (2^n_refl)")
    rng = np.random.default_rng(seed)
    r_w = np.empty((n_w, 3))
    for ax in range(3):
        if ax < n_refl:
            r_w[:, ax] = rng.uniform(0.3, 0.5 * box, n_w)
        else:
            r_w[:, ax] = rng.uniform(-0.5 * box, 0.5 * box, n_w)
    r_full = np.empty((g * n_w, 3))
    for h in range(g):
        sign = np.array([-1.0 if (h >> ax) & 1 else 1.0 for ax in range(3)])
        r_full[h * n_w:(h + 1) * n_w] = r_w * sign[None, :]
    n_v, n_c = int(nv_irrep.sum()), int(nc_irrep.sum())
    phi_v_w = rng.standard_normal((n_w, n_v)) / np.sqrt(g * n_w)
    phi_c_w = rng.standard_normal((n_w, n_c)) / np.sqrt(g * n_w)
    eps_v = rng.uniform(-10.0, -5.0, n_v)
    eps_c = rng.uniform(-3.0, 20.0, n_c)
    irrep_v = np.repeat(np.arange(g, dtype=np.int32), nv_irrep)
    irrep_c = np.repeat(np.arange(g, dtype=np.int32), nc_irrep)
    omega = np.linspace(-20.0, 20.0, n_omega)
    return SymmetricProblem(n_refl, nv_irrep, nc_irrep, r_w, r_full, phi_v_w, phi_c_w, irrep_v, irrep_c, eps_v, eps_c, omega)
