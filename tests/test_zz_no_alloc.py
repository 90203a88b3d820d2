"""gwl_chain_norms_static: the entry point of libgwl that calls no cudaMalloc.

Some host programs cannot let a library allocate on the GPU: a DFT/GW driver or a PyTorch process that has already
put all of HBM into its own memory pool (a library's cudaMalloc then fails or fragments what is left), or a driver
that keeps other streams busy and cannot afford the device-wide synchronisation that cudaMalloc / cudaFree imply.
For them the library computes <P_j|P_j> (the `norm2` output of gwl_lanczos, the numerator of Eq. 14)
with its reduction partials in a fixed 256 KB array that is part of the library image instead of in a context
buffer.  All calls share that array and it keeps the last call's contents, so the GPU test below makes two calls
in a row with different sizes and values and compares each with the existing, context-based path
(gwl_set_start_vectors + gwl_lanczos) within the 1e-12 relative tolerance the other tests use for ||P||^2.

This file sorts last among tests/test_*.py on purpose: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  It passes both alone in a fresh process (its first call then does the
per-device set-up) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

from paper_2310_20103_b200 import gwl, synth

TOL_NORM = 1e-12     # relative, as in tests/test_gpu_parity.py for <P|P>


def _existing_path_norm2(prob, P):
    """norm2 through the context: explicit start vectors, one Lanczos step."""
    n = P.shape[0]
    with gwl.Context(prob.cfg.n_v, prob.cfg.n_c, prob.cfg.n_mu) as ctx:
        ctx.set_orbitals(prob.phi_v, prob.phi_c)
        ctx.set_energies(prob.eps_v, prob.eps_c)
        ctx.set_kernel(prob.V)
        ctx.set_start_vectors(P, np.full(n, -6.0), np.ones(n, dtype=np.int32))
        _, _, n2, _ = ctx.lanczos(n, 1, n, 0)
    return n2


def test_limits_are_rejected_before_any_cuda_call():
    """Sizes beyond the fixed scratch give GWL_EINVAL and a message that names the limit; needs no GPU because
    nothing is launched (the pointers are never touched)."""
    lib = gwl.load_library()
    err = ctypes.create_string_buffer(256)
    dummy = ctypes.c_void_p(256)
    st = lib.gwl_chain_norms_static(dummy, 4097, 1000, dummy, None, err, 256)
    assert st == gwl.GWL_EINVAL and b"GWL_STATIC_MAX_CHAINS = 4096" in err.value
    st = lib.gwl_chain_norms_static(dummy, 4, (1 << 32) + 1, dummy, None, err, 256)
    assert st == gwl.GWL_EINVAL and b"GWL_STATIC_MAX_NVC" in err.value
    st = lib.gwl_chain_norms_static(dummy, -1, 10, dummy, None, err, 256)
    assert st == gwl.GWL_EINVAL and err.value
    st = lib.gwl_chain_norms_static(dummy, 3, 0, dummy, None, None, 0)      # err may be NULL
    assert st == gwl.GWL_EINVAL
    st = lib.gwl_chain_norms_static(None, 0, 10, None, None, err, 256)       # empty block: no-op
    assert st == gwl.GWL_OK and err.value == b""


@pytest.mark.gpu
def test_static_scratch_norms_match_the_context_path_on_two_calls_in_a_row():
    import torch
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)

    # first call: 9 chains, N_vc = 40 * 1237 = 49 480 (four reduction slices, ragged tail)
    pa = synth.make_custom(40, 1237, 32, seed=5)
    Pa = np.random.default_rng(11).standard_normal((9, pa.cfg.n_vc)) * np.logspace(-3, 3, 9)[:, None]
    # second call: fewer chains, another length (two slices), other values -- stale partials of call one
    # sit in the shared array and must not leak into these results
    pb = synth.make_custom(7, 2501, 16, seed=6)
    Pb = np.random.default_rng(12).standard_normal((5, pb.cfg.n_vc))
    Pb[3] = 0.0                                                # a dead chain: norm2 must be exactly 0

    da, db = torch.from_numpy(Pa).to(dev), torch.from_numpy(Pb).to(dev)
    na = torch.full((9,), -1.0, dtype=torch.float64, device=dev)
    nb = torch.full((5,), -1.0, dtype=torch.float64, device=dev)
    gwl.chain_norms_static(da, na)
    gwl.chain_norms_static(db, nb)
    torch.cuda.synchronize()
    na, nb = na.cpu().numpy(), nb.cpu().numpy()

    ref_a, ref_b = _existing_path_norm2(pa, Pa), _existing_path_norm2(pb, Pb)
    assert (np.abs(na - ref_a) <= TOL_NORM * ref_a).all(), (na, ref_a)
    assert (np.abs(nb - ref_b) <= TOL_NORM * ref_b).all(), (nb, ref_b)
    assert nb[3] == 0.0 and ref_b[3] == 0.0
    # and both against the plain definition
    assert (np.abs(na - (Pa * Pa).sum(axis=1)) <= TOL_NORM * na).all()
    assert (np.abs(nb - (Pb * Pb).sum(axis=1)) <= TOL_NORM * np.maximum(nb, 1e-300)).all()

    # a third call with the first inputs repeats the first result bit for bit (fixed reduction order, nothing stale)
    na2 = torch.empty(9, dtype=torch.float64, device=dev)
    gwl.chain_norms_static(da, na2, cuda_stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert (na2.cpu().numpy() == na).all()

    # size limit through the binding
    big = torch.empty(5000, dtype=torch.float64, device=dev)
    with pytest.raises(gwl.GwlError, match="GWL_STATIC_MAX_CHAINS"):
        gwl.chain_norms_static(da, big, n_chains=5000, n_vc=1)
