"""CPU-side checks of the boundary: libgwl.so builds, loads without a GPU or driver, exports every
symbol include/gwl.h declares, fails loudly without a device, and the binding validates its arguments."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2310_20103_b200 import gwl, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    if not os.path.exists(gwl.LIB_PATH):
        from paper_2310_20103_b200 import build
        build.build()
    return gwl.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "gwl.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gwl_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 17
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/gwl.h but not exported by libgwl.so"
    assert sorted(gwl.SIGNATURES) == names


def test_no_libcuda_dependency():
    """The library must load on a driver-less box: only the static CUDA runtime, no libcuda.so link."""
    import subprocess
    out = subprocess.run(["ldd", gwl.LIB_PATH], capture_output=True, text=True).stdout
    assert "libcuda.so" not in out and "libcudart" not in out and "libtorch" not in out


def test_create_validates_and_fails_loudly_without_gpu(lib):
    h = ctypes.c_void_p()
    assert lib.gwl_create(None, 1, 1, 1) == gwl.GWL_EINVAL
    assert lib.gwl_create(ctypes.byref(h), 0, 1, 1) == gwl.GWL_EINVAL
    assert lib.gwl_create(ctypes.byref(h), 1, -3, 1) == gwl.GWL_EINVAL
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if not has_gpu:
        assert lib.gwl_create(ctypes.byref(h), 2, 2, 2) == gwl.GWL_ECUDA
        assert not h.value
        with pytest.raises(gwl.GwlError):
            gwl.Context(2, 2, 2)
    # complex contexts: n_k * n_v beyond GWL_TDC_MAX_KV is refused at creation (it is a grid dimension of the complex GEMMs)
    assert lib.gwl_tdc_create(ctypes.byref(h), 64, 1100, 8, 16, 1) == gwl.GWL_EINVAL and not h.value
    lib.gwl_destroy(None)                       # NULL-safe
    assert lib.gwl_last_error(None) == b""
    assert lib.gwl_set_pointer_mode(None, 0) == gwl.GWL_EINVAL
    assert lib.gwl_probe_fp64_peak(7, None) == gwl.GWL_EINVAL


def test_missing_library_is_an_error(tmp_path, monkeypatch):
    monkeypatch.setattr(gwl, "_lib", None)
    with pytest.raises(gwl.GwlError):
        gwl.load_library(str(tmp_path / "nope.so"))
    monkeypatch.setattr(gwl, "_lib", None)


def test_synth_configs_match_baseline():
    sizes = [(c.n_v, c.n_c, c.n_mu, c.n_chains, c.block, c.steps, c.n_omega) for c in synth.CONFIGS]
    assert sizes == [(8, 24, 192, 4, 4, 60, 201), (64, 256, 1536, 64, 64, 200, 401),
                     (256, 1024, 6144, 256, 256, 300, 401), (512, 2048, 12288, 512, 256, 300, 401),
                     (1024, 4096, 20480, 256, 128, 200, 801)]
    p = synth.make_problem(0)
    q = synth.make_problem(0)
    assert np.array_equal(p.phi_c, q.phi_c) and np.array_equal(p.V, q.V)      # seeded
    assert p.eps_c.min() - p.eps_v.max() >= 2.0
    assert np.all(np.diff(p.eps_v) > 0) and np.all(np.diff(p.eps_c) > 0)
    assert abs(p.V[0, 0] - 28.8) < 1e-12 and np.abs(p.V - p.V.T).max() == 0
    assert np.linalg.eigvalsh(p.V).min() > 0
    assert abs(np.mean(p.phi_c ** 2) * p.cfg.n_mu - 1) < 0.1
    s = synth.make_problem(synth.Config("s", 2, 2, 500, 40.0, True, (-12, -4), (-2, 25), 1, 1, 1, 1, 3))
    assert np.linalg.norm(s.r, axis=1).max() <= 20.0                               # diameter 40 (Q16)
    assert abs(synth.CONFIGS[2].flop_per_vector() - 6.52e9) < 0.01e9


def test_fit_sqrt_polynomial_through_the_c_abi(lib):
    """gwl_fit_sqrt_polynomial called through ctypes (host arithmetic, no GPU): equals the oracle's lstsq fit, and rejects
    bad arguments.  PAPER.md:85, :284, :317."""
    from oracle import gw_oracle as orc
    for g, lo, hi in ((7, 5.0, 1125.0), (1, 0.3, 0.9), (64, 1.0, 4.0e4)):
        c = np.zeros(g + 1)
        assert lib.gwl_fit_sqrt_polynomial(g, lo, hi, c.ctypes.data_as(ctypes.c_void_p)) == gwl.GWL_OK
        ref = orc.fit_sqrt_chebyshev(g, lo, hi)
        assert np.abs(c - ref).max() <= 1e-12 * np.abs(ref).max()
    c = np.zeros(8)
    p = c.ctypes.data_as(ctypes.c_void_p)
    for g, lo, hi, ptr in ((0, 1.0, 2.0, p), (65, 1.0, 2.0, p), (3, 0.0, 2.0, p), (3, 2.0, 2.0, p), (3, 1.0, 2.0, None)):
        assert lib.gwl_fit_sqrt_polynomial(g, lo, hi, ptr) == gwl.GWL_EINVAL
    assert lib.gwl_sqrt_fit_range(None, 0, 0.02, None, None) == gwl.GWL_EINVAL


def test_polyfit_helper_closed_form_equals_least_squares():
    """paper_2310_20103_b200/polyfit.py (a call-through to gwl_fit_sqrt_polynomial) against the oracle's lstsq fit and
    against sqrt itself on the range."""
    import numpy as np
    from oracle import gw_oracle as orc
    from paper_2310_20103_b200 import polyfit
    lo, hi = polyfit.default_range(np.array([-10.0, -5.5]), np.array([-3.0, 20.0]))
    assert abs(lo - 0.8 * 2.5 ** 2) < 1e-12 and abs(hi - 1.25 * 30.0 ** 2) < 1e-9
    for g in (1, 7, 8, 16):
        c = polyfit.sqrt_chebyshev(g, lo, hi)
        ref = orc.fit_sqrt_chebyshev(g, lo, hi)
        assert np.abs(c - ref).max() <= 1e-12 * np.abs(ref).max()
    x = np.linspace(lo, hi, 200)
    err = np.abs(orc.poly_eval_scalar(polyfit.sqrt_chebyshev(8, lo, hi), lo, hi, x) - np.sqrt(x)) / np.sqrt(x)
    assert err.max() < 0.2 and err[50:].max() < 0.01
