"""Thin ctypes binding over libgwl.so (include/gwl.h).  Argument marshalling only: every step of the path
runs in the library's CUDA kernels.  There is no CPU fallback -- if libgwl.so is missing or the call
fails, a GwlError is raised.

Host mode (default): numpy float64 arrays in, numpy arrays out.
Device mode (`ctx.set_pointer_mode(1)`): torch CUDA float64 tensors in/out, nothing is copied.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_int32, c_int64, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgwl.so")

GWL_OK, GWL_EINVAL, GWL_ESTATE, GWL_ENOMEM, GWL_ECUDA = range(5)
GWL_RPA, GWL_TDA = 0, 1
_STATUS = {0: "GWL_OK", 1: "GWL_EINVAL", 2: "GWL_ESTATE", 3: "GWL_ENOMEM", 4: "GWL_ECUDA"}

# name -> (restype, argtypes); every symbol include/gwl.h declares
SIGNATURES = {
    "gwl_create": (c_int, [POINTER(c_void_p), c_int64, c_int64, c_int64]),
    "gwl_destroy": (None, [c_void_p]),
    "gwl_last_error": (c_char_p, [c_void_p]),
    "gwl_set_pointer_mode": (c_int, [c_void_p, c_int]),
    "gwl_set_stream": (c_int, [c_void_p, c_void_p]),
    "gwl_set_orbitals": (c_int, [c_void_p, c_void_p, c_void_p]),
    "gwl_set_energies": (c_int, [c_void_p, c_void_p, c_void_p]),
    "gwl_set_kernel": (c_int, [c_void_p, c_void_p]),
    "gwl_set_polynomial": (c_int, [c_void_p, c_int, c_void_p, c_double, c_double]),
    "gwl_set_approximation": (c_int, [c_void_p, c_int]),
    "gwl_fit_sqrt_polynomial": (c_int, [c_int, c_double, c_double, c_void_p]),
    "gwl_sqrt_fit_range": (c_int, [c_void_p, c_int64, c_double, POINTER(c_double), POINTER(c_double)]),
    "gwl_spectrum_bounds": (c_int, [c_void_p, c_int64, POINTER(c_double), POINTER(c_double)]),
    "gwl_casida_matvec": (c_int, [c_void_p, c_void_p, c_void_p, c_int64]),
    "gwl_set_chains": (c_int, [c_void_p, c_int64, c_void_p, c_void_p]),
    "gwl_set_start_vectors": (c_int, [c_void_p, c_int64, c_void_p, c_void_p, c_void_p]),
    "gwl_lanczos": (c_int, [c_void_p, c_int64, c_int64, c_int64, c_int, c_void_p, c_void_p, c_void_p, c_void_p]),
    "gwl_resolvent": (c_int, [c_void_p, c_void_p, c_int64, c_void_p]),
    "gwl_selfenergy": (c_int, [c_void_p, c_void_p, c_int64, c_double, c_void_p, c_void_p]),
    "gwl_selfenergy_state": (c_int, [c_void_p, c_int32, c_int64, c_int64, c_int, c_void_p, c_int64, c_double, c_void_p]),
    "gwl_exchange": (c_int, [c_void_p, c_int64, c_void_p, c_void_p]),
    "gwl_qp_solve": (c_int, [c_void_p, c_int64, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int64, c_void_p,
                             c_void_p, c_void_p]),
    "gwl_tdc_create": (c_int, [POINTER(c_void_p), c_int64, c_int64, c_int64, c_int64, c_int64]),
    "gwl_tdc_set_orbitals": (c_int, [c_void_p, c_void_p, c_void_p]),
    "gwl_tdc_set_energies": (c_int, [c_void_p, c_void_p, c_void_p]),
    "gwl_tdc_set_chains": (c_int, [c_void_p, c_int64, c_void_p]),
    "gwl_tdc_matvec": (c_int, [c_void_p, c_void_p, c_void_p, c_int64]),
    "gwl_tdc_matvec_rpa": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_int64]),
    "gwl_tdc_selfenergy_state": (c_int, [c_void_p, c_int32, c_int32, c_int32, c_int64, c_int64, c_int, c_void_p, c_int64, c_double,
                                         c_void_p]),
    "gwl_sym_create": (c_int, [POINTER(c_void_p), c_int, c_void_p, c_void_p, c_int64]),
    "gwl_sym_set_orbitals": (c_int, [c_void_p, c_void_p, c_void_p]),
    "gwl_sym_set_kernel": (c_int, [c_void_p, c_void_p]),
    "gwl_sym_select": (c_int, [c_void_p, c_int, POINTER(c_int64)]),
    "gwl_sym_matvec": (c_int, [c_void_p, c_void_p, c_void_p, c_int64]),
    "gwl_sym_selfenergy_state": (c_int, [c_void_p, c_int32, c_int64, c_int64, c_int, c_void_p, c_int64, c_double, c_void_p]),
    "gwl_isdf_build": (c_int, [c_void_p, c_int64, c_void_p, c_void_p, c_void_p, c_double, c_double, c_void_p, c_void_p,
                               c_void_p]),
    "gwl_isdf_select_points": (c_int, [c_void_p, c_int64, c_void_p, c_void_p, c_void_p, c_int64, c_void_p, POINTER(c_int32)]),
    "gwl_get_timing": (c_int, [c_void_p, POINTER(c_double), POINTER(c_double), POINTER(c_double)]),
    "gwl_set_profiling": (c_int, [c_void_p, c_int]),
    "gwl_get_kernel_times": (c_int, [c_void_p, POINTER(c_double), POINTER(c_int64)]),
    "gwl_get_launch_count": (c_int, [c_void_p, POINTER(c_int64)]),
    "gwl_probe_fp64_peak": (c_int, [c_int, POINTER(c_double)]),
    "gwl_chain_norms_static": (c_int, [c_void_p, c_int64, c_int64, c_void_p, c_void_p, c_char_p, c_int64]),
}


KERNEL_CLASSES = ("gemm_fwd_KX", "gemm_V", "gemm_bwd_KtW", "splitk_reduce", "scale_axpy_dot", "lanczos_update",
                  "reorth", "spectral")


class GwlError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


_lib = None


def load_library(path: str = LIB_PATH):
    """Loads libgwl.so (built by `python -m paper_2310_20103_b200.build`); raises if it is absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(path):
            raise GwlError(GWL_ESTATE, f"{path} not found: build it with `python -m paper_2310_20103_b200.build` "
                                       "(there is no CPU fallback)")
        lib = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _host(a, dtype=np.float64):
    return np.ascontiguousarray(a, dtype=dtype)


def _ptr(a):
    if a is None:
        return None
    if _is_torch(a):
        return c_void_p(a.data_ptr())
    return c_void_p(a.ctypes.data)


def probe_fp64_peak(kind: int = 0) -> float:
    """TFLOP/s of a register-resident DMMA (kind 0) or DFMA (kind 1) loop on the current device."""
    lib = load_library()
    out = c_double(0.0)
    st = lib.gwl_probe_fp64_peak(kind, byref(out))
    if st != GWL_OK:
        raise GwlError(st, "gwl_probe_fp64_peak failed")
    return out.value


def chain_norms_static(p, norm2, n_chains: int | None = None, n_vc: int | None = None, cuda_stream: int | None = None):
    """norm2[j] = <P_j|P_j> through gwl_chain_norms_static, the entry point for callers that must not trigger a
    cudaMalloc (all of HBM already in the caller's pool, or other streams that a device-wide synchronisation would
    stall).  p [n_chains, n_vc] and norm2 [n_chains] are contiguous torch CUDA float64 tensors on the current device;
    norm2 is written in place on `cuda_stream` (default: the legacy default stream) and returned.  The scratch is a
    fixed 256 KB array inside libgwl.so shared by all calls: do not let two calls overlap on one GPU.  Sizes may be
    given explicitly when p is a flat buffer; limits: n_chains <= 4096, n_vc <= 2^32 (GwlError otherwise)."""
    lib = load_library()
    if n_chains is None or n_vc is None:
        if p.dim() != 2:
            raise GwlError(GWL_EINVAL, "chain_norms_static: p must be [n_chains, n_vc] (or pass the sizes)")
        n_chains, n_vc = p.shape
    if not (_is_torch(p) and _is_torch(norm2) and p.is_cuda and norm2.is_cuda and p.is_contiguous()
            and norm2.is_contiguous()) or p.numel() < n_chains * n_vc or norm2.numel() < n_chains:
        raise GwlError(GWL_EINVAL, "chain_norms_static: p, norm2 must be contiguous torch CUDA float64 tensors of "
                                   "at least n_chains * n_vc and n_chains elements")
    err = ctypes.create_string_buffer(256)
    st = lib.gwl_chain_norms_static(_ptr(p), int(n_chains), int(n_vc), _ptr(norm2), c_void_p(cuda_stream or 0), err, 256)
    if st != GWL_OK:
        raise GwlError(st, err.value.decode())
    return norm2


def fit_sqrt_polynomial(g: int, lo: float, hi: float) -> np.ndarray:
    """cheb[0..g] of p_g(x) ~ sqrt(x) on [lo, hi] (gwl_fit_sqrt_polynomial: host arithmetic inside libgwl.so)."""
    c = np.zeros(int(g) + 1 if g >= 0 else 1)
    st = load_library().gwl_fit_sqrt_polynomial(int(g), float(lo), float(hi), _ptr(c))
    if st != GWL_OK:
        raise GwlError(st, "gwl_fit_sqrt_polynomial: need 1 <= g <= 64 and 0 < lo < hi")
    return c


class Context:
    """gwl_ctx wrapper.  Method names follow the C ABI without the gwl_ prefix."""

    def __init__(self, n_v: int, n_c: int, n_mu: int):
        self._lib = load_library()
        self._h = c_void_p()
        self.n_v, self.n_c, self.n_mu = int(n_v), int(n_c), int(n_mu)
        self.n_vc = self.n_v * self.n_c
        self.device_ptrs = 0
        st = self._lib.gwl_create(byref(self._h), n_v, n_c, n_mu)
        if st != GWL_OK:
            self._h = c_void_p()
            raise GwlError(st, "gwl_create failed (no CUDA device, or bad sizes)")

    # -- plumbing ---------------------------------------------------------------------------------
    def _ck(self, st):
        if st != GWL_OK:
            msg = self._lib.gwl_last_error(self._h)
            raise GwlError(st, msg.decode() if msg else "")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.gwl_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def last_error(self) -> str:
        return self._lib.gwl_last_error(self._h).decode()

    def set_pointer_mode(self, device_ptrs: int):
        self._ck(self._lib.gwl_set_pointer_mode(self._h, int(device_ptrs)))
        self.device_ptrs = int(device_ptrs)

    def set_stream(self, cuda_stream: int | None):
        self._ck(self._lib.gwl_set_stream(self._h, c_void_p(cuda_stream or 0)))

    # -- inputs -----------------------------------------------------------------------------------
    def set_orbitals(self, phi_v, phi_c):
        pv, pc = _host(phi_v), _host(phi_c)
        if pv.shape != (self.n_mu, self.n_v) or pc.shape != (self.n_mu, self.n_c):
            raise GwlError(GWL_EINVAL, "set_orbitals: phi_v must be [n_mu, n_v], phi_c [n_mu, n_c]")
        self._ck(self._lib.gwl_set_orbitals(self._h, _ptr(pv), _ptr(pc)))

    def set_energies(self, eps_v, eps_c):
        ev, ec = _host(eps_v), _host(eps_c)
        if ev.shape != (self.n_v,) or ec.shape != (self.n_c,):
            raise GwlError(GWL_EINVAL, "set_energies: eps_v must be [n_v], eps_c [n_c]")
        self._ck(self._lib.gwl_set_energies(self._h, _ptr(ev), _ptr(ec)))

    def set_kernel(self, V):
        Vh = _host(V)
        if Vh.shape != (self.n_mu, self.n_mu):
            raise GwlError(GWL_EINVAL, "set_kernel: V must be [n_mu, n_mu]")
        self._ck(self._lib.gwl_set_kernel(self._h, _ptr(Vh)))

    def set_polynomial(self, g: int, cheb=None, lo: float = 0.0, hi: float = 0.0):
        c = None if cheb is None else _host(cheb)
        if g > 0 and (c is None or c.shape != (g + 1,)):
            raise GwlError(GWL_EINVAL, "set_polynomial: cheb must have g+1 entries")
        self._ck(self._lib.gwl_set_polynomial(self._h, int(g), _ptr(c), float(lo), float(hi)))

    def set_approximation(self, approximation: int):
        """0 = RPA (operator C, default), 1 = Tamm-Dancoff (operator A)."""
        self._ck(self._lib.gwl_set_approximation(self._h, int(approximation)))

    def sqrt_fit_range(self, steps: int = 40, margin: float = 0.02):
        """(lo, hi) for gwl_set_polynomial: steps = 0 the paper's heuristic range, else from gwl_spectrum_bounds."""
        lo, hi = c_double(0.0), c_double(0.0)
        self._ck(self._lib.gwl_sqrt_fit_range(self._h, int(steps), float(margin), byref(lo), byref(hi)))
        return lo.value, hi.value

    def spectrum_bounds(self, steps: int = 40):
        """(lam_min, lam_max) estimates of the operator's spectrum from a short Lanczos run."""
        lo, hi = c_double(), c_double()
        self._ck(self._lib.gwl_spectrum_bounds(self._h, int(steps), byref(lo), byref(hi)))
        return lo.value, hi.value

    def isdf_build(self, phi_v_grid, phi_c_grid, r, weight: float, soft: float, idx, want_zeta: bool = True):
        """ISDF front end: fits zeta at the interpolation points idx, builds (alpha|beta) and installs
        the orbitals at those points and the kernel in this context.  Returns (zeta_t [n_mu, n_r] or None, V [n_mu, n_mu])."""
        pv, pc, rr, ix = _host(phi_v_grid), _host(phi_c_grid), _host(r), _host(idx, np.int32)
        n_r = rr.shape[0]
        if pv.shape != (n_r, self.n_v) or pc.shape != (n_r, self.n_c) or rr.shape != (n_r, 3) or ix.shape != (self.n_mu,):
            raise GwlError(GWL_EINVAL, "isdf_build: phi_v_grid [n_r, n_v], phi_c_grid [n_r, n_c], r [n_r, 3], idx [n_mu]")
        zt = np.zeros((self.n_mu, n_r)) if want_zeta else None
        V = np.zeros((self.n_mu, self.n_mu))
        self._ck(self._lib.gwl_isdf_build(self._h, n_r, _ptr(pv), _ptr(pc), _ptr(rr), float(weight), float(soft), _ptr(ix),
                                          _ptr(zt), _ptr(V)))
        return zt, V

    def isdf_select_points(self, r, weight, init_idx, max_iters: int = 50):
        """Weighted k-means (CVT) interpolation points; returns (idx [n_mu] int32, iterations done)."""
        rr, w, ii = _host(r), _host(weight), _host(init_idx, np.int32)
        n_r = rr.shape[0]
        if rr.shape != (n_r, 3) or w.shape != (n_r,) or ii.shape != (self.n_mu,):
            raise GwlError(GWL_EINVAL, "isdf_select_points: r [n_r, 3], weight [n_r], init_idx [n_mu]")
        idx = np.zeros(self.n_mu, dtype=np.int32)
        done = c_int32(0)
        self._ck(self._lib.gwl_isdf_select_points(self._h, n_r, _ptr(rr), _ptr(w), _ptr(ii), int(max_iters), _ptr(idx),
                                                  byref(done)))
        return idx, done.value

    # -- the path ---------------------------------------------------------------------------------
    def casida_matvec(self, x, y=None):
        """y = C x.  Host mode: x numpy [nvec, n_v, n_c] (or [nvec, n_vc]) -> numpy of the same shape.
        Device mode: x, y torch CUDA float64 tensors, contiguous; y is written in place and returned."""
        if self.device_ptrs:
            if y is None or not _is_torch(x) or not _is_torch(y):
                raise GwlError(GWL_EINVAL, "casida_matvec (device mode): x and y must be torch CUDA tensors")
            if not (x.is_contiguous() and y.is_contiguous()) or x.numel() != y.numel() or x.numel() % self.n_vc:
                raise GwlError(GWL_EINVAL, "casida_matvec: x, y must be contiguous [nvec, n_v, n_c]")
            nvec = x.numel() // self.n_vc
            self._ck(self._lib.gwl_casida_matvec(self._h, _ptr(x), _ptr(y), nvec))
            return y
        xh = _host(x)
        if xh.size % self.n_vc:
            raise GwlError(GWL_EINVAL, "casida_matvec: x must be [nvec, n_v, n_c]")
        nvec = xh.size // self.n_vc
        yh = np.empty_like(xh)
        self._ck(self._lib.gwl_casida_matvec(self._h, _ptr(xh), _ptr(yh), nvec))
        return yh

    def set_chains(self, n_idx, m_idx):
        n, m = _host(n_idx, np.int32), _host(m_idx, np.int32)
        if n.shape != m.shape or n.ndim != 1:
            raise GwlError(GWL_EINVAL, "set_chains: n_idx and m_idx must be 1-d and of equal length")
        self._ck(self._lib.gwl_set_chains(self._h, n.size, _ptr(n), _ptr(m)))

    def set_start_vectors(self, p, eps_n, sgn_n):
        e, s = _host(eps_n), _host(sgn_n, np.int32)
        if self.device_ptrs:
            n = p.numel() // self.n_vc
            pp = p
        else:
            pp = _host(p)
            n = pp.size // self.n_vc
        if e.shape != (n,) or s.shape != (n,):
            raise GwlError(GWL_EINVAL, "set_start_vectors: eps_n and sgn_n must have one entry per chain")
        self._ck(self._lib.gwl_set_start_vectors(self._h, n, _ptr(pp), _ptr(e), _ptr(s)))

    def lanczos(self, n_chains: int, steps: int, block: int, reorth: int = 0, out=None):
        """Returns (alpha[n_chains, steps], beta[n_chains, steps], norm2[n_chains], len[n_chains]).
        Device mode: pass out=(alpha, beta, norm2, len) torch CUDA tensors (or None to skip the copy-out)."""
        if self.device_ptrs:
            a = b = n2 = ln = None
            if out is not None:
                a, b, n2, ln = out
            self._ck(self._lib.gwl_lanczos(self._h, n_chains, steps, block, reorth, _ptr(a), _ptr(b), _ptr(n2), _ptr(ln)))
            return out
        a = np.zeros((n_chains, steps))
        b = np.zeros((n_chains, steps))
        n2 = np.zeros(n_chains)
        ln = np.zeros(n_chains, dtype=np.int32)
        self._ck(self._lib.gwl_lanczos(self._h, n_chains, steps, block, reorth, _ptr(a), _ptr(b), _ptr(n2), _ptr(ln)))
        return a, b, n2, ln

    def resolvent(self, zeta, n_chains: int | None = None, out=None):
        """r[chain, i] = <P|(zeta_i - Op)^-1|P> (complex).  Host mode: zeta complex numpy array."""
        if self.device_ptrs:
            n_zeta = zeta.numel() // 2
            self._ck(self._lib.gwl_resolvent(self._h, _ptr(zeta), n_zeta, _ptr(out)))
            return out
        z = np.ascontiguousarray(zeta, dtype=np.complex128)
        r = np.zeros((n_chains, z.size), dtype=np.complex128)
        self._ck(self._lib.gwl_resolvent(self._h, _ptr(z), z.size, _ptr(r)))
        return r

    def selfenergy(self, omega, eta: float, n_chains: int | None = None, want_sum: bool = True, out=None):
        """Host mode: returns (sigma[n_chains, n_omega] complex, sigma_sum[n_omega] complex or None).
        Device mode: out=(sigma [n_chains, n_omega, 2] or None, sigma_sum [n_omega, 2] or None)."""
        if self.device_ptrs:
            sg, ss = out if out is not None else (None, None)
            self._ck(self._lib.gwl_selfenergy(self._h, _ptr(omega), omega.numel(), float(eta), _ptr(sg), _ptr(ss)))
            return out
        om = _host(omega)
        sg = np.zeros((n_chains, om.size), dtype=np.complex128)
        ss = np.zeros(om.size, dtype=np.complex128) if want_sum else None
        self._ck(self._lib.gwl_selfenergy(self._h, _ptr(om), om.size, float(eta), _ptr(sg), _ptr(ss)))
        return sg, ss

    def selfenergy_state(self, m_idx: int, steps: int, block: int, reorth: int, omega, eta: float, out=None):
        """Sigma^corr_mm(omega) summed over all n (Eq. 10).  Host mode: returns complex numpy [n_omega].
        Device mode: omega and out [n_omega, 2] are torch CUDA tensors; out is returned."""
        if self.device_ptrs:
            self._ck(self._lib.gwl_selfenergy_state(self._h, int(m_idx), steps, block, reorth, _ptr(omega),
                                                    omega.numel(), float(eta), _ptr(out)))
            return out
        om = _host(omega)
        ss = np.zeros(om.size, dtype=np.complex128)
        self._ck(self._lib.gwl_selfenergy_state(self._h, int(m_idx), steps, block, reorth, _ptr(om), om.size,
                                                float(eta), _ptr(ss)))
        return ss

    def exchange(self, m_idx, out=None):
        """Sigma^ex_mm (Eq. 6) for the orbitals m_idx.  Host mode: numpy [n_states]; device mode: out torch tensor."""
        m = _host(m_idx, np.int32)
        if m.ndim != 1:
            raise GwlError(GWL_EINVAL, "exchange: m_idx must be 1-d")
        if self.device_ptrs:
            self._ck(self._lib.gwl_exchange(self._h, m.size, _ptr(m), _ptr(out)))
            return out
        sx = np.zeros(m.size)
        self._ck(self._lib.gwl_exchange(self._h, m.size, _ptr(m), _ptr(sx)))
        return sx

    def qp_solve(self, eps_m, vxc_m, sigma_x, sigma_c, omega, out=None):
        """Newton-Raphson solution of E(omega) = omega.  Host mode: sigma_c complex [n_states, n_omega];
        returns (e_qp, z_qp, iters).  Device mode: sigma_x, sigma_c [n_states, n_omega, 2], omega and
        out=(e_qp, z_qp, iters or None) are torch CUDA tensors."""
        e, v = _host(eps_m), _host(vxc_m)
        if e.ndim != 1 or e.shape != v.shape:
            raise GwlError(GWL_EINVAL, "qp_solve: eps_m and vxc_m must be 1-d and of equal length")
        n = e.size
        if self.device_ptrs:
            eq, zq, it = out
            self._ck(self._lib.gwl_qp_solve(self._h, n, _ptr(e), _ptr(v), _ptr(sigma_x), _ptr(sigma_c), _ptr(omega),
                                            omega.numel(), _ptr(eq), _ptr(zq), _ptr(it)))
            return out
        sx, om = _host(sigma_x), _host(omega)
        sc = np.ascontiguousarray(sigma_c, dtype=np.complex128)
        if sx.shape != (n,) or sc.shape != (n, om.size):
            raise GwlError(GWL_EINVAL, "qp_solve: sigma_x must be [n_states], sigma_c [n_states, n_omega]")
        eq, zq, it = np.zeros(n), np.zeros(n), np.zeros(n, dtype=np.int32)
        self._ck(self._lib.gwl_qp_solve(self._h, n, _ptr(e), _ptr(v), _ptr(sx), _ptr(sc), _ptr(om), om.size, _ptr(eq),
                                        _ptr(zq), _ptr(it)))
        return eq, zq, it

    def get_timing(self):
        a, b, c = c_double(), c_double(), c_double()
        self._ck(self._lib.gwl_get_timing(self._h, byref(a), byref(b), byref(c)))
        return a.value, b.value, c.value

    def set_profiling(self, level: int):
        self._ck(self._lib.gwl_set_profiling(self._h, int(level)))

    def get_kernel_times(self):
        """{class name: (ms, launches)} since the start of the last lanczos call (profiling level 2)."""
        n = len(KERNEL_CLASSES)
        ms = (c_double * n)()
        cnt = (c_int64 * n)()
        self._ck(self._lib.gwl_get_kernel_times(self._h, ms, cnt))
        return {KERNEL_CLASSES[i]: (ms[i], cnt[i]) for i in range(n)}

    def get_launch_count(self) -> int:
        n = c_int64()
        self._ck(self._lib.gwl_get_launch_count(self._h, byref(n)))
        return n.value


class TdcContext(Context):
    """Complex-orbital (periodic Tamm-Dancoff) context, gwl_tdc_* (SURVEY.md 8(f)-3).
    lanczos / resolvent / selfenergy / timing calls are the inherited ones."""

    def __init__(self, n_k: int, n_v: int, n_c: int, n_mu: int, n_q: int = 1):
        self._lib = load_library()
        self._h = c_void_p()
        self.n_k, self.n_v, self.n_c, self.n_mu, self.n_q = int(n_k), int(n_v), int(n_c), int(n_mu), int(n_q)
        self.n_kvc = self.n_k * self.n_v * self.n_c
        self.n_vc = 2 * self.n_kvc                        # real entries of one (planar) Lanczos vector
        self.device_ptrs = 0
        st = self._lib.gwl_tdc_create(byref(self._h), n_k, n_v, n_c, n_mu, n_q)
        if st != GWL_OK:
            self._h = c_void_p()
            raise GwlError(st, "gwl_tdc_create failed (no CUDA device, or bad sizes)")

    def set_orbitals(self, psi_v, psi_cq):
        pv = np.ascontiguousarray(psi_v, dtype=np.complex128)
        pc = np.ascontiguousarray(psi_cq, dtype=np.complex128)
        if pv.shape != (self.n_k, self.n_mu, self.n_v) or pc.shape != (self.n_k, self.n_mu, self.n_c):
            raise GwlError(GWL_EINVAL, "set_orbitals: psi_v must be [n_k, n_mu, n_v], psi_cq [n_k, n_mu, n_c] complex")
        self._ck(self._lib.gwl_tdc_set_orbitals(self._h, _ptr(pv), _ptr(pc)))

    def set_energies(self, eps_v, eps_cq):
        ev, ec = _host(eps_v), _host(eps_cq)
        if ev.shape != (self.n_k, self.n_v) or ec.shape != (self.n_k, self.n_c):
            raise GwlError(GWL_EINVAL, "set_energies: eps_v must be [n_k, n_v], eps_cq [n_k, n_c]")
        self._ck(self._lib.gwl_tdc_set_energies(self._h, _ptr(ev), _ptr(ec)))

    def set_chains(self, chains):
        ch = _host(chains, np.int32)
        if ch.ndim != 2 or ch.shape[1] != 4:
            raise GwlError(GWL_EINVAL, "set_chains: chains must be [n_chains, 4] = (k slot of n, n, k slot of m, m)")
        self._ck(self._lib.gwl_tdc_set_chains(self._h, ch.shape[0], _ptr(ch)))

    def matvec(self, x, y=None):
        """y = A(q) x.  Host mode: x complex numpy [nvec, n_k, n_v, n_c] (or [nvec, n_kvc]).  Device mode: x, y torch
        CUDA complex128 tensors, contiguous."""
        if self.device_ptrs:
            nvec = x.numel() // self.n_kvc
            self._ck(self._lib.gwl_tdc_matvec(self._h, _ptr(x), _ptr(y), nvec))
            return y
        xh = np.ascontiguousarray(x, dtype=np.complex128)
        if xh.size % self.n_kvc:
            raise GwlError(GWL_EINVAL, "matvec: x must be [nvec, n_k, n_v, n_c]")
        yh = np.empty_like(xh)
        self._ck(self._lib.gwl_tdc_matvec(self._h, _ptr(xh), _ptr(yh), xh.size // self.n_kvc))
        return yh

    def selfenergy_state(self, kn: int, km: int, m_idx: int, steps: int, block: int, reorth: int, omega, eta: float, out=None):
        """The q-term of Sigma_{mk,mk}(omega) summed over all n of slot kn (PAPER.md:288 / :310).  Host mode: complex numpy
        [n_omega]; device mode: omega and out [n_omega, 2] torch CUDA tensors."""
        if self.device_ptrs:
            self._ck(self._lib.gwl_tdc_selfenergy_state(self._h, int(kn), int(km), int(m_idx), steps, block, reorth, _ptr(omega),
                                                        omega.numel(), float(eta), _ptr(out)))
            return out
        om = _host(omega)
        ss = np.zeros(om.size, dtype=np.complex128)
        self._ck(self._lib.gwl_tdc_selfenergy_state(self._h, int(kn), int(km), int(m_idx), steps, block, reorth, _ptr(om), om.size,
                                                    float(eta), _ptr(ss)))
        return ss

    def matvec_rpa(self, x, y, ox=None, oy=None):
        """[ox; oy] = Omega^ [x; y] = [A x + B y; B^* x + A^* y].  Host mode: complex numpy arrays
        [nvec, n_kvc]; device mode: torch CUDA complex128 tensors (ox, oy given)."""
        if self.device_ptrs:
            nvec = x.numel() // self.n_kvc
            self._ck(self._lib.gwl_tdc_matvec_rpa(self._h, _ptr(x), _ptr(y), _ptr(ox), _ptr(oy), nvec))
            return ox, oy
        xh = np.ascontiguousarray(x, dtype=np.complex128)
        yh = np.ascontiguousarray(y, dtype=np.complex128)
        if xh.size % self.n_kvc or xh.shape != yh.shape:
            raise GwlError(GWL_EINVAL, "matvec_rpa: x and y must both be [nvec, n_k, n_v, n_c]")
        oxh, oyh = np.empty_like(xh), np.empty_like(yh)
        self._ck(self._lib.gwl_tdc_matvec_rpa(self._h, _ptr(xh), _ptr(yh), _ptr(oxh), _ptr(oyh), xh.size // self.n_kvc))
        return oxh, oyh


class SymContext(Context):
    """Symmetry-block context, gwl_sym_* (reading Q25): an abelian point group of
    order 2^n_gen, orbitals sorted by irrep.  After select(gamma) the inherited set_chains / lanczos / resolvent /
    selfenergy / set_polynomial calls act on block gamma."""

    def __init__(self, n_gen: int, nv_irrep, nc_irrep, n_mu_w: int):
        self._lib = load_library()
        self._h = c_void_p()
        self.nv_irrep, self.nc_irrep = _host(nv_irrep, np.int32), _host(nc_irrep, np.int32)
        self.g = 1 << int(n_gen)
        if self.nv_irrep.shape != (self.g,) or self.nc_irrep.shape != (self.g,):
            raise GwlError(GWL_EINVAL, "SymContext: nv_irrep and nc_irrep need 2^n_gen entries")
        self.n_v, self.n_c, self.n_mu = int(self.nv_irrep.sum()), int(self.nc_irrep.sum()), int(n_mu_w)
        self.n_vc = 0                                      # pairs of the selected block
        self.device_ptrs = 0
        st = self._lib.gwl_sym_create(byref(self._h), int(n_gen), _ptr(self.nv_irrep), _ptr(self.nc_irrep), int(n_mu_w))
        if st != GWL_OK:
            self._h = c_void_p()
            raise GwlError(st, "gwl_sym_create failed (no CUDA device, or bad sizes)")

    def set_orbitals(self, phi_v_w, phi_c_w):
        pv, pc = _host(phi_v_w), _host(phi_c_w)
        if pv.shape != (self.n_mu, self.n_v) or pc.shape != (self.n_mu, self.n_c):
            raise GwlError(GWL_EINVAL, "set_orbitals: phi_v_w must be [n_mu_w, N_v], phi_c_w [n_mu_w, N_c]")
        self._ck(self._lib.gwl_sym_set_orbitals(self._h, _ptr(pv), _ptr(pc)))

    def set_kernel(self, V_wf):
        Vh = _host(V_wf)
        if Vh.shape != (self.n_mu, self.g, self.n_mu):
            raise GwlError(GWL_EINVAL, "set_kernel: V_wf must be [n_mu_w, g, n_mu_w]")
        self._ck(self._lib.gwl_sym_set_kernel(self._h, _ptr(Vh)))

    def select(self, gamma: int) -> int:
        n = c_int64(0)
        self._ck(self._lib.gwl_sym_select(self._h, int(gamma), byref(n)))
        self.n_vc = n.value
        return n.value

    def matvec(self, x, y=None):
        """y = C_gamma x on the selected block.  Host mode: numpy [nvec, n_pairs]; device mode: torch CUDA tensors."""
        if self.device_ptrs:
            self._ck(self._lib.gwl_sym_matvec(self._h, _ptr(x), _ptr(y), x.numel() // self.n_vc))
            return y
        xh = _host(x)
        if self.n_vc == 0 or xh.size % self.n_vc:
            raise GwlError(GWL_EINVAL, "matvec: x must be [nvec, n_pairs of the selected block]")
        yh = np.empty_like(xh)
        self._ck(self._lib.gwl_sym_matvec(self._h, _ptr(xh), _ptr(yh), xh.size // self.n_vc))
        return yh

    def selfenergy_state(self, m_idx: int, steps: int, block: int, reorth: int, omega, eta: float, out=None):
        if self.device_ptrs:
            self._ck(self._lib.gwl_sym_selfenergy_state(self._h, int(m_idx), steps, block, reorth, _ptr(omega), omega.numel(),
                                                        float(eta), _ptr(out)))
            return out
        om = _host(omega)
        ss = np.zeros(om.size, dtype=np.complex128)
        self._ck(self._lib.gwl_sym_selfenergy_state(self._h, int(m_idx), steps, block, reorth, _ptr(om), om.size, float(eta),
                                                    _ptr(ss)))
        return ss


def context_from_problem(prob) -> Context:
    """Creates a context and uploads the inputs of a synth.Problem (orbitals, energies, kernel, chains)."""
    cfg = prob.cfg
    ctx = Context(cfg.n_v, cfg.n_c, cfg.n_mu)
    ctx.set_orbitals(prob.phi_v, prob.phi_c)
    ctx.set_energies(prob.eps_v, prob.eps_c)
    ctx.set_kernel(prob.V)
    ctx.set_chains(prob.n_idx, prob.m_idx)
    return ctx
