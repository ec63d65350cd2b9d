"""Thin ctypes binding of libtdvp.so (include/tdvp.h).  Argument marshalling only: every step of
the path runs in the library's CUDA kernels.  PyTorch is used for device memory and streams.

The function names are those of the C ABI.  The stateless calls take complex128 CUDA tensors
(C-contiguous) and return / fill CUDA tensors; `Chain` wraps a `tdvp_handle` created by
`tdvp_create(mpo, mps)`.

There is no CPU fallback: if libtdvp.so is missing or cannot be loaded, importing a symbol from
here raises.  Build it with `python -m paper_1907_12044_b200.build`.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_longlong, c_void_p

import numpy as np
import torch

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libtdvp.so")

TDVP_OK, TDVP_EINVAL, TDVP_ENOMEM, TDVP_ECUDA, TDVP_ESTATE = 0, -1, -2, -3, -4
TDVP_FLAG_SKIP_CANONICAL_CHECK = 1
TDVP_FLAG_NO_GRAPH = 2
TDVP_MAX_KRYLOV = 64

# every symbol include/tdvp.h declares (tests check that the library exports each of them)
EXPORTED_SYMBOLS = [
    "tdvp_default_options", "tdvp_create_context", "tdvp_create", "tdvp_destroy",
    "tdvp_apply_heff", "tdvp_update_env", "tdvp_apply_bond", "tdvp_expm_heff", "tdvp_expm_bond",
    "tdvp_qr_gauge", "tdvp_svd_bond", "tdvp_apply_heff_host", "tdvp_apply_heff_site", "tdvp_update_env_site",
    "tdvp_step_ps", "tdvp_step_mu", "tdvp_step_mu_cmf", "tdvp_mu_derivative", "tdvp_set_gauge", "tdvp_observe", "tdvp_populations",
    "tdvp_norm_energy", "tdvp_get_mps", "tdvp_set_mps", "tdvp_get_centre", "tdvp_sync",
    "tdvp_last_error", "tdvp_probe_fp64_tensor_peak", "tdvp_probe_dmma_issue", "tdvp_set_gemm_products", "tdvp_get_gemm_products", "tdvp_launch_count", "tdvp_profile_enable",
    "tdvp_profile_read", "tdvp_pc_rk4_warmup", "tdvp_build_vibronic_mpo", "tdvp_step_ps2", "tdvp_qr_gauge_noalloc",
]


class tdvp_options(ctypes.Structure):
    _fields_ = [("krylov_dim", c_int), ("krylov_tol", c_double), ("mu_eps", c_double),
                ("w_zero_tol", c_double), ("flags", c_int)]


class TdvpError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libtdvp error %d: %s" % (code, msg))
        self.code = code


def _load():
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            "libtdvp.so not found at %s: the CUDA extension is not built and there is no CPU "
            "fallback.  Run `python -m paper_1907_12044_b200.build`." % _LIB_PATH)
    lib = ctypes.CDLL(_LIB_PATH)
    P = c_void_p
    sig = {
        "tdvp_default_options": (None, [POINTER(tdvp_options)]),
        "tdvp_create_context": (c_int, [POINTER(P), POINTER(tdvp_options), P]),
        "tdvp_create": (c_int, [POINTER(P), c_int, POINTER(c_int), POINTER(c_int), POINTER(P),
                                POINTER(c_int), POINTER(P), c_int, POINTER(tdvp_options), P]),
        "tdvp_destroy": (c_int, [P]),
        "tdvp_apply_heff": (c_int, [P, c_int, c_int, c_int, c_int, c_int, P, P, P, P, P]),
        "tdvp_apply_heff_host": (c_int, [P, c_int, c_int, c_int, c_int, c_int, P, P, P, P, P]),
        "tdvp_update_env": (c_int, [P, c_int, c_int, c_int, c_int, c_int, c_int, P, P, P, P]),
        "tdvp_apply_bond": (c_int, [P, c_int, c_int, c_int, P, P, P, P]),
        "tdvp_expm_heff": (c_int, [P, c_int, c_int, c_int, c_int, c_int, P, P, P, c_double, c_double,
                                   P, P, POINTER(c_int)]),
        "tdvp_expm_bond": (c_int, [P, c_int, c_int, c_int, P, P, c_double, c_double, P, P, POINTER(c_int)]),
        "tdvp_qr_gauge": (c_int, [P, c_int, c_int, c_int, c_int, P, P, P]),
        "tdvp_qr_gauge_noalloc": (c_int, [P, c_int, c_int, c_int, c_int, P, P, P]),
        "tdvp_svd_bond": (c_int, [P, c_int, c_int, c_int, P, P, P, P]),
        "tdvp_apply_heff_site": (c_int, [P, c_int, P, P]),
        "tdvp_update_env_site": (c_int, [P, c_int, c_int]),
        "tdvp_step_ps": (c_int, [P, c_double]),
        "tdvp_step_ps2": (c_int, [P, c_double]),
        "tdvp_step_mu": (c_int, [P, c_double, POINTER(c_double)]),
        "tdvp_step_mu_cmf": (c_int, [P, c_double, c_int]),
        "tdvp_mu_derivative": (c_int, [P, POINTER(P)]),
        "tdvp_set_gauge": (c_int, [P, c_int]),
        "tdvp_observe": (c_int, [P, c_int, P, P]),
        "tdvp_populations": (c_int, [P, c_int, POINTER(c_double)]),
        "tdvp_norm_energy": (c_int, [P, POINTER(c_double), POINTER(c_double)]),
        "tdvp_get_mps": (c_int, [P, c_int, P, POINTER(c_int), POINTER(c_int)]),
        "tdvp_set_mps": (c_int, [P, POINTER(P), c_int]),
        "tdvp_get_centre": (c_int, [P]),
        "tdvp_sync": (c_int, [P]),
        "tdvp_last_error": (c_char_p, [P]),
        "tdvp_probe_fp64_tensor_peak": (c_int, [c_int, POINTER(c_double)]),
        "tdvp_probe_dmma_issue": (c_int, [c_int, c_int, POINTER(c_double)]),
        "tdvp_launch_count": (c_longlong, []),
        "tdvp_set_gemm_products": (c_int, [c_int]),
        "tdvp_get_gemm_products": (c_int, []),
        "tdvp_profile_enable": (c_int, [c_int]),
        "tdvp_profile_read": (c_int, [POINTER(c_double), POINTER(c_longlong)]),
        "tdvp_build_vibronic_mpo": (c_int, [c_int, c_int, c_int, c_int, POINTER(c_double), POINTER(c_double), POINTER(c_double),
                                            POINTER(c_double), c_double, POINTER(c_int), POINTER(c_int), POINTER(c_int), POINTER(P)]),
        "tdvp_pc_rk4_warmup": (c_int, [P, c_int, POINTER(c_int), POINTER(c_int), POINTER(P), POINTER(c_int), POINTER(P),
                                       c_double, c_int, c_int, c_int, POINTER(c_int), POINTER(P)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    return lib


_lib = _load()


def library_path() -> str:
    return _LIB_PATH


def _check(rc, handle=None):
    if rc != TDVP_OK:
        msg = _lib.tdvp_last_error(handle)
        raise TdvpError(rc, msg.decode() if msg else "")


def _dev(t: torch.Tensor, shape=None) -> int:
    if not (t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()):
        raise TypeError("expected a contiguous complex128 CUDA tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError("expected shape %s, got %s" % (tuple(shape), tuple(t.shape)))
    return t.data_ptr()


def _hptr(h):
    return h._h if isinstance(h, (Context, Chain)) else h


def make_options(krylov_dim=10, krylov_tol=0.0, mu_eps=1e-10, w_zero_tol=0.0, flags=0) -> tdvp_options:
    o = tdvp_options()
    _lib.tdvp_default_options(byref(o))
    o.krylov_dim, o.krylov_tol, o.mu_eps, o.w_zero_tol, o.flags = krylov_dim, krylov_tol, mu_eps, w_zero_tol, flags
    return o


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return c_void_p(stream.cuda_stream)


class Context:
    """tdvp_create_context: a stream + workspace for the stateless calls."""

    def __init__(self, options: tdvp_options | None = None, stream=None):
        self._h = c_void_p()
        _check(_lib.tdvp_create_context(byref(self._h), byref(options) if options else None, _stream_ptr(stream)))

    def tdvp_sync(self):
        _check(_lib.tdvp_sync(self._h), self._h)

    def close(self):
        if self._h:
            _lib.tdvp_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def tdvp_create_context(options=None, stream=None) -> Context:
    return Context(options, stream)


# ---- stateless contractions ------------------------------------------------------------------

def tdvp_apply_heff(L, W, A, R, out=None, handle=None):
    Ml, Dl, _ = L.shape
    Mr, Dr, _ = R.shape
    d = A.shape[1]
    if out is None:
        out = torch.empty((Ml, d, Mr), dtype=torch.complex128, device=A.device)
    h = _hptr(handle)
    _check(_lib.tdvp_apply_heff(h, Ml, Mr, d, Dl, Dr, _dev(L, (Ml, Dl, Ml)), _dev(W, (Dl, d, d, Dr)),
                                _dev(A, (Ml, d, Mr)), _dev(R, (Mr, Dr, Mr)), _dev(out, (Ml, d, Mr))), h)
    return out


def tdvp_apply_heff_host(L, W, A, R, out, handle=None):
    """HOST numpy complex128 arrays in and out: H2D copies, the apply, D2H copy, blocking."""
    Ml, Dl, _ = L.shape
    Mr, Dr, _ = R.shape
    d = A.shape[1]
    for x in (L, W, A, R, out):
        if not (isinstance(x, np.ndarray) and x.dtype == np.complex128 and x.flags.c_contiguous):
            raise TypeError("expected C-contiguous complex128 numpy arrays")
    h = _hptr(handle)
    _check(_lib.tdvp_apply_heff_host(h, Ml, Mr, d, Dl, Dr, L.ctypes.data, W.ctypes.data, A.ctypes.data,
                                     R.ctypes.data, out.ctypes.data), h)
    return out


def tdvp_update_env(side, env_in, W, A, env_out=None, handle=None):
    Ml, d, Mr = A.shape
    Dl, _, _, Dr = W.shape
    shp_in = (Ml, Dl, Ml) if side == 0 else (Mr, Dr, Mr)
    shp_out = (Mr, Dr, Mr) if side == 0 else (Ml, Dl, Ml)
    if env_out is None:
        env_out = torch.empty(shp_out, dtype=torch.complex128, device=A.device)
    h = _hptr(handle)
    _check(_lib.tdvp_update_env(h, side, Ml, Mr, d, Dl, Dr, _dev(env_in, shp_in), _dev(W, (Dl, d, d, Dr)),
                                _dev(A), _dev(env_out, shp_out)), h)
    return env_out


def tdvp_apply_bond(L, D, R, out=None, handle=None):
    Ml, Dw, _ = L.shape
    Mr = R.shape[0]
    if out is None:
        out = torch.empty((Ml, Mr), dtype=torch.complex128, device=D.device)
    h = _hptr(handle)
    _check(_lib.tdvp_apply_bond(h, Ml, Mr, Dw, _dev(L, (Ml, Dw, Ml)), _dev(D, (Ml, Mr)), _dev(R, (Mr, Dw, Mr)),
                                _dev(out, (Ml, Mr))), h)
    return out


def tdvp_expm_heff(L, W, R, z, v, y=None, handle=None, want_dim=False):
    Ml, Dl, _ = L.shape
    Mr, Dr, _ = R.shape
    d = v.shape[1]
    if y is None:
        y = torch.empty_like(v)
    h = _hptr(handle)
    m = c_int(0)
    _check(_lib.tdvp_expm_heff(h, Ml, Mr, d, Dl, Dr, _dev(L, (Ml, Dl, Ml)), _dev(W, (Dl, d, d, Dr)),
                               _dev(R, (Mr, Dr, Mr)), float(np.real(z)), float(np.imag(z)), _dev(v, (Ml, d, Mr)),
                               _dev(y, (Ml, d, Mr)), byref(m) if want_dim else None), h)
    return (y, m.value) if want_dim else y


def tdvp_expm_bond(L, R, z, v, y=None, handle=None, want_dim=False):
    Ml, Dw, _ = L.shape
    Mr = R.shape[0]
    if y is None:
        y = torch.empty_like(v)
    h = _hptr(handle)
    m = c_int(0)
    _check(_lib.tdvp_expm_bond(h, Ml, Mr, Dw, _dev(L, (Ml, Dw, Ml)), _dev(R, (Mr, Dw, Mr)), float(np.real(z)),
                               float(np.imag(z)), _dev(v, (Ml, Mr)), _dev(y, (Ml, Mr)),
                               byref(m) if want_dim else None), h)
    return (y, m.value) if want_dim else y


def tdvp_qr_gauge(side, C, handle=None):
    Ml, d, Mr = C.shape
    Q = torch.empty_like(C)
    n = Mr if side == 0 else Ml
    D = torch.empty((n, n), dtype=torch.complex128, device=C.device)
    h = _hptr(handle)
    _check(_lib.tdvp_qr_gauge(h, side, Ml, d, Mr, _dev(C), _dev(Q), _dev(D)), h)
    return Q, D


def tdvp_qr_gauge_noalloc(side, C, Q, D, stream=None):
    """tdvp_qr_gauge without any allocation (include/tdvp.h): the caller passes the outputs too --
    Q like C, D [n, n] with n = Mr (side 0) or Ml (side 1); scratch is the library's static 6 MiB block."""
    Ml, d, Mr = C.shape
    n = Mr if side == 0 else Ml
    _check(_lib.tdvp_qr_gauge_noalloc(_stream_ptr(stream), side, Ml, d, Mr, _dev(C), _dev(Q, (Ml, d, Mr)), _dev(D, (n, n))))
    return Q, D


def tdvp_svd_bond(C, handle=None):
    """C[Ml,d,Mr] viewed as Ml x (d*Mr) = U diag(lam) Vh; returns (U[Ml,Ml], lam[Ml] float64, Vh[Ml,d,Mr])."""
    Ml, d, Mr = C.shape
    U = torch.empty((Ml, Ml), dtype=torch.complex128, device=C.device)
    lam = torch.empty((Ml,), dtype=torch.float64, device=C.device)
    Vh = torch.empty_like(C)
    h = _hptr(handle)
    _check(_lib.tdvp_svd_bond(h, Ml, d, Mr, _dev(C), _dev(U), c_void_p(lam.data_ptr()), _dev(Vh)), h)
    return U, lam, Vh


CM1_TO_RAD_PER_FS = 1.8836515673e-4        # 2 pi c: energies in cm^-1 -> angular frequencies in rad/fs (reading c5)


def tdvp_build_vibronic_mpo(E, J, omega, huang_rhys, n_ph, layout="A", energy_unit=CM1_TO_RAD_PER_FS):
    """Frenkel-Holstein Hamiltonian (Eq. 45) -> list of HOST numpy MPO site tensors W_i[Dl, d, d, Dr]
    (include/tdvp.h).  Host-only: needs no GPU."""
    E = np.ascontiguousarray(E, dtype=np.float64)
    J = np.ascontiguousarray(J, dtype=np.float64)
    om = np.ascontiguousarray(omega, dtype=np.float64)
    S = np.ascontiguousarray(huang_rhys, dtype=np.float64)
    n_el = E.shape[0]
    n_modes = om.shape[1] if om.ndim == 2 else 0
    lay = {"A": 0, "B": 1}[layout]
    dp = lambda a: a.ctypes.data_as(POINTER(c_double))
    n = c_int(0)
    cap = n_el * (1 + max(n_modes, 0)) + 1
    phys, bond = (c_int * cap)(), (c_int * (cap + 1))()
    _check(_lib.tdvp_build_vibronic_mpo(lay, n_el, n_modes, int(n_ph), dp(E), dp(J), dp(om), dp(S), float(energy_unit),
                                        byref(n), phys, bond, None))
    ns = n.value
    out = [np.empty((bond[i], phys[i], phys[i], bond[i + 1]), dtype=np.complex128) for i in range(ns)]
    PA = c_void_p * ns
    _check(_lib.tdvp_build_vibronic_mpo(lay, n_el, n_modes, int(n_ph), dp(E), dp(J), dp(om), dp(S), float(energy_unit),
                                        byref(n), phys, bond, PA(*[o.ctypes.data for o in out])))
    return out


def tdvp_pc_rk4_warmup(mpo, mps, tau, n_steps, M_max, M_out, handle=None):
    """P&C-RK4 warm-up (include/tdvp.h): HOST numpy MPO / MPS in, list of HOST numpy site tensors out
    (right-canonical, centre at site 0, bonds min(M_out, what the shapes allow))."""
    n = len(mps)
    keep = [np.ascontiguousarray(t, dtype=np.complex128) for t in list(mpo) + list(mps)]
    phys = [int(A.shape[1]) for A in mps]
    mpo_bond = [int(W.shape[0]) for W in mpo] + [int(mpo[-1].shape[3])]
    mps_bond = [int(A.shape[0]) for A in mps] + [int(mps[-1].shape[2])]
    left, right = [1] * (n + 1), [1] * (n + 1)
    for i in range(n):
        left[i + 1] = min(left[i] * phys[i], 1 << 40)
    for i in range(n - 1, -1, -1):
        right[i] = min(right[i + 1] * phys[i], 1 << 40)
    cap = [int(min(M_out, left[i], right[i])) for i in range(n + 1)]
    outs = [np.zeros(cap[i] * phys[i] * cap[i + 1], dtype=np.complex128) for i in range(n)]
    PA, IA, IB = c_void_p * n, c_int * n, c_int * (n + 1)
    bonds = IB()
    h = _hptr(handle)
    _check(_lib.tdvp_pc_rk4_warmup(h, n, IA(*phys), IB(*mpo_bond), PA(*[t.ctypes.data for t in keep[:n]]), IB(*mps_bond),
                                   PA(*[t.ctypes.data for t in keep[n:]]), float(tau), int(n_steps), int(M_max), int(M_out),
                                   bonds, PA(*[o.ctypes.data for o in outs])), h)
    b = list(bonds)
    return [outs[i][:b[i] * phys[i] * b[i + 1]].reshape(b[i], phys[i], b[i + 1]).copy() for i in range(n)]


def tdvp_probe_fp64_tensor_peak(iters=20000) -> float:
    t = c_double(0.0)
    _check(_lib.tdvp_probe_fp64_tensor_peak(iters, byref(t)))
    return t.value


PROFILE_PHASES = ("zgemm", "wstage", "vector", "qr", "svd")


def tdvp_probe_dmma_issue(fillers, iters=4000) -> float:
    t = c_double(0.0)
    _check(_lib.tdvp_probe_dmma_issue(int(fillers), iters, byref(t)))
    return t.value


def tdvp_profile_enable(on: bool):
    _check(_lib.tdvp_profile_enable(1 if on else 0))


def tdvp_profile_read():
    """{phase: (milliseconds, brackets)} since the last read; blocks on the device."""
    ms = (c_double * len(PROFILE_PHASES))()
    cnt = (c_longlong * len(PROFILE_PHASES))()
    _check(_lib.tdvp_profile_read(ms, cnt))
    return {name: (ms[i], int(cnt[i])) for i, name in enumerate(PROFILE_PHASES)}


def tdvp_set_gemm_products(products: int) -> None:
    """3 (default) or 4 real DMMA products per complex product in the GEMM stages (include/tdvp.h)."""
    _check(_lib.tdvp_set_gemm_products(int(products)))


def tdvp_get_gemm_products() -> int:
    return int(_lib.tdvp_get_gemm_products())


def tdvp_launch_count() -> int:
    return int(_lib.tdvp_launch_count())


# ---- resident chain --------------------------------------------------------------------------

class Chain:
    """tdvp_create(mpo, mps): the resident MPS + MPO + environment cache of one chain."""

    def __init__(self, mpo, mps, options: tdvp_options | None = None, stream=None):
        """mpo[i]: W_i[Dl,d,d,Dr], mps[i]: A_i[Ml,d,Mr]; numpy complex128 (HOST) or torch CUDA
        complex128 tensors (DEVICE) -- all of one kind.  MPS right-canonical, centre at site 0."""
        n = len(mps)
        assert len(mpo) == n
        on_device = isinstance(mps[0], torch.Tensor)
        self.n = n
        self.phys = [int(A.shape[1]) for A in mps]
        self.mpo_bond = [int(W.shape[0]) for W in mpo] + [int(mpo[-1].shape[3])]
        self.mps_bond = [int(A.shape[0]) for A in mps] + [int(mps[-1].shape[2])]
        if on_device:
            keep = [t.contiguous() for t in list(mpo) + list(mps)]
            ptrs = [_dev(t) for t in keep]
        else:
            keep = [np.ascontiguousarray(t, dtype=np.complex128) for t in list(mpo) + list(mps)]
            ptrs = [t.ctypes.data for t in keep]
        PA = c_void_p * n
        self._h = c_void_p()
        IA, IB = c_int * n, c_int * (n + 1)
        _check(_lib.tdvp_create(byref(self._h), n, IA(*self.phys), IB(*self.mpo_bond), PA(*ptrs[:n]),
                                IB(*self.mps_bond), PA(*ptrs[n:]), 1 if on_device else 0,
                                byref(options) if options else None, _stream_ptr(stream)))

    def close(self):
        if self._h:
            _lib.tdvp_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def tdvp_step_ps(self, dt):
        _check(_lib.tdvp_step_ps(self._h, float(dt)), self._h)

    def tdvp_step_ps2(self, dt):
        _check(_lib.tdvp_step_ps2(self._h, float(dt)), self._h)

    def tdvp_step_mu(self, dt, want_err=False):
        e = c_double(0.0)
        _check(_lib.tdvp_step_mu(self._h, float(dt), byref(e) if want_err else None), self._h)
        return e.value if want_err else None

    def tdvp_step_mu_cmf(self, dt, n_sub):
        _check(_lib.tdvp_step_mu_cmf(self._h, float(dt), int(n_sub)), self._h)

    def tdvp_mu_derivative(self):
        """Time derivatives of the resident (left-canonical) MPS, as HOST numpy arrays."""
        outs = [np.empty((self.mps_bond[i], self.phys[i], self.mps_bond[i + 1]), dtype=np.complex128)
                for i in range(self.n)]
        PA = c_void_p * self.n
        _check(_lib.tdvp_mu_derivative(self._h, PA(*[o.ctypes.data for o in outs])), self._h)
        return outs

    def tdvp_set_gauge(self, centre):
        _check(_lib.tdvp_set_gauge(self._h, int(centre)), self._h)

    def tdvp_get_centre(self):
        c = _lib.tdvp_get_centre(self._h)
        if c < 0:
            _check(c, self._h)
        return c

    def tdvp_apply_heff_site(self, site, A, out=None):
        if out is None:
            out = torch.empty_like(A)
        shp = (self.mps_bond[site], self.phys[site], self.mps_bond[site + 1])
        _check(_lib.tdvp_apply_heff_site(self._h, site, _dev(A, shp), _dev(out, shp)), self._h)
        return out

    def tdvp_update_env_site(self, site, side):
        _check(_lib.tdvp_update_env_site(self._h, site, side), self._h)

    def tdvp_observe(self, site, op):
        op = np.ascontiguousarray(op, dtype=np.complex128)
        assert op.shape == (self.phys[site], self.phys[site])
        out = np.zeros(1, dtype=np.complex128)
        _check(_lib.tdvp_observe(self._h, site, op.ctypes.data, out.ctypes.data), self._h)
        return complex(out[0])

    def tdvp_populations(self, site=0):
        out = (c_double * self.phys[site])()
        _check(_lib.tdvp_populations(self._h, site, out), self._h)
        return np.array(out[:], dtype=np.float64)

    def tdvp_norm_energy(self):
        nrm, en = c_double(0.0), c_double(0.0)
        _check(_lib.tdvp_norm_energy(self._h, byref(nrm), byref(en)), self._h)
        return nrm.value, en.value

    def tdvp_get_mps(self, site=None):
        if site is None:
            return [self.tdvp_get_mps(i) for i in range(self.n)]
        out = np.empty((self.mps_bond[site], self.phys[site], self.mps_bond[site + 1]), dtype=np.complex128)
        _check(_lib.tdvp_get_mps(self._h, site, out.ctypes.data, None, None), self._h)
        return out

    def tdvp_set_mps(self, mps, centre=0):
        keep = [np.ascontiguousarray(t, dtype=np.complex128) for t in mps]
        for i, t in enumerate(keep):
            assert t.shape == (self.mps_bond[i], self.phys[i], self.mps_bond[i + 1])
        PA = c_void_p * self.n
        _check(_lib.tdvp_set_mps(self._h, PA(*[t.ctypes.data for t in keep]), int(centre)), self._h)

    def tdvp_sync(self):
        _check(_lib.tdvp_sync(self._h), self._h)


def tdvp_create(mpo, mps, options=None, stream=None) -> Chain:
    return Chain(mpo, mps, options, stream)
