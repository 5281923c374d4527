"""Thin ctypes binding of libpyro.so (include/pyro.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used
here for device memory and streams.  There is no CPU fallback: if libpyro.so is missing
or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpyro.so")

EXPORTS = (
    "pyro_mech_create", "pyro_mech_destroy", "pyro_mech_set_newton", "pyro_get_temperature",
    "pyro_get_temperature_from_enthalpy", "pyro_get_density", "pyro_get_pressure",
    "pyro_get_net_production_rates", "pyro_get_jacobian", "pyro_reactor_rk4", "pyro_reactor_rk4_static", "pyro_reactor_cn", "pyro_reactor_cn_work_doubles", "pyro_source_terms", "pyro_source_terms_host", "pyro_mech_info", "pyro_probe_fp64_peak", "pyro_probe_dmma_peak", "pyro_probe_indexed_rmw",
    "pyro_status_string", "pyro_last_error_string", "pyro_transport_create", "pyro_transport_destroy",
    "pyro_get_transport",
)

PYRO_OK = 0
RK4_STATIC_MAX_DOUBLES = 4194304   # PYRO_RK4_STATIC_MAX_DOUBLES of pyro.h
STATUS_NAMES = {0: "PYRO_OK", 1: "PYRO_ERR_NULL", 2: "PYRO_ERR_BAD_SIZE", 3: "PYRO_ERR_BAD_MECH",
                4: "PYRO_ERR_TOO_LARGE", 5: "PYRO_ERR_ALIGN", 6: "PYRO_ERR_CUDA", 7: "PYRO_ERR_UNSUPPORTED"}


class PyroError(RuntimeError):
    def __init__(self, status, detail):
        self.status = int(status)
        super().__init__(f"{STATUS_NAMES.get(self.status, self.status)}: {detail}")


class MechDesc(C.Structure):
    """Mirror of pyro_mech_desc."""
    _fields_ = [
        ("n_species", C.c_int32), ("n_reactions", C.c_int32), ("n_elements", C.c_int32),
        ("mol_weight", C.c_void_p), ("nasa_lo", C.c_void_p), ("nasa_hi", C.c_void_p), ("t_mid", C.c_void_p),
        ("elem_comp", C.c_void_p),
        ("reac_ptr", C.c_void_p), ("reac_species", C.c_void_p), ("reac_coeff", C.c_void_p),
        ("prod_ptr", C.c_void_p), ("prod_species", C.c_void_p), ("prod_coeff", C.c_void_p),
        ("A", C.c_void_p), ("b", C.c_void_p), ("theta", C.c_void_p),
        ("type", C.c_void_p), ("reversible", C.c_void_p),
        ("eff_default", C.c_void_p), ("eff_ptr", C.c_void_p), ("eff_species", C.c_void_p),
        ("eff_value", C.c_void_p),
        ("A0", C.c_void_p), ("b0", C.c_void_p), ("theta0", C.c_void_p), ("troe", C.c_void_p),
    ]


_lib = None


def probe_dmma_peak(device=0, millis=200.0):
    """Measured mma.sync.m8n8k4.f64 peak of the device in TFLOP/s."""
    out = C.c_double(0.0)
    _check(load_library().pyro_probe_dmma_peak(int(device), float(millis), C.byref(out)))
    return float(out.value)


def probe_indexed_rmw(device=0, warps_per_sm=8, mode=1):
    """SM cycles per iteration of sixteen indexed read-modify-writes per thread (mode 0 shared memory, 1 tensor memory,
    2 tensor-memory loads only)."""
    out = C.c_double(0.0)
    _check(load_library().pyro_probe_indexed_rmw(int(device), int(warps_per_sm), int(mode), C.byref(out)))
    return float(out.value)


class TransportDesc(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("mol_weight", C.c_void_p), ("visc", C.c_void_p), ("cond", C.c_void_p),
                ("diff", C.c_void_p)]


def load_library():
    """Loads libpyro.so (building it with nvcc first if the sources are newer)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        from . import build
        build.build_libpyro()
    lib = C.CDLL(LIB_PATH)
    vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
    lib.pyro_mech_create.argtypes = [C.POINTER(MechDesc), C.c_int, C.POINTER(vp)]
    lib.pyro_mech_destroy.argtypes = [vp]
    lib.pyro_mech_set_newton.argtypes = [vp, dbl, C.c_int]
    lib.pyro_get_temperature.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp, vp]
    lib.pyro_get_temperature_from_enthalpy.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp]
    lib.pyro_get_density.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
    lib.pyro_get_pressure.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
    lib.pyro_get_net_production_rates.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp]
    lib.pyro_get_jacobian.argtypes = [vp, i64, i64, vp, vp, vp, C.c_int, vp, vp, vp]
    lib.pyro_reactor_rk4.argtypes = [vp, i64, i64, vp, vp, vp, vp, dbl, C.c_int32, vp, vp, vp]
    lib.pyro_reactor_rk4_static.argtypes = [vp, i64, i64, vp, vp, vp, vp, dbl, C.c_int32, vp, vp]
    lib.pyro_reactor_cn.argtypes = [vp, i64, i64, vp, vp, vp, vp, dbl, C.c_int32, C.c_int32, dbl, vp, vp, vp]
    lib.pyro_reactor_cn_work_doubles.argtypes = [vp, i64, C.POINTER(i64)]
    lib.pyro_source_terms.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.pyro_source_terms_host.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp, C.POINTER(i64)]
    lib.pyro_transport_create.argtypes = [C.POINTER(TransportDesc), C.c_int, C.POINTER(vp)]
    lib.pyro_transport_destroy.argtypes = [vp]
    lib.pyro_get_transport.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, vp]
    lib.pyro_mech_info.argtypes = [vp, C.POINTER(i64), C.c_int]
    lib.pyro_probe_fp64_peak.argtypes = [C.c_int, dbl, C.POINTER(dbl)]
    lib.pyro_probe_dmma_peak.argtypes = [C.c_int, dbl, C.POINTER(dbl)]
    lib.pyro_probe_indexed_rmw.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(dbl)]
    lib.pyro_status_string.argtypes = [C.c_int]
    lib.pyro_status_string.restype = C.c_char_p
    lib.pyro_last_error_string.restype = C.c_char_p
    _lib = lib
    return lib


def _check(status):
    if status != PYRO_OK:
        raise PyroError(status, load_library().pyro_last_error_string().decode())


def make_desc(mech):
    """pyro_mech_desc from an object with the attributes of `inputs.Mechanism`.
    Returns (desc, keepalive)."""
    keep = []

    def arr(x, dt):
        if x is None:
            return None
        a = np.ascontiguousarray(np.asarray(x), dtype=dt)
        keep.append(a)
        return a.ctypes.data

    d = MechDesc()
    d.n_species = int(mech.n_species)
    d.n_reactions = int(mech.n_reactions)
    ec = getattr(mech, "elem_comp", None)
    d.n_elements = 0 if ec is None else int(np.asarray(ec).shape[1])
    d.elem_comp = arr(ec, np.int32) if d.n_elements else None
    for name in ("mol_weight", "nasa_lo", "nasa_hi", "t_mid", "A", "b", "theta", "eff_default", "eff_value",
                 "A0", "b0", "theta0", "troe"):
        setattr(d, name, arr(getattr(mech, name), np.float64))
    for name in ("reac_ptr", "reac_species", "reac_coeff", "prod_ptr", "prod_species", "prod_coeff",
                 "eff_ptr", "eff_species"):
        setattr(d, name, arr(getattr(mech, name), np.int32))
    d.type = arr(mech.rtype, np.uint8)
    d.reversible = arr(mech.reversible, np.uint8)
    return d, keep


_INFO_KEYS = ("n_species", "n_reactions", "n_plain", "n_extended", "table_bytes", "tables_in_shared",
              "block_threads", "smem_bytes", "blocks_per_sm", "registers", "local_bytes", "sm_count",
              "points_per_thread", "tmem_columns", "b_in_tmem")


def _ptr(t):
    return None if t is None else t.data_ptr()


def _stream(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


class Mechanism:
    """Owns a pyro_mech handle.  Field arguments are torch CUDA float64 tensors
    (Y, omega of shape [n_species, ld] with points contiguous)."""

    def __init__(self, mech, device=0):
        lib = load_library()
        desc, keep = make_desc(mech)
        h = C.c_void_p()
        _check(lib.pyro_mech_create(C.byref(desc), int(device), C.byref(h)))
        self._h = h
        self._lib = lib
        self.device = int(device)
        self.n_species = int(mech.n_species)
        self.n_reactions = int(mech.n_reactions)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.pyro_mech_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self):
        out = (C.c_int64 * 15)()
        n = self._lib.pyro_mech_info(self._h, out, 15)
        if n < 0:
            _check(-n)
        return dict(zip(_INFO_KEYS, [int(v) for v in out[:n]]))

    def set_newton(self, abs_tol_K=1e-6, max_iter=10):
        _check(self._lib.pyro_mech_set_newton(self._h, float(abs_tol_K), int(max_iter)))

    def get_temperature(self, e, Y, T_guess, rho=None, out=None, n_not_converged=None, stream=None):
        """pyro_get_temperature: T from (e, Y, T_guess); returns T."""
        import torch
        n = e.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        if out is None:
            out = torch.empty_like(e)
        _check(self._lib.pyro_get_temperature(self._h, n, ld, _ptr(rho), _ptr(e), _ptr(Y), _ptr(T_guess),
                                              _ptr(out), _ptr(n_not_converged), _stream(stream)))
        return out

    def get_temperature_from_enthalpy(self, h, Y, T_guess, out=None, n_not_converged=None, stream=None):
        """pyro_get_temperature_from_enthalpy: T from (h, Y, T_guess); returns T."""
        import torch
        n = h.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        if out is None:
            out = torch.empty_like(h)
        _check(self._lib.pyro_get_temperature_from_enthalpy(self._h, n, ld, _ptr(h), _ptr(Y), _ptr(T_guess),
                                                            _ptr(out), _ptr(n_not_converged), _stream(stream)))
        return out

    def _eos(self, fn, a, T, Y, out, stream):
        import torch
        n = a.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        if out is None:
            out = torch.empty_like(a)
        _check(fn(self._h, n, ld, _ptr(a), _ptr(T), _ptr(Y), _ptr(out), _stream(stream)))
        return out

    def get_density(self, p, T, Y, out=None, stream=None):
        """pyro_get_density: rho from (p, T, Y); returns rho."""
        return self._eos(self._lib.pyro_get_density, p, T, Y, out, stream)

    def get_pressure(self, rho, T, Y, out=None, stream=None):
        """pyro_get_pressure: p from (rho, T, Y); returns p."""
        return self._eos(self._lib.pyro_get_pressure, rho, T, Y, out, stream)

    def get_net_production_rates(self, rho, T, Y, out=None, stream=None):
        """pyro_get_net_production_rates: omega from (rho, T, Y); returns omega."""
        import torch
        n = rho.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        if out is None:
            out = torch.empty_like(Y)
        assert out.stride(0) == ld or n == 0
        _check(self._lib.pyro_get_net_production_rates(self._h, n, ld, _ptr(rho), _ptr(T), _ptr(Y), _ptr(out),
                                                       _stream(stream)))
        return out

    def source_terms(self, rho, e, Y, T_guess, T_out=None, omega_out=None, n_not_converged=None, stream=None):
        """pyro_source_terms: (rho, e, Y, T_guess) -> (T, omega) in one launch; returns (T, omega)."""
        import torch
        n = rho.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        if T_out is None:
            T_out = torch.empty_like(e)
        if omega_out is None:
            omega_out = torch.empty_like(Y)
        assert omega_out.stride(0) == ld or n == 0
        _check(self._lib.pyro_source_terms(self._h, n, ld, _ptr(rho), _ptr(e), _ptr(Y), _ptr(T_guess), _ptr(T_out),
                                           _ptr(omega_out), _ptr(n_not_converged), _stream(stream)))
        return T_out, omega_out

    def reactor_rk4(self, rho, e, Y, T, dt, n_steps, work=None, n_not_converged=None, stream=None):
        """pyro_reactor_rk4: marches Y (in place) by n_steps RK4 steps of size dt; T: guess in, final temperature out."""
        import torch
        n = rho.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        if work is None:
            work = torch.empty_like(Y)
        assert work.stride(0) == ld or n == 0
        _check(self._lib.pyro_reactor_rk4(self._h, n, ld, _ptr(rho), _ptr(e), _ptr(Y), _ptr(T), float(dt), int(n_steps),
                                          _ptr(work), _ptr(n_not_converged), _stream(stream)))
        return Y, T

    def reactor_rk4_static(self, rho, e, Y, T, dt, n_steps, n_not_converged=None, stream=None):
        """pyro_reactor_rk4_static: reactor_rk4 for callers that may not allocate device memory.  Nothing is allocated
        here either (no torch tensor is created): the scratch is the fixed array inside libpyro.so, which limits
        n_species * ceil32(n) to RK4_STATIC_MAX_DOUBLES and must not be used by two overlapping calls on one device."""
        n = rho.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        _check(self._lib.pyro_reactor_rk4_static(self._h, n, ld, _ptr(rho), _ptr(e), _ptr(Y), _ptr(T), float(dt),
                                                 int(n_steps), _ptr(n_not_converged), _stream(stream)))
        return Y, T

    def reactor_cn(self, rho, e, Y, T, dt, n_steps, newton_iters=4, update_tol=1e-10, work=None, n_not_converged=None,
                   stream=None):
        """pyro_reactor_cn: marches Y (in place) by n_steps Crank-Nicolson steps; T: guess in, temperature of the last
        Newton iterate out."""
        import torch
        n = rho.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        need = C.c_int64(0)
        _check(self._lib.pyro_reactor_cn_work_doubles(self._h, ld, C.byref(need)))
        need = int(need.value)
        if work is None:
            work = torch.empty(need, dtype=torch.float64, device=Y.device)
        assert work.numel() >= need
        _check(self._lib.pyro_reactor_cn(self._h, n, ld, _ptr(rho), _ptr(e), _ptr(Y), _ptr(T), float(dt), int(n_steps),
                                         int(newton_iters), float(update_tol), _ptr(work), _ptr(n_not_converged),
                                         _stream(stream)))
        return Y, T

    def get_jacobian(self, rho, T, Y, mode=0, out=None, dSdT=None, want_dSdT=True, stream=None):
        """pyro_get_jacobian: J[i, k, p] = dS_i/dY_k (mode 0: fixed (rho, T); mode 1: fixed (rho, e)) and
        dSdT[i, p]; returns (J, dSdT).  J has shape [n_species, n_species, ld]."""
        import torch
        n = rho.shape[0]
        ns = Y.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        if out is None:
            out = torch.empty((ns, ns, ld), dtype=torch.float64, device=Y.device)
        assert out.is_contiguous() and out.shape[2] == ld
        if dSdT is None and want_dSdT:
            dSdT = torch.empty((ns, ld), dtype=torch.float64, device=Y.device)
        _check(self._lib.pyro_get_jacobian(self._h, n, ld, _ptr(rho), _ptr(T), _ptr(Y), int(mode), _ptr(out),
                                           _ptr(dSdT), _stream(stream)))
        return out[:, :, :n], (None if dSdT is None else dSdT[:, :n])

    def source_terms_host(self, rho, e, Y, T_guess, T_out, omega_out):
        """pyro_source_terms_host on HOST buffers (numpy arrays or CPU torch tensors, float64,
        preferably pinned).  Returns the Newton non-convergence count."""
        def hp(x):
            return x.ctypes.data if isinstance(x, np.ndarray) else x.data_ptr()

        def ld_of(x, n):
            if isinstance(x, np.ndarray):
                return x.strides[0] // 8 if x.ndim == 2 and n > 0 else n
            return x.stride(0) if x.dim() == 2 and n > 0 else n
        n = rho.shape[0]
        ld = ld_of(Y, n)
        assert ld_of(omega_out, n) == ld
        bad = C.c_int64(0)
        _check(self._lib.pyro_source_terms_host(self._h, n, ld, hp(rho), hp(e), hp(Y), hp(T_guess), hp(T_out),
                                                hp(omega_out), C.byref(bad)))
        return int(bad.value)


def probe_fp64_peak(device=0, millis=200.0):
    """Measured DFMA peak of the device in TFLOP/s (2 flops per FMA)."""
    out = C.c_double(0.0)
    _check(load_library().pyro_probe_fp64_peak(int(device), float(millis), C.byref(out)))
    return float(out.value)


class Transport:
    """Owns a pyro_transport handle (mixture-averaged transport fits of one species set)."""

    def __init__(self, tr, device=0):
        self._lib = load_library()
        keep = [np.ascontiguousarray(np.asarray(getattr(tr, k)), dtype=np.float64)
                for k in ("mol_weight", "visc", "cond", "diff")]
        self.n_species = int(keep[0].shape[0])
        desc = TransportDesc(self.n_species, *[a.ctypes.data for a in keep])
        h = C.c_void_p()
        _check(self._lib.pyro_transport_create(C.byref(desc), int(device), C.byref(h)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._lib.pyro_transport_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def get_transport(self, T, Y, mu=None, kappa=None, D=None, stream=None):
        """pyro_get_transport: (mu [n], kappa [n], D_km [n_species, ld]) from (T, Y)."""
        import torch
        n = T.shape[0]
        ld = Y.stride(0) if Y.dim() == 2 and n > 0 else n
        mu = torch.empty_like(T) if mu is None else mu
        kappa = torch.empty_like(T) if kappa is None else kappa
        D = torch.empty_like(Y) if D is None else D
        assert D.stride(0) == ld or n == 0
        _check(self._lib.pyro_get_transport(self._h, n, ld, _ptr(T), _ptr(Y), _ptr(mu), _ptr(kappa), _ptr(D), _stream(stream)))
        return mu, kappa, D
