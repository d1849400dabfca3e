"""Thin ctypes binding of librtcc (include/rtcc.h): argument marshalling only -- every step of the hot path
runs in the CUDA kernels behind the C ABI.  There is no CPU fallback: if the library is missing or a call
fails, an exception is raised.

Arrays may be numpy arrays (the context is then created with RTCC_HOST_PTRS and the library copies) or
torch CUDA tensors (device pointers, no copies).  Complex arrays are complex128.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "librtcc.so")
_lib = None

RTCC_HOST_PTRS = 1
SYMBOLS = [
    "rtcc_create", "rtcc_destroy", "rtcc_sizes", "rtcc_residual", "rtcc_residual_energy", "rtcc_set_amplitudes",
    "rtcc_get_amplitudes", "rtcc_set_solver", "rtcc_step", "rtcc_cumulant", "rtcc_last_micro_iterations", "rtcc_time",
    "rtcc_counters", "rtcc_reset_counters", "rtcc_set_timing", "rtcc_ladder_timing", "rtcc_fp64_peak",
    "rtcc_debug_buffer", "rtcc_debug_gemm", "rtcc_last_cuda_error", "rtcc_strerror", "rtcc_build_fock", "rtcc_spectral_function",
    "rtcc_set_default_option", "rtcc_ladder_plan", "rtcc_ladder_occupancy", "rtcc_save", "rtcc_load", "rtcc_problem_sizes",
    "rtcc_get_state", "rtcc_set_state",
]


class RtccError(RuntimeError):
    def __init__(self, code, what, cuda=0):
        super().__init__(f"{what}: error {code} ({strerror(code)})" + (f", cudaError {cuda}" if cuda else ""))
        self.code = code


def load():
    """dlopen librtcc.so (built by paper_2301_04249_b200.build / __graft_entry__.build); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise RuntimeError(f"{_LIBPATH} not found: run `python -m paper_2301_04249_b200.build` (no CPU fallback exists)")
        lib = ctypes.CDLL(_LIBPATH)
        vp, i, d, ll = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_longlong
        P = ctypes.POINTER
        lib.rtcc_create.argtypes = [P(vp), i, i, i, i, i, vp, vp, ctypes.c_uint, vp]
        lib.rtcc_destroy.argtypes = [vp]; lib.rtcc_destroy.restype = None
        lib.rtcc_sizes.argtypes = [vp, P(ll), P(ll), P(ll)]
        lib.rtcc_residual.argtypes = [vp, vp, vp, vp, vp]
        lib.rtcc_residual_energy.argtypes = [vp, P(d)]
        lib.rtcc_set_amplitudes.argtypes = [vp, vp, vp, d, P(d)]
        lib.rtcc_get_amplitudes.argtypes = [vp, vp, vp]
        lib.rtcc_set_solver.argtypes = [vp, i, d, i, i]
        lib.rtcc_step.argtypes = [vp, d]
        lib.rtcc_cumulant.argtypes = [vp, P(d)]
        lib.rtcc_last_micro_iterations.argtypes = [vp]
        lib.rtcc_time.argtypes = [vp]; lib.rtcc_time.restype = d
        lib.rtcc_counters.argtypes = [vp, P(ll), P(d)]
        lib.rtcc_reset_counters.argtypes = [vp]
        lib.rtcc_set_timing.argtypes = [vp, i]
        lib.rtcc_ladder_timing.argtypes = [vp, P(d), P(d), P(d)]
        lib.rtcc_fp64_peak.argtypes = [P(d)]
        lib.rtcc_debug_buffer.argtypes = [vp, ctypes.c_char_p, vp, ll]; lib.rtcc_debug_buffer.restype = ll
        lib.rtcc_debug_gemm.argtypes = [i, i, i, vp, vp, vp, d, d, i]
        lib.rtcc_build_fock.argtypes = [i, i, vp, vp, i, i, vp, ctypes.c_uint, vp]
        lib.rtcc_spectral_function.argtypes = [i, d, vp, d, d, d, i, vp, vp, vp]
        lib.rtcc_set_default_option.argtypes = [ctypes.c_char_p, i]
        lib.rtcc_ladder_plan.argtypes = [vp, i, P(i)]
        lib.rtcc_ladder_occupancy.argtypes = [vp, P(i)]
        lib.rtcc_problem_sizes.argtypes = [i, i, i, i, i, P(ll)]
        lib.rtcc_save.argtypes = [vp, ctypes.c_char_p]
        lib.rtcc_load.argtypes = [vp, ctypes.c_char_p]
        lib.rtcc_get_state.argtypes = [vp, vp, vp, vp, vp, P(d)]
        lib.rtcc_set_state.argtypes = [vp, vp, vp, vp, vp, P(d)]
        lib.rtcc_last_cuda_error.argtypes = [vp]
        lib.rtcc_strerror.argtypes = [i]; lib.rtcc_strerror.restype = ctypes.c_char_p
        _lib = lib
    return _lib


def strerror(code: int) -> str:
    return load().rtcc_strerror(int(code)).decode()


def problem_sizes(oa, ob, va, vb, n_chol):
    """Size accounting without a context (include/rtcc.h: rtcc_problem_sizes); needs no GPU."""
    buf = (ctypes.c_longlong * 6)()
    rc = load().rtcc_problem_sizes(oa, ob, va, vb, n_chol, buf)
    if rc:
        raise RtccError(rc, "rtcc_problem_sizes")
    keys = ("n_t1", "n_t2", "t2_unpacked_elements", "cholesky_doubles", "bytes_standard", "bytes_lean")
    return dict(zip(keys, list(buf)))


def set_default_option(name: str, value: int = 0):
    """Process-wide tuning default for contexts created afterwards (include/rtcc.h: rtcc_set_default_option)."""
    rc = load().rtcc_set_default_option(name.encode(), int(value))
    if rc:
        raise RtccError(rc, f"rtcc_set_default_option({name})")


def _is_torch(x):
    return type(x).__module__.startswith("torch")


def _ptr(x):
    if _is_torch(x):
        return ctypes.c_void_p(x.data_ptr())
    return ctypes.c_void_p(x.ctypes.data)


def fp64_peak() -> float:
    """Measured FP64 DMMA peak of the current device in TFLOP/s."""
    v = ctypes.c_double(0.0)
    rc = load().rtcc_fp64_peak(ctypes.byref(v))
    if rc:
        raise RtccError(rc, "rtcc_fp64_peak")
    return v.value


def debug_gemm(A: np.ndarray, B: np.ndarray, C: np.ndarray | None = None, alpha=1.0, beta=0.0):
    """Test hook: alpha*A@B + beta*C through the tensor-core contraction kernel (real or complex128)."""
    cplx = np.iscomplexobj(A) or np.iscomplexobj(B)
    M, K = A.shape
    N = B.shape[1]
    if cplx:
        pa = np.ascontiguousarray(np.stack([A.real, A.imag]).astype(np.float64))
        pb = np.ascontiguousarray(np.stack([B.real, B.imag]).astype(np.float64))
        pc = np.zeros((2, M, N)) if C is None else np.ascontiguousarray(np.stack([C.real, C.imag]).astype(np.float64))
    else:
        pa = np.ascontiguousarray(A, dtype=np.float64)
        pb = np.ascontiguousarray(B, dtype=np.float64)
        pc = np.zeros((M, N)) if C is None else np.array(C, dtype=np.float64)
    rc = load().rtcc_debug_gemm(M, N, K, _ptr(pa), _ptr(pb), _ptr(pc), float(alpha), float(beta), int(cplx))
    if rc:
        raise RtccError(rc, "rtcc_debug_gemm")
    return pc[0] + 1j * pc[1] if cplx else pc


def build_fock(L, eps, core_spin: int, core_index: int):
    """(N-1) Fock matrix f_pq = eps_p delta_pq - v_pc^qc from L[2,K,n,n] and eps[2,n]; numpy in, numpy out,
    or torch CUDA tensors in, torch out."""
    dev = _is_torch(L)
    if dev:
        import torch
        K, n = L.shape[1], L.shape[2]
        fock = torch.empty((2, n, n), dtype=torch.float64, device=L.device)
        eps = eps.contiguous()
    else:
        L = np.ascontiguousarray(L, dtype=np.float64); eps = np.ascontiguousarray(eps, dtype=np.float64)
        K, n = L.shape[1], L.shape[2]
        fock = np.empty((2, n, n))
    rc = load().rtcc_build_fock(n, K, _ptr(L), _ptr(eps), int(core_spin), int(core_index), _ptr(fock), 0 if dev else RTCC_HOST_PTRS, None)
    if rc:
        raise RtccError(rc, "rtcc_build_fock")
    return fock


def spectral_function(C, dt, eps_c, e_corr, eta, omega):
    """G(tau_k) (complex array) and A(omega) from the recorded cumulant C(k dt) (Eqs. 3-4); host arrays."""
    C = np.ascontiguousarray(C, dtype=np.complex128)
    omega = np.ascontiguousarray(omega, dtype=np.float64)
    G = np.empty(C.size, dtype=np.complex128)
    A = np.empty(omega.size)
    rc = load().rtcc_spectral_function(C.size, float(dt), _ptr(C), float(eps_c), float(e_corr), float(eta), omega.size, _ptr(omega), _ptr(G), _ptr(A))
    if rc:
        raise RtccError(rc, "rtcc_spectral_function")
    return G, A


class Rtcc:
    """One (N-1)-electron RT-EOM-CCSD problem on the current CUDA device (see include/rtcc.h)."""

    def __init__(self, oa, ob, va, vb, n_chol, L, fock, stream=None):
        lib = load()
        self._lib = lib
        self.device_mode = _is_torch(L)
        if self.device_mode:
            import torch
            assert L.is_cuda and fock.is_cuda and L.dtype == torch.float64 and L.is_contiguous() and fock.is_contiguous()
        else:
            L = np.ascontiguousarray(L, dtype=np.float64)
            fock = np.ascontiguousarray(fock, dtype=np.float64)
        self.dims = (oa, ob, va, vb, n_chol)
        h = ctypes.c_void_p()
        flags = 0 if self.device_mode else RTCC_HOST_PTRS
        rc = lib.rtcc_create(ctypes.byref(h), oa, ob, va, vb, n_chol, _ptr(L), _ptr(fock), flags,
                             ctypes.c_void_p(stream or 0))
        if rc:
            raise RtccError(rc, "rtcc_create", lib.rtcc_last_cuda_error(None))
        self._h = h
        a, b, w = ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_longlong()
        lib.rtcc_sizes(h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(w))
        self.n_t1, self.n_t2, self.workspace_bytes = a.value, b.value, w.value

    def close(self):
        if getattr(self, "_h", None):
            self._lib.rtcc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc, what):
        if rc:
            raise RtccError(rc, what, self._lib.rtcc_last_cuda_error(self._h))

    def _new(self, n):
        if self.device_mode:
            import torch
            return torch.empty(n, dtype=torch.complex128, device="cuda")
        return np.empty(n, dtype=np.complex128)

    def _chk(self, x, n):
        if self.device_mode:
            assert _is_torch(x) and x.is_cuda and x.is_contiguous() and x.numel() == n
            return x
        x = np.ascontiguousarray(x, dtype=np.complex128)
        assert x.size == n
        return x

    def residual(self, t1, t2, r1=None, r2=None):
        """R1, R2 (packed) at the given packed amplitudes; E via residual_energy()."""
        t1 = self._chk(t1, self.n_t1); t2 = self._chk(t2, self.n_t2)
        r1 = self._new(self.n_t1) if r1 is None else r1
        r2 = self._new(self.n_t2) if r2 is None else r2
        self._ck(self._lib.rtcc_residual(self._h, _ptr(t1), _ptr(t2), _ptr(r1), _ptr(r2)), "rtcc_residual")
        return r1, r2

    def residual_energy(self) -> complex:
        out = (ctypes.c_double * 2)()
        self._ck(self._lib.rtcc_residual_energy(self._h, out), "rtcc_residual_energy")
        return complex(out[0], out[1])

    def set_amplitudes(self, t1, t2, time=0.0, C=0j):
        t1 = self._chk(t1, self.n_t1); t2 = self._chk(t2, self.n_t2)
        c = (ctypes.c_double * 2)(complex(C).real, complex(C).imag)
        self._ck(self._lib.rtcc_set_amplitudes(self._h, _ptr(t1), _ptr(t2), float(time), c), "rtcc_set_amplitudes")

    def get_amplitudes(self):
        t1, t2 = self._new(self.n_t1), self._new(self.n_t2)
        self._ck(self._lib.rtcc_get_amplitudes(self._h, _ptr(t1), _ptr(t2)), "rtcc_get_amplitudes")
        return t1, t2

    def save(self, path: str):
        """Checkpoint T(tau), R(T(tau)), tau, C, E and the solver settings."""
        self._ck(self._lib.rtcc_save(self._h, os.fsencode(path)), "rtcc_save")

    def load(self, path: str):
        self._ck(self._lib.rtcc_load(self._h, os.fsencode(path)), "rtcc_load")

    def get_state(self, out=None):
        """(t1, t2, r1, r2, tau, C, E): the propagation state T(tau), R(T(tau)) and its scalars, through memory.
        `out` = (t1, t2, r1, r2) arrays to fill instead of new ones."""
        t1, t2, r1, r2 = out if out is not None else (self._new(self.n_t1), self._new(self.n_t2), self._new(self.n_t1), self._new(self.n_t2))
        sc = (ctypes.c_double * 5)()
        self._ck(self._lib.rtcc_get_state(self._h, _ptr(t1), _ptr(t2), _ptr(r1), _ptr(r2), sc), "rtcc_get_state")
        return t1, t2, r1, r2, sc[0], complex(sc[1], sc[2]), complex(sc[3], sc[4])

    def set_state(self, t1, t2, r1, r2, time, C, E):
        """Install a state taken with get_state (no residual evaluation)."""
        t1 = self._chk(t1, self.n_t1); t2 = self._chk(t2, self.n_t2); r1 = self._chk(r1, self.n_t1); r2 = self._chk(r2, self.n_t2)
        sc = (ctypes.c_double * 5)(float(time), complex(C).real, complex(C).imag, complex(E).real, complex(E).imag)
        self._ck(self._lib.rtcc_set_state(self._h, _ptr(t1), _ptr(t2), _ptr(r1), _ptr(r2), sc), "rtcc_set_state")

    def set_solver(self, mode=0, tol=1e-4, max_micro=200, fixed_micro=0):
        self._ck(self._lib.rtcc_set_solver(self._h, mode, tol, max_micro, fixed_micro), "rtcc_set_solver")

    def step(self, dt: float) -> int:
        self._ck(self._lib.rtcc_step(self._h, float(dt)), "rtcc_step")
        return self._lib.rtcc_last_micro_iterations(self._h)

    def cumulant(self):
        """(C, E) at the current time."""
        out = (ctypes.c_double * 4)()
        self._ck(self._lib.rtcc_cumulant(self._h, out), "rtcc_cumulant")
        return complex(out[0], out[1]), complex(out[2], out[3])

    @property
    def time(self) -> float:
        return self._lib.rtcc_time(self._h)

    def counters(self):
        a, f = ctypes.c_longlong(), ctypes.c_double()
        self._ck(self._lib.rtcc_counters(self._h, ctypes.byref(a), ctypes.byref(f)), "rtcc_counters")
        return a.value, f.value

    def reset_counters(self):
        self._ck(self._lib.rtcc_reset_counters(self._h), "rtcc_reset_counters")

    def set_timing(self, on: bool):
        self._ck(self._lib.rtcc_set_timing(self._h, int(on)), "rtcc_set_timing")

    def ladder_timing(self):
        """(ms, executed flops, model flops) of the pp-ladder kernels of the last timed residual."""
        a, b, c = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        self._ck(self._lib.rtcc_ladder_timing(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)), "rtcc_ladder_timing")
        return a.value, b.value, c.value

    def ladder_plan(self):
        """Per spin case with a non-empty block: dict of the pp-ladder launch plan (include/rtcc.h: rtcc_ladder_plan)."""
        keys = ("columns", "tile", "col_tiles", "cluster", "groups", "ef_slices", "row_tiles", "active_sms")
        out = []
        for k in range(3):
            buf = (ctypes.c_int * 8)()
            if self._lib.rtcc_ladder_plan(self._h, k, buf):
                break
            out.append(dict(zip(keys, list(buf))))
        return out

    def ladder_occupancy(self):
        buf = (ctypes.c_int * 17)()
        self._ck(self._lib.rtcc_ladder_occupancy(self._h, buf), "rtcc_ladder_occupancy")
        return list(buf)

    def debug_buffer(self, name: str) -> np.ndarray:
        n = self._lib.rtcc_debug_buffer(self._h, name.encode(), None, 0)
        if n < 0:
            raise RtccError(int(n), f"rtcc_debug_buffer({name})")
        out = np.empty(n, dtype=np.float64)
        self._lib.rtcc_debug_buffer(self._h, name.encode(), _ptr(out), n)
        return out
