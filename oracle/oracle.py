"""CPU oracle for the RT-EOM-CCSD hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this module.  It shares no code with, and never
imports, the CUDA path (``paper_2301_04249_b200``).

Layers:
  O-1  per-spin Cholesky vectors / Fock matrix -> spin-orbital <pq||rs>, f
  O-2  residuals R1, R2 and E (PAPER.md:76-79 Eqs. 7-8; :58-63 Eqs. 5-6) -- ``rtcc_oracle.c``
  O-3  first-order Adams-Moulton step with fixed-point micro-iterations (PAPER.md:93 Eq. 9, :97, :103)
  O-4  cumulant C(t) by the trapezoid rule (PAPER.md:58 Eq. 5; :89)

Packed amplitude layout (the boundary's, include/rtcc.h): t1 = [alpha (o_a x v_a, a fastest) | beta];
t2 = [aa packed | bb packed | ab full]; same-spin element (i<j, a<b) at pair(i,j)*P(v)+pair(a,b),
pair(x,y) = y(y-1)/2 + x; ab element (i,J,a,B) at ((i*o_b+J)*v_a+a)*v_b+B.

Parity status: every function here is pinned by tests/test_oracle_pins.py (P-0..P-9 of SURVEY.md 8(c)).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rtcc_oracle.c")
_LIB = os.path.join(_HERE, "librtcc_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile rtcc_oracle.c with gcc (-O2, OpenMP).  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        i = ctypes.c_int
        lib.orc_num_threads.restype = i
        lib.orc_build_so.argtypes = [i, i, i, i, i, dp, dp, dp, dp]
        lib.orc_build_so.restype = None
        lib.orc_eri_chem.argtypes = [i, i, dp, i, i, i, i]
        lib.orc_eri_chem.restype = ctypes.c_double
        lib.orc_eri_antisym.argtypes = [i, i, dp, dp]
        lib.orc_eri_antisym.restype = None
        lib.orc_residual.argtypes = [i, i, dp, dp, dp, dp, dp, dp, dp]
        lib.orc_residual.restype = i
        _lib = lib
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def num_threads() -> int:
    return int(_load().orc_num_threads())


def npair(n: int) -> int:
    return n * (n - 1) // 2


def pair(x, y):
    """pair(x,y) = y(y-1)/2 + x for x < y."""
    return y * (y - 1) // 2 + x


@dataclass
class Dims:
    oa: int
    ob: int
    va: int
    vb: int
    K: int

    @property
    def n(self):
        return self.oa + self.va

    @property
    def no(self):
        return self.oa + self.ob

    @property
    def nv(self):
        return self.va + self.vb

    @property
    def n_t1(self):
        return self.oa * self.va + self.ob * self.vb

    @property
    def n_t2(self):
        return (npair(self.oa) * npair(self.va) + npair(self.ob) * npair(self.vb)
                + self.oa * self.ob * self.va * self.vb)


def t2_bytes_unpacked(oa, ob, va, vb) -> int:
    """Bytes of ONE T2 in the paper's storage: three unpacked spin blocks, complex128
    ("only three spin cases"; Table 2 PAPER.md:143-150 is reproduced by this count)."""
    return 16 * (oa * oa * va * va + ob * ob * vb * vb + oa * ob * va * vb)


# ----------------------------------------------------------------------------- index maps
def unpack(d: Dims, t1p: np.ndarray, t2p: np.ndarray):
    """Packed blocks -> spin-orbital t1[i,a], t2[i,j,a,b].
    Spin-orbital order [alpha occ | beta occ | alpha virt | beta virt]; t2 filled by antisymmetry;
    spin-forbidden elements are exactly zero."""
    oa, ob, va, vb = d.oa, d.ob, d.va, d.vb
    no, nv = d.no, d.nv
    t1 = np.zeros((no, nv), dtype=np.complex128)
    t2 = np.zeros((no, no, nv, nv), dtype=np.complex128)
    t1[:oa, :va] = t1p[: oa * va].reshape(oa, va)
    t1[oa:, va:] = t1p[oa * va:].reshape(ob, vb)
    off = 0
    for (o, v, io, iv) in ((oa, va, 0, 0), (ob, vb, oa, va)):
        pv = npair(v)
        for j in range(o):
            for i in range(j):
                for b in range(v):
                    for a in range(b):
                        x = t2p[off + pair(i, j) * pv + pair(a, b)]
                        I, J, A, B = io + i, io + j, iv + a, iv + b
                        t2[I, J, A, B] = x
                        t2[J, I, A, B] = -x
                        t2[I, J, B, A] = -x
                        t2[J, I, B, A] = x
        off += npair(o) * pv
    ab = t2p[off:].reshape(oa, ob, va, vb)
    for i in range(oa):
        for J in range(ob):
            blk = ab[i, J]                       # [a, B]
            t2[i, oa + J, :va, va:] = blk
            t2[oa + J, i, :va, va:] = -blk
            t2[i, oa + J, va:, :va] = -blk.T
            t2[oa + J, i, va:, :va] = blk.T
    return t1, t2


def pack(d: Dims, r1: np.ndarray, r2: np.ndarray):
    """Spin-orbital r1[i,a], r2[i,j,a,b] -> packed blocks (inverse of unpack on the unique elements)."""
    oa, ob, va, vb = d.oa, d.ob, d.va, d.vb
    r1p = np.concatenate([r1[:oa, :va].reshape(-1), r1[oa:, va:].reshape(-1)])
    out = np.empty(d.n_t2, dtype=np.complex128)
    off = 0
    for (o, v, io, iv) in ((oa, va, 0, 0), (ob, vb, oa, va)):
        pv = npair(v)
        for j in range(o):
            for i in range(j):
                for b in range(v):
                    for a in range(b):
                        out[off + pair(i, j) * pv + pair(a, b)] = r2[io + i, io + j, iv + a, iv + b]
        off += npair(o) * pv
    out[off:] = r2[:oa, oa:, :va, va:].reshape(-1)
    return r1p, out


# ----------------------------------------------------------------------------- problem
class Problem:
    """Spin-orbital statement of one (N-1)-electron problem: f[N,N], <pq||rs>[N,N,N,N]."""

    def __init__(self, oa, ob, va, vb, K, L, fock):
        lib = _load()
        self.d = Dims(oa, ob, va, vb, K)
        n = oa + va
        if ob + vb != n:
            raise ValueError("o_alpha+v_alpha must equal o_beta+v_beta")
        L = np.ascontiguousarray(L, dtype=np.float64).reshape(2, K, n, n)
        fock = np.ascontiguousarray(fock, dtype=np.float64).reshape(2, n, n)
        N = 2 * n
        self.N = N
        self.Lso = np.zeros((K, N, N))
        self.f = np.zeros((N, N))
        lib.orc_build_so(oa, ob, va, vb, K, _dp(L), _dp(fock), _dp(self.Lso), _dp(self.f))
        self.g = np.empty((N, N, N, N))
        lib.orc_eri_antisym(N, K, _dp(self.Lso), _dp(self.g))

    def eri_chem(self, p, q, r, s) -> float:
        return float(_load().orc_eri_chem(self.N, self.d.K, _dp(self.Lso), p, q, r, s))

    def residual_so(self, t1, t2):
        """R1[i,a], R2[i,j,a,b], E from spin-orbital amplitudes (Eqs. 7-8, 5)."""
        d = self.d
        t1 = np.ascontiguousarray(t1, dtype=np.complex128)
        t2 = np.ascontiguousarray(t2, dtype=np.complex128)
        r1 = np.empty_like(t1)
        r2 = np.empty_like(t2)
        E = np.zeros(1, dtype=np.complex128)
        rc = _load().orc_residual(d.no, d.nv, _dp(self.f), _dp(self.g), _dp(t1), _dp(t2),
                                  _dp(r1), _dp(r2), _dp(E))
        if rc != 0:
            raise MemoryError("oracle scratch allocation failed")
        return r1, r2, complex(E[0])

    def residual(self, t1p, t2p):
        """Packed in, packed out: r1, r2, E."""
        t1, t2 = unpack(self.d, np.asarray(t1p), np.asarray(t2p))
        r1, r2, E = self.residual_so(t1, t2)
        r1p, r2p = pack(self.d, r1, r2)
        return r1p, r2p, E


class Propagator:
    """O-3 / O-4: dt/dtau = +i R(t) (Eq. 2), first-order Adams-Moulton (Eq. 9) solved by fixed-point
    iteration from the previous amplitudes, cumulant by the trapezoid rule (Eq. 5).

    mode 0: plain iteration  t(k+1) = B + (i dt/2) R(t(k)),            B = t + (i dt/2) R(t)
    mode 1: denominator-preconditioned iteration (same fixed point):
            t(k+1) = (B + (i dt/2)(R(t(k)) - D o t(k))) / (1 - i dt D/2),
            D_i^a = f_aa - f_ii, D_ij^ab = f_aa + f_bb - f_ii - f_jj  (R = D o t + rest for diagonal f).
    Convergence: max |t(k+1) - t(k)| over the unique (packed) elements < tol, or exactly fixed_micro
    iterations when fixed_micro > 0.
    """

    def __init__(self, prob: Problem, mode=0, tol=1e-4, max_micro=200, fixed_micro=0):
        self.p = prob
        d = prob.d
        self.t1 = np.zeros(d.n_t1, dtype=np.complex128)
        self.t2 = np.zeros(d.n_t2, dtype=np.complex128)
        self.time = 0.0
        self.C = 0.0 + 0.0j
        self.mode, self.tol, self.max_micro, self.fixed_micro = mode, tol, max_micro, fixed_micro
        self.r1, self.r2, self.E = prob.residual(self.t1, self.t2)
        self.last_micro = 0
        self.D1, self.D2 = self._denominators()

    def _denominators(self):
        d = self.p.d
        eps = np.diag(self.p.f)
        eo, ev = eps[: d.no], eps[d.no:]
        D1 = ev[None, :] - eo[:, None]
        D2 = (ev[None, None, :, None] + ev[None, None, None, :]
              - eo[:, None, None, None] - eo[None, :, None, None])
        return pack(d, D1.astype(np.complex128), D2.astype(np.complex128))

    def set_state(self, t1p, t2p, time=0.0, C=0.0):
        self.t1 = np.array(t1p, dtype=np.complex128)
        self.t2 = np.array(t2p, dtype=np.complex128)
        self.time, self.C = float(time), complex(C)
        self.r1, self.r2, self.E = self.p.residual(self.t1, self.t2)

    def step(self, dt: float) -> int:
        h = 0.5j * dt
        B1 = self.t1 + h * self.r1
        B2 = self.t2 + h * self.r2
        x1, x2 = self.t1, self.t2
        r1, r2 = self.r1, self.r2
        k = 0
        while True:
            if self.mode == 0:
                y1 = B1 + h * r1
                y2 = B2 + h * r2
            else:
                y1 = (B1 + h * (r1 - self.D1 * x1)) / (1.0 - h * self.D1)
                y2 = (B2 + h * (r2 - self.D2 * x2)) / (1.0 - h * self.D2)
            k += 1
            delta = max(np.max(np.abs(y1 - x1), initial=0.0), np.max(np.abs(y2 - x2), initial=0.0))
            x1, x2 = y1, y2
            if not np.isfinite(delta):
                raise FloatingPointError("non-finite amplitudes")
            r1, r2, E = self.p.residual(x1, x2)
            if self.fixed_micro > 0:
                if k >= self.fixed_micro:
                    break
            elif delta < self.tol:
                break
            elif k >= self.max_micro:
                raise RuntimeError("micro-iterations did not converge")
        self.C += h * (self.E + E)
        self.t1, self.t2, self.r1, self.r2, self.E = x1, x2, r1, r2, E
        self.time += dt
        self.last_micro = k
        return k


# ----------------------------------------------------------------------------- NEXT-3 / NEXT-2
def build_fock_n1(L, eps, core_spin: int, core_index: int):
    """(N-1)-electron Fock matrix f_pq = eps_p delta_pq - v_pc^qc, v_pq^rs = <pq||rs>, written
    out per spin: f^s_pq = eps^s_p delta_pq - (pq|cc) + delta(s, s_c) (pc|cq), (pq|rs) = sum_Q L_pq L_rs.
    L[2,K,n,n], eps[2,n] -> fock[2,n,n].  Pinned against -<pc||qc> of the spin-orbital tensor (test_fock_n1_*)."""
    L = np.asarray(L, dtype=np.float64)
    eps = np.asarray(eps, dtype=np.float64)
    n = L.shape[2]
    fock = np.zeros((2, n, n))
    Lcc = L[core_spin][:, core_index, core_index]
    for s in range(2):
        fock[s] = np.diag(eps[s]) - np.einsum("Qpq,Q->pq", L[s], Lcc)
        if s == core_spin:
            fock[s] += np.einsum("Qp,Qq->pq", L[s][:, :, core_index], L[s][:, core_index, :])
    return fock


def green_function(C, dt, eps_c, e_corr):
    """G_c^R(tau_k) = -i exp(-i (eps_c + E_N^corr) tau_k) exp(C(tau_k)), tau_k = k dt >= 0   (Eqs. 3-4)."""
    C = np.asarray(C, dtype=np.complex128)
    tau = dt * np.arange(C.size)
    return -1j * np.exp(-1j * (eps_c + e_corr) * tau) * np.exp(C)


def spectral_function(C, dt, eps_c, e_corr, eta, omega):
    """A_c(omega) = -(1/pi) Im G_c^R(omega), G(omega) = int_0^T G(tau) exp(i omega tau - eta tau) dtau by the
    trapezoid rule on the recorded grid (reading R14: eta is the caller's Lorentzian half width)."""
    G = green_function(C, dt, eps_c, e_corr)
    tau = dt * np.arange(G.size)
    w = np.full(G.size, dt)
    w[0] = w[-1] = 0.5 * dt
    out = np.empty(len(omega))
    for k, om in enumerate(np.asarray(omega, dtype=np.float64)):
        out[k] = -np.imag(np.sum(w * G * np.exp((1j * om - eta) * tau))) / np.pi
    return G, out
