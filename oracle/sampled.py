"""Sampled-element CPU oracle (tier B of SURVEY.md 8(c)) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

For problem sizes where the full 4-index tensor <pq||rs> of ``oracle.py`` does not fit (or takes minutes), this module
evaluates the SAME spin-orbital working equations (Eqs. 7-8) for individual output
elements R2[i,j,a,b] / R1[i,a], producing every integral it needs on demand as a direct sum over the Cholesky vectors,
<pq||rs> = sum_Q (L_pr L_qs - L_ps L_qr).  Plain numpy einsum, fp64, no blocking beyond "only the
index slices this element touches".  It shares no code with the CUDA path and does not import it.

Pinned by tests/test_oracle_pins.py::test_sampled_oracle_matches_full_oracle (agreement with the determinant-pinned
tier-A oracle to 1e-13 on complex amplitudes with a general Fock matrix).

``SampledOracleC`` (rtcc_sampled.c) evaluates the same elements with plain C loops straight off the packed blocks; it is
the one that fits BASELINE.json configs 3-5.  Pinned the same way (test_sampled_c_oracle_matches_full_oracle).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

from . import oracle as orc


class _PackedIndex:
    """Packed t2 / t1 position -> spin-orbital indices (shared by both sampled oracles; needs self.d)."""

    def so_of_packed_t2(self, k):
        d = self.d
        nss = [orc.npair(d.oa) * orc.npair(d.va), orc.npair(d.ob) * orc.npair(d.vb)]
        off_o, off_v = [0, d.oa], [0, d.va]
        for s, (o, v) in enumerate(((d.oa, d.va), (d.ob, d.vb))):
            if k < nss[s]:
                pij, pab = divmod(k, orc.npair(v))
                j = int((1 + np.sqrt(1 + 8 * pij)) // 2)
                while orc.pair(0, j) > pij:
                    j -= 1
                while orc.pair(0, j + 1) <= pij:
                    j += 1
                i = pij - orc.pair(0, j)
                b = int((1 + np.sqrt(1 + 8 * pab)) // 2)
                while orc.pair(0, b) > pab:
                    b -= 1
                while orc.pair(0, b + 1) <= pab:
                    b += 1
                a = pab - orc.pair(0, b)
                return off_o[s] + i, off_o[s] + j, off_v[s] + a, off_v[s] + b
            k -= nss[s]
        B = k % d.vb; k //= d.vb
        a = k % d.va; k //= d.va
        J = k % d.ob; i = k // d.ob
        return i, d.oa + J, a, d.va + B

    def so_of_packed_t1(self, k):
        d = self.d
        if k < d.oa * d.va:
            return divmod(k, d.va)
        i, a = divmod(k - d.oa * d.va, d.vb)
        return d.oa + i, d.va + a

    def packed_of_so_t2(self, i, j, a, b):
        """Inverse of so_of_packed_t2 for a canonical element (same spin: i<j, a<b; mixed: i alpha, j beta, a alpha, b beta)."""
        d = self.d
        naa = orc.npair(d.oa) * orc.npair(d.va)
        nbb = orc.npair(d.ob) * orc.npair(d.vb)
        if j < d.oa:
            return orc.pair(i, j) * orc.npair(d.va) + orc.pair(a, b)
        if i >= d.oa:
            return naa + orc.pair(i - d.oa, j - d.oa) * orc.npair(d.vb) + orc.pair(a - d.va, b - d.va)
        return naa + nbb + ((i * d.ob + (j - d.oa)) * d.va + a) * d.vb + (b - d.va)


class SampledOracle(_PackedIndex):
    def __init__(self, oa, ob, va, vb, K, L, fock, t1p, t2p):
        self.d = d = orc.Dims(oa, ob, va, vb, K)
        n = oa + va
        N = 2 * n
        self.no, self.nv, self.N = d.no, d.nv, N
        L = np.asarray(L, dtype=np.float64).reshape(2, K, n, n)
        fock = np.asarray(fock, dtype=np.float64).reshape(2, n, n)
        # spin-orbital order [alpha occ | beta occ | alpha virt | beta virt]   (O-1)
        idx = [np.concatenate([np.arange(0, oa), d.no + np.arange(0, va)]),
               np.concatenate([oa + np.arange(0, ob), d.no + va + np.arange(0, vb)])]
        self.Lso = np.zeros((K, N, N))
        self.f = np.zeros((N, N))
        for s in range(2):
            self.Lso[:, idx[s][:, None], idx[s][None, :]] = L[s]
            self.f[idx[s][:, None], idx[s][None, :]] = fock[s]
        self.t1, self.t2 = orc.unpack(d, np.asarray(t1p), np.asarray(t2p))
        no = self.no
        self.Loo, self.Lov = self.Lso[:, :no, :no], self.Lso[:, :no, no:]
        self.Lvo, self.Lvv = self.Lso[:, no:, :no], self.Lso[:, no:, no:]
        t1, t2 = self.t1, self.t2
        # <mn||ef> (o^2 v^2: small) and the one-body intermediates, exactly as O-2 defines them
        d_menf = np.tensordot(self.Lov, self.Lov, axes=(0, 0))            # (me|nf) = sum_Q L_me L_nf   [m,e,n,f]
        self.oovv = oovv = d_menf.transpose(0, 2, 1, 3) - d_menf.transpose(0, 2, 3, 1)      # <mn||ef> = (me|nf) - (mf|ne)
        tt = np.einsum("ia,jb->ijab", t1, t1)
        self.tau = t2 + tt - tt.transpose(0, 1, 3, 2)
        taut = t2 + 0.5 * (tt - tt.transpose(0, 1, 3, 2))
        f = self.f
        fov, foo, fvv = f[:no, no:], f[:no, :no], f[no:, no:]
        # F_ae = f_ae - 1/2 f_me t_m^a + t_m^f <ma||fe> - 1/2 tau~_mn^af <mn||ef>
        # (<ma||fe> = -<ma||ef>; one virtual index a at a time so that no o v^3 object is held)
        self.Fae = fvv - 0.5 * np.einsum("me,ma->ae", fov, t1) - 0.5 * np.einsum("mnaf,mnef->ae", taut, oovv)
        for a in range(self.nv):
            self.Fae[a] -= np.einsum("mf,mef->e", t1, self._g_m_a_ef(a))
        # F_mi = f_mi + 1/2 t_i^e f_me + t_n^e <mn||ie> + 1/2 tau~_in^ef <mn||ef>
        d_mine = np.tensordot(self.Loo, self.Lov, axes=(0, 0))            # (mi|ne)   [m,i,n,e]
        g_mnie = d_mine.transpose(0, 2, 1, 3) - d_mine.transpose(2, 0, 1, 3)               # <mn||ie> = (mi|ne) - (me|ni)
        self.g_mnie = g_mnie
        self.Fmi = (foo + 0.5 * np.einsum("ie,me->mi", t1, fov) + np.einsum("ne,mnie->mi", t1, g_mnie)
                    + 0.5 * np.einsum("inef,mnef->mi", taut, oovv))
        # F_me = f_me + t_n^f <mn||ef>
        self.Fme = fov + np.einsum("nf,mnef->me", t1, oovv)

    # ---- integral slices, each a direct sum over Q
    def _g_ab_ef(self, a, b):          # <ab||ef> for all e,f
        Lvv = self.Lvv
        return np.einsum("Qe,Qf->ef", Lvv[:, a, :], Lvv[:, b, :]) - np.einsum("Qf,Qe->ef", Lvv[:, a, :], Lvv[:, b, :])

    def _g_m_a_ef(self, a):            # <ma||ef> for all m,e,f
        d_meaf = np.tensordot(self.Lov, self.Lvv[:, a, :], axes=(0, 0))   # (me|af)   [m,e,f]
        return d_meaf - d_meaf.transpose(0, 2, 1)                         # <ma||ef> = (me|af) - (mf|ae)

    def _W_mbej(self, b, j):           # W_mbej for all m,e   (b, j fixed)
        t1, t2, no = self.t1, self.t2, self.no
        g_mbej = np.einsum("Qme,Q->me", self.Lov, self.Lvo[:, b, j]) - np.einsum("Qm,Qe->me", self.Loo[:, :, j], self.Lvv[:, b, :])
        g_mbef = self._g_m_a_ef(b)                                           # <mb||ef>
        d_menj = np.tensordot(self.Lov, self.Loo[:, :, j], axes=(0, 0))   # (me|nj)   [m,e,n]
        g_mnej = d_menj.transpose(0, 2, 1) - d_menj.transpose(2, 0, 1)   # <mn||ej> = (me|nj) - (mj|ne)
        W = g_mbej + np.einsum("f,mef->me", t1[j], g_mbef) - np.einsum("n,mne->me", t1[:, b], g_mnej)
        W -= np.einsum("nf,mnef->me", 0.5 * t2[j, :, :, b] + np.outer(t1[:, b], t1[j]), self.oovv)
        return W, g_mbej

    def r2(self, i, j, a, b):
        """R2_ij^ab (spin-orbital indices; a, b count from the first virtual)."""
        t1, t2, tau, no = self.t1, self.t2, self.tau, self.no
        oovv = self.oovv
        x = oovv[i, j, a, b]
        # P(ab) t_ij^ae (F_be - 1/2 t_m^b F_me)
        Fb = self.Fae[b] - 0.5 * t1[:, b] @ self.Fme
        Fa = self.Fae[a] - 0.5 * t1[:, a] @ self.Fme
        x += t2[i, j, a, :] @ Fb - t2[i, j, b, :] @ Fa
        # - P(ij) t_im^ab (F_mj + 1/2 t_j^e F_me)
        Fj = self.Fmi[:, j] + 0.5 * self.Fme @ t1[j]
        Fi = self.Fmi[:, i] + 0.5 * self.Fme @ t1[i]
        x -= t2[i, :, a, b] @ Fj - t2[j, :, a, b] @ Fi
        # 1/2 tau_mn^ab W_mnij
        g_mnij = np.einsum("Qm,Qn->mn", self.Loo[:, :, i], self.Loo[:, :, j]) - np.einsum("Qm,Qn->mn", self.Loo[:, :, j], self.Loo[:, :, i])
        Wmn = (g_mnij + np.einsum("e,mne->mn", t1[j], self.g_mnie[:, :, i, :]) - np.einsum("e,mne->mn", t1[i], self.g_mnie[:, :, j, :])
               + 0.25 * np.einsum("ef,mnef->mn", tau[i, j], oovv))
        x += 0.5 * np.sum(tau[:, :, a, b] * Wmn)
        # 1/2 tau_ij^ef W_abef
        Wef = (self._g_ab_ef(a, b) + np.einsum("m,mef->ef", t1[:, b], self._g_m_a_ef(a)) - np.einsum("m,mef->ef", t1[:, a], self._g_m_a_ef(b))
               + 0.25 * np.einsum("mn,mnef->ef", tau[:, :, a, b], oovv))
        x += 0.5 * np.sum(tau[i, j] * Wef)
        # P(ij)P(ab) ( t_im^ae W_mbej - t_i^e t_m^a <mb||ej> )
        for (ii, jj, aa, bb, sg) in ((i, j, a, b, 1.0), (j, i, a, b, -1.0), (i, j, b, a, -1.0), (j, i, b, a, 1.0)):
            W, g = self._W_mbej(bb, jj)
            x += sg * (np.sum(t2[ii, :, aa, :] * W) - t1[:, aa] @ g @ t1[ii])
        # P(ij) t_i^e <ab||ej>  - P(ab) t_m^a <mb||ij>
        g_abej = lambda jj: (np.einsum("Qe,Q->e", self.Lvv[:, a, :], self.Lvo[:, b, jj]) - np.einsum("Q,Qe->e", self.Lvo[:, a, jj], self.Lvv[:, b, :]))
        x += t1[i] @ g_abej(j) - t1[j] @ g_abej(i)
        g_mbij = lambda bb: (np.einsum("Qm,Q->m", self.Loo[:, :, i], self.Lvo[:, bb, j]) - np.einsum("Qm,Q->m", self.Loo[:, :, j], self.Lvo[:, bb, i]))
        x -= t1[:, a] @ g_mbij(b) - t1[:, b] @ g_mbij(a)
        return complex(x)

    def r1(self, i, a):
        """R1_i^a."""
        t1, t2, no = self.t1, self.t2, self.no
        x = self.f[i, no + a] + t1[i] @ self.Fae[a] - t1[:, a] @ self.Fmi[:, i] + np.sum(t2[i, :, a, :] * self.Fme)
        g_naif = np.einsum("Qn,Qf->nf", self.Loo[:, :, i], self.Lvv[:, a, :]) - np.einsum("Qnf,Q->nf", self.Lov, self.Lvo[:, a, i])
        x -= np.sum(t1 * g_naif)
        x -= 0.5 * np.sum(t2[i] * self._g_m_a_ef(a))
        d_nemi = np.tensordot(self.Lov, self.Loo[:, :, i], axes=(0, 0))   # (ne|mi)   [n,e,m]
        g_nmei = d_nemi.transpose(0, 2, 1) - d_nemi.transpose(2, 0, 1)   # <nm||ei> = (ne|mi) - (ni|me)
        x -= 0.5 * np.einsum("mne,nme->", t2[:, :, a, :], g_nmei)
        return complex(x)

    def energy(self):
        f, no = self.f, self.no
        return complex(np.sum(f[:no, no:] * self.t1) + 0.25 * np.sum(self.oovv * self.t2)
                       + 0.5 * np.einsum("ijab,ia,jb->", self.oovv, self.t1, self.t1))


# ----------------------------------------------------------------------------------------------------------------------
_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "rtcc_sampled.c")
_CLIB = os.path.join(_HERE, "librtcc_sampled.so")
_clib = None


def build(force: bool = False) -> str:
    """Compile rtcc_sampled.c with gcc (-O2, OpenMP).  Returns the .so path."""
    if force or not os.path.exists(_CLIB) or os.path.getmtime(_CLIB) < os.path.getmtime(_CSRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _CLIB, _CSRC, "-lm"])
    return _CLIB


def _cload():
    global _clib
    if _clib is None:
        build()
        lib = ctypes.CDLL(_CLIB)
        dp, i, vp = ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_void_p
        lib.sorc_num_threads.restype = i
        lib.sorc_create.argtypes = [i, i, i, i, i, dp, dp, dp, dp]
        lib.sorc_create.restype = vp
        lib.sorc_destroy.argtypes = [vp]
        lib.sorc_destroy.restype = None
        lib.sorc_drop_slices.argtypes = [vp]
        lib.sorc_drop_slices.restype = None
        lib.sorc_r2.argtypes = [vp, i, i, i, i, dp]
        lib.sorc_r2.restype = i
        lib.sorc_r1.argtypes = [vp, i, i, dp]
        lib.sorc_r1.restype = i
        lib.sorc_energy.argtypes = [vp, dp]
        lib.sorc_energy.restype = None
        _clib = lib
    return _clib


class SampledOracleC(_PackedIndex):
    """Same elements as ``SampledOracle`` from rtcc_sampled.c: plain C loops straight off the packed blocks and the per-spin
    Cholesky vectors, so that BASELINE.json configs 3-5 (where the numpy version's spin-orbital copies of t2 do not fit in
    host memory) can be checked.  Pinned to the full oracle in tests/test_oracle_pins.py."""

    def __init__(self, oa, ob, va, vb, K, L, fock, t1p, t2p):
        self.d = orc.Dims(oa, ob, va, vb, K)
        n = oa + va
        L = np.ascontiguousarray(L, dtype=np.float64).reshape(2, K, n, n)
        fock = np.ascontiguousarray(fock, dtype=np.float64).reshape(2, n, n)
        t1p = np.ascontiguousarray(t1p, dtype=np.complex128)
        t2p = np.ascontiguousarray(t2p, dtype=np.complex128)
        assert t1p.size == self.d.n_t1 and t2p.size == self.d.n_t2
        dp = ctypes.POINTER(ctypes.c_double)
        self._lib = _cload()
        self._h = self._lib.sorc_create(oa, ob, va, vb, K, L.ctypes.data_as(dp), fock.ctypes.data_as(dp),
                                        t1p.ctypes.data_as(dp), t2p.ctypes.data_as(dp))
        if not self._h:
            raise MemoryError("sampled oracle: allocation failed")
        self._out = np.zeros(2)
        self._dp = self._out.ctypes.data_as(dp)

    def close(self):
        if self._h:
            self._lib.sorc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def drop_slices(self):
        self._lib.sorc_drop_slices(self._h)

    def r2(self, i, j, a, b):
        if self._lib.sorc_r2(self._h, int(i), int(j), int(a), int(b), self._dp):
            raise MemoryError("sampled oracle: allocation failed")
        return complex(self._out[0], self._out[1])

    def r1(self, i, a):
        if self._lib.sorc_r1(self._h, int(i), int(a), self._dp):
            raise MemoryError("sampled oracle: allocation failed")
        return complex(self._out[0], self._out[1])

    def energy(self):
        self._lib.sorc_energy(self._h, self._dp)
        return complex(self._out[0], self._out[1])
