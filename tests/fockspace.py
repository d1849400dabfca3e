"""Determinant-space (Fock-space) brute force used to pin the oracle.

Independent of oracle/ and of the CUDA path: second-quantised operators as sparse matrices on the
2^N-dimensional Fock space (Jordan-Wigner signs), H = sum h_pq p+ q + 1/4 sum <pq||rs> p+ q+ s r
(PAPER.md:41), T_n with the (1/n!)^2 prefactor.
"""
import numpy as np
import scipy.sparse as sp


class FockSpace:
    def __init__(self, N):
        self.N = N
        dim = 1 << N
        self.dim = dim
        self.a = []          # annihilators
        idx = np.arange(dim)
        for p in range(N):
            occ = (idx >> p) & 1
            src = idx[occ == 1]
            dst = src ^ (1 << p)
            # sign = (-1)^(number of occupied orbitals below p)
            below = src & ((1 << p) - 1)
            par = np.zeros_like(below)
            x = below.copy()
            while np.any(x):
                par ^= x & 1
                x >>= 1
            sign = 1.0 - 2.0 * par
            self.a.append(sp.csr_matrix((sign, (dst, src)), shape=(dim, dim)))
        self.ad = [m.T.tocsr() for m in self.a]

    def det(self, occ):
        v = np.zeros(self.dim, dtype=np.complex128)
        k = 0
        for p in occ:
            k |= 1 << p
        v[k] = 1.0
        return v

    def one_body(self, h):
        N = self.N
        H = sp.csr_matrix((self.dim, self.dim), dtype=np.complex128)
        for p in range(N):
            for q in range(N):
                if h[p, q] != 0:
                    H = H + h[p, q] * (self.ad[p] @ self.a[q])
        return H

    def two_body(self, g):
        """1/4 sum_pqrs g[p,q,r,s] p+ q+ s r."""
        N = self.N
        H = sp.csr_matrix((self.dim, self.dim), dtype=np.complex128)
        for p in range(N):
            for q in range(N):
                if p == q:
                    continue
                D = sp.csr_matrix((self.dim, self.dim), dtype=np.complex128)
                for r in range(N):
                    for s in range(N):
                        if r != s and g[p, q, r, s] != 0:
                            D = D + g[p, q, r, s] * (self.a[s] @ self.a[r])
                H = H + 0.25 * (self.ad[p] @ self.ad[q] @ D)
        return H

    def cluster(self, no, t1, t2):
        """T = sum t_i^a a+ i + 1/4 sum t_ij^ab a+ b+ j i (virtual a is spin-orbital no+a)."""
        nv = self.N - no
        T = sp.csr_matrix((self.dim, self.dim), dtype=np.complex128)
        for i in range(no):
            for a in range(nv):
                if t1[i, a] != 0:
                    T = T + t1[i, a] * (self.ad[no + a] @ self.a[i])
        for i in range(no):
            for j in range(no):
                for a in range(nv):
                    for b in range(nv):
                        if t2[i, j, a, b] != 0:
                            T = T + 0.25 * t2[i, j, a, b] * (
                                self.ad[no + a] @ self.ad[no + b] @ self.a[j] @ self.a[i])
        return T


def hamiltonian(fs, no, f, g):
    """H with h = f - sum_{i occ} <pi||qi>  (f is the Fock matrix of the reference determinant)."""
    h = f - np.einsum("piqi->pq", g[:, :no, :, :no])
    return (fs.one_body(h) + fs.two_body(g)).tocsr()


def expT_apply(T, v, sign=1.0):
    out = v.copy()
    term = v.copy()
    k = 1
    while True:
        term = sign * (T @ term) / k
        if not np.any(term):
            break
        out = out + term
        k += 1
        if k > 64:
            raise RuntimeError("T not nilpotent?")
    return out


def cc_projections(fs, no, f, g, t1, t2):
    """R1[i,a], R2[i,j,a,b], E = <mu| e^{-T} H_N e^{T} |Phi> (equal to the connected form of Eqs. 5,7,8)."""
    nv = fs.N - no
    H = hamiltonian(fs, no, f, g)
    phi = fs.det(range(no))
    Eref = np.vdot(phi, H @ phi)
    T = fs.cluster(no, t1, t2)
    w = expT_apply(T, phi)
    w = H @ w - Eref * w
    w = expT_apply(T, w, sign=-1.0)
    E = np.vdot(phi, w)
    R1 = np.zeros((no, nv), dtype=np.complex128)
    R2 = np.zeros((no, no, nv, nv), dtype=np.complex128)
    for i in range(no):
        for a in range(nv):
            bra = fs.ad[no + a] @ (fs.a[i] @ phi)
            R1[i, a] = np.vdot(bra, w)
    for i in range(no):
        for j in range(no):
            for a in range(nv):
                for b in range(nv):
                    bra = fs.ad[no + a] @ (fs.ad[no + b] @ (fs.a[j] @ (fs.a[i] @ phi)))
                    R2[i, j, a, b] = np.vdot(bra, w)
    return R1, R2, E
