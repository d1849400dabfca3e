"""Pins of the CPU oracle against what the paper and the mathematics fix.
None of these tests touches the CUDA path."""
import os

import numpy as np
import pytest
import scipy.linalg

from oracle import oracle as orc
from tests.fockspace import FockSpace, cc_projections, hamiltonian

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def rand_problem(oa, ob, va, vb, K, seed, sigma=0.3, offdiag=0.1, same_spatial=False):
    """Seeded spin-structured real symmetric L[2,K,n,n], general real symmetric fock[2,n,n]."""
    rng = np.random.default_rng(seed)
    n = oa + va
    L = rng.standard_normal((2, K, n, n)) * sigma
    L = 0.5 * (L + L.transpose(0, 1, 3, 2))
    fock = np.zeros((2, n, n))
    for s, o in ((0, oa), (1, ob)):
        eps = np.concatenate([np.sort(rng.uniform(-1.5, -0.3, o)), np.sort(rng.uniform(0.1, 3.0, n - o))])
        A = rng.standard_normal((n, n)) * offdiag
        fock[s] = np.diag(eps) + 0.5 * (A + A.T)
    if same_spatial:
        L[1] = L[0]
        fock[1] = fock[0]
    return L, fock


def rand_amps(d, seed, scale=0.1, real=False):
    rng = np.random.default_rng(seed)
    t1 = scale * (rng.standard_normal(d.n_t1) + (0 if real else 1j) * rng.standard_normal(d.n_t1))
    t2 = scale * (rng.standard_normal(d.n_t2) + (0 if real else 1j) * rng.standard_normal(d.n_t2))
    return t1.astype(np.complex128), t2.astype(np.complex128)


# ------------------------------------------------------------------ P-9: the paper's only worked numbers
def test_table2_t2_sizes():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "table2_t2_sizes.txt")) if not l.startswith("#")]
    assert len(rows) == 4
    for name, oa, ob, va, vb, gb in rows:
        got = orc.t2_bytes_unpacked(int(oa), int(ob), int(va), int(vb)) / 2.0 ** 30
        # printed to one decimal; benzene-ammonia prints 5.8 for 5.74
        assert abs(got - float(gb)) < 0.07, (name, got, gb)


# ------------------------------------------------------------------ index maps
def test_pack_unpack_roundtrip_and_antisymmetry():
    d = orc.Dims(2, 3, 4, 3, 1)
    t1p, t2p = rand_amps(d, 1)
    t1, t2 = orc.unpack(d, t1p, t2p)
    assert np.array_equal(t2, -t2.transpose(1, 0, 2, 3))
    assert np.array_equal(t2, -t2.transpose(0, 1, 3, 2))
    # spin-forbidden elements exactly zero: spin(i)+spin(j) must equal spin(a)+spin(b)
    so = np.array([0] * d.oa + [1] * d.ob)
    sv = np.array([0] * d.va + [1] * d.vb)
    forb = (so[:, None, None, None] + so[None, :, None, None]) != (sv[None, None, :, None] + sv[None, None, None, :])
    assert np.all(t2[forb] == 0)
    assert np.all(t1[: d.oa, d.va:] == 0) and np.all(t1[d.oa:, : d.va] == 0)
    r1p, r2p = orc.pack(d, t1, t2)
    assert np.array_equal(r1p, t1p) and np.array_equal(r2p, t2p)
    # number of non-zero spin-orbital elements = 4*same-spin unique + 4*ab
    nz = np.count_nonzero(t2)
    paa = orc.npair(d.oa) * orc.npair(d.va) + orc.npair(d.ob) * orc.npair(d.vb)
    assert nz == 4 * paa + 4 * d.oa * d.ob * d.va * d.vb
    # explicit element addresses of the boundary layout
    assert orc.pair(0, 1) == 0 and orc.pair(0, 2) == 1 and orc.pair(1, 2) == 2 and orc.pair(2, 3) == 5
    off_ab = paa
    i, J, a, B = 1, 2, 3, 1
    assert t2[i, d.oa + J, a, d.va + B] == t2p[off_ab + ((i * d.ob + J) * d.va + a) * d.vb + B]
    off_bb = orc.npair(d.oa) * orc.npair(d.va)
    assert t2[d.oa + 0, d.oa + 2, d.va + 1, d.va + 2] == t2p[off_bb + orc.pair(0, 2) * orc.npair(d.vb) + orc.pair(1, 2)]


# ------------------------------------------------------------------ P-1: Cholesky reconstruction
def test_cholesky_reconstruction_and_symmetries():
    oa, ob, va, vb, K = 2, 3, 4, 3, 7
    L, fock = rand_problem(oa, ob, va, vb, K, 11)
    p = orc.Problem(oa, ob, va, vb, K, L, fock)
    N = p.N
    # direct contraction with numpy on the spin-orbital vectors
    chem = np.einsum("Qpq,Qrs->pqrs", p.Lso, p.Lso)
    g = chem.transpose(0, 2, 1, 3) - chem.transpose(0, 2, 3, 1)      # <pq||rs> = (pr|qs) - (ps|qr)
    assert np.allclose(p.g, g, atol=1e-13)
    rng = np.random.default_rng(0)
    for _ in range(50):
        a, b, c, e = rng.integers(0, N, 4)
        assert abs(p.eri_chem(a, b, c, e) - chem[a, b, c, e]) < 1e-13
    assert np.allclose(p.g, -p.g.transpose(1, 0, 2, 3), atol=1e-14)
    assert np.allclose(p.g, -p.g.transpose(0, 1, 3, 2), atol=1e-14)
    assert np.allclose(p.g, p.g.transpose(2, 3, 0, 1), atol=1e-14)
    # spin structure: L^Q_pq = 0 unless spins equal; per-spin blocks land where O-1 says
    assert np.array_equal(p.Lso[:, :oa, :oa], L[0][:, :oa, :oa])
    assert np.array_equal(p.Lso[:, oa:oa + ob, oa + ob + va:], L[1][:, :ob, ob:])
    assert np.all(p.Lso[:, :oa, oa:oa + ob] == 0)
    assert np.array_equal(p.f[oa + ob:oa + ob + va, :oa], fock[0][oa:, :oa])


# ------------------------------------------------------------------ P-0: determinant-space brute force
@pytest.mark.parametrize("dims", [(1, 2, 3, 2), (2, 2, 2, 2), (2, 1, 2, 3), (2, 0, 2, 4), (2, 2, 3, 3)])
def test_residual_matches_determinant_space(dims):
    oa, ob, va, vb = dims
    K = 5
    L, fock = rand_problem(oa, ob, va, vb, K, 100 + sum(dims), sigma=0.4, offdiag=0.2)
    p = orc.Problem(oa, ob, va, vb, K, L, fock)
    t1p, t2p = rand_amps(p.d, 7, scale=0.3)
    t1, t2 = orc.unpack(p.d, t1p, t2p)
    r1, r2, E = p.residual_so(t1, t2)
    fs = FockSpace(p.N)
    R1, R2, Eb = cc_projections(fs, p.d.no, p.f, p.g, t1, t2)
    scale = max(np.abs(R2).max(), 1.0)
    assert np.abs(r1 - R1).max() < 1e-12 * scale
    assert np.abs(r2 - R2).max() < 1e-12 * scale
    assert abs(E - Eb) < 1e-12 * max(abs(Eb), 1.0)


# ------------------------------------------------------------------ P-2: exact two-electron dynamics
def _exact_two_electron(p, tau):
    """C(tau) = ln <Phi|exp(+i H_N tau)|Phi> and the exact amplitudes (CCSD is exact for 2 electrons)."""
    fs = FockSpace(p.N)
    no = p.d.no
    H = hamiltonian(fs, no, p.f, p.g).toarray()
    phi = fs.det(range(no))
    Eref = np.vdot(phi, H @ phi).real
    HN = H - Eref * np.eye(fs.dim)
    psi = scipy.linalg.expm(1j * tau * HN) @ phi
    c0 = np.vdot(phi, psi)
    nv = p.d.nv
    t1 = np.zeros((no, nv), dtype=complex)
    for i in range(no):
        for a in range(nv):
            t1[i, a] = np.vdot(fs.ad[no + a] @ (fs.a[i] @ phi), psi) / c0
    t2 = np.zeros((no, no, nv, nv), dtype=complex)
    for i in range(no):
        for j in range(no):
            for a in range(nv):
                for b in range(nv):
                    c = np.vdot(fs.ad[no + a] @ (fs.ad[no + b] @ (fs.a[j] @ (fs.a[i] @ phi))), psi) / c0
                    t2[i, j, a, b] = c - (t1[i, a] * t1[j, b] - t1[i, b] * t1[j, a])
    return np.log(c0), t1, t2


@pytest.mark.parametrize("dims", [(1, 1, 2, 2), (2, 0, 2, 4)])
def test_exact_two_electron_dynamics_second_order(dims):
    oa, ob, va, vb = dims
    L, fock = rand_problem(oa, ob, va, vb, 4, 5, sigma=0.35, offdiag=0.15)
    p = orc.Problem(oa, ob, va, vb, 4, L, fock)
    tau = 0.8
    Cex, t1ex, t2ex = _exact_two_electron(p, tau)
    errs = []
    for nsteps in (20, 40, 80):
        pr = orc.Propagator(p, mode=0, tol=1e-13, max_micro=500)
        for _ in range(nsteps):
            pr.step(tau / nsteps)
        errs.append(abs(pr.C - Cex))
        t1, t2 = orc.unpack(p.d, pr.t1, pr.t2)
        terr = max(np.abs(t1 - t1ex).max(), np.abs(t2 - t2ex).max())
    assert errs[-1] < 2e-5 and terr < 5e-4
    # implicit trapezoid is second-order accurate: error falls 4x per halving
    assert 3.6 < errs[0] / errs[1] < 4.4 and 3.6 < errs[1] / errs[2] < 4.4
    # the preconditioned micro-iteration reaches the same fixed point
    pr1 = orc.Propagator(p, mode=1, tol=1e-13, max_micro=500)
    for _ in range(80):
        pr1.step(tau / 80)
    assert abs(pr1.C - pr.C) < 1e-11
    # time reversal: C(-tau) = conj C(tau)
    prm = orc.Propagator(p, mode=0, tol=1e-13, max_micro=500)
    for _ in range(20):
        prm.step(-tau / 20)
    prp = orc.Propagator(p, mode=0, tol=1e-13, max_micro=500)
    for _ in range(20):
        prp.step(tau / 20)
    assert abs(prm.C - np.conj(prp.C)) < 1e-12


# ------------------------------------------------------------------ P-3: stationary limit = FCI
@pytest.mark.parametrize("dims", [(1, 1, 2, 2), (2, 0, 2, 4), (1, 1, 3, 3)])
def test_stationary_limit_is_fci(dims):
    oa, ob, va, vb = dims
    L, fock = rand_problem(oa, ob, va, vb, 4, 21, sigma=0.3, offdiag=0.05)
    p = orc.Problem(oa, ob, va, vb, 4, L, fock)
    pr = orc.Propagator(p)                      # only for the denominators
    t1 = np.zeros(p.d.n_t1, dtype=complex)
    t2 = np.zeros(p.d.n_t2, dtype=complex)
    for _ in range(400):
        r1, r2, E = p.residual(t1, t2)
        if max(np.abs(r1).max(initial=0), np.abs(r2).max(initial=0)) < 1e-13:
            break
        t1 = t1 - r1 / pr.D1
        t2 = t2 - r2 / pr.D2
    assert max(np.abs(r1).max(initial=0), np.abs(r2).max(initial=0)) < 1e-12
    assert abs(E.imag) < 1e-13                  # real amplitudes give a real energy
    fs = FockSpace(p.N)
    H = hamiltonian(fs, p.d.no, p.f, p.g).toarray()
    phi = fs.det(range(p.d.no))
    Eref = np.vdot(phi, H @ phi).real
    # sector with the reference's particle number and S_z
    spins = np.array([0] * oa + [1] * ob + [0] * va + [1] * vb)
    keep = []
    for k in range(fs.dim):
        bits = [(k >> q) & 1 for q in range(p.N)]
        if sum(bits) == p.d.no and sum(b for b, s in zip(bits, spins) if s == 0) == oa:
            keep.append(k)
    w = np.linalg.eigvalsh(H[np.ix_(keep, keep)].real)
    assert abs((Eref + E.real) - w[0]) < 1e-11


# ------------------------------------------------------------------ P-4: t = 0 and short time
def test_t0_and_short_time():
    oa, ob, va, vb, K = 2, 2, 3, 3, 6
    L, fock = rand_problem(oa, ob, va, vb, K, 31, sigma=0.2, offdiag=0.1)
    p = orc.Problem(oa, ob, va, vb, K, L, fock)
    d = p.d
    z1 = np.zeros((d.no, d.nv), dtype=complex)
    z2 = np.zeros((d.no, d.no, d.nv, d.nv), dtype=complex)
    r1, r2, E = p.residual_so(z1, z2)
    assert E == 0
    for i in range(d.no):
        for a in range(d.nv):
            assert r1[i, a] == p.f[i, d.no + a]
            for j in range(d.no):
                for b in range(d.nv):
                    A, B = d.no + a, d.no + b
                    ref = p.eri_chem(A, i, B, j) - p.eri_chem(A, j, B, i)     # <ab||ij> = (ai|bj) - (aj|bi)
                    assert abs(r2[i, j, a, b] - ref) < 1e-14
    # C(tau) = -(tau^2/2) [ sum_{i<j,a<b} <ab||ij>^2 + sum_ia f_ia^2 ] + O(tau^3)
    s = 0.25 * np.sum(p.g[: d.no, : d.no, d.no:, d.no:] ** 2) + np.sum(p.f[: d.no, d.no:] ** 2)
    tau = 2e-3
    pr = orc.Propagator(p, mode=0, tol=1e-15, max_micro=100)
    for _ in range(4):
        pr.step(tau / 4)
    lead = -0.5 * tau ** 2 * s
    assert abs(pr.C.real - lead) < 2e-2 * abs(lead)
    assert abs(pr.C.imag) < 2e-2 * abs(lead)


# ------------------------------------------------------------------ P-5: weak-coupling closed form
def _weak_coupling_err(sig, nsteps=25, dt=0.05):
    oa, ob, va, vb, K = 2, 2, 3, 3, 6
    L, fock = rand_problem(oa, ob, va, vb, K, 41, sigma=sig, offdiag=0.0)
    p = orc.Problem(oa, ob, va, vb, K, L, fock)
    d = p.d
    pr = orc.Propagator(p, mode=0, tol=1e-15, max_micro=300)
    for _ in range(nsteps):
        pr.step(dt)
    # discrete linear model: t_{n+1} = ((1 + i dt D/2) t_n + i dt v)/(1 - i dt D/2), E = sum_{i<j,a<b} v t
    eps = np.diag(p.f)
    Clin = 0.0
    Ccont = 0.0
    tau = nsteps * dt
    for i in range(d.no):
        for j in range(i + 1, d.no):
            for a in range(d.nv):
                for b in range(a + 1, d.nv):
                    v = p.g[d.no + a, d.no + b, i, j]
                    D = eps[d.no + a] + eps[d.no + b] - eps[i] - eps[j]
                    t = 0.0
                    c = 0.0
                    for _ in range(nsteps):
                        tn = ((1 + 0.5j * dt * D) * t + 1j * dt * v) / (1 - 0.5j * dt * D)
                        c += 0.5j * dt * (v * t + v * tn)
                        t = tn
                    Clin += c
                    Ccont += (v * v / D ** 2) * (np.exp(1j * D * tau) - 1 - 1j * D * tau)
    return abs(pr.C - Clin) / abs(Clin), abs(Clin - Ccont) / abs(Ccont)


def test_weak_coupling_closed_form():
    e1, disc1 = _weak_coupling_err(0.06)
    e2, disc2 = _weak_coupling_err(0.03)
    assert e1 < 5e-2 and e2 < 1.3e-2
    assert 3.0 < e1 / e2 < 5.0           # deviation from the linear model scales as sigma^2
    assert disc1 < 2e-2                   # AM1 + trapezoid approaches the continuous closed form


# ------------------------------------------------------------------ P-6: invariants
def test_invariants():
    oa, ob, va, vb, K = 2, 3, 4, 3, 6
    L, fock = rand_problem(oa, ob, va, vb, K, 51)
    p = orc.Problem(oa, ob, va, vb, K, L, fock)
    d = p.d
    t1p, t2p = rand_amps(d, 3, scale=0.2)
    t1, t2 = orc.unpack(d, t1p, t2p)
    r1, r2, E = p.residual_so(t1, t2)
    tol = 1e-13 * np.abs(r2).max()
    assert np.abs(r2 + r2.transpose(1, 0, 2, 3)).max() < tol
    assert np.abs(r2 + r2.transpose(0, 1, 3, 2)).max() < tol
    so = np.array([0] * oa + [1] * ob)
    sv = np.array([0] * va + [1] * vb)
    forb = (so[:, None, None, None] + so[None, :, None, None]) != (sv[None, None, :, None] + sv[None, None, None, :])
    assert np.abs(r2[forb]).max() < tol
    assert np.abs(r1[:oa, va:]).max() < tol and np.abs(r1[oa:, :va]).max() < tol
    # R(conj t) = conj R(t); real t gives real R
    c1, c2, Ec = p.residual_so(np.conj(t1), np.conj(t2))
    assert np.abs(c1 - np.conj(r1)).max() < tol and np.abs(c2 - np.conj(r2)).max() < tol
    assert abs(Ec - np.conj(E)) < 1e-14
    q1, q2, Eq = p.residual_so(t1.real + 0j, t2.real + 0j)
    assert np.abs(q1.imag).max() == 0 and np.abs(q2.imag).max() == 0
    # linearised Jacobian at t=0, J_mu,nu = <mu|H_N|nu> - <mu|tau_nu H_N|Phi>, is symmetric on the packed
    # (orthonormal-determinant) space when f_ov = 0 (the second term then vanishes): <Y, J X> = <X, J Y>
    fock0 = fock.copy()
    fock0[0][:oa, oa:] = 0; fock0[0][oa:, :oa] = 0
    fock0[1][:ob, ob:] = 0; fock0[1][ob:, :ob] = 0
    p = orc.Problem(oa, ob, va, vb, K, L, fock0)
    x1, x2 = rand_amps(d, 8, scale=1.0, real=True)
    y1, y2 = rand_amps(d, 9, scale=1.0, real=True)
    h = 1e-4

    def J(v1, v2):
        a1, a2, _ = p.residual(h * v1, h * v2)
        b1, b2, _ = p.residual(-h * v1, -h * v2)
        return (a1 - b1) / (2 * h), (a2 - b2) / (2 * h)
    jx1, jx2 = J(x1, x2)
    jy1, jy2 = J(y1, y2)
    lhs = np.dot(y1, jx1) + np.dot(y2, jx2)
    rhs = np.dot(x1, jy1) + np.dot(x2, jy2)
    assert abs(lhs - rhs) < 1e-7 * abs(lhs)


def test_spin_symmetric_case():
    # o_a=o_b, v_a=v_b, same L and fock for both spins, t_aa = t_bb  =>  R_aa = R_bb
    oa = ob = 2
    va = vb = 3
    L, fock = rand_problem(oa, ob, va, vb, 5, 61, same_spatial=True)
    p = orc.Problem(oa, ob, va, vb, 5, L, fock)
    d = p.d
    t1p, t2p = rand_amps(d, 4, scale=0.2)
    n1 = oa * va
    t1p[n1:] = t1p[:n1]
    nss = orc.npair(oa) * orc.npair(va)
    t2p[nss:2 * nss] = t2p[:nss]
    ab = t2p[2 * nss:].reshape(oa, ob, va, vb)
    ab[:] = 0.5 * (ab + ab.transpose(1, 0, 3, 2))      # t_iJ^aB = t_Ji^Ba
    r1, r2, _ = p.residual(t1p, t2p)
    assert np.abs(r1[:n1] - r1[n1:]).max() < 1e-13
    assert np.abs(r2[:nss] - r2[nss:2 * nss]).max() < 1e-13


# ------------------------------------------------------------------ P-7: separability
def test_separability():
    # two subsystems with disjoint orbitals and disjoint Q ranges: C_AB = C_A + C_B
    dA, dB = (1, 1, 2, 2), (1, 2, 3, 2)
    KA, KB = 3, 4
    LA, fA = rand_problem(*dA, KA, 71, sigma=0.3, offdiag=0.1)
    LB, fB = rand_problem(*dB, KB, 72, sigma=0.3, offdiag=0.1)
    oa, ob, va, vb = (dA[0] + dB[0], dA[1] + dB[1], dA[2] + dB[2], dA[3] + dB[3])
    n = oa + va
    K = KA + KB
    L = np.zeros((2, K, n, n))
    fock = np.zeros((2, n, n))
    for s in range(2):
        oA, oB = dA[s], dB[s]
        nA, nB = dA[0] + dA[2], dB[0] + dB[2]
        idxA = list(range(oA)) + list(range(oA + oB, oA + oB + (nA - oA)))
        idxB = list(range(oA, oA + oB)) + list(range(oA + oB + (nA - oA), n))
        L[s][:KA][np.ix_(range(KA), idxA, idxA)] = LA[s]
        L[s][KA:][np.ix_(range(KB), idxB, idxB)] = LB[s]
        fock[s][np.ix_(idxA, idxA)] = fA[s]
        fock[s][np.ix_(idxB, idxB)] = fB[s]
    C = []
    for (dd, KK, LL, ff) in ((dA, KA, LA, fA), (dB, KB, LB, fB), ((oa, ob, va, vb), K, L, fock)):
        pr = orc.Propagator(orc.Problem(*dd, KK, LL, ff), mode=0, tol=1e-14, max_micro=300)
        for _ in range(5):
            pr.step(0.05)
        C.append(pr.C)
    assert abs(C[2] - (C[0] + C[1])) < 1e-13
    assert abs(C[0]) > 1e-6 and abs(C[1]) > 1e-6


# ------------------------------------------------------------------ tier B: sampled-element oracle vs tier A
def test_sampled_oracle_matches_full_oracle():
    """The on-demand-integral evaluation of single residual elements (oracle/sampled.py) must reproduce the full
    spin-orbital oracle (pinned above by determinant-space brute force) on complex amplitudes, general Fock."""
    from oracle.sampled import SampledOracle
    for (oa, ob, va, vb, K, seed) in [(2, 3, 4, 3, 5, 21), (3, 1, 2, 4, 4, 22), (2, 2, 3, 3, 6, 23)]:
        L, fock = rand_problem(oa, ob, va, vb, K, seed)
        prob = orc.Problem(oa, ob, va, vb, K, L, fock)
        t1p, t2p = rand_amps(prob.d, seed + 100)
        r1p, r2p, E = prob.residual(t1p, t2p)
        so = SampledOracle(oa, ob, va, vb, K, L, fock, t1p, t2p)
        assert abs(so.energy() - E) < 1e-13
        for k in range(prob.d.n_t2):                  # every packed element, through the packed -> spin-orbital map
            i, j, a, b = so.so_of_packed_t2(k)
            assert abs(so.r2(i, j, a, b) - r2p[k]) < 1e-13, (k, i, j, a, b)
        for k in range(prob.d.n_t1):
            i, a = so.so_of_packed_t1(k)
            assert abs(so.r1(i, a) - r1p[k]) < 1e-13
        # antisymmetry of the sampled values themselves
        i, j, a, b = so.so_of_packed_t2(0)
        assert abs(so.r2(j, i, a, b) + so.r2(i, j, a, b)) < 1e-13


def test_sampled_c_oracle_matches_full_oracle():
    """rtcc_sampled.c (the tier-B oracle that fits configs 3-5) against tier A: EVERY packed element of R1 and R2 and E, complex
    amplitudes, general Fock matrix, shapes with o_s in {0, 1}, v_s = 1 and unequal spins; then spin-orbital elements outside
    the packed set (antisymmetric partners, a spin-forbidden one) to pin the accessors' sign and spin rules."""
    from oracle.sampled import SampledOracleC
    shapes = [(2, 3, 4, 3, 5, 21), (3, 1, 2, 4, 4, 22), (2, 2, 3, 3, 6, 23), (2, 0, 3, 5, 4, 24), (1, 2, 2, 1, 3, 25), (3, 3, 5, 5, 7, 26)]
    for (oa, ob, va, vb, K, seed) in shapes:
        L, fock = rand_problem(oa, ob, va, vb, K, seed)
        prob = orc.Problem(oa, ob, va, vb, K, L, fock)
        t1p, t2p = rand_amps(prob.d, seed + 100)
        r1p, r2p, E = prob.residual(t1p, t2p)
        scale = max(np.abs(r2p).max(initial=0), np.abs(r1p).max(initial=0), 1.0)
        so = SampledOracleC(oa, ob, va, vb, K, L, fock, t1p, t2p)
        assert abs(so.energy() - E) < 1e-13 * max(1.0, abs(E))
        for k in range(prob.d.n_t2):
            i, j, a, b = so.so_of_packed_t2(k)
            assert so.packed_of_so_t2(i, j, a, b) == k
            assert abs(so.r2(i, j, a, b) - r2p[k]) < 2e-13 * scale, (k, i, j, a, b)
        for k in range(prob.d.n_t1):
            i, a = so.so_of_packed_t1(k)
            assert abs(so.r1(i, a) - r1p[k]) < 2e-13 * scale
        if prob.d.n_t2:
            t1, t2 = orc.unpack(prob.d, t1p, t2p)
            r1so, r2so, _ = prob.residual_so(t1, t2)
            i, j, a, b = so.so_of_packed_t2(prob.d.n_t2 - 1)
            for (p, q, r, s) in ((j, i, a, b), (i, j, b, a), (j, i, b, a)):
                assert abs(so.r2(p, q, r, s) - r2so[p, q, r, s]) < 2e-13 * scale
            if oa and ob:
                assert so.r2(0, oa, 0, 1 if va > 1 else 0) == 0 or va == 1      # (alpha beta | alpha alpha): spin-forbidden
        so.close()


def test_sampled_c_oracle_matches_numpy_sampled_oracle_beyond_tier_a():
    """A size the full oracle cannot hold comfortably (N = 60 spin-orbitals): the two independently written sampled oracles
    (numpy einsum vs C loops) agree on a spread of elements from all three spin blocks."""
    from oracle.sampled import SampledOracle, SampledOracleC
    oa, ob, va, vb, K = 4, 5, 26, 25, 31
    L, fock = rand_problem(oa, ob, va, vb, K, 41)
    d = orc.Dims(oa, ob, va, vb, K)
    t1p, t2p = rand_amps(d, 141)
    a_, c_ = SampledOracle(oa, ob, va, vb, K, L, fock, t1p, t2p), SampledOracleC(oa, ob, va, vb, K, L, fock, t1p, t2p)
    assert abs(a_.energy() - c_.energy()) < 1e-12
    rng = np.random.default_rng(5)
    for k in list(rng.integers(0, d.n_t2, 12)) + [0, d.n_t2 - 1]:
        idx = a_.so_of_packed_t2(int(k))
        assert abs(a_.r2(*idx) - c_.r2(*idx)) < 1e-12 * max(1.0, abs(a_.r2(*idx)))
    for k in (0, d.n_t1 - 1, d.n_t1 // 2):
        idx = a_.so_of_packed_t1(int(k))
        assert abs(a_.r1(*idx) - c_.r1(*idx)) < 1e-12
    c_.close()


# ------------------------------------------------------------------ NEXT-3: (N-1) Fock matrix
def test_fock_n1_is_eps_minus_antisymmetrised_core_integral():
    """f_pq = eps_p delta_pq - <pc||qc>: the per-spin Coulomb/exchange formula must equal the spin-orbital definition
    evaluated with the (independently pinned) antisymmetrised tensor of the C oracle, for the hole in either spin."""
    oa, ob, va, vb, K = 2, 3, 4, 3, 6
    L, fock_any = rand_problem(oa, ob, va, vb, K, 31)
    prob = orc.Problem(oa, ob, va, vb, K, L, fock_any)
    n = oa + va
    rng = np.random.default_rng(3)
    eps = rng.uniform(-2, 2, (2, n))
    so = lambda s, p: (p if p < (ob if s else oa) else prob.d.no + (va if s else 0) + p - (ob if s else oa)) + (oa if s and p < ob else 0)
    for cs, ci in ((0, oa), (1, 0), (0, 1)):
        f = orc.build_fock_n1(L, eps, cs, ci)
        c = so(cs, ci)
        for s in range(2):
            for p in range(n):
                for q in range(n):
                    ref = (eps[s, p] if p == q else 0.0) - prob.g[so(s, p), c, so(s, q), c]
                    assert abs(f[s, p, q] - ref) < 1e-13
        assert np.allclose(f, f.transpose(0, 2, 1))


# ------------------------------------------------------------------ NEXT-2: Green's function / spectral function, Eqs. 3-4
def test_spectral_function_closed_forms():
    """C = 0: a single Lorentzian (eta/pi)/((w-e0)^2+eta^2) at e0 = eps_c + E_corr.  C = b (exp(-i W tau) - 1): the Poisson
    satellite series exp(-b) sum_n b^n/n! Lorentzian(w - e0 - n W) (cumulant textbook result).  Long, finely sampled record."""
    dt, nt, eta = 0.01, 40001, 0.05
    tau = dt * np.arange(nt)
    om = np.linspace(-3.0, 1.0, 81)
    e0 = -1.3
    lor = lambda x: (eta / np.pi) / (x * x + eta * eta)
    G, A = orc.spectral_function(np.zeros(nt, complex), dt, -1.0, -0.3, eta, om)
    assert np.abs(G[0] + 1j) < 1e-15 and np.allclose(np.abs(G), 1.0)
    assert np.abs(A - lor(om - e0)).max() < 2e-4
    b, W = 0.4, 0.7
    C = b * (np.exp(-1j * W * tau) - 1.0)
    _, A2 = orc.spectral_function(C, dt, -1.0, -0.3, eta, om)
    from math import factorial
    ref = sum(np.exp(-b) * b ** k / factorial(k) * lor(om - e0 - k * W) for k in range(25))
    assert np.abs(A2 - ref).max() < 2e-4
    assert abs(np.trapezoid(A2, om) - np.trapezoid(ref, om)) < 1e-3


# ------------------------------------------------------------------ fixed_micro and set_state of the propagator
def test_fixed_micro_is_k_sweeps_of_a_contraction_towards_the_implicit_solution():
    """Eq. 9 is implicit in T(tau+dt); PAPER.md:103 solves it by fixed-point sweeps.  With fixed_micro = k the oracle
    must do exactly k sweeps: the distance to the converged step (pinned by the exact two-electron dynamics above) then shrinks
    geometrically in k, by about the same factor per sweep, in both iteration modes; k sweeps of mode 0 started from t and one more
    differ by exactly one application of the map (checked through the residual the oracle reports)."""
    oa, ob, va, vb, K = 2, 1, 2, 3, 4
    L, fock = rand_problem(oa, ob, va, vb, K, seed=5, sigma=0.25, offdiag=0.0)
    prob = orc.Problem(oa, ob, va, vb, K, L, fock)
    dt = 0.2
    for mode in (0, 1):
        ref = orc.Propagator(prob, mode=mode, tol=1e-15, max_micro=500)
        ref.step(dt)
        errs = []
        for k in range(1, 8):
            p = orc.Propagator(prob, mode=mode, fixed_micro=k)
            assert p.step(dt) == k and p.last_micro == k
            errs.append(max(np.abs(p.t1 - ref.t1).max(), np.abs(p.t2 - ref.t2).max()))
            if mode == 0 and k >= 2:
                # the k-th iterate is B + (i dt/2) R(iterate k-1): R(t(k-1)) is what the (k-1)-sweep propagator reports
                h = 0.5j * dt
                assert np.allclose(p.t2, h * prob.residual(np.zeros_like(p.t1), np.zeros_like(p.t2))[1] + h * prev.r2, rtol=0, atol=1e-15)
            prev = p
        ratios = [errs[i + 1] / errs[i] for i in range(len(errs) - 1)]
        assert errs[0] > 1e-6 and all(r < 0.8 for r in ratios), (mode, errs)
        assert max(ratios[1:]) < 4.0 * min(ratios[1:]), (mode, ratios)
        assert errs[-1] < errs[0] * max(ratios) ** 5 * 1.01


def test_set_state_continues_like_the_uninterrupted_run():
    """Propagator.set_state (the oracle side of the restart tests): a second propagator started from the amplitudes, time and
    cumulant of the first continues to the same amplitudes and cumulant as the uninterrupted run, and its E at the restart point is
    the energy functional of those amplitudes."""
    oa, ob, va, vb, K = 2, 2, 2, 2, 3
    L, fock = rand_problem(oa, ob, va, vb, K, seed=8, sigma=0.2)
    prob = orc.Problem(oa, ob, va, vb, K, L, fock)
    a = orc.Propagator(prob, mode=0, tol=1e-13, max_micro=300)
    for _ in range(3):
        a.step(0.05)
    b = orc.Propagator(prob, mode=0, tol=1e-13, max_micro=300)
    b.set_state(a.t1, a.t2, a.time, a.C)
    assert b.E == prob.residual(a.t1, a.t2)[2] and b.time == a.time and b.C == a.C
    for _ in range(3):
        a.step(0.05); b.step(0.05)
    assert np.array_equal(a.t1, b.t1) and np.array_equal(a.t2, b.t2) and a.C == b.C and abs(a.time - 0.3) < 1e-15
