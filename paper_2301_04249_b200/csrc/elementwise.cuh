// elementwise.cuh -- bandwidth-bound kernels of the RT-EOM-CCSD hot path: spin-block unpacking of the
// packed boundary amplitudes into the contraction layouts, assembly / antisymmetrisation of the
// residual (PAPER.md:133 spin-explicit blocks), the Adams-Moulton update (Eq. 9) and the
// deterministic reductions for the cumulant rate (Eqs. 5-6).
//
// Complex arrays inside the library are "row-planar": element (r, c) of a matrix with `cols` columns
// has its real part at r*2*cols + c and its imaginary part at r*2*cols + cols + c, so every row is a
// Re|Im-stacked real row (north_star: "stacking Re and Im").  Packed boundary arrays are interleaved.
#pragma once
#include <cuda_runtime.h>

namespace rtcc {

struct Dims {
    int o[2], v[2], n, NQ;
    int n1a, n1b, n1;        // spin-conserving ov pairs: alpha (i,a) then beta
    int nA, nB;              // spin-flip pairs: A = (i alpha, B beta), B = (I beta, a alpha)
    int po[2], pv[2];        // P(o), P(v)
    int oo;                  // o_alpha * o_beta
    long long off_t1[2];     // offsets (complex elements) into packed t1
    long long off_t2[3];     // aa, bb, ab offsets into packed t2
    long long n_t1, n_t2;
};

__host__ __device__ inline long long pair_index(int x, int y) { return (long long)y * (y - 1) / 2 + x; }

struct c128 { double re, im; };

// antisymmetric same-spin amplitude t_{im}^{ae} from the packed block
__device__ __forceinline__ c128 ss_amp(const double* t2p, long long off, int pv, int i, int m, int a, int e)
{
    c128 z = {0.0, 0.0};
    if (i == m || a == e) return z;
    double s = 1.0;
    if (i > m) { int t = i; i = m; m = t; s = -s; }
    if (a > e) { int t = a; a = e; e = t; s = -s; }
    long long k = off + pair_index(i, m) * pv + pair_index(a, e);
    z.re = s * t2p[2 * k]; z.im = s * t2p[2 * k + 1];
    return z;
}
__device__ __forceinline__ c128 ab_amp(const double* t2p, const Dims& d, int i, int J, int a, int B)
{
    long long k = d.off_t2[2] + (((long long)i * d.o[1] + J) * d.v[0] + a) * d.v[1] + B;
    c128 z = {t2p[2 * k], t2p[2 * k + 1]};
    return z;
}

// tile-major zero-padded slabs of the bare vectors for the ladder's bulk copies (see ladder.cuh):
//   rows of PR orbitals x PC virtual columns, pitch PR*PC+4:  T[pt][ct][Qt][16 k][pi*PC + ci]
__global__ void k_tile_L(int NQ, int n, int o, int v, int PR, int PC, int nCt, int nQt, const double* __restrict__ L, double* __restrict__ T)
{
    const long long tot = (long long)NQ * n * v;
    const int pitch = PR * PC + 4;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        int ee = (int)(x % v); long long r = x / v; int p = (int)(r % n); int Q = (int)(r / n);
        long long blk = ((long long)(p / PR) * nCt + ee / PC) * nQt + Q / 16;
        T[(blk * 16 + Q % 16) * pitch + (p % PR) * PC + ee % PC] = L[((long long)Q * n + p) * n + o + ee];
    }
}
// index of amplitude (e, f, col) in the ladder's tile-major X: Xt[et][ft][ct][8 kt][16][nt2+4]
__device__ __forceinline__ long long xt_index(int e, int f, int col, int nFt, int ncol, int nt2)
{
    const int k2 = (e % 16) * 8 + (f % 8);
    long long t = (((long long)(e / 16) * nFt + f / 8) * ncol + col / nt2) * 8 + k2 / 16;
    return (t * 16 + k2 % 16) * (nt2 + 4) + col % nt2;
}

// t1 packed -> planar t1r[pl][x], x in sc pair order (alpha (i,a) then beta)
__global__ void k_unpack_t1(Dims d, const double* __restrict__ t1p, double* __restrict__ t1r)
{
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < d.n1; x += (long long)gridDim.x * blockDim.x) {
        t1r[x] = t1p[2 * x];
        t1r[d.n1 + x] = t1p[2 * x + 1];
    }
}

// Right operand of the three-multiplication complex product: for a planar matrix W (rows x [Re cols | Im cols]) writes
// Wd = Im - Re (rows x cols, dense) and replaces the Im plane by Re + Im.
__global__ void k_r3m_W(long long rows, long long cols, double* __restrict__ W, double* __restrict__ Wd)
{
    const long long tot = rows * cols;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        const long long r = x / cols, c = x - r * cols;
        const double re = W[r * 2 * cols + c], im = W[r * 2 * cols + cols + c];
        Wd[x] = im - re;
        W[r * 2 * cols + cols + c] = re + im;
    }
}

// Tiled unpacking of the pair-space amplitude matrices (north_star: "coalesced ... shared-memory staging").  Every packed
// amplitude is read ONCE, as a 16-byte complex element with the packed layout's fastest index across the threads, and written
// to all the places the pair-space matrices hold it -- directly where the destination's fastest index is the source's, through
// a 32 x 33 shared-memory tile (transposed) where it is the other one.  T_sc and T_AB are symmetric / share their elements:
//   alpha-beta amplitude t = tab[i,M,a,E]:  Tsc[(a i a),(b M E)] = Tsc[(b M E),(a i a)] = t,   T_AB[(i,E),(M,a)] = -t
//   same-spin amplitude t = t_{i<m}^{a<e}:  T[(i,a),(m,e)] = T[(m,e),(i,a)] = t,  T[(i,e),(m,a)] = T[(m,a),(i,e)] = -t
// (elements with i == m or a == e are zero: the buffers are cleared once at creation and those places never written).
// Ts / TsAB (optional): Re + Im of every element, the left operand of the three-multiplication complex product.
constexpr int UP_T = 32;
__global__ void __launch_bounds__(256) k_unpack_ab(Dims d, const double* __restrict__ t2p, double* __restrict__ Tsc, double* __restrict__ TAB,
                                                   double* __restrict__ Ts, double* __restrict__ TsAB)
{
    __shared__ double sre[UP_T][UP_T + 1], sim[UP_T][UP_T + 1];
    const int oa = d.o[0], ob = d.o[1], va = d.v[0], vb = d.v[1];
    const int nAt = (va + UP_T - 1) / UP_T, nEt = (vb + UP_T - 1) / UP_T;
    const long long nitem = (long long)oa * ob * nAt * nEt;
    const long long n1 = d.n1, ld = 2 * n1, nB = d.nB;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const double2* __restrict__ src = reinterpret_cast<const double2*>(t2p) + d.off_t2[2];
    for (long long it = blockIdx.x; it < nitem; it += gridDim.x) {
        long long k = it;
        const int E0 = (int)(k % nEt) * UP_T; k /= nEt;
        const int a0 = (int)(k % nAt) * UP_T; k /= nAt;
        const int M = (int)(k % ob), i = (int)(k / ob);
        const long long base = ((long long)i * ob + M) * va;
        __syncthreads();
        double2 zz[UP_T / 8];                           // all loads of the tile first: they are in flight together
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int a = a0 + ty + 8 * q, E = E0 + tx;
            zz[q] = (a < va && E < vb) ? src[(base + a) * vb + E] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int a = a0 + ty + 8 * q, E = E0 + tx;
            const double2 z = zz[q];
            if (a < va && E < vb) {
                const long long r = (long long)i * va + a, c = d.n1a + (long long)M * vb + E;
                Tsc[r * ld + c] = z.x;
                Tsc[r * ld + n1 + c] = z.y;
                if (Ts) Ts[r * n1 + c] = z.x + z.y;
            }
            sre[ty + 8 * q][tx] = z.x; sim[ty + 8 * q][tx] = z.y;
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int E = E0 + ty + 8 * q, a = a0 + tx;
            if (a < va && E < vb) {
                const double re = sre[tx][ty + 8 * q], im = sim[tx][ty + 8 * q];
                const long long r = d.n1a + (long long)M * vb + E, c = (long long)i * va + a;
                Tsc[r * ld + c] = re;
                Tsc[r * ld + n1 + c] = im;
                if (Ts) Ts[r * n1 + c] = re + im;
                const long long rA = (long long)i * vb + E, cA = (long long)M * va + a;
                TAB[rA * 2 * nB + cA] = -re;
                TAB[rA * 2 * nB + nB + cA] = -im;
                if (TsAB) TsAB[rA * nB + cA] = -re - im;
            }
        }
    }
}
__global__ void __launch_bounds__(256) k_unpack_ss(Dims d, int s, const int2* __restrict__ opairs, const double* __restrict__ t2p,
                                                   double* __restrict__ Tsc, double* __restrict__ Ts)
{
    __shared__ double sre[UP_T][UP_T + 1], sim[UP_T][UP_T + 1];
    const int v = d.v[s], po = d.po[s], pv = d.pv[s];
    const int nT = (v + UP_T - 1) / UP_T, ntri = nT * (nT + 1) / 2;
    const long long nitem = (long long)po * ntri;
    const long long n1 = d.n1, ld = 2 * n1, off = s ? d.n1a : 0;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const double2* __restrict__ src = reinterpret_cast<const double2*>(t2p) + d.off_t2[s];
    for (long long it = blockIdx.x; it < nitem; it += gridDim.x) {
        const int pim = (int)(it / ntri); int tt = (int)(it - (long long)pim * ntri);
        int et = 0;                                          // tile pair (at <= et) from the triangular index
        while ((et + 1) * (et + 2) / 2 <= tt) ++et;
        const int at = tt - et * (et + 1) / 2;
        const int a0 = at * UP_T, e0 = et * UP_T;
        const int2 im_ = opairs[pim];
        const long long ri = off + (long long)im_.x * v, rm = off + (long long)im_.y * v;    // first row / column of (i,.) and (m,.)
        __syncthreads();
        double2 zz[UP_T / 8];
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int e = e0 + ty + 8 * q, a = a0 + tx;
            zz[q] = (a < e && e < v) ? src[(long long)pim * pv + pair_index(a, e)] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int e = e0 + ty + 8 * q, a = a0 + tx;
            const double2 z = zz[q];
            if (a < e && e < v) {
                // destinations whose fastest index is a:  T[(i,e),(m,a)] = -t,  T[(m,e),(i,a)] = +t
                long long r = ri + e, c = rm + a;
                Tsc[r * ld + c] = -z.x; Tsc[r * ld + n1 + c] = -z.y;
                if (Ts) Ts[r * n1 + c] = -z.x - z.y;
                r = rm + e; c = ri + a;
                Tsc[r * ld + c] = z.x; Tsc[r * ld + n1 + c] = z.y;
                if (Ts) Ts[r * n1 + c] = z.x + z.y;
            }
            sre[ty + 8 * q][tx] = z.x; sim[ty + 8 * q][tx] = z.y;
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int a = a0 + ty + 8 * q, e = e0 + tx;
            if (a < e && e < v) {
                const double re = sre[tx][ty + 8 * q], im = sim[tx][ty + 8 * q];
                // destinations whose fastest index is e:  T[(i,a),(m,e)] = +t,  T[(m,a),(i,e)] = -t
                long long r = ri + a, c = rm + e;
                Tsc[r * ld + c] = re; Tsc[r * ld + n1 + c] = im;
                if (Ts) Ts[r * n1 + c] = re + im;
                r = rm + a; c = ri + e;
                Tsc[r * ld + c] = -re; Tsc[r * ld + n1 + c] = -im;
                if (Ts) Ts[r * n1 + c] = -re - im;
            }
        }
    }
}

// Ladder operands by tiled transposition (same scheme as k_unpack_*): the packed blocks are [(occupied pair)][(virtual pair)]
// with the virtual pair fastest, the ladder wants [(virtual pair)][Re | Im][(occupied pair)].  A CTA reads a 32 x 32 tile with
// the virtual pair across the threads (16-byte elements), turns it in shared memory and writes with the occupied pair across
// the threads: the planar X, the tile-major zero-padded X of the ladder kernels and tau.
// X_ab[(e,F)][pl][(i,J)] = tab[i,J,e,F];  tau_ab = X + t1a[i,e] t1b[J,F]
__global__ void __launch_bounds__(256) k_build_Xab(Dims d, const double* __restrict__ t2p, const double* __restrict__ t1r,
                                                   double* __restrict__ X, double* __restrict__ Xt, int nFt, int ncol, int nt2, double* __restrict__ tau)
{
    __shared__ double sre[UP_T][UP_T + 1], sim[UP_T][UP_T + 1];
    const int va = d.v[0], vb = d.v[1], ob = d.o[1];
    const long long vv = (long long)va * vb, oo = d.oo, n1 = d.n1;
    const int nCt = (int)((oo + UP_T - 1) / UP_T);
    const long long nRt = (vv + UP_T - 1) / UP_T, nitem = nRt * nCt;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const double2* __restrict__ src = reinterpret_cast<const double2*>(t2p) + d.off_t2[2];
    for (long long it = blockIdx.x; it < nitem; it += gridDim.x) {
        const long long r0 = (it / nCt) * UP_T; const int c0 = (int)(it % nCt) * UP_T;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int col = c0 + ty + 8 * q; const long long row = r0 + tx;
            double2 z = make_double2(0.0, 0.0);
            if (col < oo && row < vv) z = src[(long long)col * vv + row];
            sre[ty + 8 * q][tx] = z.x; sim[ty + 8 * q][tx] = z.y;
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const long long row = r0 + ty + 8 * q; const int col = c0 + tx;
            if (col < oo && row < vv) {
                const double re = sre[tx][ty + 8 * q], im = sim[tx][ty + 8 * q];
                const int e = (int)(row / vb), F = (int)(row - (long long)e * vb), i = col / ob, J = col - i * ob;
                const long long xa = (long long)i * va + e, xb = d.n1a + (long long)J * vb + F;
                const double ar = t1r[xa], ai = t1r[n1 + xa], br = t1r[xb], bi = t1r[n1 + xb];
                X[row * 2 * oo + col] = re;
                X[row * 2 * oo + oo + col] = im;
                Xt[xt_index(e, F, col, nFt, ncol, nt2)] = re;
                Xt[xt_index(e, F, (int)oo + col, nFt, ncol, nt2)] = im;
                tau[row * 2 * oo + col] = re + ar * br - ai * bi;
                tau[row * 2 * oo + oo + col] = im + ar * bi + ai * br;
            }
        }
    }
}

// X_ss[(e,f)][pl][(i<j)] = t_{ij}^{ef} = -X_ss[(f,e)];  tau = X + t1[i,e] t1[j,f] - t1[i,f] t1[j,e].  Rows e == f are zero: the
// buffers are cleared at creation and those rows never written.  anti: rows e >= f of the tile-major X stay zero as well.
__global__ void __launch_bounds__(256) k_build_Xss(Dims d, int s, const double* __restrict__ t2p, const double* __restrict__ t1r,
                                                   const int2* __restrict__ opairs, const int2* __restrict__ vpairs, double* __restrict__ X,
                                                   double* __restrict__ Xt, int nFt, int ncol, int nt2, double* __restrict__ tau, int anti)
{
    __shared__ double sre[UP_T][UP_T + 1], sim[UP_T][UP_T + 1];
    const int v = d.v[s], po = d.po[s], pv = d.pv[s];
    const long long o1 = s ? d.n1a : 0, n1 = d.n1;
    const int nCt = (po + UP_T - 1) / UP_T, nRt = (pv + UP_T - 1) / UP_T;
    const long long nitem = (long long)nRt * nCt;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const double2* __restrict__ src = reinterpret_cast<const double2*>(t2p) + d.off_t2[s];
    for (long long it = blockIdx.x; it < nitem; it += gridDim.x) {
        const int r0 = (int)(it / nCt) * UP_T, c0 = (int)(it % nCt) * UP_T;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int col = c0 + ty + 8 * q, pr = r0 + tx;
            double2 z = make_double2(0.0, 0.0);
            if (col < po && pr < pv) z = src[(long long)col * pv + pr];
            sre[ty + 8 * q][tx] = z.x; sim[ty + 8 * q][tx] = z.y;
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < UP_T / 8; ++q) {
            const int pr = r0 + ty + 8 * q, col = c0 + tx;
            if (col < po && pr < pv) {
                const double re = sre[tx][ty + 8 * q], im = sim[tx][ty + 8 * q];
                const int2 ef = vpairs[pr], ij = opairs[col];
                const int e = ef.x, f = ef.y;                       // e < f
                const long long ie = o1 + (long long)ij.x * v + e, jf = o1 + (long long)ij.y * v + f;
                const long long iff = o1 + (long long)ij.x * v + f, je = o1 + (long long)ij.y * v + e;
                const double tr = t1r[ie] * t1r[jf] - t1r[n1 + ie] * t1r[n1 + jf] - (t1r[iff] * t1r[je] - t1r[n1 + iff] * t1r[n1 + je]);
                const double ti = t1r[ie] * t1r[n1 + jf] + t1r[n1 + ie] * t1r[jf] - (t1r[iff] * t1r[n1 + je] + t1r[n1 + iff] * t1r[je]);
                const long long ra = ((long long)e * v + f) * 2 * po, rb = ((long long)f * v + e) * 2 * po;
                X[ra + col] = re; X[ra + po + col] = im;
                X[rb + col] = -re; X[rb + po + col] = -im;
                tau[ra + col] = re + tr; tau[ra + po + col] = im + ti;
                tau[rb + col] = -re - tr; tau[rb + po + col] = -im - ti;
                Xt[xt_index(e, f, col, nFt, ncol, nt2)] = re;
                Xt[xt_index(e, f, po + col, nFt, ncol, nt2)] = im;
                if (!anti) {
                    Xt[xt_index(f, e, col, nFt, ncol, nt2)] = -re;
                    Xt[xt_index(f, e, po + col, nFt, ncol, nt2)] = -im;
                }
            }
        }
    }
}

// Nq[Q][pl][(s,i,a)] = Mq + Lt[s][pl][Q][o+a][i]      (N^Q_ia = L~^Q_ai + M^Q_ia)
__global__ void k_add_Lvo(Dims d, const double* __restrict__ Lt0, const double* __restrict__ Lt1, const double* __restrict__ Mq, double* __restrict__ Nq)
{
    const long long tot = (long long)d.NQ * 2 * d.n1;
    const long long nn = (long long)d.n * d.n, plane = (long long)d.NQ * nn;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        long long Q = x / (2 * d.n1); int r = (int)(x - Q * 2 * d.n1);
        int pl = r >= d.n1; int c = pl ? r - d.n1 : r;
        int s = c >= d.n1a; int cc = s ? c - d.n1a : c;
        int i = cc / d.v[s], a = cc - i * d.v[s];
        const double* Lt = s ? Lt1 : Lt0;
        Nq[x] = Mq[x] + Lt[pl * plane + Q * nn + (long long)(d.o[s] + a) * d.n + i];
    }
}

// W[(m,e)][pl][(j,b)] += -1/2 delta_mj Fvv[b][e] + 1/2 delta_be Foo[m][j]
// (Fvv / Foo are the vv / oo blocks of the two dressed-Fock buffers; rows are (m of spin so, e of spin sv))
// Only columns with j in [jlo, jhi) are touched (a column slab of W holds those j; coff is then relative to the slab).
__global__ void k_add_Fd(int om, int ve, int n, const double* __restrict__ Fo, int oo_, const double* __restrict__ Fv, int ov_,
                         double* __restrict__ W, long long ldW, long long poff, long long roff, long long coff, int jlo, int jhi)
{
    // Fo: dressed Fock of the occupied index' spin (planar [2][n][n]), oo_ = its o; Fv likewise for the virtual index
    const long long nn = (long long)n * n;
    const long long tot1 = (long long)om * ve * ve, tot2 = (long long)om * om * ve;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot1 + tot2; x += (long long)gridDim.x * blockDim.x) {
        for (int pl = 0; pl < 2; ++pl) {
            if (x < tot1) {          // (m, e, b): j = m
                int m = (int)(x / ((long long)ve * ve)); int r = (int)(x - (long long)m * ve * ve);
                int e = r / ve, b = r - e * ve;
                if (m < jlo || m >= jhi) continue;
                double f = Fv[pl * nn + (long long)(ov_ + b) * n + ov_ + e];
                // b == e also gets the Foo[m][m] piece here so that each W element is touched by one thread only
                double add = -0.5 * f;
                if (b == e) add += 0.5 * Fo[pl * nn + (long long)m * n + m];
                W[(roff + (long long)m * ve + e) * ldW + pl * poff + coff + (long long)m * ve + b] += add;
            } else {                 // (m, j != m, e): b = e
                long long y = x - tot1;
                int m = (int)(y / ((long long)om * ve)); int r = (int)(y - (long long)m * om * ve);
                int j = r / ve, e = r - j * ve;
                if (j == m || j < jlo || j >= jhi) continue;
                double f = Fo[pl * nn + (long long)m * n + j];
                W[(roff + (long long)m * ve + e) * ldW + pl * poff + coff + (long long)j * ve + e] += 0.5 * f;
            }
        }
    }
}

// same-spin o^4 pieces: Wp[(m<n)][pl][(i<j)] = W4[(m,n)][(i,j)] - W4[(m,n)][(j,i)];  Yoop = rows (m,n) of Y
__global__ void k_ss_prep(int o, int po, int n, const int2* __restrict__ opairs, const double* __restrict__ W4,
                          const double* __restrict__ Y, double* __restrict__ Wp, double* __restrict__ Yoop)
{
    const long long tot = (long long)po * po;
    const int o2 = o * o;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        int r = (int)(x / po), c = (int)(x - (long long)r * po);
        int2 mn = opairs[r], ij = opairs[c];
        long long row = (long long)(mn.x * o + mn.y) * 2 * o2;
        for (int pl = 0; pl < 2; ++pl) {
            Wp[(long long)r * 2 * po + pl * po + c] = W4[row + pl * o2 + ij.x * o + ij.y] - W4[row + pl * o2 + ij.y * o + ij.x];
            Yoop[(long long)r * 2 * po + pl * po + c] = Y[((long long)mn.x * n + mn.y) * 2 * po + pl * po + c];
        }
    }
}

struct AsmArgs {
    const double *Zsc, *ZAB, *ZBA, *Yab, *Yss[2], *Zv[2], *r1buf, *Ft[2];
    const int2 *opairs[2], *vpairs[2];
    double *r1p, *r2p;
};

// residual in the packed boundary layout (interleaved complex):
//   r2 = P(ij)P(ab) Z + ladder pieces, r1 = r1buf + f~_ai
__global__ void k_assemble(Dims d, AsmArgs A)
{
    const long long nss0 = (long long)d.po[0] * d.pv[0], nss1 = (long long)d.po[1] * d.pv[1];
    const long long tot = d.n_t2 + d.n_t1;
    const long long ld = 2LL * d.n1;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        double out[2];
        if (x >= d.n_t2) {
            long long k = x - d.n_t2;
            int s = k >= d.n1a; int cc = (int)(s ? k - d.n1a : k);
            int i = cc / d.v[s], a = cc - i * d.v[s];
            const long long nn = (long long)d.n * d.n;
            for (int pl = 0; pl < 2; ++pl)
                out[pl] = A.r1buf[pl * (long long)d.n1 + k] + A.Ft[s][pl * nn + (long long)(d.o[s] + a) * d.n + i];
            A.r1p[2 * k] = out[0]; A.r1p[2 * k + 1] = out[1];
            continue;
        }
        if (x < nss0 + nss1) {
            int s = x >= nss0; long long k = s ? x - nss0 : x;
            int pij = (int)(k / d.pv[s]), pab = (int)(k - (long long)pij * d.pv[s]);
            int2 ij = A.opairs[s][pij], ab = A.vpairs[s][pab];
            const int v = d.v[s], po = d.po[s], o = d.o[s];
            const long long off = s ? d.n1a : 0;
            long long ia = off + ij.x * v + ab.x, jb = off + ij.y * v + ab.y, ja = off + ij.y * v + ab.x, ib = off + ij.x * v + ab.y;
            for (int pl = 0; pl < 2; ++pl) {
                long long p = pl * (long long)d.n1;
                double z = A.Zsc[ia * ld + p + jb] - A.Zsc[ja * ld + p + ib] - A.Zsc[ib * ld + p + ja] + A.Zsc[jb * ld + p + ia];
                z += A.Yss[s][((long long)(o + ab.x) * d.n + o + ab.y) * 2 * po + pl * po + pij];
                z += -A.Zv[s][((long long)ab.x * v + ab.y) * 2 * po + pl * po + pij] + A.Zv[s][((long long)ab.y * v + ab.x) * 2 * po + pl * po + pij];
                out[pl] = z;
            }
        } else {
            long long k = x - nss0 - nss1;
            int B = (int)(k % d.v[1]); k /= d.v[1];
            int a = (int)(k % d.v[0]); k /= d.v[0];
            int J = (int)(k % d.o[1]); int i = (int)(k / d.o[1]);
            long long ia = (long long)i * d.v[0] + a, JB = d.n1a + (long long)J * d.v[1] + B;
            long long iB = (long long)i * d.v[1] + B, Ja = (long long)J * d.v[0] + a;
            for (int pl = 0; pl < 2; ++pl) {
                double z = A.Zsc[ia * ld + pl * (long long)d.n1 + JB] + A.Zsc[JB * ld + pl * (long long)d.n1 + ia];
                z -= A.ZAB[iB * 2 * d.nB + pl * (long long)d.nB + Ja];
                z -= A.ZBA[Ja * 2 * d.nA + pl * (long long)d.nA + iB];
                z += A.Yab[((long long)(d.o[0] + a) * d.n + d.o[1] + B) * 2 * d.oo + pl * d.oo + i * d.o[1] + J];
                out[pl] = z;
            }
        }
        A.r2p[2 * x] = out[0]; A.r2p[2 * x + 1] = out[1];
    }
}

// Tiled assembly (north_star: "coalesced ... with shared-memory staging").  Every source of a residual element is contiguous
// in a DIFFERENT index (the pair-space matrices in the column's virtual index, the ladder output in the occupied pair), so a
// thread-per-element gather reads one 32-byte sector per 8 bytes used.  Here a CTA owns a 3-D tile, sweeps it once per
// contiguity class with the matching index fastest across the threads (full sectors), accumulates in shared memory, and
// writes the packed output with its own fastest index.  Summation order per element is fixed: bit-reproducible.
constexpr int AS_TJ = 8, AS_TA = 16, AS_TB = 16, AS_PB = AS_TB + 1;
// Each sweep first issues all of a thread's loads (AS_NIT independent 8-byte loads per source, kept in registers), then
// accumulates: the loads of a sweep are in flight together instead of one dependent round trip per element.
constexpr int AS_NIT = 2 * AS_TJ * AS_TA * AS_TB / 256;
// alpha-beta block: r2[i,J,a,B] = Zsc[ia,JB] + Zsc[JB,ia] - Z_AB[iB,Ja] - Z_BA[Ja,iB] + Y[(a,B)][(i,J)]
__global__ void __launch_bounds__(256) k_assemble_ab(Dims d, AsmArgs A)
{
    __shared__ double acc[2][AS_TJ][AS_TA][AS_PB];
    const int oa = d.o[0], ob = d.o[1], va = d.v[0], vb = d.v[1];
    const int nJt = (ob + AS_TJ - 1) / AS_TJ, nAt = (va + AS_TA - 1) / AS_TA, nBt = (vb + AS_TB - 1) / AS_TB;
    const long long ntile = (long long)oa * nJt * nAt * nBt;
    const long long ld = 2LL * d.n1, nss = (long long)d.po[0] * d.pv[0] + (long long)d.po[1] * d.pv[1];
    const long long n1 = d.n1, nA = d.nA, nB = d.nB, oo = d.oo;
    const int tid = threadIdx.x;
    const double* __restrict__ Zsc = A.Zsc;
    const double* __restrict__ ZAB = A.ZAB;
    const double* __restrict__ ZBA = A.ZBA;
    const double* __restrict__ Yab = A.Yab;
    for (long long t = blockIdx.x; t < ntile; t += gridDim.x) {
        long long k = t;
        const int B0 = (int)(k % nBt) * AS_TB; k /= nBt;
        const int a0 = (int)(k % nAt) * AS_TA; k /= nAt;
        const int J0 = (int)(k % nJt) * AS_TJ; const int i = (int)(k / nJt);
        double val[AS_NIT];
        __syncthreads();
        // class "B fastest": Zsc[ia,JB] - Z_BA[Ja,iB]
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            const int b = x % AS_TB, a = (x / AS_TB) % AS_TA, j = (x / (AS_TB * AS_TA)) % AS_TJ, pl = x / (AS_TB * AS_TA * AS_TJ);
            const int B = B0 + b, aa = a0 + a, J = J0 + j;
            double v = 0.0;
            if (B < vb && aa < va && J < ob) {
                const long long ia = (long long)i * va + aa, JB = d.n1a + (long long)J * vb + B, iB = (long long)i * vb + B, Ja = (long long)J * va + aa;
                v = Zsc[ia * ld + pl * n1 + JB] - ZBA[Ja * 2 * nA + pl * nA + iB];
            }
            val[it] = v;
        }
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            acc[x / (AS_TB * AS_TA * AS_TJ)][(x / (AS_TB * AS_TA)) % AS_TJ][(x / AS_TB) % AS_TA][x % AS_TB] = val[it];
        }
        __syncthreads();
        // class "a fastest": Zsc[JB,ia] - Z_AB[iB,Ja]
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            const int a = x % AS_TA, b = (x / AS_TA) % AS_TB, j = (x / (AS_TB * AS_TA)) % AS_TJ, pl = x / (AS_TB * AS_TA * AS_TJ);
            const int B = B0 + b, aa = a0 + a, J = J0 + j;
            double v = 0.0;
            if (B < vb && aa < va && J < ob) {
                const long long ia = (long long)i * va + aa, JB = d.n1a + (long long)J * vb + B, iB = (long long)i * vb + B, Ja = (long long)J * va + aa;
                v = Zsc[JB * ld + pl * n1 + ia] - ZAB[iB * 2 * nB + pl * nB + Ja];
            }
            val[it] = v;
        }
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            acc[x / (AS_TB * AS_TA * AS_TJ)][(x / (AS_TB * AS_TA)) % AS_TJ][x % AS_TA][(x / AS_TA) % AS_TB] += val[it];
        }
        __syncthreads();
        // class "J fastest": ladder output Y[(a,B)][(i,J)]
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            const int j = x % AS_TJ, b = (x / AS_TJ) % AS_TB, a = (x / (AS_TJ * AS_TB)) % AS_TA, pl = x / (AS_TB * AS_TA * AS_TJ);
            const int B = B0 + b, aa = a0 + a, J = J0 + j;
            double v = 0.0;
            if (B < vb && aa < va && J < ob)
                v = Yab[((long long)(oa + aa) * d.n + ob + B) * 2 * oo + pl * oo + (long long)i * ob + J];
            val[it] = v;
        }
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            acc[x / (AS_TB * AS_TA * AS_TJ)][x % AS_TJ][(x / (AS_TJ * AS_TB)) % AS_TA][(x / AS_TJ) % AS_TB] += val[it];
        }
        __syncthreads();
        // packed output, B fastest, (re, im) interleaved
        for (int x = tid; x < AS_TJ * AS_TA * AS_TB; x += 256) {
            const int b = x % AS_TB, a = (x / AS_TB) % AS_TA, j = x / (AS_TB * AS_TA);
            const int B = B0 + b, aa = a0 + a, J = J0 + j;
            if (B < vb && aa < va && J < ob) {
                const long long o = nss + (((long long)i * ob + J) * va + aa) * vb + B;
                reinterpret_cast<double2*>(A.r2p)[o] = make_double2(acc[0][j][a][b], acc[1][j][a][b]);
            }
        }
    }
}
// same-spin block of spin s: r2[(i<j),(a<b)] = Z[ia,jb] - Z[ja,ib] - Z[ib,ja] + Z[jb,ia] + Y[(a,b)][(ij)] - Zv[a][b][(ij)] + Zv[b][a][(ij)]
__global__ void __launch_bounds__(256) k_assemble_ss(Dims d, int s, AsmArgs A)
{
    __shared__ double acc[2][AS_TJ][AS_TA][AS_PB];
    const int o = d.o[s], v = d.v[s], po = d.po[s], pv = d.pv[s];
    const int nPt = (po + AS_TJ - 1) / AS_TJ, nAt = (v + AS_TA - 1) / AS_TA, nBt = (v + AS_TB - 1) / AS_TB;
    const long long ntile = (long long)nPt * nAt * nBt;
    const long long ld = 2LL * d.n1, n1 = d.n1, off = s ? d.n1a : 0, obase = s ? (long long)d.po[0] * d.pv[0] : 0;
    const int tid = threadIdx.x;
    const int2* __restrict__ op = A.opairs[s];
    const double* __restrict__ Zsc = A.Zsc;
    const double* __restrict__ Yss = A.Yss[s];
    const double* __restrict__ Zv = A.Zv[s];
    for (long long t = blockIdx.x; t < ntile; t += gridDim.x) {
        long long k = t;
        const int b0 = (int)(k % nBt) * AS_TB; k /= nBt;
        const int a0 = (int)(k % nAt) * AS_TA; const int p0 = (int)(k / nAt) * AS_TJ;
        if (a0 >= b0 + AS_TB) continue;                    // no a < b in this tile (block-uniform)
        double val[AS_NIT];
        __syncthreads();
        // class "b fastest": Z[ia,jb] - Z[ja,ib]
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            const int b = x % AS_TB, a = (x / AS_TB) % AS_TA, j = (x / (AS_TB * AS_TA)) % AS_TJ, pl = x / (AS_TB * AS_TA * AS_TJ);
            const int bb = b0 + b, aa = a0 + a, pij = p0 + j;
            double w = 0.0;
            if (aa < bb && bb < v && pij < po) {
                const int2 ij = op[pij];
                const long long ia = off + (long long)ij.x * v + aa, jb = off + (long long)ij.y * v + bb, ja = off + (long long)ij.y * v + aa, ib = off + (long long)ij.x * v + bb;
                w = Zsc[ia * ld + pl * n1 + jb] - Zsc[ja * ld + pl * n1 + ib];
            }
            val[it] = w;
        }
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            acc[x / (AS_TB * AS_TA * AS_TJ)][(x / (AS_TB * AS_TA)) % AS_TJ][(x / AS_TB) % AS_TA][x % AS_TB] = val[it];
        }
        __syncthreads();
        // class "a fastest": - Z[ib,ja] + Z[jb,ia]
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            const int a = x % AS_TA, b = (x / AS_TA) % AS_TB, j = (x / (AS_TB * AS_TA)) % AS_TJ, pl = x / (AS_TB * AS_TA * AS_TJ);
            const int bb = b0 + b, aa = a0 + a, pij = p0 + j;
            double w = 0.0;
            if (aa < bb && bb < v && pij < po) {
                const int2 ij = op[pij];
                const long long ia = off + (long long)ij.x * v + aa, jb = off + (long long)ij.y * v + bb, ja = off + (long long)ij.y * v + aa, ib = off + (long long)ij.x * v + bb;
                w = -Zsc[ib * ld + pl * n1 + ja] + Zsc[jb * ld + pl * n1 + ia];
            }
            val[it] = w;
        }
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            acc[x / (AS_TB * AS_TA * AS_TJ)][(x / (AS_TB * AS_TA)) % AS_TJ][x % AS_TA][(x / AS_TA) % AS_TB] += val[it];
        }
        __syncthreads();
        // class "pair (ij) fastest": ladder output and its T1 corrections
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            const int j = x % AS_TJ, b = (x / AS_TJ) % AS_TB, a = (x / (AS_TJ * AS_TB)) % AS_TA, pl = x / (AS_TB * AS_TA * AS_TJ);
            const int bb = b0 + b, aa = a0 + a, pij = p0 + j;
            double w = 0.0;
            if (aa < bb && bb < v && pij < po) {
                const long long c = pl * (long long)po + pij;
                w = Yss[((long long)(o + aa) * d.n + o + bb) * 2 * po + c] - Zv[((long long)aa * v + bb) * 2 * po + c] + Zv[((long long)bb * v + aa) * 2 * po + c];
            }
            val[it] = w;
        }
#pragma unroll
        for (int it = 0; it < AS_NIT; ++it) {
            const int x = tid + it * 256;
            acc[x / (AS_TB * AS_TA * AS_TJ)][x % AS_TJ][(x / (AS_TJ * AS_TB)) % AS_TA][(x / AS_TJ) % AS_TB] += val[it];
        }
        __syncthreads();
        // packed output: pair(a,b) = b(b-1)/2 + a, a fastest
        for (int x = tid; x < AS_TJ * AS_TA * AS_TB; x += 256) {
            const int a = x % AS_TA, b = (x / AS_TA) % AS_TB, j = x / (AS_TB * AS_TA);
            const int bb = b0 + b, aa = a0 + a, pij = p0 + j;
            if (aa < bb && bb < v && pij < po) {
                const long long ox = obase + (long long)pij * pv + pair_index(aa, bb);
                reinterpret_cast<double2*>(A.r2p)[ox] = make_double2(acc[0][j][a][b], acc[1][j][a][b]);
            }
        }
    }
}
// singles: r1 = r1buf + f~_ai
__global__ void k_assemble_r1(Dims d, AsmArgs A)
{
    const long long nn = (long long)d.n * d.n;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < d.n_t1; k += (long long)gridDim.x * blockDim.x) {
        const int s = k >= d.n1a; const int cc = (int)(s ? k - d.n1a : k);
        const int i = cc / d.v[s], a = cc - i * d.v[s];
        A.r1p[2 * k] = A.r1buf[k] + A.Ft[s][(long long)(d.o[s] + a) * d.n + i];
        A.r1p[2 * k + 1] = A.r1buf[d.n1 + k] + A.Ft[s][nn + (long long)(d.o[s] + a) * d.n + i];
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Low-memory ("lean") pipeline: BASELINE.json config 5 does not fit 180 GB with the pair-space matrices held whole
// (Table 2: the paper's storage argument is three amplitude-sized tensors plus the Cholesky
// vectors).  There the same-spin pair-space blocks are the only unpacked amplitudes, the alpha-beta block is read in place
// from the packed boundary layout through strides, the ring intermediates W and Z live in column slabs that are folded
// into the packed residual slab by slab, and the ladder's buffers reuse the memory of the ring phase.

// Tss[(i,a)][pl][(m,e)] = t_{im}^{ae} for one spin (planar, n1s x 2 n1s)
__global__ void k_build_Tss(Dims d, int s, const double* __restrict__ t2p, double* __restrict__ T)
{
    const int v = d.v[s];
    const long long n1s = (long long)d.o[s] * v, tot = n1s * n1s;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        const long long r = x / n1s, c = x - r * n1s;
        const int i = (int)(r / v), a = (int)(r - (long long)i * v), m = (int)(c / v), e = (int)(c - (long long)m * v);
        c128 z = ss_amp(t2p, d.off_t2[s], d.pv[s], i, m, a, e);
        T[r * 2 * n1s + c] = z.re;
        T[r * 2 * n1s + n1s + c] = z.im;
    }
}

// tile-major ladder amplitudes only (no planar copy, no tau): alpha-beta and same-spin
__global__ void k_build_Xt_ab(Dims d, const double* __restrict__ t2p, double* __restrict__ Xt, int nFt, int ncol, int nt2)
{
    const long long tot = (long long)d.v[0] * d.v[1] * d.oo;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        // x runs over the packed order (i, J, e, F) so that the reads are contiguous
        const long long vv = (long long)d.v[0] * d.v[1];
        const int col = (int)(x / vv); const long long ef = x - (long long)col * vv;
        const int e = (int)(ef / d.v[1]), F = (int)(ef - (long long)e * d.v[1]);
        const long long k = d.off_t2[2] + x;
        Xt[xt_index(e, F, col, nFt, ncol, nt2)] = t2p[2 * k];
        Xt[xt_index(e, F, d.oo + col, nFt, ncol, nt2)] = t2p[2 * k + 1];
    }
}
__global__ void k_build_Xt_ss(Dims d, int s, const double* __restrict__ t2p, const int2* __restrict__ opairs, double* __restrict__ Xt, int nFt, int ncol, int nt2, int anti)
{
    const int v = d.v[s], po = d.po[s];
    const long long tot = (long long)v * v * po;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        const long long row = x / po; const int col = (int)(x - row * po);
        const int e = (int)(row / v), f = (int)(row - (long long)e * v);
        const int2 ij = opairs[col];
        if (anti && e >= f) continue;         // antisymmetrised ladder: those rows stay zero
        c128 z = ss_amp(t2p, d.off_t2[s], d.pv[s], ij.x, ij.y, e, f);
        Xt[xt_index(e, f, col, nFt, ncol, nt2)] = z.re;
        Xt[xt_index(e, f, po + col, nFt, ncol, nt2)] = z.im;
    }
}

// V[(m,N)][pl][(i,J)] = Woo[(m,N)][pl][(i,J)] + Y[(m, N) row of the all-orbital ladder output][pl][(i,J)]   (alpha-beta o^4 pieces)
__global__ void k_add_oo_rows(int oa, int ob, int n, long long oo, const double* __restrict__ Woo, const double* __restrict__ Y, double* __restrict__ V)
{
    const long long tot = oo * 2 * oo;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        const long long r = x / (2 * oo), c = x - r * 2 * oo;
        const int m = (int)(r / ob), N = (int)(r - (long long)m * ob);
        V[x] = Woo[x] + Y[((long long)m * n + N) * 2 * oo + c];
    }
}
// same spin: Vp[(m<n)][pl][(i<j)] = W4 antisymmetrised + Y rows (m,n);  Yoo[(m,n)][pl][(i<j)] = antisymmetric unpacking of the Y rows (m<n)
__global__ void k_ss_prep_lean(int o, int po, int n, const int2* __restrict__ opairs, const double* __restrict__ W4,
                               const double* __restrict__ Y, double* __restrict__ Vp, double* __restrict__ Yoo)
{
    const long long tot = (long long)po * po;
    const int o2 = o * o;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(x / po), c = (int)(x - (long long)r * po);
        const int2 mn = opairs[r], ij = opairs[c];
        const long long row = (long long)(mn.x * o + mn.y) * 2 * o2;
        for (int pl = 0; pl < 2; ++pl) {
            const double y = Y[((long long)mn.x * n + mn.y) * 2 * po + pl * po + c];
            Vp[(long long)r * 2 * po + pl * po + c] = W4[row + pl * o2 + ij.x * o + ij.y] - W4[row + pl * o2 + ij.y * o + ij.x] + y;
            Yoo[((long long)mn.x * o + mn.y) * 2 * po + pl * po + c] = y;
            Yoo[((long long)mn.y * o + mn.x) * 2 * po + pl * po + c] = -y;
        }
    }
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < (long long)o * 2 * po; x += (long long)gridDim.x * blockDim.x) {
        const int m = (int)(x / (2 * po)); const long long c = x - (long long)m * 2 * po;
        Yoo[((long long)m * o + m) * 2 * po + c] = 0.0;
    }
}
// offsets of the ladder-output rows (o+a, o+b), a < b, by packed virtual pair index
__global__ void k_pair_row_table(int o, int n, int pv, long long ld, const int2* __restrict__ vpairs, long long* __restrict__ tab)
{
    for (int x = blockIdx.x * blockDim.x + threadIdx.x; x < pv; x += gridDim.x * blockDim.x) {
        const int2 ab = vpairs[x];
        tab[x] = ((long long)(o + ab.x) * n + o + ab.y) * ld;
    }
}

// Fold one slab of a ring intermediate into the packed residual:  r2 (+)= signed sum of the slab's elements each packed
// element depends on.  kind 0/1: columns (j,b) of spin kind with j in [j0, j1) of Z_sc (rows: all n1 pairs);
// kind 2: Z_AB[(i,B),(J,a)] whole, kind 3: Z_BA[(J,a),(i,B)] whole (both subtracted from the alpha-beta block).
// Z is planar with row pitch 2*wc (wc = columns held).  Every packed element is owned by one thread: no atomics.
__global__ void k_fold_slab(Dims d, int kind, int j0, int j1, const double* __restrict__ Z, long long wc,
                            const int2* __restrict__ op, const int2* __restrict__ vp, double* __restrict__ r2p)
{
    const long long nss0 = (long long)d.po[0] * d.pv[0], nss1 = (long long)d.po[1] * d.pv[1];
    const long long nab = (long long)d.oo * d.v[0] * d.v[1];
    const long long ld = 2 * wc;
    if (kind <= 1) {
        const int s = kind, v = d.v[s];
        const long long rbase = s ? d.n1a : 0;          // row offset of spin-s pairs in the n1 rows
        const long long c0 = (long long)j0 * v;
        // same-spin block of spin s: Z[ia,jb] - Z[ja,ib] - Z[ib,ja] + Z[jb,ia]
        const long long nss = s ? nss1 : nss0, off = s ? nss0 : 0;
        for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < nss; x += (long long)gridDim.x * blockDim.x) {
            const int pij = (int)(x / d.pv[s]), pab = (int)(x - (long long)pij * d.pv[s]);
            const int2 ij = op[pij], ab = vp[pab];
            double re = 0.0, im = 0.0;
            bool any = false;
            // terms (row occupied, row virtual, column occupied, column virtual, sign)
            const int t[4][5] = {{ij.x, ab.x, ij.y, ab.y, 1}, {ij.y, ab.x, ij.x, ab.y, -1}, {ij.x, ab.y, ij.y, ab.x, -1}, {ij.y, ab.y, ij.x, ab.x, 1}};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (t[k][2] >= j0 && t[k][2] < j1) {
                    const long long row = rbase + (long long)t[k][0] * v + t[k][1], col = (long long)t[k][2] * v + t[k][3] - c0;
                    re += t[k][4] * Z[row * ld + col]; im += t[k][4] * Z[row * ld + wc + col];
                    any = true;
                }
            }
            if (any) { r2p[2 * (off + x)] += re; r2p[2 * (off + x) + 1] += im; }
        }
        // alpha-beta block: Z[ia,JB] (column beta) or Z[JB,ia] (column alpha)
        for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < nab; x += (long long)gridDim.x * blockDim.x) {
            long long k = x;
            const int B = (int)(k % d.v[1]); k /= d.v[1];
            const int a = (int)(k % d.v[0]); k /= d.v[0];
            const int J = (int)(k % d.o[1]); const int i = (int)(k / d.o[1]);
            long long row, col; int jc;
            if (s == 1) { row = (long long)i * d.v[0] + a; col = (long long)J * d.v[1] + B; jc = J; }
            else { row = d.n1a + (long long)J * d.v[1] + B; col = (long long)i * d.v[0] + a; jc = i; }
            if (jc < j0 || jc >= j1) continue;
            col -= c0;
            r2p[2 * (nss0 + nss1 + x)] += Z[row * ld + col];
            r2p[2 * (nss0 + nss1 + x) + 1] += Z[row * ld + wc + col];
        }
    } else {
        for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < nab; x += (long long)gridDim.x * blockDim.x) {
            long long k = x;
            const int B = (int)(k % d.v[1]); k /= d.v[1];
            const int a = (int)(k % d.v[0]); k /= d.v[0];
            const int J = (int)(k % d.o[1]); const int i = (int)(k / d.o[1]);
            const long long iB = (long long)i * d.v[1] + B, Ja = (long long)J * d.v[0] + a;
            const long long row = kind == 2 ? iB : Ja, col = kind == 2 ? Ja : iB;
            r2p[2 * (nss0 + nss1 + x)] -= Z[row * ld + col];
            r2p[2 * (nss0 + nss1 + x) + 1] -= Z[row * ld + wc + col];
        }
    }
}

// last pass of the lean assembly: r2 += ladder pieces (the T1 and o^4 corrections are already inside Y), r1 = r1buf + f~_ai
__global__ void k_fold_ladder(Dims d, AsmArgs A)
{
    const long long nss0 = (long long)d.po[0] * d.pv[0], nss1 = (long long)d.po[1] * d.pv[1];
    const long long tot = d.n_t2 + d.n_t1;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        if (x >= d.n_t2) {
            const long long k = x - d.n_t2;
            const int s = k >= d.n1a; const int cc = (int)(s ? k - d.n1a : k);
            const int i = cc / d.v[s], a = cc - i * d.v[s];
            const long long nn = (long long)d.n * d.n;
            for (int pl = 0; pl < 2; ++pl)
                A.r1p[2 * k + pl] = A.r1buf[pl * (long long)d.n1 + k] + A.Ft[s][pl * nn + (long long)(d.o[s] + a) * d.n + i];
            continue;
        }
        if (x < nss0 + nss1) {
            const int s = x >= nss0; const long long k = s ? x - nss0 : x;
            const int pij = (int)(k / d.pv[s]), pab = (int)(k - (long long)pij * d.pv[s]);
            const int2 ab = A.vpairs[s][pab];
            const int po = d.po[s], o = d.o[s];
            for (int pl = 0; pl < 2; ++pl)
                A.r2p[2 * x + pl] += A.Yss[s][((long long)(o + ab.x) * d.n + o + ab.y) * 2 * po + pl * po + pij];
        } else {
            long long k = x - nss0 - nss1;
            const int B = (int)(k % d.v[1]); k /= d.v[1];
            const int a = (int)(k % d.v[0]); k /= d.v[0];
            const int J = (int)(k % d.o[1]); const int i = (int)(k / d.o[1]);
            for (int pl = 0; pl < 2; ++pl)
                A.r2p[2 * x + pl] += A.Yab[((long long)(d.o[0] + a) * d.n + d.o[1] + B) * 2 * d.oo + pl * d.oo + i * d.o[1] + J];
        }
    }
}

// ---------------------------------------------------------------- reductions (deterministic)
constexpr int RED_BLOCKS = 296, RED_THREADS = 256;

__device__ __forceinline__ double block_sum(double v, double* sh)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) for (int i = 0; i < (int)(blockDim.x >> 5); ++i) r += sh[i];
    return r;      // valid on thread 0
}
__device__ __forceinline__ double block_max(double v, double* sh)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) for (int i = 0; i < (int)(blockDim.x >> 5); ++i) r = fmax(r, sh[i]);
    return r;
}

// Fused T1 dressing for problems whose n x n Cholesky slice fits in shared memory (one CTA per Cholesky vector, both
// spins):  L~^Q = (1 - T) L^Q (1 + T)  and  gamma^Q = sum_s sum_ie L^Q_ie t_i^e.  Replaces the
// copy + two skinny GEMMs per spin of the general path; same arithmetic, fixed summation order.
struct DressArgs { const double* L[2]; double* Lt[2]; const double* t1r; double* gam; };
__global__ void __launch_bounds__(256) k_dress(Dims d, DressArgs A)
{
    extern __shared__ double sm[];
    const int n = d.n, ld = n | 1, Q = blockIdx.x, tid = threadIdx.x;
    const long long nn = (long long)n * n, plane = (long long)d.NQ * nn;
    __shared__ double red[32];
    double gr = 0.0, gi = 0.0;
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = s ? d.n1a : 0;
        double* Ls = sm;                       // [n][ld]
        double* tr = Ls + (size_t)n * ld;      // [o][v]
        double* ti = tr + (size_t)o * v;
        double* Br = ti + (size_t)o * v;       // [n][o]   (L T)[p][i] = sum_e L[p][o+e] t_i^e
        double* Bi = Br + (size_t)n * o;
        __syncthreads();
        const double* Lg = A.L[s] + Q * nn;
        for (int x = tid; x < n * n; x += 256) Ls[(x / n) * ld + x % n] = Lg[x];
        for (int x = tid; x < o * v; x += 256) { tr[x] = A.t1r[off1 + x]; ti[x] = A.t1r[d.n1 + off1 + x]; }
        __syncthreads();
        for (int x = tid; x < n * o; x += 256) {
            const int p = x / o, i = x - p * o;
            double ar = 0.0, ai = 0.0;
            for (int e = 0; e < v; ++e) { const double l = Ls[p * ld + o + e]; ar += l * tr[i * v + e]; ai += l * ti[i * v + e]; }
            Br[x] = ar; Bi[x] = ai;
        }
        for (int x = tid; x < o * v; x += 256) { const int i = x / v, e = x - i * v; const double l = Ls[i * ld + o + e]; gr += l * tr[x]; gi += l * ti[x]; }
        __syncthreads();
        double* Or = A.Lt[s] + Q * nn;
        double* Oi = Or + plane;
        for (int x = tid; x < n * n; x += 256) {
            const int p = x / n, q = x - p * n;
            double vr = Ls[p * ld + q], vi = 0.0;
            if (q < o) { vr += Br[p * o + q]; vi = Bi[p * o + q]; }
            if (p >= o) {                      // row a: subtract sum_m t_m^a (L Y)[m][q]
                const int a = p - o;
                for (int m = 0; m < o; ++m) {
                    double yr = Ls[m * ld + q], yi = 0.0;
                    if (q < o) { yr += Br[m * o + q]; yi = Bi[m * o + q]; }
                    const double xr = tr[m * v + a], xi = ti[m * v + a];
                    vr -= xr * yr - xi * yi;
                    vi -= xr * yi + xi * yr;
                }
            }
            Or[x] = vr; Oi[x] = vi;
        }
    }
    const double a = block_sum(gr, red);
    const double b = block_sum(gi, red);
    if (tid == 0) { A.gam[Q] = a; A.gam[d.NQ + Q] = b; }
}
inline size_t dress_smem(const Dims& d)
{
    size_t m = 0;
    for (int s = 0; s < 2; ++s) {
        size_t x = (size_t)d.n * (d.n | 1) + 2 * (size_t)d.o[s] * d.v[s] + 2 * (size_t)d.n * d.o[s];
        if (x > m) m = x;
    }
    return m * sizeof(double);
}

// ---------------------------------------------------------------------------------------------------------------
// Fused small-problem kernels for the dressed Fock matrix, the F intermediates and the singles (SURVEY.md 8(a) a2, a6,
// a7): sums over the Cholesky index are split into NCH chunks (one CTA each, fixed order inside), the chunk partials
// are added in fixed order by k_reduce_chunks, and a one-CTA-per-spin kernel finishes.  Same arithmetic as the tcgemm
// path they replace; used when the per-thread element counts fit (FUSE_MAXE).
constexpr int FUSE_T = 512, FUSE_MAXE = 12;

__global__ void k_reduce_chunks(const double* __restrict__ in, double* __restrict__ out, int nchunk, long long len)
{
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < len; x += (long long)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int c = 0; c < nchunk; ++c) s += in[c * len + x];
        out[x] = s;
    }
}

// part[chunk][s][0..3][n*n]: J = sum_Q gamma^Q L^Q (re, im),  Ex = sum_Q sum_i L~^Q_pi L~^Q_iq (re, im)
__global__ void __launch_bounds__(FUSE_T) k_fock_partial(Dims d, const double* __restrict__ L0, const double* __restrict__ L1,
                                                         const double* __restrict__ Lt0, const double* __restrict__ Lt1,
                                                         const double* __restrict__ gam, int nch, double* __restrict__ part)
{
    extern __shared__ double sm[];
    const int s = blockIdx.y, c = blockIdx.x, tid = threadIdx.x;
    const int n = d.n, o = d.o[s];
    const long long nn = (long long)n * n, plane = (long long)d.NQ * nn;
    const double* L = s ? L1 : L0;
    const double* Lt = s ? Lt1 : Lt0;
    double* Ar = sm;                 // L~[p][i]   [n][o]
    double* Ai = Ar + n * o;
    double* Br = Ai + n * o;         // L~[i][q]   [o][n]
    double* Bi = Br + o * n;
    double jr[FUSE_MAXE], ji[FUSE_MAXE], xr[FUSE_MAXE], xi[FUSE_MAXE];
#pragma unroll
    for (int k = 0; k < FUSE_MAXE; ++k) jr[k] = ji[k] = xr[k] = xi[k] = 0.0;
    const int Q0 = (int)((long long)c * d.NQ / nch), Q1 = (int)((long long)(c + 1) * d.NQ / nch);
    for (int Q = Q0; Q < Q1; ++Q) {
        __syncthreads();
        for (int x = tid; x < n * o; x += FUSE_T) {
            const int p = x / o, i = x - p * o;
            Ar[x] = Lt[Q * nn + (long long)p * n + i]; Ai[x] = Lt[plane + Q * nn + (long long)p * n + i];
        }
        for (int x = tid; x < o * n; x += FUSE_T) { Br[x] = Lt[Q * nn + x]; Bi[x] = Lt[plane + Q * nn + x]; }
        __syncthreads();
        const double gr = gam[Q], gi = gam[d.NQ + Q];
#pragma unroll
        for (int k = 0; k < FUSE_MAXE; ++k) {
            const int e = tid + k * FUSE_T;
            if (e < nn) {
                const int p = e / n, q = e - p * n;
                const double l = L[Q * nn + e];
                jr[k] += gr * l; ji[k] += gi * l;
                double ar = 0.0, ai = 0.0;
                for (int i = 0; i < o; ++i) {
                    const double pr = Ar[p * o + i], pi = Ai[p * o + i], qr = Br[i * n + q], qi = Bi[i * n + q];
                    ar += pr * qr - pi * qi; ai += pr * qi + pi * qr;
                }
                xr[k] += ar; xi[k] += ai;
            }
        }
    }
    double* out = part + ((long long)c * 2 + s) * 4 * nn;
#pragma unroll
    for (int k = 0; k < FUSE_MAXE; ++k) {
        const int e = tid + k * FUSE_T;
        if (e < nn) { out[e] = jr[k]; out[nn + e] = ji[k]; out[2 * nn + e] = xr[k]; out[3 * nn + e] = xi[k]; }
    }
}

// f~ = X (Fb + J) Y - Ex   from the reduced sums red[s][0..3][n*n]; writes the planar Ft[s]
struct FockFinishArgs { const double* Fb[2]; double* Ft[2]; const double* red; const double* t1r; };
__global__ void __launch_bounds__(FUSE_T) k_fock_finish(Dims d, FockFinishArgs A)
{
    extern __shared__ double sm[];
    const int s = blockIdx.x, tid = threadIdx.x;
    const int n = d.n, o = d.o[s], v = d.v[s];
    const long long nn = (long long)n * n, off1 = s ? d.n1a : 0;
    double* Fr = sm;                 // F0 = Fb + J   [n][n]
    double* Fi = Fr + nn;
    double* tr = Fi + nn;            // [o][v]
    double* ti = tr + o * v;
    double* Gr = ti + o * v;         // (F0 T)[p][i]  [n][o]
    double* Gi = Gr + n * o;
    const double* red = A.red + (long long)s * 4 * nn;
    for (int x = tid; x < nn; x += FUSE_T) { Fr[x] = A.Fb[s][x] + red[x]; Fi[x] = red[nn + x]; }
    for (int x = tid; x < o * v; x += FUSE_T) { tr[x] = A.t1r[off1 + x]; ti[x] = A.t1r[d.n1 + off1 + x]; }
    __syncthreads();
    for (int x = tid; x < n * o; x += FUSE_T) {
        const int p = x / o, i = x - p * o;
        double ar = 0.0, ai = 0.0;
        for (int e = 0; e < v; ++e) {
            const double fr = Fr[p * n + o + e], fi = Fi[p * n + o + e], xr = tr[i * v + e], xi = ti[i * v + e];
            ar += fr * xr - fi * xi; ai += fr * xi + fi * xr;
        }
        Gr[x] = ar; Gi[x] = ai;
    }
    __syncthreads();
    for (int x = tid; x < n * o; x += FUSE_T) { const int p = x / o, i = x - p * o; Fr[p * n + i] += Gr[x]; Fi[p * n + i] += Gi[x]; }
    __syncthreads();
    double* Or = A.Ft[s];
    double* Oi = Or + nn;
    for (int x = tid; x < nn; x += FUSE_T) {
        const int p = x / n, q = x - p * n;
        double vr = Fr[x], vi = Fi[x];
        if (p >= o) {
            const int a = p - o;
            for (int m = 0; m < o; ++m) {
                const double xr = tr[m * v + a], xi = ti[m * v + a], yr = Fr[m * n + q], yi = Fi[m * n + q];
                vr -= xr * yr - xi * yi; vi -= xr * yi + xi * yr;
            }
        }
        Or[x] = vr - red[2 * nn + x]; Oi[x] = vi - red[3 * nn + x];
    }
}

// part[chunk][s][pl][SZ]:  [0, v*v): -sum_Q,m L_me M_ma  (a,e);  then o*o: +sum_Q,e L_me M_ie (m,i);
//                          then o*v: -sum_Q,n M_na L~_ni + sum_Q,f M_if L~_af  (i,a)
__global__ void __launch_bounds__(FUSE_T) k_postm_partial(Dims d, const double* __restrict__ L0, const double* __restrict__ L1,
                                                          const double* __restrict__ Lt0, const double* __restrict__ Lt1,
                                                          const double* __restrict__ Mq, int nch, long long SZ, double* __restrict__ part)
{
    extern __shared__ double sm[];
    const int s = blockIdx.y, c = blockIdx.x, tid = threadIdx.x;
    const int n = d.n, o = d.o[s], v = d.v[s];
    const long long nn = (long long)n * n, plane = (long long)d.NQ * nn, off1 = s ? d.n1a : 0, ld1 = 2LL * d.n1;
    const double* L = s ? L1 : L0;
    const double* Lt = s ? Lt1 : Lt0;
    double* Lov = sm;                    // [o][v]
    double* Mr = Lov + o * v;            // [o][v]
    double* Mi = Mr + o * v;
    double* Or_ = Mi + o * v;            // L~oo [o][o]
    double* Oi_ = Or_ + o * o;
    double* Vr = Oi_ + o * o;            // L~vv [v][v]
    double* Vi = Vr + v * v;
    double far_[FUSE_MAXE], fai[FUSE_MAXE], fmr = 0.0, fmi = 0.0, r1r[2] = {0.0, 0.0}, r1i[2] = {0.0, 0.0};
#pragma unroll
    for (int k = 0; k < FUSE_MAXE; ++k) far_[k] = fai[k] = 0.0;
    const int Q0 = (int)((long long)c * d.NQ / nch), Q1 = (int)((long long)(c + 1) * d.NQ / nch);
    for (int Q = Q0; Q < Q1; ++Q) {
        __syncthreads();
        for (int x = tid; x < o * v; x += FUSE_T) {
            const int m = x / v, e = x - m * v;
            Lov[x] = L[Q * nn + (long long)m * n + o + e];
            Mr[x] = Mq[Q * ld1 + off1 + x]; Mi[x] = Mq[Q * ld1 + d.n1 + off1 + x];
        }
        for (int x = tid; x < o * o; x += FUSE_T) {
            const int m = x / o, i = x - m * o;
            Or_[x] = Lt[Q * nn + (long long)m * n + i]; Oi_[x] = Lt[plane + Q * nn + (long long)m * n + i];
        }
        for (int x = tid; x < v * v; x += FUSE_T) {
            const int a = x / v, f = x - a * v;
            Vr[x] = Lt[Q * nn + (long long)(o + a) * n + o + f]; Vi[x] = Lt[plane + Q * nn + (long long)(o + a) * n + o + f];
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < FUSE_MAXE; ++k) {
            const int x = tid + k * FUSE_T;
            if (x < v * v) {
                const int a = x / v, e = x - a * v;
                double ar = 0.0, ai = 0.0;
                for (int m = 0; m < o; ++m) { const double l = Lov[m * v + e]; ar += l * Mr[m * v + a]; ai += l * Mi[m * v + a]; }
                far_[k] -= ar; fai[k] -= ai;
            }
        }
        if (tid < o * o) {
            const int m = tid / o, i = tid - m * o;
            double ar = 0.0, ai = 0.0;
            for (int e = 0; e < v; ++e) { const double l = Lov[m * v + e]; ar += l * Mr[i * v + e]; ai += l * Mi[i * v + e]; }
            fmr += ar; fmi += ai;
        }
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const int x = tid + k * FUSE_T;
            if (x < o * v) {
                const int i = x / v, a = x - i * v;
                double ar = 0.0, ai = 0.0;
                for (int m = 0; m < o; ++m) {
                    const double mr = Mr[m * v + a], mi = Mi[m * v + a], lr = Or_[m * o + i], li = Oi_[m * o + i];
                    ar -= mr * lr - mi * li; ai -= mr * li + mi * lr;
                }
                for (int f = 0; f < v; ++f) {
                    const double mr = Mr[i * v + f], mi = Mi[i * v + f], lr = Vr[a * v + f], li = Vi[a * v + f];
                    ar += mr * lr - mi * li; ai += mr * li + mi * lr;
                }
                r1r[k] += ar; r1i[k] += ai;
            }
        }
    }
    double* out = part + ((long long)c * 2 + s) * 2 * SZ;
#pragma unroll
    for (int k = 0; k < FUSE_MAXE; ++k) {
        const int x = tid + k * FUSE_T;
        if (x < v * v) { out[x] = far_[k]; out[SZ + x] = fai[k]; }
    }
    if (tid < o * o) { out[v * v + tid] = fmr; out[SZ + v * v + tid] = fmi; }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const int x = tid + k * FUSE_T;
        if (x < o * v) { out[v * v + o * o + x] = r1r[k]; out[SZ + v * v + o * o + x] = r1i[k]; }
    }
}

// Ft vv += F_ae part, Ft oo += F_mi part, r1buf += singles part   (red[s][pl][SZ])
__global__ void k_postm_finish(Dims d, const double* __restrict__ red, long long SZ, double* __restrict__ Ft0, double* __restrict__ Ft1,
                               double* __restrict__ r1buf)
{
    const int n = d.n;
    const long long nn = (long long)n * n;
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = s ? d.n1a : 0;
        double* Ft = s ? Ft1 : Ft0;
        const long long tot = (long long)v * v + o * o + o * v;
        for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < 2 * tot; x += (long long)gridDim.x * blockDim.x) {
            const int pl = x >= tot; const long long y = pl ? x - tot : x;
            const double val = red[((long long)s * 2 + pl) * SZ + y];
            if (y < (long long)v * v) { const int a = (int)(y / v), e = (int)(y - (long long)a * v); Ft[pl * nn + (long long)(o + a) * n + o + e] += val; }
            else if (y < (long long)v * v + o * o) { const long long z = y - (long long)v * v; const int m = (int)(z / o), i = (int)(z - (long long)m * o); Ft[pl * nn + (long long)m * n + i] += val; }
            else { const long long z = y - (long long)v * v - o * o; r1buf[pl * (long long)d.n1 + off1 + z] += val; }
        }
    }
}

// r1buf[x] = sum_(s,m,e) Tsc[x][(m,e)] f~_me     (one warp per row; complex x complex)
__global__ void __launch_bounds__(256) k_tsc_matvec(Dims d, const double* __restrict__ Tsc, const double* __restrict__ Ft0,
                                                     const double* __restrict__ Ft1, double* __restrict__ r1buf)
{
    const int n = d.n, n1 = d.n1, lane = threadIdx.x & 31;
    const long long nn = (long long)n * n;
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (row >= n1) return;
    const double* Tr = Tsc + (long long)row * 2 * n1;
    const double* Ti = Tr + n1;
    double ar = 0.0, ai = 0.0;
    for (int c = lane; c < n1; c += 32) {
        const int s = c >= d.n1a; const int cc = s ? c - d.n1a : c;
        const int m = cc / d.v[s], e = cc - m * d.v[s];
        const double* F = s ? Ft1 : Ft0;
        const double fr = F[(long long)m * n + d.o[s] + e], fi = F[nn + (long long)m * n + d.o[s] + e];
        const double tr = Tr[c], ti = Ti[c];
        ar += tr * fr - ti * fi; ai += tr * fi + ti * fr;
    }
    for (int o = 16; o > 0; o >>= 1) { ar += __shfl_down_sync(0xffffffffu, ar, o); ai += __shfl_down_sync(0xffffffffu, ai, o); }
    if (lane == 0) { r1buf[row] = ar; r1buf[n1 + row] = ai; }
}

struct EnergyArgs {
    const double* L[2]; const double* Lt[2]; const double* fock[2];   // bare vectors, dressed vectors (planar), bare Fock
    const double* t1r; const double* Mq; const double* gam; double* partial;   // partial[RED_BLOCKS][2]
    unsigned* counter; double* out;                                             // last block: out[0..1] = sum of the partials
};

// E = sum f_ia t_i^a + 1/2 [ sum_Q,ia L_ia M_ia + sum_Q gamma_Q^2 - sum_s sum_Q,ij U_ji U_ij ],  U = L~_oo - L_oo
// (Eq. 5 integrand PAPER.md:58).  Mq must still hold the bare M^Q (before k_add_Lvo).
__global__ void __launch_bounds__(RED_THREADS) k_energy(Dims d, EnergyArgs A)
{
    __shared__ double sh[32];
    double sr = 0.0, si = 0.0;
    const long long nn = (long long)d.n * d.n, plane = (long long)d.NQ * nn;
    const long long nT = d.n1, nM = (long long)d.NQ * d.n1, nG = d.NQ;
    const long long nU0 = (long long)d.NQ * d.o[0] * d.o[0], nU1 = (long long)d.NQ * d.o[1] * d.o[1];
    const long long tot = nT + nM + nG + nU0 + nU1;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        long long y = x;
        if (y < nT) {
            int s = y >= d.n1a; int cc = (int)(s ? y - d.n1a : y);
            int i = cc / d.v[s], a = cc - i * d.v[s];
            double f = A.fock[s][(long long)i * d.n + d.o[s] + a];
            sr += f * A.t1r[y]; si += f * A.t1r[d.n1 + y];
            continue;
        }
        y -= nT;
        if (y < nM) {
            long long Q = y / d.n1; int c = (int)(y - Q * d.n1);
            int s = c >= d.n1a; int cc = s ? c - d.n1a : c;
            int i = cc / d.v[s], a = cc - i * d.v[s];
            double l = 0.5 * A.L[s][Q * nn + (long long)i * d.n + d.o[s] + a];
            sr += l * A.Mq[Q * 2 * d.n1 + c]; si += l * A.Mq[Q * 2 * d.n1 + d.n1 + c];
            continue;
        }
        y -= nM;
        if (y < nG) {
            double gr = A.gam[y], gi = A.gam[d.NQ + y];
            sr += 0.5 * (gr * gr - gi * gi); si += gr * gi;
            continue;
        }
        y -= nG;
        int s = 0;
        if (y >= nU0) { y -= nU0; s = 1; }
        const int o = d.o[s];
        long long Q = y / (o * o); int r = (int)(y - Q * o * o);
        int i = r / o, j = r - i * o;
        long long ij = Q * nn + (long long)i * d.n + j, ji = Q * nn + (long long)j * d.n + i;
        double ur = A.Lt[s][ij] - A.L[s][ij], ui = A.Lt[s][plane + ij];
        double wr = A.Lt[s][ji] - A.L[s][ji], wi = A.Lt[s][plane + ji];
        sr -= 0.5 * (ur * wr - ui * wi); si -= 0.5 * (ur * wi + ui * wr);
    }
    double a = block_sum(sr, sh);
    double b = block_sum(si, sh);
    __shared__ bool last;
    if (threadIdx.x == 0) {
        A.partial[2 * blockIdx.x] = a; A.partial[2 * blockIdx.x + 1] = b;
        __threadfence();
        last = atomicAdd(A.counter, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (last) {          // the last block adds the block sums in a fixed order (thread t: blocks t, t + 256, ...; then the block tree)
        __threadfence();
        double pa = 0.0, pb = 0.0;
        for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) { pa += A.partial[2 * i]; pb += A.partial[2 * i + 1]; }
        pa = block_sum(pa, sh);
        pb = block_sum(pb, sh);
        if (threadIdx.x == 0) { A.out[0] = pa; A.out[1] = pb; *A.counter = 0u; }
    }
}

// y = a + (hr + i*hi) * r over n complex (interleaved) elements
__global__ void k_caxpy(long long n, const double* __restrict__ a, const double* __restrict__ r, double hr, double hi,
                        double* __restrict__ y)
{
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < n; x += (long long)gridDim.x * blockDim.x) {
        double2 av = reinterpret_cast<const double2*>(a)[x], rv = reinterpret_cast<const double2*>(r)[x];
        double2 o;
        o.x = av.x + hr * rv.x - hi * rv.y;
        o.y = av.y + hr * rv.y + hi * rv.x;
        reinterpret_cast<double2*>(y)[x] = o;
    }
}

// The packed amplitude vector [t1 alpha | t1 beta | aa | bb | ab] as five row x column segments; the orbital-energy
// denominator of an element is colE[col] - rowE[row] (D_i^a = f_aa - f_ii, D_ij^ab = f_aa + f_bb - f_ii - f_jj), read from
// small per-segment tables instead of an amplitude-sized array.
struct AmpSegs {
    long long off[6];            // segment s holds elements off[s] .. off[s+1]
    int ncol[5];
    const double* rowE[5];
    const double* colE[5];
};
// rowE / colE tables (one launch at setup): tab = [oa | ob | po_a | po_b | oa*ob | va | vb | pv_a | pv_b | va*vb]
__global__ void k_build_denominator_tables(Dims d, const double* __restrict__ f0, const double* __restrict__ f1,
                                           const int2* __restrict__ op0, const int2* __restrict__ op1,
                                           const int2* __restrict__ vp0, const int2* __restrict__ vp1, double* __restrict__ tab)
{
    const int n = d.n;
    const long long cnt[10] = {d.o[0], d.o[1], d.po[0], d.po[1], d.oo, d.v[0], d.v[1], d.pv[0], d.pv[1], (long long)d.v[0] * d.v[1]};
    long long tot = 0;
    for (int k = 0; k < 10; ++k) tot += cnt[k];
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
        long long y = x; int k = 0;
        while (y >= cnt[k]) { y -= cnt[k]; ++k; }
        const int oa = d.o[0], ob = d.o[1];
        auto eo = [&](int s, int i) { const double* f = s ? f1 : f0; return f[(long long)i * n + i]; };
        auto ev = [&](int s, int a) { const double* f = s ? f1 : f0; const int o = s ? ob : oa; return f[(long long)(o + a) * n + o + a]; };
        double v;
        switch (k) {
            case 0: v = eo(0, (int)y); break;
            case 1: v = eo(1, (int)y); break;
            case 2: { int2 ij = op0[y]; v = eo(0, ij.x) + eo(0, ij.y); break; }
            case 3: { int2 ij = op1[y]; v = eo(1, ij.x) + eo(1, ij.y); break; }
            case 4: v = eo(0, (int)(y / ob)) + eo(1, (int)(y % ob)); break;
            case 5: v = ev(0, (int)y); break;
            case 6: v = ev(1, (int)y); break;
            case 7: { int2 ab = vp0[y]; v = ev(0, ab.x) + ev(0, ab.y); break; }
            case 8: { int2 ab = vp1[y]; v = ev(1, ab.x) + ev(1, ab.y); break; }
            default: v = ev(0, (int)(y / d.v[1])) + ev(1, (int)(y % d.v[1])); break;
        }
        tab[x] = v;
    }
}

// Adams-Moulton micro-iteration (Eq. 9):
//   mode 0:  y = B + h R(x)                       h = i dt/2
//   mode 1:  y = (B + h (R(x) - D x)) / (1 - h D) D = orbital-energy denominator (same fixed point)
// writes y and the block maxima of |y - x| (a non-finite value is reported as +inf); the last block to finish reduces the
// block maxima to out_delta[0] (max is order-independent, so this stays bit-reproducible).
// first != 0: x = t(tau), R = R(t(tau)) and B = t + h R is formed here and stored OVER R (Bv == R): the Adams-Moulton history is
// then three amplitude-sized vectors (t, B, iterate) plus the residual of the iterate.
// Aliasing: xin may be y (in-place iterate), Bv may be R (first): none of the four is __restrict__; every element is read
// before it is written, by the same thread.
constexpr int AM_CHUNK = 8;
__global__ void __launch_bounds__(RED_THREADS) k_am_update(long long n, AmpSegs sg, double* Bv, const double* R, const double* xin, int mode, int first,
                                                           double dt_half, double* y, double* __restrict__ bmax, unsigned* __restrict__ counter,
                                                           double* __restrict__ out_delta)
{
    __shared__ double sh[32];
    __shared__ bool last;
    double mx = 0.0;
    const long long per = (long long)RED_THREADS * AM_CHUNK;
    for (long long c0 = blockIdx.x * per; c0 < n; c0 += (long long)gridDim.x * per) {
        long long x = c0 + threadIdx.x;
        int seg = 0; long long row = 0; int col = 0;
        if (mode != 0 && x < n) {
            while (x >= sg.off[seg + 1]) ++seg;
            const long long y0 = x - sg.off[seg];
            row = y0 / sg.ncol[seg]; col = (int)(y0 - row * sg.ncol[seg]);
        }
#pragma unroll 2
        for (int j = 0; j < AM_CHUNK; ++j, x += RED_THREADS) {
            if (x >= n) break;
            double2 r = reinterpret_cast<const double2*>(R)[x];
            double2 t = reinterpret_cast<const double2*>(xin)[x], b, o;
            if (first) {
                b.x = t.x - dt_half * r.y;
                b.y = t.y + dt_half * r.x;
                reinterpret_cast<double2*>(Bv)[x] = b;
            } else b = reinterpret_cast<const double2*>(Bv)[x];
            if (mode == 0) {
                o.x = b.x - dt_half * r.y;
                o.y = b.y + dt_half * r.x;
            } else {
                const double D = sg.colE[seg][col] - sg.rowE[seg][row];
                double gr = r.x - D * t.x, gi = r.y - D * t.y;          // R - D x
                double nr = b.x - dt_half * gi, ni = b.y + dt_half * gr; // B + h (R - D x)
                double c = dt_half * D;                                   // 1 - h D = 1 - i c
                double den = 1.0 / (1.0 + c * c);
                o.x = (nr - c * ni) * den;                                // (nr + i ni)(1 + i c)/(1+c^2)
                o.y = (ni + c * nr) * den;
                const long long xn = x + RED_THREADS;                     // (segment, row, column) of the next element
                if (xn < n) {
                    if (xn >= sg.off[seg + 1] || sg.ncol[seg] < RED_THREADS) {
                        while (xn >= sg.off[seg + 1]) ++seg;
                        const long long y0 = xn - sg.off[seg];
                        row = y0 / sg.ncol[seg]; col = (int)(y0 - row * sg.ncol[seg]);
                    } else {
                        col += RED_THREADS;
                        if (col >= sg.ncol[seg]) { col -= sg.ncol[seg]; ++row; }
                    }
                }
            }
            reinterpret_cast<double2*>(y)[x] = o;
            double dx = o.x - t.x, dy = o.y - t.y;
            double a = sqrt(dx * dx + dy * dy);
            if (!(a == a) || isinf(a)) a = INFINITY;
            mx = fmax(mx, a);
        }
    }
    double m = block_max(mx, sh);
    if (threadIdx.x == 0) {
        bmax[blockIdx.x] = m;
        __threadfence();
        last = atomicAdd(counter, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (last) {
        __threadfence();
        double v = 0.0;
        for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) v = fmax(v, bmax[i]);
        v = block_max(v, sh);
        if (threadIdx.x == 0) { out_delta[0] = v; *counter = 0u; }
    }
}

// (N-1) Fock matrix, PAPER.md:48 (see include/rtcc.h: rtcc_build_fock)
__global__ void k_build_fock(int n, int NQ, const double* __restrict__ L, const double* __restrict__ eps, int cs, int ci,
                             double* __restrict__ fock)
{
    const long long nn = (long long)n * n;
    for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < 2 * nn; x += (long long)gridDim.x * blockDim.x) {
        const int s = (int)(x / nn); const long long r = x - s * nn;
        const int p = (int)(r / n), q = (int)(r - (long long)p * n);
        const double* Ls = L + (long long)s * NQ * nn;
        const double* Lc = L + (long long)cs * NQ * nn;
        double coul = 0.0, exch = 0.0;
        for (int Q = 0; Q < NQ; ++Q) {
            coul += Ls[Q * nn + r] * Lc[Q * nn + (long long)ci * n + ci];
            if (s == cs) exch += Ls[Q * nn + (long long)p * n + ci] * Ls[Q * nn + (long long)ci * n + q];
        }
        fock[x] = (p == q ? eps[s * n + p] : 0.0) - coul + exch;
    }
}

// G(tau_k) and A(omega): one block per frequency, fixed-order block reduction (see include/rtcc.h: rtcc_spectral_function)
__global__ void k_green(int nt, double dt, const double* __restrict__ C, double e0, double* __restrict__ G)
{
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nt; k += gridDim.x * blockDim.x) {
        const double tau = k * dt, m = exp(C[2 * k]), ph = C[2 * k + 1] - e0 * tau;      // exp(C) exp(-i e0 tau)
        const double zr = m * cos(ph), zi = m * sin(ph);
        G[2 * k] = zi; G[2 * k + 1] = -zr;                                                // times -i
    }
}
__global__ void __launch_bounds__(RED_THREADS) k_spectral(int nt, double dt, const double* __restrict__ G, double eta, int nw,
                                                           const double* __restrict__ omega, double* __restrict__ A)
{
    __shared__ double sh[32];
    const int w = blockIdx.x;
    if (w >= nw) return;
    const double om = omega[w];
    double acc = 0.0;                      // Im of the integral
    for (int k = threadIdx.x; k < nt; k += blockDim.x) {
        const double tau = k * dt, wgt = (k == 0 || k == nt - 1) ? 0.5 * dt : dt, d = exp(-eta * tau);
        const double c = cos(om * tau), s = sin(om * tau);
        acc += wgt * d * (G[2 * k] * s + G[2 * k + 1] * c);
    }
    const double r = block_sum(acc, sh);
    if (threadIdx.x == 0) A[w] = -r / 3.14159265358979323846;
}

// FP64 tensor-pipe peak probe: register-resident DMMA loop (denominator of the contraction roofline)
__global__ void __launch_bounds__(256) k_dmma_peak(double* out, int iters, double seed)
{
    double acc[16][2], a[4], b[4];
    for (int i = 0; i < 16; ++i) acc[i][0] = acc[i][1] = 0.0;
    for (int i = 0; i < 4; ++i) { a[i] = seed * (threadIdx.x + i); b[i] = seed * (i + 1); }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                             : "+d"(acc[i * 4 + j][0]), "+d"(acc[i * 4 + j][1]) : "d"(a[i]), "d"(b[j]));
    }
    double s = 0.0;
    for (int i = 0; i < 16; ++i) s += acc[i][0] + acc[i][1];
    out[blockIdx.x * (long long)blockDim.x + threadIdx.x] = s;
}

}  // namespace rtcc
