// ladder.cuh -- the o^2 v^4 particle-particle ladder as two chained FP64 tensor-core contractions,
// the four-virtual-index integrals formed tile by tile from the Cholesky vectors and never stored
// ("R(V,V,O,O) = alpha * v(V,V,V,V) * t2(V,V,O,O)", :129-131 Cholesky vectors;
//  BASELINE.json north_star bullet 2).
//
//   Y[(p,q)][x] = sum_{e,f} ( sum_Q LA[Q][p][e] * LB[Q][q][f] ) * X[(e,f)][x]
//
// p, q run over ALL orbitals of their spin (occupied rows deliver the T1-dressing corrections and
// the o^4 intermediate of the hole-hole ladder for free), e, f over virtuals,
// x over the Re|Im-stacked occupied pairs.  The three spin cases (ab, aa, bb) run in ONE launch.
// A work item = (spin case, 8x8 tile of (p,q) rows, column tile, slice of the (e,f) plane); the
// CTA walks its slice in chunks of 16x8 (e,f):
//   GEMM-1  W[(p,e),(q,f)] = sum_Q LA^T LB          (128 x 64 x n_chol, DMMA, accumulators in registers)
//   re-index W -> shared memory as A-operand [(p,q)][(e,f)]   (64 x 128)
//   GEMM-2  acc[(p,q)][x] += W * X[(e,f) chunk][x]  (64 x NT2 x 128, DMMA)
// Both GEMMs stream their global operands through one 3-stage cp.async pipeline whose producer keeps
// running pointers (no divisions, no 64-bit multiplies in the steady state).  When the (e,f) plane is
// sliced (small problems: more items than SMs), each slice writes its own partial buffer and
// ladder_reduce_kernel sums them in a fixed order -- no atomics, bit-reproducible.
#pragma once
#include "tcgemm.cuh"

namespace rtcc {

struct LadderCase {
    const double* LA; const double* LB;   // bare Cholesky vectors of the two spins, [NQ][n][n]
    long long sQA, sQB;                   // stride between Cholesky vectors
    int ldA, ldB;                         // row pitch (orbital count n)
    int offA, offB;                       // first virtual column (o_sigma)
    int nA, nB;                           // number of rows p / q
    int vA, vB;                           // number of virtuals e / f
    const double* X; long long ldX;       // [(e*vB+f)][N2]
    int N2;
    double* Y; long long ldY;             // [(p*nB+q)][N2]
    double* Ypart;                        // [nsplit][nA*nB][ldY] when nsplit > 1
    const int2* tiles; int ntiles;        // (p0,q0) row tiles
    int nsplit;                           // slices of the (e,f) chunk list
    int nt2;                              // column tile width: 64 or 128
    int ncol;                             // column tiles
    int item0;                            // first work item of this case
};
struct LadderBatch {
    LadderCase c[3];
    int ncase, NQ, nitems;
};

constexpr int LD_PP = 8, LD_PQ = 8, LD_PE = 16, LD_PF = 8;
constexpr int LD_M1 = LD_PP * LD_PE;      // 128
constexpr int LD_N1 = LD_PQ * LD_PF;      // 64
constexpr int LD_R = LD_PP * LD_PQ;       // 64 rows
constexpr int LD_K2 = LD_PE * LD_PF;      // 128
constexpr int LD_BK = 16, LD_ST = 3;
constexpr int LD_LDA1 = LD_M1 + 4, LD_LDB1 = LD_N1 + 4, LD_LDW = LD_K2 + 4;
constexpr int LD_STAGE = LD_BK * (LD_LDA1 + LD_LDB1);      // >= 16*(128+4)

constexpr size_t ladder_smem() { return sizeof(double) * (LD_ST * (size_t)LD_STAGE + (size_t)LD_R * LD_LDW); }

template <int NT2>
__device__ __forceinline__ void ladder_body(const LadderCase& g, const int NQ, const int p0, const int q0, const int x0,
                                            const int ch_begin, const int ch_end, double* __restrict__ Yout, double* smem)
{
    constexpr int NTH = 256;
    constexpr int LDX2 = NT2 + 4;
    constexpr int WGN = NT2 / 32;               // GEMM-2 warp grid: (8/WGN) x WGN, warp tile WM2 x 32
    constexpr int WGM = 8 / WGN;
    constexpr int WM2 = LD_R / WGM;             // 32 (NT2=128) or 16 (NT2=64)
    constexpr int TM2 = WM2 / 8;
    constexpr int RPP = NTH / NT2;              // X rows per pass: 2 or 4
    double* stg = smem;
    double* Ws = smem + LD_ST * LD_STAGE;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lr = lane >> 2, lc = lane & 3;
    const int nFt = (g.vB + LD_PF - 1) / LD_PF;
    const int T1 = (NQ + LD_BK - 1) / LD_BK;
    constexpr int T2 = LD_K2 / LD_BK;
    const int tpc = T1 + T2;
    const int total = (ch_end - ch_begin) * tpc;

    // ---- producer state (running pointers)
    const int mA = tid % LD_M1, kA0 = tid / LD_M1;           // A1: 2 k-rows per pass, 8 passes
    const int nB = tid % LD_N1, kB0 = tid / LD_N1;           // B1: 4 k-rows per pass, 4 passes
    const int pA = mA / LD_PE, eA = mA % LD_PE, qB = nB / LD_PF, fB = nB % LD_PF;
    const bool rowA = p0 + pA < g.nA, rowB = q0 + qB < g.nB;
    const double* baseA = g.LA + (long long)(p0 + pA) * g.ldA + g.offA + eA + kA0 * g.sQA;
    const double* baseB = g.LB + (long long)(q0 + qB) * g.ldB + g.offB + fB + kB0 * g.sQB;
    const long long stepA = 2 * g.sQA, stepB = 4 * g.sQB;
    const int cX = tid % NT2, kX0 = tid / NT2;
    const bool colX = x0 + cX < g.N2;
    const long long sF = g.ldX, sE = g.ldX * g.vB;
    const double* baseX = g.X + x0 + cX;
    int p_ch = ch_begin, p_r = 0;
    int p_e0 = (ch_begin / nFt) * LD_PE, p_f0 = (ch_begin % nFt) * LD_PF;
    const double* curA = baseA + p_e0;
    const double* curB = baseB + p_f0;

    auto produce = [&](int stage) {
        double* sb = stg + stage * LD_STAGE;
        if (p_r < T1) {
            const int kb = p_r * LD_BK;
            {
                const bool mv = rowA && (p_e0 + eA < g.vA);
                const double* s = curA;
                double* d = sb + kA0 * LD_LDA1 + mA;
#pragma unroll
                for (int j = 0; j < LD_BK / 2; ++j) {
                    const bool v = mv && (kb + kA0 + 2 * j < NQ);
                    cp_async8(d + 2 * j * LD_LDA1, v ? s : g.LA, v);
                    s += stepA;
                }
                curA = s;
            }
            {
                const bool nv = rowB && (p_f0 + fB < g.vB);
                const double* s = curB;
                double* d = sb + LD_BK * LD_LDA1 + kB0 * LD_LDB1 + nB;
#pragma unroll
                for (int j = 0; j < LD_BK / 4; ++j) {
                    const bool v = nv && (kb + kB0 + 4 * j < NQ);
                    cp_async8(d + 4 * j * LD_LDB1, v ? s : g.LB, v);
                    s += stepB;
                }
                curB = s;
            }
        } else {
            // rows kb..kb+15 of the chunk = (e, f) with e = e0 + kb/8 + {0,1}, f = f0 + 0..7
            const int kb = (p_r - T1) * LD_BK;
            const int eb = p_e0 + (kb >> 3);
            const double* P0 = baseX + ((long long)eb * g.vB + p_f0) * g.ldX;
            double* d = sb + kX0 * LDX2 + cX;
#pragma unroll
            for (int j = 0; j < LD_BK / RPP; ++j) {
                const int kk = kX0 + RPP * j;                 // compile-time pattern: kk>>3, kk&7
                const int de = (RPP * j + (RPP - 1)) >> 3;    // same for every kX0 < RPP because RPP divides 8
                const int ff = kk & 7;
                const bool v = colX && (eb + de < g.vA) && (p_f0 + ff < g.vB);
                const double* s = P0 + de * sE + ff * sF;
                cp_async8(d + RPP * j * LDX2, v ? s : g.X, v);
            }
        }
        if (++p_r == tpc) {
            p_r = 0; ++p_ch;
            p_f0 += LD_PF;
            if (p_f0 >= nFt * LD_PF) { p_f0 = 0; p_e0 += LD_PE; }
            curA = baseA + p_e0;
            curB = baseB + p_f0;
        }
    };

    double acc2[TM2][4][2];
#pragma unroll
    for (int i = 0; i < TM2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;
    double acc1[4][4][2];

    // GEMM-1 warp grid 4 x 2 (32 x 32 each); GEMM-2 warp grid WGM x WGN (WM2 x 32 each)
    const int w1m = (warp >> 1) * 32, w1n = (warp & 1) * 32;
    const int w2m = (warp / WGN) * WM2, w2n = (warp % WGN) * 32;

    int issued = 0;
#pragma unroll
    for (int s = 0; s < LD_ST - 1; ++s) {
        if (issued < total) { produce(s); ++issued; }
        cp_async_commit();
    }
    int r = 0, cstage = 0, pstage = LD_ST - 1;
    for (int s = 0; s < total; ++s) {
        cp_async_wait<LD_ST - 2>();
        __syncthreads();
        if (issued < total) { produce(pstage); ++issued; }
        cp_async_commit();
        if (++pstage == LD_ST) pstage = 0;
        const double* sb = stg + cstage * LD_STAGE;
        if (++cstage == LD_ST) cstage = 0;
        if (r < T1) {
            if (r == 0) {
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) acc1[i][j][0] = acc1[i][j][1] = 0.0;
            }
            const double* as = sb + lc * LD_LDA1 + w1m + lr;
            const double* bs = sb + LD_BK * LD_LDA1 + lc * LD_LDB1 + w1n + lr;
#pragma unroll
            for (int ks = 0; ks < LD_BK / 4; ++ks) {
                double a[4], b[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) a[i] = as[ks * 4 * LD_LDA1 + 8 * i];
#pragma unroll
                for (int j = 0; j < 4; ++j) b[j] = bs[ks * 4 * LD_LDB1 + 8 * j];
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) dmma884(acc1[i][j][0], acc1[i][j][1], a[i], b[j]);
            }
            if (r == T1 - 1) {
                // W[(p,e),(q,f)] -> Ws[(p,q)][(e,f)].  The previous chunk's GEMM-2 finished reading Ws
                // at least one __syncthreads ago (T1 >= 1 tiles of GEMM-1 lie in between).
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int m = w1m + 8 * i + lr;
                    const int p = m / LD_PE, e = m % LD_PE;
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int n = w1n + 8 * j + 2 * lc;          // n, n+1: same q, f and f+1
                        const int q = n / LD_PF, f = n % LD_PF;
                        *reinterpret_cast<double2*>(&Ws[(p * LD_PQ + q) * LD_LDW + e * LD_PF + f]) =
                            make_double2(acc1[i][j][0], acc1[i][j][1]);
                    }
                }
            }
        } else {
            const int kb = (r - T1) * LD_BK;
            const double* ws = Ws + (w2m + lr) * LD_LDW + kb + lc;
            const double* xs = sb + lc * LDX2 + w2n + lr;
#pragma unroll
            for (int ks = 0; ks < LD_BK / 4; ++ks) {
                double a[TM2], b[4];
#pragma unroll
                for (int i = 0; i < TM2; ++i) a[i] = ws[8 * i * LD_LDW + ks * 4];
#pragma unroll
                for (int j = 0; j < 4; ++j) b[j] = xs[ks * 4 * LDX2 + 8 * j];
#pragma unroll
                for (int i = 0; i < TM2; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) dmma884(acc2[i][j][0], acc2[i][j][1], a[i], b[j]);
            }
        }
        if (++r == tpc) r = 0;
    }
    cp_async_wait<0>();

#pragma unroll
    for (int i = 0; i < TM2; ++i) {
        const int row = w2m + 8 * i + lr;
        const int p = p0 + row / LD_PQ, q = q0 + row % LD_PQ;
        if (p >= g.nA || q >= g.nB) continue;
        double* y = Yout + ((long long)p * g.nB + q) * g.ldY;
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const int x = x0 + w2n + 8 * j + 2 * lc + c;
                if (x < g.N2) y[x] = acc2[i][j][c];
            }
    }
}

__global__ void __launch_bounds__(256) ladder_kernel(const LadderBatch b)
{
    extern __shared__ double smem[];
    int item = blockIdx.x, ci = 0;
    if (b.ncase > 1 && item >= b.c[1].item0) ci = 1;
    if (b.ncase > 2 && item >= b.c[2].item0) ci = 2;
    const LadderCase& g = b.c[ci];
    item -= g.item0;
    const int split = item % g.nsplit; item /= g.nsplit;
    const int col = item % g.ncol;
    const int tile = item / g.ncol;
    const int2 tl = g.tiles[tile];
    const int nEt = (g.vA + LD_PE - 1) / LD_PE, nFt = (g.vB + LD_PF - 1) / LD_PF;
    const int nchunk = nEt * nFt;
    const int ch0 = (int)((long long)split * nchunk / g.nsplit), ch1 = (int)((long long)(split + 1) * nchunk / g.nsplit);
    double* Yout = g.nsplit > 1 ? g.Ypart + (long long)split * g.nA * g.nB * g.ldY : g.Y;
    if (g.nt2 == 64) ladder_body<64>(g, b.NQ, tl.x, tl.y, col * 64, ch0, ch1, Yout, smem);
    else ladder_body<128>(g, b.NQ, tl.x, tl.y, col * 128, ch0, ch1, Yout, smem);
}

// Y = sum over slices of Ypart (fixed order)
__global__ void ladder_reduce_kernel(const LadderBatch b)
{
    for (int ci = 0; ci < b.ncase; ++ci) {
        const LadderCase& g = b.c[ci];
        if (g.nsplit <= 1) continue;
        const long long tot = (long long)g.nA * g.nB * g.ldY;
        for (long long x = blockIdx.x * (long long)blockDim.x + threadIdx.x; x < tot; x += (long long)gridDim.x * blockDim.x) {
            double s = 0.0;
            for (int k = 0; k < g.nsplit; ++k) s += g.Ypart[k * tot + x];
            g.Y[x] = s;
        }
    }
}

// Host side: choose column tile width and the (e,f) slicing so that the items fill the SMs evenly.
inline void ladder_plan(LadderBatch& b, int num_sms, int max_split)
{
    long long rows = 0;
    for (int i = 0; i < b.ncase; ++i) {
        LadderCase& g = b.c[i];
        g.nt2 = g.N2 <= 64 ? 64 : 128;
        g.ncol = (g.N2 + g.nt2 - 1) / g.nt2;
        rows += (long long)g.ntiles * g.ncol;
    }
    int best = 1;
    if (rows < 8LL * num_sms) {
        double beff = 0.0;
        for (int S = 1; S <= max_split; ++S) {
            double w = (double)rows * S / num_sms;
            double eff = w / ceil(w);
            if (eff > beff + 0.02) { beff = eff; best = S; }
        }
    }
    int item = 0;
    for (int i = 0; i < b.ncase; ++i) {
        LadderCase& g = b.c[i];
        const int nchunk = ((g.vA + LD_PE - 1) / LD_PE) * ((g.vB + LD_PF - 1) / LD_PF);
        g.nsplit = best < nchunk ? best : (nchunk > 0 ? nchunk : 1);
        g.item0 = item;
        item += g.ntiles * g.ncol * g.nsplit;
    }
    b.nitems = item;
}

// executed tensor-pipe flops of one launch
inline double ladder_flops(const LadderBatch& b)
{
    double f = 0.0;
    for (int i = 0; i < b.ncase; ++i) {
        const LadderCase& g = b.c[i];
        double rows = 64.0 * g.ntiles, ef = (double)g.vA * g.vB;
        f += 2.0 * rows * ef * ((double)b.NQ * g.ncol + (double)g.ncol * g.nt2);
    }
    return f;
}

inline int ladder_launch(const LadderBatch& b, cudaStream_t st, int num_sms)
{
    if (b.nitems <= 0) return 0;
    ladder_kernel<<<b.nitems, 256, ladder_smem(), st>>>(b);
    bool red = false;
    for (int i = 0; i < b.ncase; ++i) red |= b.c[i].nsplit > 1;
    if (red) { ladder_reduce_kernel<<<num_sms * 4, 256, 0, st>>>(b); return 2; }
    return 1;
}

inline cudaError_t ladder_init()
{
    return cudaFuncSetAttribute(ladder_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ladder_smem());
}

}  // namespace rtcc
