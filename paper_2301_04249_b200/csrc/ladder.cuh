// ladder.cuh -- the o^2 v^4 particle-particle ladder as two chained FP64 tensor-core contractions,
// the four-virtual-index integrals formed tile by tile from the Cholesky vectors and never stored
// ("R(V,V,O,O) = alpha * v(V,V,V,V) * t2(V,V,O,O)", :129-131 Cholesky vectors;
//  BASELINE.json north_star bullet 2).
//
//   Y[(p,q)][x] = sum_{e,f} ( sum_Q LA[Q][p][e] * LB[Q][q][f] ) * X[(e,f)][x]
//
// p, q run over ALL orbitals of their spin (occupied rows deliver the T1-dressing corrections and
// the o^4 intermediate of the hole-hole ladder for free), e, f over virtuals,
// x over the Re|Im-stacked occupied pairs.  One CTA owns a tile of 8x8 (p,q) rows and NT2 columns
// and walks the (e,f) plane in chunks of 16x8:
//   GEMM-1  W[(p,e),(q,f)] = sum_Q LA^T LB          (128 x 64 x n_chol, DMMA, accumulators in registers)
//   re-index W -> shared memory as A-operand [(p,q)][(e,f)]   (64 x 128)
//   GEMM-2  acc[(p,q)][x] += W * X[(e,f) chunk][x]  (64 x NT2 x 128, DMMA)
// Both GEMMs stream their global operands through one 3-stage cp.async pipeline.
#pragma once
#include "tcgemm.cuh"

namespace rtcc {

struct LadderArgs {
    const double* LA; const double* LB;   // [NQ][nA][ldA] / [NQ][nB][ldB] slices of the bare vectors
    long long sQA, sQB;                   // stride between Cholesky vectors
    int ldA, ldB;                         // row pitch (orbital count n)
    int offA, offB;                       // first virtual column (o_sigma)
    int nA, nB;                           // number of rows p / q
    int vA, vB;                           // number of virtuals e / f
    int NQ;
    const double* X; long long ldX;       // [(e*vB+f)][N2]
    int N2;
    double* Y; long long ldY;             // [(p*nB+q)][N2]
    const int2* tiles; int ntiles;        // (p0,q0) row tiles
};

constexpr int LD_PP = 8, LD_PQ = 8, LD_PE = 16, LD_PF = 8;
constexpr int LD_M1 = LD_PP * LD_PE;      // 128
constexpr int LD_N1 = LD_PQ * LD_PF;      // 64
constexpr int LD_R = LD_PP * LD_PQ;       // 64 rows
constexpr int LD_K2 = LD_PE * LD_PF;      // 128
constexpr int LD_BK = 16, LD_ST = 3;
constexpr int LD_LDA1 = LD_M1 + 4, LD_LDB1 = LD_N1 + 4, LD_LDW = LD_K2 + 4;

template <int NT2> constexpr size_t ladder_smem()
{
    constexpr size_t stage1 = (size_t)LD_BK * (LD_LDA1 + LD_LDB1);
    constexpr size_t stage2 = (size_t)LD_BK * (NT2 + 4);
    constexpr size_t stage = stage1 > stage2 ? stage1 : stage2;
    return sizeof(double) * (LD_ST * stage + (size_t)LD_R * LD_LDW);
}

template <int NT2>
__global__ void __launch_bounds__(256) ladder_kernel(const LadderArgs g)
{
    constexpr int NTH = 256;
    constexpr int LDX2 = NT2 + 4;
    constexpr size_t stage1 = (size_t)LD_BK * (LD_LDA1 + LD_LDB1);
    constexpr size_t stage2 = (size_t)LD_BK * LDX2;
    constexpr size_t STAGE = stage1 > stage2 ? stage1 : stage2;
    constexpr int WN2 = NT2 / 4;          // GEMM-2 warp tile 32 x WN2
    constexpr int TN2 = WN2 / 8;
    extern __shared__ double smem[];
    double* stg = smem;                               // [ST][STAGE]
    double* Ws = smem + LD_ST * STAGE;                // [64][LDW]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lr = lane >> 2, lc = lane & 3;
    const int2 tl = g.tiles[blockIdx.x];
    const int p0 = tl.x, q0 = tl.y;
    const int x0 = blockIdx.y * NT2;

    const int nEt = (g.vA + LD_PE - 1) / LD_PE, nFt = (g.vB + LD_PF - 1) / LD_PF;
    const int nchunk = nEt * nFt;
    const int T1 = (g.NQ + LD_BK - 1) / LD_BK, T2 = LD_K2 / LD_BK;
    const int tpc = T1 + T2;
    const int total = nchunk * tpc;

    auto load_tile = [&](int s, int stage) {
        const int ch = s / tpc, r = s - ch * tpc;
        const int e0 = (ch / nFt) * LD_PE, f0 = (ch % nFt) * LD_PF;
        double* sb = stg + stage * STAGE;
        if (r < T1) {
            // Cholesky-vector tiles: A1[k][(p,e)], B1[k][(q,f)]
            double* as = sb;
            double* bs = sb + LD_BK * LD_LDA1;
            const int kb = r * LD_BK;
            {
                const int m = tid % LD_M1, k0 = tid / LD_M1;       // 2 k-rows per pass
                const int p = m / LD_PE, e = m % LD_PE;
                const bool mv = (p0 + p < g.nA) && (e0 + e < g.vA);
                const double* src = g.LA + (long long)(p0 + p) * g.ldA + g.offA + e0 + e;
#pragma unroll
                for (int j = 0; j < LD_BK / 2; ++j) {
                    int kk = k0 + 2 * j, Q = kb + kk;
                    bool v = mv && Q < g.NQ;
                    cp_async8(as + kk * LD_LDA1 + m, v ? (src + Q * g.sQA) : g.LA, v);
                }
            }
            {
                const int n = tid % LD_N1, k0 = tid / LD_N1;       // 4 k-rows per pass
                const int q = n / LD_PF, f = n % LD_PF;
                const bool nv = (q0 + q < g.nB) && (f0 + f < g.vB);
                const double* src = g.LB + (long long)(q0 + q) * g.ldB + g.offB + f0 + f;
#pragma unroll
                for (int j = 0; j < LD_BK / 4; ++j) {
                    int kk = k0 + 4 * j, Q = kb + kk;
                    bool v = nv && Q < g.NQ;
                    cp_async8(bs + kk * LD_LDB1 + n, v ? (src + Q * g.sQB) : g.LB, v);
                }
            }
        } else {
            // amplitude tile X[(e,f) rows kb..kb+15][x0..x0+NT2)
            const int kb = (r - T1) * LD_BK;
            constexpr int RPP = NTH / NT2;                 // rows per pass
            const int c = tid % NT2, k0 = tid / NT2;
            const bool cv = x0 + c < g.N2;
#pragma unroll
            for (int j = 0; j < LD_BK / RPP; ++j) {
                int kk = k0 + RPP * j, k2 = kb + kk;
                int e = e0 + k2 / LD_PF, f = f0 + k2 % LD_PF;
                bool v = cv && e < g.vA && f < g.vB;
                const double* src = g.X + ((long long)e * g.vB + f) * g.ldX + x0 + c;
                cp_async8(sb + kk * LDX2 + c, v ? src : g.X, v);
            }
        }
    };

    double acc2[4][TN2][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < TN2; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;
    double acc1[4][4][2];

    // GEMM-1 warp grid 4 x 2 (32 x 32 each); GEMM-2 warp grid 2 x 4 (32 x WN2 each)
    const int w1m = (warp >> 1) * 32, w1n = (warp & 1) * 32;
    const int w2m = (warp >> 2) * 32, w2n = (warp & 3) * WN2;

#pragma unroll
    for (int s = 0; s < LD_ST - 1; ++s) {
        if (s < total) load_tile(s, s);
        cp_async_commit();
    }
    int r = 0;                                    // position inside the chunk
    for (int s = 0; s < total; ++s) {
        cp_async_wait<LD_ST - 2>();
        __syncthreads();
        {
            int sn = s + LD_ST - 1;
            if (sn < total) load_tile(sn, sn % LD_ST);
            cp_async_commit();
        }
        const double* sb = stg + (s % LD_ST) * STAGE;
        if (r < T1) {
            if (r == 0) {
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) acc1[i][j][0] = acc1[i][j][1] = 0.0;
            }
            const double* as = sb;
            const double* bs = sb + LD_BK * LD_LDA1;
#pragma unroll
            for (int ks = 0; ks < LD_BK / 4; ++ks) {
                double a[4], b[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) a[i] = as[(ks * 4 + lc) * LD_LDA1 + w1m + 8 * i + lr];
#pragma unroll
                for (int j = 0; j < 4; ++j) b[j] = bs[(ks * 4 + lc) * LD_LDB1 + w1n + 8 * j + lr];
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
                    int m = w1m + 8 * i + lr;
                    int p = m / LD_PE, e = m % LD_PE;
#pragma unroll
                    for (int j = 0; j < 4; ++j)
#pragma unroll
                        for (int c = 0; c < 2; ++c) {
                            int n = w1n + 8 * j + 2 * lc + c;
                            int q = n / LD_PF, f = n % LD_PF;
                            Ws[(p * LD_PQ + q) * LD_LDW + e * LD_PF + f] = acc1[i][j][c];
                        }
                }
            }
        } else {
            const int kb = (r - T1) * LD_BK;
#pragma unroll
            for (int ks = 0; ks < LD_BK / 4; ++ks) {
                double a[4], b[TN2];
#pragma unroll
                for (int i = 0; i < 4; ++i) a[i] = Ws[(w2m + 8 * i + lr) * LD_LDW + kb + ks * 4 + lc];
#pragma unroll
                for (int j = 0; j < TN2; ++j) b[j] = sb[(ks * 4 + lc) * LDX2 + w2n + 8 * j + lr];
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < TN2; ++j) dmma884(acc2[i][j][0], acc2[i][j][1], a[i], b[j]);
            }
        }
        if (++r == tpc) r = 0;
    }
    cp_async_wait<0>();

#pragma unroll
    for (int i = 0; i < 4; ++i) {
        int row = w2m + 8 * i + lr;
        int p = p0 + row / LD_PQ, q = q0 + row % LD_PQ;
        if (p >= g.nA || q >= g.nB) continue;
        double* y = g.Y + ((long long)p * g.nB + q) * g.ldY;
#pragma unroll
        for (int j = 0; j < TN2; ++j)
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                int x = x0 + w2n + 8 * j + 2 * lc + c;
                if (x < g.N2) y[x] = acc2[i][j][c];
            }
    }
}

inline int ladder_launch(const LadderArgs& g, cudaStream_t st, double* flops_out = nullptr)
{
    if (g.ntiles <= 0 || g.N2 <= 0) return 0;
    constexpr int NT2 = 128;
    dim3 grid(g.ntiles, (g.N2 + NT2 - 1) / NT2);
    ladder_kernel<NT2><<<grid, 256, ladder_smem<NT2>(), st>>>(g);
    if (flops_out) {
        double rows = 64.0 * g.ntiles, ef = (double)g.vA * g.vB;
        *flops_out += 2.0 * rows * ef * ((double)g.NQ * grid.y + g.N2);
    }
    return 1;
}

// executed tensor-pipe flops of one launch (same count ladder_launch adds)
inline void ladder_launch_flops(const LadderArgs& g, double* out)
{
    if (g.ntiles <= 0 || g.N2 <= 0) return;
    const int ny = (g.N2 + 127) / 128;
    double rows = 64.0 * g.ntiles, ef = (double)g.vA * g.vB;
    *out += 2.0 * rows * ef * ((double)g.NQ * ny + g.N2);
}

inline cudaError_t ladder_init()
{
    return cudaFuncSetAttribute(ladder_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ladder_smem<128>());
}

}  // namespace rtcc
