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
// Both GEMMs stream their global operands through one 4-stage ring filled by a dedicated producer warp with
// 1-D bulk async copies (cp.async.bulk, TMA engine) from zero-padded operand slabs, completion tracked by
// mbarriers; the 8 consumer warps execute only LDS + DMMA.  When the (e,f) plane is
// sliced (small problems: more items than SMs), each slice writes its own partial buffer and
// ladder_reduce_kernel sums them in a fixed order -- no atomics, bit-reproducible.
#pragma once
#include "tcgemm.cuh"

namespace rtcc {

struct LadderCase {
    // Tile-major, zero-padded slabs of the bare Cholesky vectors' virtual columns, laid out exactly as the
    // shared-memory stage wants them (row pitch == 4 mod 16 doubles), so that each pipeline tile is ONE bulk copy:
    //   LA[pt][et][Qt][16 k][8 p x 16 e (+4 pad)]      LB[qt][ft][Qt][16 k][8 q x 8 f (+4 pad)]
    const double* LA; const double* LB;
    int nA, nB;                           // number of rows p / q (unpadded)
    int vA, vB;                           // number of virtuals e / f (unpadded)
    // amplitudes, tile-major and zero padded: Xt[et][ft][ct][8 kt][16 rows (e_in*8+f_in)][nt2 (+4 pad)]
    const double* X;
    int N2;
    double* Y; long long ldY;             // [(p*nB+q)][N2]
    double* Ypart;                        // [nsplit][nA*nB][ldY] when nsplit > 1
    const int2* tiles; int ntiles;        // (p0,q0) row tiles
    int nsplit;                           // slices of the (e,f) chunk list
    int nt2;                              // column tile width: 64 or 128
    int ncol;                             // column tiles
    int cl;                               // CTAs per cluster sharing one W chunk (1: plain kernel); ncol > 1 only
    int ngrp;                             // column-tile groups of cl tiles each
    int item0;                            // first work item of this case
};
struct LadderBatch {
    LadderCase c[3];
    int ncase, NQ, nitems;                // NQ: padded to a multiple of 16
};

constexpr int LD_PP = 8, LD_PQ = 8, LD_PE = 16, LD_PF = 8;
constexpr int LD_M1 = LD_PP * LD_PE;      // 128
constexpr int LD_N1 = LD_PQ * LD_PF;      // 64
constexpr int LD_R = LD_PP * LD_PQ;       // 64 rows
constexpr int LD_K2 = LD_PE * LD_PF;      // 128
constexpr int LD_BK = 16, LD_ST = 4;
constexpr int LD_LDA1 = LD_M1 + 4, LD_LDB1 = LD_N1 + 4, LD_LDW = LD_K2 + 4;
constexpr int LD_STAGE = LD_BK * (LD_LDA1 + LD_LDB1);      // >= 16*(128+4)
constexpr int LD_NCONS = 256, LD_NTH = 288;               // 8 consumer warps + 1 producer warp

constexpr size_t ladder_smem() { return sizeof(double) * (LD_ST * (size_t)LD_STAGE + (size_t)LD_R * LD_LDW) + 2 * LD_ST * sizeof(unsigned long long); }

// 1-D bulk async copy global -> shared (TMA engine), completion counted in bytes on an mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void bar_consumers() { asm volatile("bar.sync 1, 256;" ::: "memory"); }

template <int NT2>
__device__ __forceinline__ void ladder_body(const LadderCase& gc, const int NQ, const int p0, const int q0, const int x0,
                                            const int ch_begin, const int ch_end, double* __restrict__ Yout, double* smem)
{
    constexpr int LDX2 = NT2 + 4;
    constexpr int WGN = NT2 / 32;               // GEMM-2 warp grid: (8/WGN) x WGN, warp tile WM2 x 32
    constexpr int WGM = 8 / WGN;
    constexpr int WM2 = LD_R / WGM;             // 32 (NT2=128) or 16 (NT2=64)
    constexpr int TM2 = WM2 / 8;
    double* stg = smem;
    double* Ws = smem + LD_ST * LD_STAGE;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(Ws + LD_R * LD_LDW);
    unsigned long long* empty = full + LD_ST;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nFt = (gc.vB + LD_PF - 1) / LD_PF;
    const int T1 = NQ / LD_BK;
    constexpr int T2 = LD_K2 / LD_BK;
    const int tpc = T1 + T2;
    const int total = (ch_end - ch_begin) * tpc;

    if (tid == 0) {
        for (int s = 0; s < LD_ST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == 8) {
        // ---------------- producer: one elected lane, one or two bulk copies per tile
        if (lane == 0) {
            const int nEt = (gc.vA + LD_PE - 1) / LD_PE;
            constexpr int BLKA = LD_BK * LD_LDA1, BLKB = LD_BK * LD_LDB1, BLKX = LD_BK * LDX2;
            const int ncol = gc.ncol, ct = x0 / NT2;
            const double* LAp = gc.LA + (long long)(p0 / LD_PP) * nEt * T1 * BLKA;
            const double* LBp = gc.LB + (long long)(q0 / LD_PQ) * nFt * T1 * BLKB;
            int et = ch_begin / nFt, ft = ch_begin % nFt, r = 0;
            const double* curA = LAp + (long long)et * T1 * BLKA;
            const double* curB = LBp + (long long)ft * T1 * BLKB;
            const double* curX = gc.X + (((long long)(et * nFt + ft) * ncol + ct) * T2) * BLKX;
            int stage = 0; unsigned par = 1;       // first pass over the ring: slots are free
            for (int it = 0; it < total; ++it) {
                mbar_wait(&empty[stage], par);
                double* sb = stg + stage * LD_STAGE;
                if (r < T1) {
                    mbar_expect_tx(&full[stage], (BLKA + BLKB) * 8);
                    bulk_g2s(sb, curA, BLKA * 8, &full[stage]);
                    bulk_g2s(sb + BLKA, curB, BLKB * 8, &full[stage]);
                    curA += BLKA; curB += BLKB;
                } else {
                    mbar_expect_tx(&full[stage], BLKX * 8);
                    bulk_g2s(sb, curX, BLKX * 8, &full[stage]);
                    curX += BLKX;
                }
                if (++r == tpc) {
                    r = 0;
                    if (++ft == nFt) { ft = 0; ++et; }
                    curA = LAp + (long long)et * T1 * BLKA;
                    curB = LBp + (long long)ft * T1 * BLKB;
                    curX = gc.X + (((long long)(et * nFt + ft) * ncol + ct) * T2) * BLKX;
                }
                if (++stage == LD_ST) { stage = 0; par ^= 1; }
            }
        }
        return;
    }

    // ---------------- consumer warps
    const int lr = lane >> 2, lc = lane & 3;
    double acc2[TM2][4][2];
#pragma unroll
    for (int i = 0; i < TM2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;
    double acc1[4][4][2];

    // GEMM-1 warp grid 4 x 2 (32 x 32 each); GEMM-2 warp grid WGM x WGN (WM2 x 32 each)
    const int w1m = (warp >> 1) * 32, w1n = (warp & 1) * 32;
    const int w2m = (warp / WGN) * WM2, w2n = (warp % WGN) * 32;

    int r = 0, stage = 0; unsigned par = 0;
    for (int it = 0; it < total; ++it) {
        mbar_wait(&full[stage], par);
        const double* sb = stg + stage * LD_STAGE;
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
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[stage]);
            if (r == T1 - 1) {
                bar_consumers();        // every consumer has finished the previous chunk's GEMM-2 reads of Ws
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
                bar_consumers();        // W chunk complete
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
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[stage]);
        }
        if (++r == tpc) r = 0;
        if (++stage == LD_ST) { stage = 0; par ^= 1; }
    }

#pragma unroll
    for (int i = 0; i < TM2; ++i) {
        const int row = w2m + 8 * i + lr;
        const int p = p0 + row / LD_PQ, q = q0 + row % LD_PQ;
        if (p >= gc.nA || q >= gc.nB) continue;
        double* y = Yout + ((long long)p * gc.nB + q) * gc.ldY;
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const int x = x0 + w2n + 8 * j + 2 * lc + c;
                if (x < gc.N2) y[x] = acc2[i][j][c];
            }
    }
}

__global__ void __launch_bounds__(LD_NTH) ladder_kernel(const LadderBatch b)
{
    extern __shared__ __align__(128) double smem[];
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

// ------------------------------------------------------------------------------------------------------------
// Wide amplitudes (more than one column tile): a thread-block CLUSTER of cl CTAs owns one (p,q) row tile.  CTA r
// keeps the accumulators of column tile r.  Each W chunk is built ONCE per cluster: the n_chol reduction of GEMM-1 is
// split across the CTAs, the partial tiles are summed through distributed shared memory in a fixed order
// (reduce-scatter + all-gather, deterministic) and every CTA then applies the complete chunk to its own columns.
constexpr int LC_ST = 3;
constexpr size_t ladder_cluster_smem()
{ return sizeof(double) * (LC_ST * (size_t)LD_STAGE + 2 * (size_t)LD_R * LD_LDW) + (2 * LC_ST + 2) * sizeof(unsigned long long); }

__device__ __forceinline__ unsigned cluster_rank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ unsigned map_shared(const void* p, unsigned rank)
{
    unsigned a = (unsigned)__cvta_generic_to_shared(p), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
__device__ __forceinline__ double2 ld_cluster2(unsigned addr)
{ double2 v; asm volatile("ld.shared::cluster.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory"); return v; }
__device__ __forceinline__ void st_cluster2(unsigned addr, double2 v)
{ asm volatile("st.shared::cluster.v2.f64 [%0], {%1,%2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory"); }
__device__ __forceinline__ void mbar_arrive_cluster(unsigned remote_addr)
{ asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(remote_addr) : "memory"); }
__device__ __forceinline__ void mbar_wait_cluster(unsigned long long* b, unsigned parity)
{
    const unsigned addr = (unsigned)__cvta_generic_to_shared(b);
    unsigned ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    } while (!ok);
}

__global__ void __launch_bounds__(LD_NTH, 1) ladder_cluster_kernel(const LadderCase g, const int NQ)
{
    constexpr int NT2 = 128, LDX2 = NT2 + 4, T2 = LD_K2 / LD_BK;
    extern __shared__ __align__(128) double smem[];
    double* stg = smem;
    double* Ws = smem + LC_ST * LD_STAGE;
    double* Ps = Ws + LD_R * LD_LDW;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(Ps + LD_R * LD_LDW);
    unsigned long long* empty = full + LC_ST;
    unsigned long long* cbar = empty + LC_ST;          // [0]: partial tiles written, [1]: reduced chunk distributed

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cl = g.cl;
    const int rank = (int)cluster_rank();
    int item = blockIdx.x / cl;
    const int split = item % g.nsplit; item /= g.nsplit;
    const int grp = item % g.ngrp;
    const int2 tl = g.tiles[item / g.ngrp];
    const int p0 = tl.x, q0 = tl.y;
    const int col = grp * cl + rank;
    const bool has_col = col < g.ncol;
    const int x0 = col * NT2;
    const int nEt = (g.vA + LD_PE - 1) / LD_PE, nFt = (g.vB + LD_PF - 1) / LD_PF;
    const int nchunk = nEt * nFt;
    const int ch0 = (int)((long long)split * nchunk / g.nsplit), ch1 = (int)((long long)(split + 1) * nchunk / g.nsplit);
    const int T1 = NQ / LD_BK;
    const int kt0 = (int)((long long)rank * T1 / cl), kt1 = (int)((long long)(rank + 1) * T1 / cl);   // my share of the n_chol reduction
    const int T1r = kt1 - kt0;

    if (tid == 0) {
        for (int s = 0; s < LC_ST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
        mbar_init(&cbar[0], 8 * cl); mbar_init(&cbar[1], 8 * cl);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    asm volatile("barrier.cluster.arrive.release.aligned;\n barrier.cluster.wait.acquire.aligned;" ::: "memory");   // every CTA's barriers exist

    if (warp == 8) {
        if (lane == 0) {
            constexpr int BLKA = LD_BK * LD_LDA1, BLKB = LD_BK * LD_LDB1, BLKX = LD_BK * LDX2;
            const double* LAp = g.LA + (long long)(p0 / LD_PP) * nEt * T1 * BLKA + (long long)kt0 * BLKA;
            const double* LBp = g.LB + (long long)(q0 / LD_PQ) * nFt * T1 * BLKB + (long long)kt0 * BLKB;
            int stage = 0; unsigned par = 1;
            auto issue_g1 = [&](int ch) {
                const int et = ch / nFt, ft = ch % nFt;
                const double* curA = LAp + (long long)et * T1 * BLKA;
                const double* curB = LBp + (long long)ft * T1 * BLKB;
                for (int t = 0; t < T1r; ++t) {
                    mbar_wait(&empty[stage], par);
                    double* sb = stg + stage * LD_STAGE;
                    mbar_expect_tx(&full[stage], (BLKA + BLKB) * 8);
                    bulk_g2s(sb, curA, BLKA * 8, &full[stage]);
                    bulk_g2s(sb + BLKA, curB, BLKB * 8, &full[stage]);
                    curA += BLKA; curB += BLKB;
                    if (++stage == LC_ST) { stage = 0; par ^= 1; }
                }
            };
            if (ch0 < ch1) issue_g1(ch0);
            for (int ch = ch0; ch < ch1; ++ch) {
                if (ch + 1 < ch1) issue_g1(ch + 1);            // consumers build the next partial while this chunk is being gathered
                if (has_col) {
                    const int et = ch / nFt, ft = ch % nFt;
                    const double* curX = g.X + (((long long)(et * nFt + ft) * g.ncol + col) * T2) * BLKX;
                    for (int t = 0; t < T2; ++t) {
                        mbar_wait(&empty[stage], par);
                        mbar_expect_tx(&full[stage], BLKX * 8);
                        bulk_g2s(stg + stage * LD_STAGE, curX, BLKX * 8, &full[stage]);
                        curX += BLKX;
                        if (++stage == LC_ST) { stage = 0; par ^= 1; }
                    }
                }
            }
        }
    } else {
    // ---------------- consumers
    const int lr = lane >> 2, lc = lane & 3;
    double acc2[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc2[i][j][0] = acc2[i][j][1] = 0.0;
    double acc1[4][4][2];
    const int w1m = (warp >> 1) * 32, w1n = (warp & 1) * 32;
    const int w2m = (warp >> 2) * 32, w2n = (warp & 3) * 32;
    // my slice of the 64 x 128 chunk in double2 units (reduce-scatter)
    constexpr int UNITS = LD_R * LD_K2 / 2;
    const int u0 = (int)((long long)rank * UNITS / cl), u1 = (int)((long long)(rank + 1) * UNITS / cl);

    int stage = 0; unsigned par = 0, cpar = 0;
    // GEMM-1 share of one chunk into acc1 (T1r tiles of the n_chol reduction)
    auto gemm1 = [&]() {
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc1[i][j][0] = acc1[i][j][1] = 0.0;
        for (int t = 0; t < T1r; ++t) {
            mbar_wait(&full[stage], par);
            const double* sb = stg + stage * LD_STAGE;
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
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[stage]);
            if (++stage == LC_ST) { stage = 0; par ^= 1; }
        }
    };
    // partial W[(p,e),(q,f)] -> Ps[(p,q)][(e,f)], then tell the whole cluster (barrier [0])
    auto publish = [&]() {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = w1m + 8 * i + lr;
            const int p = m / LD_PE, e = m % LD_PE;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int n = w1n + 8 * j + 2 * lc;
                const int q = n / LD_PF, f = n % LD_PF;
                *reinterpret_cast<double2*>(&Ps[(p * LD_PQ + q) * LD_LDW + e * LD_PF + f]) = make_double2(acc1[i][j][0], acc1[i][j][1]);
            }
        }
        __syncwarp();
        if (lane == 0)
            for (int r = 0; r < cl; ++r) mbar_arrive_cluster(map_shared(&cbar[0], r));      // release at cluster scope
    };
    if (ch0 < ch1) { gemm1(); publish(); }
    for (int ch = ch0; ch < ch1; ++ch) {
        mbar_wait_cluster(&cbar[0], cpar);
        // reduce my slice over the cl partial tiles (fixed order) and hand the result to every CTA of the cluster
        for (int u = u0 + (tid & 255); u < u1; u += LD_NCONS) {
            const int row = u / (LD_K2 / 2), c2 = u % (LD_K2 / 2);
            const int off = row * LD_LDW + 2 * c2;
            double2 s = make_double2(0.0, 0.0);
            for (int r = 0; r < cl; ++r) {
                double2 v = ld_cluster2(map_shared(Ps + off, r));
                s.x += v.x; s.y += v.y;
            }
            for (int r = 0; r < cl; ++r) st_cluster2(map_shared(Ws + off, r), s);
        }
        __syncwarp();
        if (lane == 0)
            for (int r = 0; r < cl; ++r) mbar_arrive_cluster(map_shared(&cbar[1], r));
        // software pipeline: the next chunk's GEMM-1 share runs while the other CTAs finish gathering this chunk
        const bool more = ch + 1 < ch1;
        if (more) gemm1();
        mbar_wait_cluster(&cbar[1], cpar);
        cpar ^= 1;
        if (has_col) {
            for (int t = 0; t < T2; ++t) {
                mbar_wait(&full[stage], par);
                const double* sb = stg + stage * LD_STAGE;
                const double* ws = Ws + (w2m + lr) * LD_LDW + t * LD_BK + lc;
                const double* xs = sb + lc * LDX2 + w2n + lr;
#pragma unroll
                for (int ks = 0; ks < LD_BK / 4; ++ks) {
                    double a[4], b[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) a[i] = ws[8 * i * LD_LDW + ks * 4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) b[j] = xs[ks * 4 * LDX2 + 8 * j];
#pragma unroll
                    for (int i = 0; i < 4; ++i)
#pragma unroll
                        for (int j = 0; j < 4; ++j) dmma884(acc2[i][j][0], acc2[i][j][1], a[i], b[j]);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[stage]);
                if (++stage == LC_ST) { stage = 0; par ^= 1; }
            }
        }
        // every CTA has finished reading Ps of this chunk (barrier [1]); my next partial may overwrite it now
        if (more) publish();
    }
    if (has_col) {
        double* Yout = g.nsplit > 1 ? g.Ypart + (long long)split * g.nA * g.nB * g.ldY : g.Y;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
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
    }
    // no CTA may retire while a sibling can still touch its shared memory
    asm volatile("barrier.cluster.arrive.release.aligned;\n barrier.cluster.wait.acquire.aligned;" ::: "memory");
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

// SMs that clusters of cl CTAs of the wide kernel can keep busy at once (0: size not schedulable); cached per size
inline int ladder_cluster_active_sms(int cl, int num_sms)
{
    static int tab[17] = {0};
    static bool done = false;
    if (!done) {
        for (int c = 2; c <= 16; ++c) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)c * 64); cfg.blockDim = dim3(LD_NTH); cfg.dynamicSmemBytes = ladder_cluster_smem();
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = (unsigned)c; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            int n = 0;
            if (cudaOccupancyMaxActiveClusters(&n, ladder_cluster_kernel, &cfg) == cudaSuccess && n > 0) tab[c] = n * c;
            cudaGetLastError();
        }
        done = true;
    }
    int a = (cl >= 2 && cl <= 16) ? tab[cl] : 0;
    return a > num_sms ? num_sms : a;
}
// cluster size for ncol column tiles: minimise  groups * (W1 + cl * W2) / active SMs   (W1: building one W chunk,
// W2: applying it to one column tile); a cluster never spans more column tiles than there are
inline int ladder_choose_cluster(int ncol, int NQ, int num_sms)
{
    int maxc = 16;
    if (const char* e = getenv("RTCC_MAX_CLUSTER")) { int v = atoi(e); if (v >= 2 && v < maxc) maxc = v; }
    const double W1 = 128.0 * 64.0 * NQ, W2 = 64.0 * 128.0 * 128.0;
    int best = 0; double bt = 1e300;
    for (int cl = 2; cl <= maxc; ++cl) {
        const int act = ladder_cluster_active_sms(cl, num_sms);
        if (act <= 0) continue;
        const int ngrp = (ncol + cl - 1) / cl;
        const int ceff = (ncol + ngrp - 1) / ngrp;          // balanced groups
        if (ceff != cl && cl <= ncol) continue;             // evaluate each balanced size once
        const double t = ngrp * (W1 + ceff * W2) / ladder_cluster_active_sms(ceff, num_sms);
        if (ladder_cluster_active_sms(ceff, num_sms) > 0 && t < bt) { bt = t; best = ceff; }
    }
    return best > 0 ? best : 2;
}

// Host side: choose column tile width, cluster shape and the (e,f) slicing so that the items fill the SMs evenly.
inline void ladder_plan(LadderBatch& b, int num_sms, int max_split)
{
    long long rows = 0;
    for (int i = 0; i < b.ncase; ++i) {
        LadderCase& g = b.c[i];
        g.nt2 = g.N2 <= 64 ? 64 : 128;
        g.ncol = (g.N2 + g.nt2 - 1) / g.nt2;
        g.cl = 1; g.ngrp = g.ncol;
        if (g.ncol > 1) {                    // balanced groups of at most max_cluster column tiles
            g.cl = ladder_choose_cluster(g.ncol, b.NQ, num_sms);
            g.ngrp = (g.ncol + g.cl - 1) / g.cl;
        }
        rows += (long long)g.ntiles * g.ngrp * g.cl;
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
    if (const char* e = getenv("RTCC_LADDER_SPLIT")) { int v = atoi(e); if (v >= 1) best = v; }   // tuning knob
    int item = 0;
    for (int i = 0; i < b.ncase; ++i) {
        LadderCase& g = b.c[i];
        const int nchunk = ((g.vA + LD_PE - 1) / LD_PE) * ((g.vB + LD_PF - 1) / LD_PF);
        g.nsplit = best < nchunk ? best : (nchunk > 0 ? nchunk : 1);
        g.item0 = item;
        if (g.cl == 1) item += g.ntiles * g.ncol * g.nsplit;     // only single-column cases run in the batched kernel
    }
    b.nitems = item;
}

// executed tensor-pipe flops of one evaluation
inline double ladder_flops(const LadderBatch& b)
{
    double f = 0.0;
    for (int i = 0; i < b.ncase; ++i) {
        const LadderCase& g = b.c[i];
        double rows = 64.0 * g.ntiles, ef = (double)g.vA * g.vB;
        f += 2.0 * rows * ef * ((double)b.NQ * g.ngrp * (g.cl == 1 ? 1.0 : 1.0) + (double)g.ncol * g.nt2);
    }
    return f;
}

inline int ladder_launch(const LadderBatch& b, cudaStream_t st, int num_sms)
{
    int launches = 0;
    bool red = false;
    if (b.nitems > 0) {
        LadderBatch pb = b;                       // cluster cases take no items of the batched kernel
        for (int i = 0; i < pb.ncase; ++i) if (pb.c[i].cl > 1) pb.c[i].ntiles = 0;
        // (item0 offsets were computed with the cluster cases contributing zero items)
        ladder_kernel<<<b.nitems, LD_NTH, ladder_smem(), st>>>(pb);
        ++launches;
    }
    for (int i = 0; i < b.ncase; ++i) {
        const LadderCase& g = b.c[i];
        red |= g.nsplit > 1;
        if (g.cl <= 1 || g.ntiles <= 0) continue;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)((long long)g.ntiles * g.ngrp * g.nsplit * g.cl));
        cfg.blockDim = dim3(LD_NTH);
        cfg.dynamicSmemBytes = ladder_cluster_smem();
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)g.cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, ladder_cluster_kernel, g, b.NQ);
        ++launches;
    }
    if (red) { ladder_reduce_kernel<<<num_sms * 4, 256, 0, st>>>(b); ++launches; }
    return launches;
}

inline cudaError_t ladder_init()
{
    cudaError_t e = cudaFuncSetAttribute(ladder_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ladder_smem());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(ladder_cluster_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ladder_cluster_smem());
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(ladder_cluster_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
}

}  // namespace rtcc
