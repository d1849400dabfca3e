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
    int cl;                               // 0: batched narrow kernel (one column tile); >= 1: wide kernel, CTAs per cluster
    int ngrp;                             // wide kernel: column-tile groups (each group rebuilds the W chunks)
    int item0;                            // first work item of this case
    int same;                             // p and q (e and f) are of the same spin: X is antisymmetric in (e,f), Y in (p,q)
    int anti;                             // wide kernel, same spin: chunks with e < f only, W antisymmetrised (see ladder_wide_kernel)
};
// (e,f) chunks of a case: all nEt x nFt, or -- antisymmetrised -- those that hold an e < f: ft >= 2 et (16 e x 8 f per chunk)
__host__ __device__ inline int ladder_nchunk(int vA, int vB, int anti)
{
    const int nEt = (vA + 15) / 16, nFt = (vB + 7) / 8;
    if (!anti) return nEt * nFt;
    int n = 0;
    for (int et = 0; et < nEt && 2 * et < nFt; ++et) n += nFt - 2 * et;
    return n;
}
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
// Wide amplitudes (more than one 128-column tile).  One CTA keeps the accumulators of up to LW_MAXC column tiles of its
// 64-row tile: the live tile in registers (FP64 DMMA accumulates in registers only), the others parked in TENSOR MEMORY
// (tcgen05.alloc / tcgen05.ld / tcgen05.st: 8 warps x 32 lanes x 256 columns = 4 parked tiles) and swapped in place when the
// CTA moves to the next tile; tiles are visited in alternating order so that a chunk ends on the tile the next one starts on.
// A thread-block CLUSTER of cl CTAs covers cl * LW_MAXC column tiles.  Every W chunk is built ONCE per cluster: CTA r builds
// the chunks g = r (mod cl) completely (all of n_chol, one cl-th of it per step so that every CTA does the same work in every
// step), writes the finished chunk into one of two shared-memory slots and sends it to the same slot of every other CTA with
// one bulk async copy through distributed shared memory (cp.async.bulk shared::cta -> shared::cluster, completion on the
// receiver's mbarrier) -- the consumer warps never touch remote memory.  Slot reuse is guarded by "credit" mbarriers at the
// builder that every consumer warp of the cluster arrives on when it has finished a chunk.  Fixed summation order
// throughout: bit-reproducible.
constexpr int LW_ST = 3;
constexpr int LW_MAXC = 5;
constexpr int LW_NTH = 384;                             // two consumer warpgroups + one producer warpgroup (register reallocation)
constexpr int LW_WSLOT = LD_R * LD_LDW;                 // doubles per W slot
constexpr int LW_NBAR = 2 * LW_ST + 4;                  // full[ST], empty[ST], wfull[2], credit[2]
constexpr size_t ladder_wide_smem()
{ return sizeof(double) * (LW_ST * (size_t)LD_STAGE + 2 * (size_t)LW_WSLOT) + LW_NBAR * sizeof(unsigned long long) + 16; }

struct LadderWide {
    LadderCase c[3];        // cases batched in one launch share the cluster size
    int ncase, NQ, cl;
};

__device__ __forceinline__ unsigned cluster_rank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ unsigned map_shared(const void* p, unsigned rank)
{
    unsigned a = (unsigned)__cvta_generic_to_shared(p), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
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
// bulk async copy from this CTA's shared memory into a peer's (addresses of the peer obtained with mapa)
__device__ __forceinline__ void bulk_s2peer(unsigned dst_cluster_addr, const void* src, unsigned bytes, unsigned bar_cluster_addr)
{
    asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_cluster_addr), "r"((unsigned)__cvta_generic_to_shared(src)), "r"(bytes), "r"(bar_cluster_addr) : "memory");
}
__device__ __forceinline__ void cluster_sync_all()
{ asm volatile("barrier.cluster.arrive.release.aligned;\n barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// ---- tensor memory: 8 consecutive 32-bit columns of this thread's lane <-> 4 doubles
__device__ __forceinline__ void tmem_ld8(unsigned taddr, unsigned (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st8(unsigned taddr, double d0, double d1, double d2, double d3)
{
    asm volatile("{\n .reg .b32 l0, h0, l1, h1, l2, h2, l3, h3;\n"
                 " mov.b64 {l0, h0}, %1;\n mov.b64 {l1, h1}, %2;\n mov.b64 {l2, h2}, %3;\n mov.b64 {l3, h3}, %4;\n"
                 " tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {l0, h0, l1, h1, l2, h2, l3, h3};\n}"
                 ::"r"(taddr), "d"(d0), "d"(d1), "d"(d2), "d"(d3) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// swap the 32 accumulators of this thread with the parked tile at taddr (64 columns), 4 doubles at a time
__device__ __forceinline__ void tmem_exchange(unsigned taddr, double (&acc)[4][4][2])
{
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            unsigned in[8];
            const unsigned a = taddr + 16 * i + 8 * h;
            tmem_ld8(a, in);
            tmem_wait_ld();
            tmem_st8(a, acc[i][2 * h][0], acc[i][2 * h][1], acc[i][2 * h + 1][0], acc[i][2 * h + 1][1]);
            acc[i][2 * h][0] = __hiloint2double((int)in[1], (int)in[0]);
            acc[i][2 * h][1] = __hiloint2double((int)in[3], (int)in[2]);
            acc[i][2 * h + 1][0] = __hiloint2double((int)in[5], (int)in[4]);
            acc[i][2 * h + 1][1] = __hiloint2double((int)in[7], (int)in[6]);
        }
    tmem_wait_st();
}
__device__ __forceinline__ void tmem_zero64(unsigned taddr)
{
#pragma unroll
    for (int i = 0; i < 8; ++i) tmem_st8(taddr + 8 * i, 0.0, 0.0, 0.0, 0.0);
    tmem_wait_st();
}

// park this thread's 32 accumulators at taddr (64 columns), same element order as tmem_exchange
__device__ __forceinline__ void tmem_put(unsigned taddr, const double (&acc)[4][4][2])
{
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int h = 0; h < 2; ++h)
            tmem_st8(taddr + 16 * i + 8 * h, acc[i][2 * h][0], acc[i][2 * h][1], acc[i][2 * h + 1][0], acc[i][2 * h + 1][1]);
    tmem_wait_st();
}

// Antisymmetrised same-spin form (LadderCase::anti).  X^{ef} = -X^{fe}, so
//   Y^{pq} = sum_{e<f} [ (pe|qf) - (pf|qe) ] X^{ef}:
// only chunks that hold an e < f are visited (rows e >= f of the tile-major X are zero), each with TWO W products -- first
// (pe|qf) from the (p0, et) x (q0, ft) operand tiles, parked in the free tensor-memory slot, then (qe|pf) = (pf|qe) from the
// (q0, et) x (p0, ft) tiles -- combined in the shared-memory slot, and ONE application: the same W-build flops as the plain form
// (which visits every (e,f)), about half the apply flops.  A CTA then holds at most 4 column tiles (one slot is the parking place).
__global__ void __launch_bounds__(LW_NTH, 1) ladder_wide_kernel(const LadderWide b)
{
    constexpr int NT2 = 128, LDX2 = NT2 + 4, T2 = LD_K2 / LD_BK;
    constexpr int BLKA = LD_BK * LD_LDA1, BLKB = LD_BK * LD_LDB1, BLKX = LD_BK * LDX2;
    extern __shared__ __align__(128) double smem[];
    double* stg = smem;
    double* Wsl = smem + LW_ST * LD_STAGE;                                   // two W slots
    unsigned long long* full = reinterpret_cast<unsigned long long*>(Wsl + 2 * LW_WSLOT);
    unsigned long long* empty = full + LW_ST;
    unsigned long long* wfull = empty + LW_ST;                                // [2]: chunk landed in slot
    unsigned long long* credit = wfull + 2;                                   // [2]: slot released by every consumer warp of the cluster
    unsigned* tmem_base_p = reinterpret_cast<unsigned*>(credit + 2);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cl = b.cl, NQ = b.NQ;
    const int rank = (int)cluster_rank();
    int item = blockIdx.x / cl;
    int ci = 0;
    if (b.ncase > 1 && item >= b.c[1].item0) ci = 1;
    if (b.ncase > 2 && item >= b.c[2].item0) ci = 2;
    const LadderCase& g = b.c[ci];
    item -= g.item0;
    const int split = item % g.nsplit; item /= g.nsplit;
    const int grp = item % g.ngrp;
    const int2 tl = g.tiles[item / g.ngrp];
    const int p0 = tl.x, q0 = tl.y;
    // column tiles of this CTA: group grp holds tiles [gt0, gt1), split evenly over the cl ranks
    const int gt0 = (int)((long long)grp * g.ncol / g.ngrp), gt1 = (int)((long long)(grp + 1) * g.ncol / g.ngrp);
    const int ct0 = gt0 + (int)((long long)rank * (gt1 - gt0) / cl), ct1 = gt0 + (int)((long long)(rank + 1) * (gt1 - gt0) / cl);
    const int Ct = ct1 - ct0;                                                 // 0 .. LW_MAXC
    const int nEt = (g.vA + LD_PE - 1) / LD_PE, nFt = (g.vB + LD_PF - 1) / LD_PF;
    const int anti = g.anti;
    const int nchunk = ladder_nchunk(g.vA, g.vB, anti);
    const int ch0 = (int)((long long)split * nchunk / g.nsplit), ch1 = (int)((long long)(split + 1) * nchunk / g.nsplit);
    const int G = ch1 - ch0;
    const int T1 = NQ / LD_BK;
    const int TB = anti ? 2 * T1 : T1;                                       // k-tiles of one W build

    if (tid == 0) {
        for (int s = 0; s < LW_ST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 8); }
        for (int s = 0; s < 2; ++s) { mbar_init(&wfull[s], 1); mbar_init(&credit[s], 8 * cl); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        // chunks 0 and 1 arrive from their builders without a preceding release of the slot: arm their barriers here
        for (int s = 0; s < 2; ++s)
            if (s < G && s % cl != rank) mbar_expect_tx(&wfull[s], LW_WSLOT * 8);
    }
    if (warp == 8) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"((unsigned)__cvta_generic_to_shared(tmem_base_p)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem_base = *tmem_base_p;
    cluster_sync_all();                                                       // every CTA's barriers exist

    // Both roles walk the same schedule.  Chunk g (0-based within [ch0, ch1)) is built by rank g % cl, published at the start
    // of step g-1 and consumed in step g.  A build is spread over the cl steps before its publication.
    if (warp >= 8) {
        // producer warpgroup: hands its registers to the consumers (the kernel is compiled for 168 registers per thread,
        // 3 warpgroups; the consumers need ~220 to keep both accumulator sets out of local memory)
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;" ::: "memory");
        if (warp == 8 && lane == 0) {
            const double* LAp = g.LA + (long long)(p0 / LD_PP) * nEt * T1 * BLKA;
            const double* LBp = g.LB + (long long)(q0 / LD_PQ) * nFt * T1 * BLKB;
            int stage = 0; unsigned par = 1;
            // second product of the antisymmetrised form: rows (q, e), columns (p, f)
            const double* LAq = g.LA + (long long)(q0 / LD_PP) * nEt * T1 * BLKA;
            const double* LBq = g.LB + (long long)(p0 / LD_PQ) * nFt * T1 * BLKB;
            auto chunk_ef = [&](int ch, int& et, int& ft) {
                if (!anti) { et = ch / nFt; ft = ch % nFt; return; }
                et = 0;
                while (ch >= nFt - 2 * et) { ch -= nFt - 2 * et; ++et; }
                ft = 2 * et + ch;
            };
            auto issue_L = [&](int ch, int k0, int k1) {
                int et, ft;
                chunk_ef(ch, et, ft);
                for (int t = k0; t < k1; ++t) {
                    const int tt = t < T1 ? t : t - T1;
                    const double* curA = (t < T1 ? LAp : LAq) + ((long long)et * T1 + tt) * BLKA;
                    const double* curB = (t < T1 ? LBp : LBq) + ((long long)ft * T1 + tt) * BLKB;
                    mbar_wait(&empty[stage], par);
                    double* sb = stg + stage * LD_STAGE;
                    mbar_expect_tx(&full[stage], (BLKA + BLKB) * 8);
                    bulk_g2s(sb, curA, BLKA * 8, &full[stage]);
                    bulk_g2s(sb + BLKA, curB, BLKB * 8, &full[stage]);
                    if (++stage == LW_ST) { stage = 0; par ^= 1; }
                }
            };
            int gb = rank, kdone = 0;
            for (int s = -2; s < G; ++s) {
                if (s >= -1 && s + 1 < G && (s + 1) % cl == rank) { gb = s + 1 + cl; kdone = 0; }
                if (gb < G && kdone < TB) {
                    const int rem = gb - 1 - s;
                    const int nk = (TB - kdone + rem - 1) / rem;
                    issue_L(ch0 + gb, kdone, kdone + nk);
                    kdone += nk;
                }
                if (s >= 0 && Ct > 0) {
                    int et, ft;
                    chunk_ef(ch0 + s, et, ft);
                    const double* Xc = g.X + ((long long)(et * nFt + ft) * g.ncol) * T2 * BLKX;
                    for (int u = 0; u < Ct; ++u) {
                        const int tile = (s & 1) ? Ct - 1 - u : u;
                        const double* curX = Xc + (long long)(ct0 + tile) * T2 * BLKX;
                        for (int t = 0; t < T2; ++t) {
                            mbar_wait(&empty[stage], par);
                            mbar_expect_tx(&full[stage], BLKX * 8);
                            bulk_g2s(stg + stage * LD_STAGE, curX, BLKX * 8, &full[stage]);
                            curX += BLKX;
                            if (++stage == LW_ST) { stage = 0; par ^= 1; }
                        }
                    }
                }
            }
        }
        __syncwarp();
    } else {
        // ---------------- consumers
        asm volatile("setmaxnreg.inc.sync.aligned.u32 232;" ::: "memory");
        const int lr = lane >> 2, lc = lane & 3;
        double acc2[4][4][2], acc1[4][4][2];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) acc2[i][j][0] = acc2[i][j][1] = acc1[i][j][0] = acc1[i][j][1] = 0.0;
        const int w1m = (warp >> 1) * 32, w1n = (warp & 1) * 32;
        const int w2m = (warp >> 2) * 32, w2n = (warp & 3) * 32;
        // this warp's tensor-memory region: lanes 32 (warp % 4) .., columns 256 (warp / 4) + 64 slot
        const unsigned tm0 = tmem_base + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)((warp >> 2) * 256);
        for (int s = 0; s + 1 < Ct; ++s) tmem_zero64(tm0 + 64 * s);      // parked tiles start at zero
        const unsigned tm_stash = tm0 + 64 * (LW_MAXC - 2);                  // antisymmetrised form: parking place of the first W product

        int stage = 0; unsigned par = 0;
        unsigned cpar = 0u;                                                   // bit sl: parity of credit[sl]
        // acc1 = W[(p,e),(q,f)] of chunk gc -> slot gc % 2 as [(p,q)][(e,f)], here and in every other CTA of the cluster
        auto publish = [&](int gc) {
            const int sl = gc & 1;
            if (gc >= 2) { mbar_wait_cluster(&credit[sl], (cpar >> sl) & 1u); cpar ^= 1u << sl; }     // every warp of the cluster is done with chunk gc-2
            double* Ws = Wsl + sl * LW_WSLOT;
            if (anti) {
                // first product back from tensor memory into its places, then the second one subtracted at the places of the
                // transposed (p,q) -- other threads' elements, hence the barrier in between
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int m = w1m + 8 * i + lr;
                    const int p = m / LD_PE, e = m % LD_PE;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        unsigned in[8];
                        tmem_ld8(tm_stash + 16 * i + 8 * h, in);
                        tmem_wait_ld();
#pragma unroll
                        for (int jj = 0; jj < 2; ++jj) {
                            const int n = w1n + 8 * (2 * h + jj) + 2 * lc;
                            const int q = n / LD_PF, f = n % LD_PF;
                            *reinterpret_cast<double2*>(&Ws[(p * LD_PQ + q) * LD_LDW + e * LD_PF + f]) =
                                make_double2(__hiloint2double((int)in[4 * jj + 1], (int)in[4 * jj]), __hiloint2double((int)in[4 * jj + 3], (int)in[4 * jj + 2]));
                        }
                    }
                }
                bar_consumers();
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int m = w1m + 8 * i + lr;
                    const int q = m / LD_PE, e = m % LD_PE;
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int n = w1n + 8 * j + 2 * lc;
                        const int p = n / LD_PF, f = n % LD_PF;
                        double2* w = reinterpret_cast<double2*>(&Ws[(p * LD_PQ + q) * LD_LDW + e * LD_PF + f]);
                        double2 v = *w;
                        v.x -= acc1[i][j][0]; v.y -= acc1[i][j][1];
                        *w = v;
                        acc1[i][j][0] = acc1[i][j][1] = 0.0;
                    }
                }
            } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int m = w1m + 8 * i + lr;
                const int p = m / LD_PE, e = m % LD_PE;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int n = w1n + 8 * j + 2 * lc;
                    const int q = n / LD_PF, f = n % LD_PF;
                    *reinterpret_cast<double2*>(&Ws[(p * LD_PQ + q) * LD_LDW + e * LD_PF + f]) = make_double2(acc1[i][j][0], acc1[i][j][1]);
                    acc1[i][j][0] = acc1[i][j][1] = 0.0;
                }
            }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");          // generic-proxy writes -> visible to the bulk copies
            bar_consumers();
            if (tid == 0) {
                for (int r = 1; r < cl; ++r) {
                    const unsigned peer = (unsigned)((rank + r) % cl);
                    bulk_s2peer(map_shared(Ws, peer), Ws, LW_WSLOT * 8, map_shared(&wfull[sl], peer));
                }
                mbar_arrive(&wfull[sl]);
            }
        };

        // steps -2 and -1 are the prologue: the first chunk of rank r is built over the steps -2 .. r-2
        int gb = rank, kdone = 0;
        for (int s = -2; s < G; ++s) {
            if (s >= -1 && s + 1 < G && (s + 1) % cl == rank) { publish(s + 1); gb = s + 1 + cl; kdone = 0; }
            if (gb < G && kdone < TB) {
                const int rem = gb - 1 - s;
                const int nk = (TB - kdone + rem - 1) / rem;
                const int kfirst = kdone;
                kdone += nk;
                for (int t = 0; t < nk; ++t) {
                    if (anti && kfirst + t == T1) {                           // first product complete: park it, start the second
                        tmem_put(tm_stash, acc1);
#pragma unroll
                        for (int i = 0; i < 4; ++i)
#pragma unroll
                            for (int j = 0; j < 4; ++j) acc1[i][j][0] = acc1[i][j][1] = 0.0;
                    }
                    mbar_wait(&full[stage], par);
                    const double* sb = stg + stage * LD_STAGE;
                    const double* as = sb + lc * LD_LDA1 + w1m + lr;
                    const double* bs = sb + LD_BK * LD_LDA1 + lc * LD_LDB1 + w1n + lr;
#pragma unroll
                    for (int ks = 0; ks < LD_BK / 4; ++ks) {
                        double a[4], bb[4];
#pragma unroll
                        for (int i = 0; i < 4; ++i) a[i] = as[ks * 4 * LD_LDA1 + 8 * i];
#pragma unroll
                        for (int j = 0; j < 4; ++j) bb[j] = bs[ks * 4 * LD_LDB1 + 8 * j];
#pragma unroll
                        for (int i = 0; i < 4; ++i)
#pragma unroll
                            for (int j = 0; j < 4; ++j) dmma884(acc1[i][j][0], acc1[i][j][1], a[i], bb[j]);
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[stage]);
                    if (++stage == LW_ST) { stage = 0; par ^= 1; }
                }
            }
            if (s < 0) continue;
            const int sl = s & 1;
            mbar_wait(&wfull[sl], (unsigned)((s >> 1) & 1));
            const double* Ws = Wsl + sl * LW_WSLOT;
            for (int u = 0; u < Ct; ++u) {
                if (u > 0) {                                                  // next tile: up in even steps, down in odd ones
                    const int prev = (s & 1) ? Ct - u : u - 1;               // live tile before the move
                    tmem_exchange(tm0 + 64 * ((s & 1) ? prev - 1 : prev), acc2);
                }
                for (int t = 0; t < T2; ++t) {
                    mbar_wait(&full[stage], par);
                    const double* sb = stg + stage * LD_STAGE;
                    const double* ws = Ws + (w2m + lr) * LD_LDW + t * LD_BK + lc;
                    const double* xs = sb + lc * LDX2 + w2n + lr;
#pragma unroll
                    for (int ks = 0; ks < LD_BK / 4; ++ks) {
                        double a[4], bb[4];
#pragma unroll
                        for (int i = 0; i < 4; ++i) a[i] = ws[8 * i * LD_LDW + ks * 4];
#pragma unroll
                        for (int j = 0; j < 4; ++j) bb[j] = xs[ks * 4 * LDX2 + 8 * j];
#pragma unroll
                        for (int i = 0; i < 4; ++i)
#pragma unroll
                            for (int j = 0; j < 4; ++j) dmma884(acc2[i][j][0], acc2[i][j][1], a[i], bb[j]);
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[stage]);
                    if (++stage == LW_ST) { stage = 0; par ^= 1; }
                }
            }
            // this warp is done with chunk s: arm the slot for chunk s+2 (if it comes from a peer) and release it to its builder
            if (s + 2 < G) {
                const int bld = (s + 2) % cl;
                __syncwarp();
                if (tid == 0 && bld != rank) mbar_expect_tx(&wfull[sl], LW_WSLOT * 8);
                if (lane == 0) mbar_arrive_cluster(map_shared(&credit[sl], (unsigned)bld));
            }
        }
        // write the Ct tiles: the live one first, then continue the alternating walk
        double* Yout = g.nsplit > 1 ? g.Ypart + (long long)split * g.nA * g.nB * g.ldY : g.Y;
        for (int u = 0; u < Ct; ++u) {
            const bool down = (G & 1) == 0 ? false : true;                    // step G would walk down if G is odd
            int tile;
            if (u > 0) {
                const int prev = down ? Ct - u : u - 1;
                tmem_exchange(tm0 + 64 * (down ? prev - 1 : prev), acc2);
            }
            tile = down ? Ct - 1 - u : u;
            const int x0 = (ct0 + tile) * NT2;
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
    // no CTA may retire while a sibling can still copy into its shared memory or arrive on its barriers
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    cluster_sync_all();
    if (warp == 8) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
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

// SMs that clusters of cl CTAs of the wide kernel can keep busy at once (0: size not schedulable)
struct LadderOcc { int act[17]; };
inline void ladder_probe_occupancy(LadderOcc& o, int num_sms)
{
    for (int c = 0; c <= 16; ++c) o.act[c] = 0;
    for (int c = 1; c <= 16; ++c) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)c * 64); cfg.blockDim = dim3(LW_NTH); cfg.dynamicSmemBytes = ladder_wide_smem();
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)c; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, ladder_wide_kernel, &cfg) == cudaSuccess && n > 0) o.act[c] = n * c > num_sms ? num_sms : n * c;
        cudaGetLastError();
    }
    if (o.act[1] <= 0) o.act[1] = num_sms;
}
// Cluster size and column groups for ncol column tiles.  A CTA holds at most LW_MAXC tiles; the W chunks are rebuilt once per
// group, so the fewest groups win, then the estimated time  (W1 + cl * ceil(tiles / cl) * W2) / active SMs  per row tile and
// chunk (W1: building one chunk, W2: applying it to one column tile; the busiest CTA of the cluster sets the pace).
struct LadderTune { int max_cluster = 16, force_cluster = 0, max_tiles = LW_MAXC, force_split = 0, overlap = 1, anti = 1; };
inline void ladder_choose_cluster(int ncol, int NQ, const LadderOcc& occ, const LadderTune& tune_in, int anti, int& cl_out, int& ngrp_out)
{
    LadderTune tune = tune_in;
    if (anti && tune.max_tiles > LW_MAXC - 1) tune.max_tiles = LW_MAXC - 1;     // one tensor-memory slot parks the first W product
    const double W1 = 128.0 * 64.0 * NQ * (anti ? 2 : 1), W2 = 64.0 * 128.0 * 128.0;
    int maxc = 16, minc = 1;
    if (tune.max_cluster >= 1 && tune.max_cluster < maxc) maxc = tune.max_cluster;
    if (tune.force_cluster >= 1 && tune.force_cluster <= 16 && occ.act[tune.force_cluster] > 0) minc = maxc = tune.force_cluster;
    const int maxt = tune.max_tiles >= 1 && tune.max_tiles < LW_MAXC ? tune.max_tiles : LW_MAXC;
    for (int ngrp = 1; ngrp <= ncol; ++ngrp) {
        const int ng = (ncol + ngrp - 1) / ngrp;            // tiles of the largest group
        int best = 0; double bt = 1e300;
        for (int cl = minc; cl <= maxc; ++cl) {
            if (occ.act[cl] <= 0 || (long long)cl * maxt < ng) continue;
            const int per = (ng + cl - 1) / cl;
            const double t = (W1 + (double)cl * per * W2) / occ.act[cl];
            if (t < bt * (1.0 - 1e-9)) { bt = t; best = cl; }
        }
        if (best > 0) { cl_out = best; ngrp_out = ngrp; return; }
    }
    cl_out = 1; ngrp_out = (ncol + maxt - 1) / maxt;
}

// Host side: column tile width, cluster shape and (e,f) slicing per spin case.  Narrow cases (one column tile) run in the batched
// kernel, wide ones in the tensor-memory kernel; max_split bounds the (e,f) slices (each slice needs a partial output buffer).
inline void ladder_plan(LadderBatch& b, int num_sms, int max_split, const LadderOcc& occ, const LadderTune& tune)
{
    long long rows = 0;
    for (int i = 0; i < b.ncase; ++i) {
        LadderCase& g = b.c[i];
        g.nt2 = g.N2 <= 64 ? 64 : 128;
        g.ncol = (g.N2 + g.nt2 - 1) / g.nt2;
        g.cl = 0; g.ngrp = 1;                 // cl = 0: batched narrow kernel
        g.anti = (g.same && g.ncol > 1 && tune.anti) ? 1 : 0;
        if (g.ncol > 1) ladder_choose_cluster(g.ncol, b.NQ, occ, tune, g.anti, g.cl, g.ngrp);
        else rows += g.ntiles;
    }
    // One launch for all wide cases when a common cluster size costs no case more than 3 % (modelled): separate launches
    // each end in a partly filled last wave.
    {
        const double W2 = 64.0 * 128.0 * 128.0;
        auto cost = [&](const LadderCase& g, int cl) {
            if (cl < 1 || cl > 16 || occ.act[cl] <= 0) return 1e300;
            const double W1 = 128.0 * 64.0 * b.NQ * (g.anti ? 2 : 1);
            const int ng = (g.ncol + g.ngrp - 1) / g.ngrp, per = (ng + cl - 1) / cl;
            int maxt = tune.max_tiles >= 1 && tune.max_tiles < LW_MAXC ? tune.max_tiles : LW_MAXC;
            if (g.anti && maxt > LW_MAXC - 1) maxt = LW_MAXC - 1;
            if (per > maxt) return 1e300;
            return (W1 + (double)cl * per * W2) / occ.act[cl];
        };
        int common = 0;
        for (int i = 0; i < b.ncase && !common; ++i) {
            const int cand = b.c[i].cl;
            if (cand <= 0) continue;
            bool ok = true;
            for (int k = 0; k < b.ncase; ++k)
                if (b.c[k].cl > 0 && cost(b.c[k], cand) > 1.03 * cost(b.c[k], b.c[k].cl)) ok = false;
            if (ok) common = cand;
        }
        if (common && tune.force_cluster < 1)
            for (int k = 0; k < b.ncase; ++k) if (b.c[k].cl > 0) b.c[k].cl = common;
    }
    // narrow cases: slices so that the items fill the SMs evenly
    int best = 1;
    if (rows > 0 && rows < 8LL * num_sms) {
        double beff = 0.0;
        for (int S = 1; S <= max_split; ++S) {
            double w = (double)rows * S / num_sms;
            double eff = w / ceil(w);
            if (eff > beff + 0.02) { beff = eff; best = S; }
        }
    }
    if (tune.force_split >= 1) best = tune.force_split;
    int item = 0;
    for (int i = 0; i < b.ncase; ++i) {
        LadderCase& g = b.c[i];
        const int nchunk = ladder_nchunk(g.vA, g.vB, g.anti);
        g.item0 = 0;
        if (g.cl == 0) {
            g.nsplit = best < nchunk ? best : (nchunk > 0 ? nchunk : 1);
            g.item0 = item;
            item += g.ntiles * g.ncol * g.nsplit;
        }
    }
    b.nitems = item;
    // wide cases: launches are grouped by cluster size; slices only when a launch has few waves
    for (int i = 0; i < b.ncase; ++i) {
        LadderCase& g = b.c[i];
        if (g.cl == 0) continue;
        bool first = true;
        for (int k = 0; k < i; ++k) first &= b.c[k].cl != g.cl;
        if (!first) continue;
        long long clusters = 0;
        for (int k = i; k < b.ncase; ++k) if (b.c[k].cl == g.cl) clusters += (long long)b.c[k].ntiles * b.c[k].ngrp;
        // wide launches are not sliced on their own: every slice needs a partial output buffer the size of Y (GBs at the
        // sizes that run here) for a gain of a few per cent in wave quantisation
        (void)clusters;
        int S = 1;
        if (tune.force_split >= 1) S = tune.force_split;
        int it = 0;
        for (int k = i; k < b.ncase; ++k) {
            LadderCase& h = b.c[k];
            if (h.cl != g.cl) continue;
            const int nchunk = ladder_nchunk(h.vA, h.vB, h.anti);
            h.nsplit = S < nchunk ? S : (nchunk > 0 ? nchunk : 1);
            h.item0 = it;
            it += h.ntiles * h.ngrp * h.nsplit;
        }
    }
}

// executed tensor-pipe flops of one evaluation
inline double ladder_flops(const LadderBatch& b)
{
    double f = 0.0;
    for (int i = 0; i < b.ncase; ++i) {
        const LadderCase& g = b.c[i];
        double rows = 64.0 * g.ntiles, ef = (double)g.vA * g.vB;
        if (g.anti) ef *= (double)ladder_nchunk(g.vA, g.vB, 1) / ladder_nchunk(g.vA, g.vB, 0);      // chunks visited; two W products each
        f += 2.0 * rows * ef * ((double)b.NQ * g.ngrp * (g.anti ? 2 : 1) + (double)g.ncol * g.nt2);
    }
    return f;
}

// side / ev_fork / ev_join (optional): the second and later wide launches go to `side` so that their CTAs fill the partly
// empty last wave of the first one (one CTA per SM: launches on one stream would each end in their own tail); `st` waits for them.
inline int ladder_launch(const LadderBatch& b, cudaStream_t st, int num_sms, cudaStream_t side = nullptr,
                         cudaEvent_t ev_fork = nullptr, cudaEvent_t ev_join = nullptr, int overlap = 1)
{
    int launches = 0;
    bool red = false;
    if (b.nitems > 0) {
        LadderBatch pb = b;                       // wide cases take no items of the batched kernel
        for (int i = 0; i < pb.ncase; ++i) if (pb.c[i].cl > 0) pb.c[i].ntiles = 0;
        ladder_kernel<<<b.nitems, LD_NTH, ladder_smem(), st>>>(pb);
        ++launches;
    }
    // the wide launches, one per cluster size
    LadderWide wl[3]; long long wcl[3]; int nwl = 0;
    for (int i = 0; i < b.ncase; ++i) {
        const LadderCase& g = b.c[i];
        red |= g.nsplit > 1;
        if (g.cl <= 0 || g.ntiles <= 0) continue;
        bool first = true;
        for (int k = 0; k < i; ++k) first &= b.c[k].cl != g.cl || b.c[k].ntiles <= 0;
        if (!first) continue;
        LadderWide& w = wl[nwl];
        w.ncase = 0; w.NQ = b.NQ; w.cl = g.cl;
        long long clusters = 0;
        for (int k = i; k < b.ncase; ++k)
            if (b.c[k].cl == g.cl && b.c[k].ntiles > 0) { w.c[w.ncase++] = b.c[k]; clusters += (long long)b.c[k].ntiles * b.c[k].ngrp * b.c[k].nsplit; }
        wcl[nwl++] = clusters;
    }
    bool forked = false;
    if (nwl > 1 && overlap && side && ev_fork && ev_join) {  // fork BEFORE the first wide launch: `side` must not wait for it
        cudaEventRecord(ev_fork, st); cudaStreamWaitEvent(side, ev_fork, 0); forked = true;
    }
    // side by side: longest CTAs first (their tail is filled by the shorter CTAs of the later launches)
    int ord[3] = {0, 1, 2};
    if (overlap) {
        double cost[3];
        for (int i = 0; i < nwl; ++i) {
            int per = 0;
            for (int k = 0; k < wl[i].ncase; ++k) {
                const LadderCase& g = wl[i].c[k];
                const int ng = (g.ncol + g.ngrp - 1) / g.ngrp, p = (ng + g.cl - 1) / g.cl;
                if (p > per) per = p;
            }
            cost[i] = 128.0 * 64.0 * b.NQ / wl[i].cl + per * 64.0 * 128.0 * 128.0;
            if (overlap == 2) cost[i] = -cost[i];
        }
        for (int i = 0; i < nwl; ++i)
            for (int k = i + 1; k < nwl; ++k)
                if (cost[ord[k]] > cost[ord[i]]) { const int t = ord[i]; ord[i] = ord[k]; ord[k] = t; }
    }
    for (int u = 0; u < nwl; ++u) {
        const int i = ord[u];
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(wcl[i] * wl[i].cl));
        cfg.blockDim = dim3(LW_NTH);
        cfg.dynamicSmemBytes = ladder_wide_smem();
        cfg.stream = (u > 0 && forked) ? side : st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)wl[i].cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, ladder_wide_kernel, wl[i]);
        ++launches;
    }
    if (forked) { cudaEventRecord(ev_join, side); cudaStreamWaitEvent(st, ev_join, 0); }
    if (red) { ladder_reduce_kernel<<<num_sms * 4, 256, 0, st>>>(b); ++launches; }
    return launches;
}

inline cudaError_t ladder_init()
{
    cudaError_t e = cudaFuncSetAttribute(ladder_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ladder_smem());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(ladder_wide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ladder_wide_smem());
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(ladder_wide_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
}

}  // namespace rtcc
