// tcgemm.cuh -- FP64 tensor-core (DMMA m8n8k4) tensor-contraction GEMM for sm_100a.
//
// C(m,n) = alpha * sum_phases s_p * sum_k A_p(m,k) B_p(k,n) + beta * C(m,n)
//
// Every index of the three operands is a two-level index (hi,lo) with independent strides, so a
// contraction over e.g. k=(Q,i) or an output scattered as [(m,e)][(j,b)] needs no transposition
// pass.  Up to two phases with signs implement complex products on planar (Re/Im) storage:
//   Re C = A_re B_re - A_im B_im,   Im C = A_re B_im + A_im B_re        (real integrals x complex
//   amplitudes need one phase only; "mixed real-complex contractions").
// Operands are staged global -> shared with 8-byte cp.async (zero-filled out of range: no
// alignment or size restrictions), three stages deep; fragments are read with conflict-free
// 64-bit LDS (row pitch == 4 mod 16 doubles) and fed to mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4, the
// only FP64 tensor shape sm_100a has -- tcgen05 has no f64 kind).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

namespace rtcc {

constexpr int TG_MAXB = 4;

struct TcGemm {
    int M, N, K;
    int Mlo, Nlo, Klo;                       // extents of the "lo" part of each index (>=1)
    long long am_hi, am_lo, ak_hi, ak_lo;    // A(m,k) strides
    long long bk_hi, bk_lo, bn_hi, bn_lo;    // B(k,n) strides
    long long cm_hi, cm_lo, cn_hi, cn_lo;    // C(m,n) strides
    int nb;                                  // descriptor batches (<= TG_MAXB)
    const double* A[TG_MAXB][2];
    const double* B[TG_MAXB][2];
    double* C[TG_MAXB];
    double* C2[TG_MAXB];                     // optional second output with the strides of C (the same product lands in both)
    signed char nphase[TG_MAXB], s0[TG_MAXB], s1[TG_MAXB];
    int nsb;                                 // strided batches
    long long sbA, sbB, sbC;
    double alpha, beta;
    int a_kfast, b_nfast;                    // which index of A / B is contiguous in memory
    int a_klin, b_klin;                      // k index of A / B is effectively single-level (set by the launcher)
    int ksplit;                              // deterministic split-K (partials in ws, reduced by a 2nd kernel)
    double* ws;
    const long long* cm_table;               // optional: offset of output row m (replaces the two-level row index of C)
    int sym_upper;                           // the product is symmetric and only C + C^T is used downstream: tiles above the diagonal
                                             // are computed and doubled, diagonal tiles computed, tiles below written as alpha*0 + beta*C
};

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc, bool valid)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ long long idx2(int x, int lo, long long s_hi, long long s_lo)
{
    if (lo >= 0x40000000) return (long long)x * s_lo;   // single-level fast path
    int h = x / lo;
    return (long long)h * s_hi + (long long)(x - h * lo) * s_lo;
}

// ---- mbarrier / async-copy helpers (shared with ladder.cuh)
__device__ __forceinline__ void mbar_init(unsigned long long* b, int count)
{ asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(b)), "r"(count)); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* b, unsigned bytes)
{ asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(b)), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_arrive(unsigned long long* b)
{ asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((unsigned)__cvta_generic_to_shared(b)) : "memory"); }
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity)
{
    const unsigned addr = (unsigned)__cvta_generic_to_shared(b);
    unsigned ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    } while (!ok);
}
// the barrier receives one arrival when all cp.async issued so far by this thread have landed
__device__ __forceinline__ void cp_async_mbar_arrive(unsigned long long* b)
{ asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"((unsigned)__cvta_generic_to_shared(b)) : "memory"); }
// 8-byte async copy, zero-filled when !valid (ignore-src predicate form: no size arithmetic)
__device__ __forceinline__ void cp_async8p(void* smem_dst, const void* gsrc, bool valid)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("{\n .reg .pred p;\n setp.eq.u32 p, %2, 0;\n cp.async.ca.shared.global [%0], [%1], 8, p;\n}" ::"r"(d), "l"(gsrc), "r"((unsigned)valid) : "memory");
}

// Warp-specialised: (BM/WM)*(BN/WN) consumer warps (LDS + DMMA only) and half as many producer warps that
// gather the tiles with 8-byte cp.async through a 4-stage mbarrier ring.
template <int BM, int BN, int WM, int WN>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 48) tcgemm_kernel(const TcGemm g)
{
    constexpr int BK = 16, ST = 4;
    constexpr int NCW = (BM / WM) * (BN / WN), NPW = NCW / 2;
    constexpr int NTH = (NCW + NPW) * 32, NP = NPW * 32;
    constexpr int LDA = BK + 4, LDB = BN + 4;
    constexpr int EA = BM * BK / NP, EB = BK * BN / NP;      // 16 each
    constexpr int TM = WM / 8, TN = WN / 8;
    static_assert(NP % BM == 0 && NP % BN == 0 && NP % BK == 0, "producer mapping");
    extern __shared__ __align__(128) double smem[];
    double* As = smem;                        // [ST][BM][LDA]
    double* Bs = smem + ST * BM * LDA;        // [ST][BK][LDB]
    long long* rowA = (long long*)(Bs + ST * BK * LDB);   // [BM] offsets (or -1)
    long long* colB = rowA + BM;                          // [BN]
    unsigned long long* full = (unsigned long long*)(colB + BN);
    unsigned long long* empty = full + ST;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int z = blockIdx.z;
    const int split = z % g.ksplit; z /= g.ksplit;
    const int sb = z % g.nsb;
    const int db = z / g.nsb;
    const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;

    for (int i = tid; i < BM; i += NTH) {
        int m = m0 + i;
        rowA[i] = (m < g.M) ? idx2(m, g.Mlo, g.am_hi, g.am_lo) : -1;
    }
    for (int i = tid; i < BN; i += NTH) {
        int n = n0 + i;
        colB[i] = (n < g.N) ? idx2(n, g.Nlo, g.bn_hi, g.bn_lo) : -1;
    }
    if (tid == 0) {
        for (int s = 0; s < ST; ++s) { mbar_init(&full[s], NP); mbar_init(&empty[s], NCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int nkt = (g.K + BK - 1) / BK;
    const int per = (nkt + g.ksplit - 1) / g.ksplit;
    const int kt0 = split * per;
    const int kt1 = min(nkt, kt0 + per);
    const bool lower = g.sym_upper && m0 > n0;
    const double symfac = (g.sym_upper && m0 < n0) ? 2.0 : 1.0;
    const int nk = lower ? 0 : max(kt1 - kt0, 0);
    const int nph = g.nphase[db];
    const int total = nk * nph;

    if (warp >= NCW) {
        // ------------------------------------------------------------ producers
        const int p = tid - NCW * 32;
        const double* Ap[2] = {g.A[db][0] + sb * g.sbA, g.A[db][1] + sb * g.sbA};
        const double* Bp[2] = {g.B[db][0] + sb * g.sbB, g.B[db][1] + sb * g.sbB};
        const bool k1a = g.a_klin, k1b = g.b_klin;      // single-level k per operand
        const int a_kfast = g.a_kfast, b_nfast = g.b_nfast;
        // kfast: this thread owns k-column (p % 16) of rows p/16 + (NP/16) j;  otherwise row p, all 16 k
        long long ra[EA];                               // row offsets (kfast) -- or ra[0] only
        if (a_kfast) {
#pragma unroll
            for (int j = 0; j < EA; ++j) ra[j] = rowA[p / BK + (NP / BK) * j];
        } else ra[0] = rowA[p % BM];
        long long cb[EB];
        if (!b_nfast) {
#pragma unroll
            for (int j = 0; j < EB; ++j) cb[j] = colB[p / BK + (NP / BK) * j];
        } else cb[0] = colB[p % BN];
        int stage = 0; unsigned par = 1;
        for (int t = 0; t < total; ++t) {
            const int ph = t >= nk ? 1 : 0;
            const int kbase = (kt0 + (t - ph * nk)) * BK;
            const double* A = Ap[ph];
            const double* B = Bp[ph];
            mbar_wait(&empty[stage], par);
            double* as = As + stage * BM * LDA;
            double* bs = Bs + stage * BK * LDB;
            if (a_kfast) {
                const int kk = p % BK, k = kbase + kk;
                const bool kv = k < g.K;
                const double* Ak = A + (kv ? (k1a ? (long long)k * g.ak_lo : idx2(k, g.Klo, g.ak_hi, g.ak_lo)) : 0);
                double* d = as + (p / BK) * LDA + kk;
#pragma unroll
                for (int j = 0; j < EA; ++j) {
                    const bool v = kv && ra[j] >= 0;
                    cp_async8p(d + (NP / BK) * j * LDA, v ? Ak + ra[j] : A, v);
                }
            } else {
                const bool rv = ra[0] >= 0;
                const double* Ar = A + (rv ? ra[0] : 0);
                const int kq = (p / BM) * EA;                    // this thread's k sub-range of the tile
                double* d = as + (p % BM) * LDA + kq;
                if (k1a) {
                    const double* s = Ar + (long long)(kbase + kq) * g.ak_lo;
#pragma unroll
                    for (int j = 0; j < EA; ++j) {
                        const bool v = rv && (kbase + kq + j < g.K);
                        cp_async8p(d + j, v ? s : A, v);
                        s += g.ak_lo;
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < EA; ++j) {
                        const bool v = rv && (kbase + kq + j < g.K);
                        cp_async8p(d + j, v ? Ar + idx2(kbase + kq + j, g.Klo, g.ak_hi, g.ak_lo) : A, v);
                    }
                }
            }
            if (b_nfast) {
                const bool cv = cb[0] >= 0;
                const double* Bc = B + (cv ? cb[0] : 0);
                const int kq = (p / BN) * EB;
                double* d = bs + kq * LDB + p % BN;
                if (k1b) {
                    const double* s = Bc + (long long)(kbase + kq) * g.bk_lo;
#pragma unroll
                    for (int j = 0; j < EB; ++j) {
                        const bool v = cv && (kbase + kq + j < g.K);
                        cp_async8p(d + j * LDB, v ? s : B, v);
                        s += g.bk_lo;
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < EB; ++j) {
                        const bool v = cv && (kbase + kq + j < g.K);
                        cp_async8p(d + j * LDB, v ? Bc + idx2(kbase + kq + j, g.Klo, g.bk_hi, g.bk_lo) : B, v);
                    }
                }
            } else {
                const int kk = p % BK, k = kbase + kk;
                const bool kv = k < g.K;
                const double* Bk = B + (kv ? (k1b ? (long long)k * g.bk_lo : idx2(k, g.Klo, g.bk_hi, g.bk_lo)) : 0);
                double* d = bs + kk * LDB + p / BK;
#pragma unroll
                for (int j = 0; j < EB; ++j) {
                    const bool v = kv && cb[j] >= 0;
                    cp_async8p(d + (NP / BK) * j, v ? Bk + cb[j] : B, v);
                }
            }
            cp_async_mbar_arrive(&full[stage]);
            if (++stage == ST) { stage = 0; par ^= 1; }
        }
        return;
    }

    // ---------------------------------------------------------------- consumers
    double acc[TM][TN][2];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int wm0 = (warp / (BN / WN)) * WM, wn0 = (warp % (BN / WN)) * WN;
    const int lr = lane >> 2, lc = lane & 3;
    const bool flip = nph == 2 && g.s0[db] != g.s1[db];
    int stage = 0; unsigned par = 0;
    for (int t = 0; t < total; ++t) {
        mbar_wait(&full[stage], par);
        if (flip && t == nk) {
#pragma unroll
            for (int i = 0; i < TM; ++i)
#pragma unroll
                for (int j = 0; j < TN; ++j) { acc[i][j][0] = -acc[i][j][0]; acc[i][j][1] = -acc[i][j][1]; }
        }
        const double* as = As + stage * BM * LDA + (wm0 + lr) * LDA + lc;
        const double* bs = Bs + stage * BK * LDB + lc * LDB + wn0 + lr;
#pragma unroll
        for (int ks = 0; ks < BK / 4; ++ks) {
            double a[TM], b[TN];
#pragma unroll
            for (int i = 0; i < TM; ++i) a[i] = as[8 * i * LDA + ks * 4];
#pragma unroll
            for (int j = 0; j < TN; ++j) b[j] = bs[ks * 4 * LDB + 8 * j];
#pragma unroll
            for (int i = 0; i < TM; ++i)
#pragma unroll
                for (int j = 0; j < TN; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[stage]);
        if (++stage == ST) { stage = 0; par ^= 1; }
    }

    const double sgn = (nph == 2) ? (double)g.s1[db] : (double)g.s0[db];
    if (g.ksplit > 1) {
        double* W = g.ws + ((long long)(db * g.nsb + sb) * g.ksplit + split) * (long long)g.M * g.N;
#pragma unroll
        for (int i = 0; i < TM; ++i) {
            int m = m0 + wm0 + 8 * i + lr;
            if (m >= g.M) continue;
#pragma unroll
            for (int j = 0; j < TN; ++j) {
                int n = n0 + wn0 + 8 * j + 2 * lc;
                if (n < g.N) W[(long long)m * g.N + n] = sgn * symfac * acc[i][j][0];
                if (n + 1 < g.N) W[(long long)m * g.N + n + 1] = sgn * symfac * acc[i][j][1];
            }
        }
        return;
    }
    double* C = g.C[db] + sb * g.sbC;
    double* C2 = g.C2[db] ? g.C2[db] + sb * g.sbC : nullptr;
    const double al = g.alpha * sgn * symfac, be = g.beta;
#pragma unroll
    for (int i = 0; i < TM; ++i) {
        int m = m0 + wm0 + 8 * i + lr;
        if (m >= g.M) continue;
        long long mo = g.cm_table ? g.cm_table[m] : idx2(m, g.Mlo, g.cm_hi, g.cm_lo);
#pragma unroll
        for (int j = 0; j < TN; ++j) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                int n = n0 + wn0 + 8 * j + 2 * lc + e;
                if (n < g.N) {
                    const long long co = mo + idx2(n, g.Nlo, g.cn_hi, g.cn_lo);
                    double* p = C + co;
                    double v = al * acc[i][j][e];
                    if (C2) {
                        double v2 = v;
                        if (be != 0.0) v2 += be * C2[co];
                        C2[co] = v2;
                    }
                    if (be != 0.0) v += be * *p;
                    *p = v;
                }
            }
        }
    }
}

// C = alpha * sum_splits ws + beta * C   (fixed summation order: deterministic)
__global__ void tcgemm_splitk_reduce(const TcGemm g)
{
    const long long MN = (long long)g.M * g.N;
    const int nbt = g.nb * g.nsb;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < MN * nbt; e += (long long)gridDim.x * blockDim.x) {
        int bt = (int)(e / MN);
        long long r = e - bt * MN;
        int m = (int)(r / g.N), n = (int)(r - (long long)m * g.N);
        int db = bt / g.nsb, sb = bt - db * g.nsb;
        const double* W = g.ws + (long long)bt * g.ksplit * MN + r;
        double s = 0.0;
        for (int k = 0; k < g.ksplit; ++k) s += W[k * MN];
        const long long co = sb * g.sbC + (g.cm_table ? g.cm_table[m] : idx2(m, g.Mlo, g.cm_hi, g.cm_lo)) + idx2(n, g.Nlo, g.cn_hi, g.cn_lo);
        double* p = g.C[db] + co;
        double v = g.alpha * s;
        if (g.C2[db]) {
            double v2 = v;
            if (g.beta != 0.0) v2 += g.beta * g.C2[db][co];
            g.C2[db][co] = v2;
        }
        if (g.beta != 0.0) v += g.beta * *p;
        *p = v;
    }
}

template <int BM, int BN> constexpr size_t tcgemm_smem()
{
    return sizeof(double) * (4 * BM * (16 + 4) + 4 * 16 * (BN + 4)) + sizeof(long long) * (BM + BN) + 8 * sizeof(unsigned long long);
}

// Host launcher.  ws_cap = capacity (doubles) of g.ws; returns number of kernels launched (1 or 2).
inline int tcgemm_launch(TcGemm g, cudaStream_t st, long long ws_cap, int num_sms, double* flops_out = nullptr, int force_tile = 0)
{
    if (g.M <= 0 || g.N <= 0 || g.nb <= 0 || g.nsb <= 0) return 0;
    if (g.Mlo <= 0 || g.Mlo >= g.M) g.Mlo = 0x40000000;
    if (g.Nlo <= 0 || g.Nlo >= g.N) g.Nlo = 0x40000000;
    g.a_klin = (g.Klo <= 0 || g.Klo >= g.K) || g.ak_hi == (long long)g.Klo * g.ak_lo;
    g.b_klin = (g.Klo <= 0 || g.Klo >= g.K) || g.bk_hi == (long long)g.Klo * g.bk_lo;
    if (g.Klo <= 0 || g.Klo >= g.K) g.Klo = 0x40000000;
    const int nbt = g.nb * g.nsb;
    const long long t128 = (long long)((g.M + 127) / 128) * ((g.N + 127) / 128) * nbt;
    // 128x128 tiles only when they fill the machine at least twice over; below that the 64x64 tiles (3 CTAs per SM, less
    // padding) measured faster (Small: ring products of dimension 907)
    bool big = t128 >= 2LL * num_sms && g.M > 64 && g.N > 64;
    if (force_tile == 64) big = false;            // rtcc_set_default_option("tile", ...): tests pin a tile configuration
    if (force_tile == 128) big = true;
    const int BM = big ? 128 : 64, BN = big ? 128 : 64;
    const long long tiles = (long long)((g.M + BM - 1) / BM) * ((g.N + BN - 1) / BN) * nbt;
    const int nkt = (g.K + 15) / 16;
    int ks = 1;
    if (g.ws && tiles * 2 <= num_sms && nkt >= 16) {
        ks = (int)(num_sms / tiles);
        if (ks > nkt / 8) ks = nkt / 8;
        while (ks > 1 && (long long)ks * nbt * g.M * g.N > ws_cap) --ks;
        if (ks < 1) ks = 1;
    }
    g.ksplit = ks;
    if (flops_out) {
        int tot_ph = 0;
        for (int b = 0; b < g.nb; ++b) tot_ph += g.nphase[b];
        const double nt = (double)((g.M + BM - 1) / BM);
        *flops_out += 2.0 * g.M * g.N * (double)g.K * tot_ph * g.nsb * (g.sym_upper ? 0.5 * (nt + 1.0) / nt : 1.0);
    }
    dim3 grid((g.M + BM - 1) / BM, (g.N + BN - 1) / BN, nbt * ks);
    if (big) {
        tcgemm_kernel<128, 128, 64, 32><<<grid, 384, tcgemm_smem<128, 128>(), st>>>(g);
    } else {
        tcgemm_kernel<64, 64, 16, 32><<<grid, 384, tcgemm_smem<64, 64>(), st>>>(g);
    }
    if (ks > 1) {
        long long tot = (long long)g.M * g.N * nbt;
        int blocks = (int)((tot + 255) / 256);
        if (blocks > num_sms * 8) blocks = num_sms * 8;
        tcgemm_splitk_reduce<<<blocks, 256, 0, st>>>(g);
        return 2;
    }
    return 1;
}

inline cudaError_t tcgemm_init()
{
    cudaError_t e = cudaFuncSetAttribute(tcgemm_kernel<128, 128, 64, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)tcgemm_smem<128, 128>());
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(tcgemm_kernel<64, 64, 16, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)tcgemm_smem<64, 64>());
}

}  // namespace rtcc
