// rtcc.cu -- context, residual pipeline, Adams-Moulton step driver and the C ABI of librtcc
// (include/rtcc.h).  The working equations are the Cholesky / T1-dressed form of the spin-orbital
// CCSD projections (Eqs. 7-8), restricted to the alpha-alpha / beta-beta / alpha-beta
// blocks; DESIGN.md section 4 derives them.  Every contraction is a tcgemm launch
// (tcgemm.cuh) except the particle-particle ladder (ladder.cuh); the rest is elementwise.cuh.
#include <cmath>
#include <cstdio>
#include <algorithm>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "../../include/rtcc.h"
#include "elementwise.cuh"
#include "ladder.cuh"
#include "tcgemm.cuh"

using namespace rtcc;

// process-wide defaults read by rtcc_create (rtcc_set_default_option, include/rtcc.h)
struct RtccOptions {
    int fused = 1, fused_fock = 1, graph = 1, prio = 1, tile = 0;
    int lean = -1, lean_slab_j = 0;              // lean: -1 automatic (when the standard layout does not fit), 0 never, 1 always
    int ring3m = -1;                             // complex ring products by three real multiplications: -1 automatic, 0 never, 1 always
    LadderTune lad;
};
static RtccOptions g_opt;
static int g_create_cuda_err = 0;            // cudaError_t of the most recent failed rtcc_create

struct rtcc_ctx {
    Dims d{};
    unsigned flags = 0;
    cudaStream_t st = nullptr;
    cudaStream_t S[8]{};                 // S[0] = st (or the capture stream), S[1..3] = helper branches
    cudaStream_t aux[7]{};
    cudaStream_t lad_side = nullptr; cudaEvent_t lad_ev[2]{};   // second wide ladder launch runs beside the first
    cudaEvent_t evs[16]{};
    int si = 0;
    int sec = 0; unsigned skipmask = 0;   // debug: RTCC_SKIP_MASK skips the GEMMs of pipeline sections (timing experiments only)
    int num_sms = 148;
    int cuda_err = 0;
    std::vector<void*> allocs;
    std::vector<std::pair<std::string, std::pair<double*, long long>>> named;
    long long bytes = 0;

    double *L[2]{}, *Lt[2]{}, *fockd[2]{}, *Fb[2]{}, *Ft[2]{}, *Kx[2]{}, *KxBA = nullptr;
    double *t1r = nullptr, *Tsc = nullptr, *Wsc = nullptr, *Zsc = nullptr;
    double *TAB = nullptr, *WBB = nullptr, *WAA = nullptr, *ZAB = nullptr, *ZBA = nullptr;
    bool ring3m = false;                                          // T.W of the ring as three real products (standard layout only)
    double *Ts_sc = nullptr, *Wd_sc = nullptr, *Ts_AB = nullptr, *Wd_BB = nullptr, *Wd_AA = nullptr;
    double *Nq = nullptr, *Mq = nullptr, *gam = nullptr, *r1buf = nullptr;
    double *Xab = nullptr, *tauab = nullptr, *Yab = nullptr, *Wooab = nullptr;
    double *LtA[2]{}, *LtB[2]{}, *Xt_ab = nullptr, *Xt_ss[2]{};   // tile-major ladder operands
    int nt2_ab = 128, nt2_ss[2]{128, 128};
    int anti_ss[2]{0, 0};                 // same-spin ladder in the antisymmetrised form: rows e >= f of the tile-major X stay zero
    double *Xss[2]{}, *tauss[2]{}, *Yss[2]{}, *W4[2]{}, *Wp[2]{}, *Yoop[2]{}, *Zv[2]{};
    int2 *opairs[2]{}, *vpairs[2]{}, *tiles_ab = nullptr, *tiles_ss[2]{};
    int ntiles_ab = 0, ntiles_ss[2]{};
    // low-memory pipeline: one arena reused by the ring phase and the ladder phase
    bool lean = false;
    double* arena = nullptr; long long arena_cap = 0;
    double *Tss[2]{}, *Wslab = nullptr, *Zslab = nullptr, *Wsf = nullptr, *Zsf = nullptr;
    int slab_j[2]{1, 1};                                         // occupied indices j per column slab, by spin
    double *Voo = nullptr, *Vp[2]{}, *Yoo[2]{};
    long long* cmp[2]{};                                         // ladder-output row offsets by packed virtual pair
    long long xt_ab_cnt = 0, xt_ss_cnt[2]{};
    LadderBatch lb{};
    LadderOcc locc{};
    RtccOptions opt{};
    double* ws = nullptr; long long ws_cap = 0;
    double *partial = nullptr, *bmax = nullptr, *scal = nullptr;   // scal: [0..1] E, [2] delta
    double* h_scal = nullptr;                                      // pinned host mirror of scal
    double *gx = nullptr, *gr = nullptr;                           // residual input / output (packed amp vectors)
    double *t_cur = nullptr, *r_cur = nullptr;                     // t(tau), R(t(tau)); during a step r_cur holds B = t + h R(t)
    double* dtab = nullptr; AmpSegs segs{};                        // orbital-energy tables behind the denominators
    unsigned* counters = nullptr;                                  // [0] energy reduction, [1] update reduction
    double *io = nullptr;                                          // staging for host-pointer mode
    long long namp = 0;                                            // n_t1 + n_t2 (complex)

    // propagation state
    double time = 0.0, C[2] = {0, 0}, E[2] = {0, 0}, E_res[2] = {0, 0};
    int mode = 0, max_micro = 200, fixed_micro = 0, last_micro = 0;
    bool state_valid = false;             // r_cur / E hold R(t_cur), E(t_cur) (evaluated by the first call that needs them)
    double tol = 1e-4;

    // instrumentation
    long long launches = 0; double flops = 0.0;
    long long res_launches = 0; double res_flops = 0.0;            // per residual evaluation
    cudaEvent_t ev_delta = nullptr;
    int timing = 0; cudaEvent_t ev[2]{}; double lad_ms = 0, lad_flops = 0, lad_model = 0;
    cudaGraphExec_t graph = nullptr;
    bool capturing = false;
    bool fused_dress = false, fused_fock = false;
    int fuse_nch = 74; long long fuse_sz = 0; size_t smem_fockp = 0, smem_fockf = 0, smem_postp = 0;
    double *fockPart = nullptr, *fockRed = nullptr, *postPart = nullptr, *postRed = nullptr;
};

namespace {

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { c->cuda_err = (int)e_; return RTCC_ECUDA; } } while (0)

template <class T> int dalloc(rtcc_ctx* c, T** p, long long count, const char* name = nullptr)
{
    if (count <= 0) count = 1;
    void* q = nullptr;
    cudaError_t e = cudaMalloc(&q, (size_t)count * sizeof(T));
    if (e != cudaSuccess) { c->cuda_err = (int)e; cudaGetLastError(); return RTCC_ENOMEM; }
    c->allocs.push_back(q);
    c->bytes += count * (long long)sizeof(T);
    *p = (T*)q;
    if (name) c->named.push_back({name, {(double*)q, count * (long long)sizeof(T) / 8}});
    return 0;
}

TcGemm G0(int M, int N, int K)
{
    TcGemm g;
    memset(&g, 0, sizeof(g));
    g.M = M; g.N = N; g.K = K;
    g.nb = 1; g.nsb = 1; g.alpha = 1.0; g.beta = 0.0; g.ksplit = 1;
    for (int b = 0; b < TG_MAXB; ++b) { g.nphase[b] = 1; g.s0[b] = 1; g.s1[b] = 1; }
    return g;
}
void setA(TcGemm& g, long long m_hi, long long m_lo, int Mlo, long long k_hi, long long k_lo, int Klo, int kfast)
{ g.am_hi = m_hi; g.am_lo = m_lo; g.Mlo = Mlo; g.ak_hi = k_hi; g.ak_lo = k_lo; g.Klo = Klo; g.a_kfast = kfast; }
void setB(TcGemm& g, long long k_hi, long long k_lo, long long n_hi, long long n_lo, int Nlo, int nfast)
{ g.bk_hi = k_hi; g.bk_lo = k_lo; g.bn_hi = n_hi; g.bn_lo = n_lo; g.Nlo = Nlo; g.b_nfast = nfast; }
void setC(TcGemm& g, long long m_hi, long long m_lo, long long n_hi, long long n_lo)
{ g.cm_hi = m_hi; g.cm_lo = m_lo; g.cn_hi = n_hi; g.cn_lo = n_lo; }
void ops_rr(TcGemm& g, const double* A, const double* B, double* C)
{ g.nb = 1; g.A[0][0] = A; g.B[0][0] = B; g.C[0] = C; }
void ops_rc(TcGemm& g, const double* A, const double* B, long long pB, double* C, long long pC)
{ g.nb = 2; for (int b = 0; b < 2; ++b) { g.A[b][0] = A; g.B[b][0] = B + b * pB; g.C[b] = C + b * pC; } }
void ops_cr(TcGemm& g, const double* A, long long pA, const double* B, double* C, long long pC)
{ g.nb = 2; for (int b = 0; b < 2; ++b) { g.A[b][0] = A + b * pA; g.B[b][0] = B; g.C[b] = C + b * pC; } }
void ops_cc(TcGemm& g, const double* A, long long pA, const double* B, long long pB, double* C, long long pC)
{
    g.nb = 2;
    g.nphase[0] = g.nphase[1] = 2;
    g.A[0][0] = A; g.B[0][0] = B; g.s0[0] = 1; g.A[0][1] = A + pA; g.B[0][1] = B + pB; g.s1[0] = -1; g.C[0] = C;
    g.A[1][0] = A; g.B[1][0] = B + pB; g.s0[1] = 1; g.A[1][1] = A + pA; g.B[1][1] = B; g.s1[1] = 1; g.C[1] = C + pC;
}
void run(rtcc_ctx* c, TcGemm& g)
{
#ifdef RTCC_DEBUG_KNOBS
    if ((c->skipmask >> c->sec) & 1u) return;      // timing experiments only (results are wrong when set)
#endif
    const long long cap = c->ws_cap / 8;
    g.ws = c->ws + c->si * cap;
    int n = tcgemm_launch(g, c->S[c->si], cap, c->num_sms, &c->flops, c->opt.tile);
    c->launches += n;
}
// C (planar, row pitch ldc, Im plane at +pc) = alpha * (T W) + beta * C with three real products (see step 9 of the pipeline).
//   Ts = Tr + Ti: element (m,k) at Ts[m * ts_m + k * ts_k];  T planar: (m,k) at T[m * t_m + k * t_k], Im plane at +pt
//   W planar with pitch ldw: Re plane Wr, its Im plane (at +pw) already holds Wr + Wi;  Wd = Wi - Wr dense with pitch ldwd
//   tr: the left operand is read transposed (m is the contiguous index)
void cplx3m(rtcc_ctx* c, int M, int N, int K, const double* Ts, int tr, long long ts_m, long long ts_k,
            const double* T, int tr2, long long t_m, long long t_k, long long pt,
            const double* W, long long ldw, long long pw, const double* Wd, long long ldwd,
            double* C, long long ldc, long long pc, double alpha, double beta)
{
    (void)tr2;
    {   // k1 into both planes
        TcGemm g = G0(M, N, K);
        setA(g, 0, ts_m, 0, 0, ts_k, 0, tr ? 0 : 1);
        setB(g, 0, ldw, 0, 1, 0, 1);
        setC(g, 0, ldc, 0, 1);
        ops_rr(g, Ts, W, C);
        g.C2[0] = C + pc;
        g.alpha = alpha; g.beta = beta;
        run(c, g);
    }
    {   // Re -= k3 = Ti (Wr + Wi)
        TcGemm g = G0(M, N, K);
        setA(g, 0, t_m, 0, 0, t_k, 0, tr ? 0 : 1);
        setB(g, 0, ldw, 0, 1, 0, 1);
        setC(g, 0, ldc, 0, 1);
        ops_rr(g, T + pt, W + pw, C);
        g.alpha = -alpha; g.beta = 1.0;
        run(c, g);
    }
    {   // Im += k2 = Tr (Wi - Wr)
        TcGemm g = G0(M, N, K);
        setA(g, 0, t_m, 0, 0, t_k, 0, tr ? 0 : 1);
        setB(g, 0, ldwd, 0, 1, 0, 1);
        setC(g, 0, ldc, 0, 1);
        ops_rr(g, T, Wd, C + pc);
        g.alpha = alpha; g.beta = 1.0;
        run(c, g);
    }
}
inline int nblk(long long n, int cap) { long long b = (n + 255) / 256; if (b < 1) b = 1; if (b > cap) b = cap; return (int)b; }
#define EW(c, kern, n, ...) do { kern<<<nblk((n), (c)->num_sms * 16), 256, 0, (c)->S[(c)->si]>>>(__VA_ARGS__); (c)->launches++; } while (0)

}  // namespace

namespace {

// ---------------------------------------------------------------------------------------------
// One evaluation of R1, R2 (Eqs. 7-8) and E (Eq. 5 integrand) at the packed amplitudes x -> r.
// Only asynchronous work on c->st (capturable into a CUDA graph).
// ---------------------------------------------------------------------------------------------
int residual_pipeline(rtcc_ctx* c, const double* x, double* r)
{
    const Dims& d = c->d;
    const int n = d.n, NQ = d.NQ, n1 = d.n1;
    const long long nn = (long long)n * n, plane = (long long)NQ * nn, ld1 = 2LL * n1;
    const double* t1p = x;
    const double* t2p = x + 2 * d.n_t1;
    // Independent parts of the evaluation run on helper streams (forked / joined with events, so the same code
    // captures into one CUDA graph with parallel branches).  Timing mode keeps everything on one stream.
    const bool par = !c->timing;
    c->S[0] = c->st;
    for (int i = 0; i < 7; ++i) c->S[i + 1] = par ? c->aux[i] : c->st;
#define ST (c->S[c->si])
#define BR(i) (c->si = (i))
#define LINK(from, to, e) do { if (par) { CK(cudaEventRecord(c->evs[e], c->S[from])); CK(cudaStreamWaitEvent(c->S[to], c->evs[e], 0)); } } while (0)
#define WAITEV(to, e) do { if (par) CK(cudaStreamWaitEvent(c->S[to], c->evs[e], 0)); } while (0)
    BR(0);

    // ---- 1. unpack the packed spin blocks into the contraction layouts
    c->sec = 1;
    EW(c, k_unpack_t1, n1, d, t1p, c->t1r);
    {   // pair-space matrices T_sc, T_AB (and Re + Im for the three-multiplication products): every packed amplitude read once
        double* Ts = c->ring3m ? c->Ts_sc : nullptr;
        const long long nab = (long long)d.oo * ((d.v[0] + UP_T - 1) / UP_T) * ((d.v[1] + UP_T - 1) / UP_T);
        if (nab > 0) {
            k_unpack_ab<<<(int)std::min<long long>(nab, (long long)c->num_sms * 16), 256, 0, ST>>>(d, t2p, c->Tsc, c->TAB, Ts, c->ring3m ? c->Ts_AB : nullptr);
            c->launches++;
        }
        for (int s = 0; s < 2; ++s) {
            const long long nT = (d.v[s] + UP_T - 1) / UP_T, nss = (long long)d.po[s] * (nT * (nT + 1) / 2);
            if (nss > 0) {
                k_unpack_ss<<<(int)std::min<long long>(nss, (long long)c->num_sms * 16), 256, 0, ST>>>(d, s, c->opairs[s], t2p, c->Tsc, Ts);
                c->launches++;
            }
        }
    }
    {
        const long long nab = (((long long)d.v[0] * d.v[1] + UP_T - 1) / UP_T) * ((d.oo + UP_T - 1) / UP_T);
        if (d.oo > 0) {
            k_build_Xab<<<(int)std::min<long long>(nab, (long long)c->num_sms * 16), 256, 0, ST>>>(d, t2p, c->t1r, c->Xab, c->Xt_ab, (d.v[1] + 7) / 8,
                                                                                       (2 * d.oo + c->nt2_ab - 1) / c->nt2_ab, c->nt2_ab, c->tauab);
            c->launches++;
        }
    }
    for (int s = 0; s < 2; ++s)
        if (d.po[s] > 0)
        {
            const long long nss = (long long)((d.pv[s] + UP_T - 1) / UP_T) * ((d.po[s] + UP_T - 1) / UP_T);
            if (nss > 0) {
                k_build_Xss<<<(int)std::min<long long>(nss, (long long)c->num_sms * 16), 256, 0, ST>>>(d, s, t2p, c->t1r, c->opairs[s], c->vpairs[s], c->Xss[s],
                    c->Xt_ss[s], (d.v[s] + 7) / 8, (2 * d.po[s] + c->nt2_ss[s] - 1) / c->nt2_ss[s], c->nt2_ss[s], c->tauss[s], c->anti_ss[s]);
                c->launches++;
            }
        }

    if (par) CK(cudaEventRecord(c->evs[0], c->S[0]));     // evs[0]: unpacked layouts ready

    // ---- 2+3. T1-dressed Cholesky vectors and gamma: one fused kernel when an n x n slice fits in shared memory
    c->sec = 2;
    if (c->fused_dress) {
        DressArgs da;
        for (int s = 0; s < 2; ++s) { da.L[s] = c->L[s]; da.Lt[s] = c->Lt[s]; }
        da.t1r = c->t1r; da.gam = c->gam;
        k_dress<<<NQ, 256, dress_smem(d), ST>>>(d, da);
        c->launches++;
        if (par) CK(cudaEventRecord(c->evs[1], c->S[0]));     // evs[1]: dressed vectors ready
    } else {
    // ---- 2. (general path) T1-dressed Cholesky vectors  L~^Q = (1-T) L^Q (1+T)
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = s ? d.n1a : 0;
        CK(cudaMemcpyAsync(c->Lt[s], c->L[s], plane * 8, cudaMemcpyDeviceToDevice, ST));
        CK(cudaMemsetAsync(c->Lt[s] + plane, 0, plane * 8, ST));
        if (o == 0) continue;
        {   // (L Y)[Q][p][i] += sum_e L[Q][p][o+e] t_i^e
            TcGemm g = G0(NQ * n, o, v);
            setA(g, 0, n, 0, 0, 1, 0, 1);
            setB(g, 0, 1, 0, v, 0, 0);
            setC(g, 0, n, 0, 1);
            ops_rc(g, c->L[s] + o, c->t1r + off1, n1, c->Lt[s], plane);
            g.beta = 1.0;
            run(c, g);
        }
        {   // rows a: L~[Q][a][q] -= sum_m t_m^a (L Y)[Q][m][q]
            TcGemm g = G0(v, NQ * n, o);
            setA(g, 0, 1, 0, 0, v, 0, 0);
            setB(g, 0, n, nn, 1, n, 1);
            setC(g, 0, n, nn, 1);
            ops_cc(g, c->t1r + off1, n1, c->Lt[s], plane, c->Lt[s] + (long long)o * n, plane);
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
    }

    if (par) CK(cudaEventRecord(c->evs[1], c->S[0]));     // evs[1]: dressed vectors ready

    // ---- 3. gamma^Q = sum_ie L^Q_ie t_i^e (both spins)
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = s ? d.n1a : 0;
        TcGemm g = G0(NQ, 1, o * v);
        setA(g, 0, nn, 0, n, 1, v, 1);
        setB(g, v, 1, 0, 0, 0, 0);
        setC(g, 0, 1, 0, 0);
        ops_rc(g, c->L[s] + o, c->t1r + off1, n1, c->gam, NQ);
        g.beta = s ? 1.0 : 0.0;
        run(c, g);
    }

    }

    // ---- 4. M^Q_ia = sum_me L^Q_me t_im^ae over the spin-conserving pair space
    c->sec = 4;
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = s ? d.n1a : 0;
        TcGemm g = G0(NQ, 2 * n1, o * v);
        setA(g, 0, nn, 0, n, 1, v, 1);
        setB(g, v * ld1, ld1, 0, 1, 0, 1);
        setC(g, 0, ld1, 0, 1);
        ops_rr(g, c->L[s] + o, c->Tsc + off1 * ld1, c->Mq);
        g.beta = s ? 1.0 : 0.0;
        run(c, g);
    }

    if (par) CK(cudaEventRecord(c->evs[6], c->S[0]));     // evs[6]: gamma, M ready

    // ---- 5. E (needs the bare M^Q)
    c->sec = 5;
    {
        EnergyArgs ea;
        for (int s = 0; s < 2; ++s) { ea.L[s] = c->L[s]; ea.Lt[s] = c->Lt[s]; ea.fock[s] = c->fockd[s]; }
        ea.t1r = c->t1r; ea.Mq = c->Mq; ea.gam = c->gam; ea.partial = c->partial;
        ea.counter = c->counters; ea.out = c->scal;
        k_energy<<<RED_BLOCKS, RED_THREADS, 0, ST>>>(d, ea);
        c->launches += 1;
    }

    // ---- 6+7 (fused path for small problems): dressed Fock, F intermediates and singles in seven launches on branch 4
    c->sec = 6;
    if (c->fused_fock) {
        const int nch = c->fuse_nch;
        const long long SZ = c->fuse_sz;
        BR(4);
        WAITEV(4, 1);
        k_fock_partial<<<dim3(nch, 2), FUSE_T, c->smem_fockp, ST>>>(d, c->L[0], c->L[1], c->Lt[0], c->Lt[1], c->gam, nch, c->fockPart);
        k_reduce_chunks<<<c->num_sms, 256, 0, ST>>>(c->fockPart, c->fockRed, nch, 8 * nn);
        FockFinishArgs fa;
        for (int s = 0; s < 2; ++s) { fa.Fb[s] = c->Fb[s]; fa.Ft[s] = c->Ft[s]; }
        fa.red = c->fockRed; fa.t1r = c->t1r;
        k_fock_finish<<<2, FUSE_T, c->smem_fockf, ST>>>(d, fa);
        k_tsc_matvec<<<(n1 + 7) / 8, 256, 0, ST>>>(d, c->Tsc, c->Ft[0], c->Ft[1], c->r1buf);
        WAITEV(4, 6);
        k_postm_partial<<<dim3(nch, 2), FUSE_T, c->smem_postp, ST>>>(d, c->L[0], c->L[1], c->Lt[0], c->Lt[1], c->Mq, nch, SZ, c->postPart);
        k_reduce_chunks<<<c->num_sms, 256, 0, ST>>>(c->postPart, c->postRed, nch, 4 * SZ);
        k_postm_finish<<<32, 256, 0, ST>>>(d, c->postRed, SZ, c->Ft[0], c->Ft[1], c->r1buf);
        c->launches += 7;
        if (par) { CK(cudaEventRecord(c->evs[2], c->S[4])); CK(cudaEventRecord(c->evs[7], c->S[4])); }
    } else {
    // ---- 6. dressed Fock  f~ = X (f + K_bare + sum_Q gamma^Q L^Q) Y - sum_Q,i L~^Q_pi L~^Q_iq
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = s ? d.n1a : 0;
        double* F = c->Ft[s];
        if (s == 1) { if (par) CK(cudaEventRecord(c->evs[2], c->S[0])); BR(4); WAITEV(4, 6); }   // evs[2]: spin-0 F ready
        CK(cudaMemcpyAsync(F, c->Fb[s], nn * 8, cudaMemcpyDeviceToDevice, ST));
        CK(cudaMemsetAsync(F + nn, 0, nn * 8, ST));
        {
            TcGemm g = G0((int)nn, 1, NQ);
            setA(g, 0, 1, 0, 0, nn, 0, 0);
            setB(g, 0, 1, 0, 0, 0, 0);
            setC(g, 0, 1, 0, 0);
            ops_rc(g, c->L[s], c->gam, NQ, F, nn);
            g.beta = 1.0;
            run(c, g);
        }
        if (o > 0) {
            {
                TcGemm g = G0(n, o, v);
                setA(g, 0, n, 0, 0, 1, 0, 1);
                setB(g, 0, 1, 0, v, 0, 0);
                setC(g, 0, n, 0, 1);
                ops_cc(g, F + o, nn, c->t1r + off1, n1, F, nn);
                g.beta = 1.0;
                run(c, g);
            }
            {
                TcGemm g = G0(v, n, o);
                setA(g, 0, 1, 0, 0, v, 0, 0);
                setB(g, 0, n, 0, 1, 0, 1);
                setC(g, 0, n, 0, 1);
                ops_cc(g, c->t1r + off1, n1, F, nn, F + (long long)o * n, nn);
                g.alpha = -1.0; g.beta = 1.0;
                run(c, g);
            }
            {
                TcGemm g = G0(n, n, NQ * o);
                setA(g, 0, n, 0, nn, 1, o, 1);
                setB(g, nn, n, 0, 1, 0, 1);
                setC(g, 0, n, 0, 1);
                ops_cc(g, c->Lt[s], plane, c->Lt[s], plane, F, nn);
                g.alpha = -1.0; g.beta = 1.0;
                run(c, g);
            }
            {   // F_ae = f~_ae - sum_Q,m L^Q_me M^Q_ma   (in place in the vv block)
                TcGemm g = G0(v, v, NQ * o);
                setA(g, 0, 1, 0, ld1, v, o, 0);
                setB(g, nn, n, 0, 1, 0, 1);
                setC(g, 0, n, 0, 1);
                ops_cr(g, c->Mq + off1, n1, c->L[s] + o, F + (long long)o * n + o, nn);
                g.alpha = -1.0; g.beta = 1.0;
                run(c, g);
            }
            {   // F_mi = f~_mi + sum_Q,e L^Q_me M^Q_ie   (in place in the oo block)
                TcGemm g = G0(o, o, NQ * v);
                setA(g, 0, n, 0, nn, 1, v, 1);
                setB(g, ld1, 1, 0, v, 0, 0);
                setC(g, 0, n, 0, 1);
                ops_rc(g, c->L[s] + o, c->Mq + off1, n1, F, nn);
                g.beta = 1.0;
                run(c, g);
            }
        }
    }

    if (par) CK(cudaEventRecord(c->evs[7], c->S[4]));     // evs[7]: spin-1 F ready
    WAITEV(4, 2);                                         // singles stay on branch 4

    // ---- 7. singles:  r1 = sum_me t_im^ae f~_me - sum_Q,n M_na L~_ni + sum_Q,f M_if L~_af   (+ f~_ai at assembly)
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = s ? d.n1a : 0;
        TcGemm g = G0(n1, 1, o * v);
        setA(g, 0, ld1, 0, v, 1, v, 1);
        setB(g, n, 1, 0, 0, 0, 0);
        setC(g, 0, 1, 0, 0);
        ops_cc(g, c->Tsc + off1, n1, c->Ft[s] + o, nn, c->r1buf, n1);
        g.beta = s ? 1.0 : 0.0;
        run(c, g);
    }
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = s ? d.n1a : 0;
        if (o == 0) continue;
        {
            TcGemm g = G0(o, v, NQ * o);
            setA(g, 0, 1, 0, nn, n, o, 0);
            setB(g, ld1, v, 0, 1, 0, 1);
            setC(g, 0, v, 0, 1);
            ops_cc(g, c->Lt[s], plane, c->Mq + off1, n1, c->r1buf + off1, n1);
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
        {
            TcGemm g = G0(o, v, NQ * v);
            setA(g, 0, v, 0, ld1, 1, v, 1);
            setB(g, nn, 1, 0, n, 0, 0);
            setC(g, 0, v, 0, 1);
            ops_cc(g, c->Mq + off1, n1, c->Lt[s] + (long long)o * n + o, plane, c->r1buf + off1, n1);
            g.beta = 1.0;
            run(c, g);
        }
    }

    }

    // ---- 8. driver + Coulomb ring channel:  Zsc = 1/2 N^T N,  N^Q_ia = L~^Q_ai + M^Q_ia
    c->sec = 8;
    BR(0);
    EW(c, k_add_Lvo, (long long)NQ * 2 * n1, d, c->Lt[0], c->Lt[1], c->Mq, c->Nq);
    {
        TcGemm g = G0(n1, n1, NQ);
        setA(g, 0, 1, 0, 0, ld1, 0, 0);
        setB(g, 0, ld1, 0, 1, 0, 1);
        setC(g, 0, ld1, 0, 1);
        ops_cc(g, c->Nq, n1, c->Nq, n1, c->Zsc, n1);
        g.alpha = 0.5;
        g.sym_upper = 1;                  // N^T N is symmetric and the assembly only uses Z + Z^T: half of the tiles
        run(c, g);
    }

    // ---- 9. exchange ring channel + F terms, spin-conserving sector:  Zsc -= T (Xd + 1/2 Kx T + Fd)
    c->sec = 9;
    BR(1);
    WAITEV(1, 1);
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s], n1s = o * v;
        const long long off1 = s ? d.n1a : 0;
        if (n1s == 0) continue;
        {
            TcGemm g = G0(n1s, 2 * n1, n1s);
            setA(g, 0, n1s, 0, 0, 1, 0, 1);
            setB(g, 0, ld1, 0, 1, 0, 1);
            setC(g, 0, ld1, 0, 1);
            ops_rr(g, c->Kx[s], c->Tsc + off1 * ld1, c->Wsc + off1 * ld1);
            g.alpha = 0.5;
            run(c, g);
        }
        {
            TcGemm g = G0(o * o, v * v, NQ);
            setA(g, n, 1, o, 0, nn, 0, 0);
            setB(g, 0, nn, n, 1, v, 1);
            setC(g, (long long)v * ld1, v, 1, ld1);
            ops_cc(g, c->Lt[s], plane, c->Lt[s] + (long long)o * n + o, plane, c->Wsc + off1 * ld1 + off1, n1);
            g.beta = 1.0;
            run(c, g);
        }
        if (s == 0 || d.n1a == 0) { WAITEV(1, 2); WAITEV(1, 7); }
        EW(c, k_add_Fd, (long long)o * v * v + (long long)o * o * v, o, v, n, c->Ft[s], o, c->Ft[s], o, c->Wsc, ld1, (long long)n1, off1, off1, 0, o);
    }
    if (c->ring3m) EW(c, k_r3m_W, (long long)n1 * n1, (long long)n1, (long long)n1, c->Wsc, c->Wd_sc);
    LINK(1, 0, 3);
    BR(0);
    if (c->ring3m) {
        // (T W) with three real products instead of four (T = Tr + i Ti, W = Wr + i Wi):
        //   k1 = (Tr + Ti) Wr,  k2 = Tr (Wi - Wr),  k3 = Ti (Wr + Wi);   Re(TW) = k1 - k3,  Im(TW) = k1 + k2
        // Ts = Tr + Ti comes from the unpack kernel, k_r3m_W left Wr + Wi in W's Im plane and Wi - Wr in Wd.
        cplx3m(c, n1, n1, n1, c->Ts_sc, 0, n1, 1, c->Tsc, 0, ld1, 1, n1, c->Wsc, ld1, n1, c->Wd_sc, n1, c->Zsc, ld1, n1, -1.0, 1.0);
    } else {
        TcGemm g = G0(n1, n1, n1);
        setA(g, 0, ld1, 0, 0, 1, 0, 1);
        setB(g, 0, ld1, 0, 1, 0, 1);
        setC(g, 0, ld1, 0, 1);
        ops_cc(g, c->Tsc, n1, c->Wsc, n1, c->Zsc, n1);
        g.alpha = -1.0; g.beta = 1.0;
        run(c, g);
    }

    // ---- 10. spin-flip sector
    c->sec = 10;
    BR(2);
    WAITEV(2, 1);
    if (d.nA > 0 && d.nB > 0) {
        const int oa = d.o[0], ob = d.o[1], va = d.v[0], vb = d.v[1], nA = d.nA, nB = d.nB;
        const long long lA = 2LL * nA, lB = 2LL * nB;
        {
            TcGemm g = G0(nB, 2 * nB, nA);
            setA(g, 0, nA, 0, 0, 1, 0, 1);
            setB(g, 0, lB, 0, 1, 0, 1);
            setC(g, 0, lB, 0, 1);
            ops_rr(g, c->KxBA, c->TAB, c->WBB);
            g.alpha = 0.5;
            run(c, g);
        }
        {
            TcGemm g = G0(ob * ob, va * va, NQ);
            setA(g, n, 1, ob, 0, nn, 0, 0);
            setB(g, 0, nn, n, 1, va, 1);
            setC(g, va * lB, va, 1, lB);
            ops_cc(g, c->Lt[1], plane, c->Lt[0] + (long long)oa * n + oa, plane, c->WBB, nB);
            g.beta = 1.0;
            run(c, g);
        }
        WAITEV(2, 2);
        WAITEV(2, 7);
        EW(c, k_add_Fd, (long long)ob * va * va + (long long)ob * ob * va, ob, va, n, c->Ft[1], ob, c->Ft[0], oa, c->WBB, lB, (long long)nB, 0LL, 0LL, 0, ob);
        if (c->ring3m) {
            EW(c, k_r3m_W, (long long)nB * nB, (long long)nB, (long long)nB, c->WBB, c->Wd_BB);
            cplx3m(c, nA, nB, nB, c->Ts_AB, 0, nB, 1, c->TAB, 0, lB, 1, nB, c->WBB, lB, nB, c->Wd_BB, nB, c->ZAB, lB, nB, -1.0, 0.0);
        } else {
            TcGemm g = G0(nA, nB, nB);
            setA(g, 0, lB, 0, 0, 1, 0, 1);
            setB(g, 0, lB, 0, 1, 0, 1);
            setC(g, 0, lB, 0, 1);
            ops_cc(g, c->TAB, nB, c->WBB, nB, c->ZAB, nB);
            g.alpha = -1.0;
            run(c, g);
        }
        {
            TcGemm g = G0(nA, nA, nB);
            setA(g, 0, 1, 0, 0, nA, 0, 0);
            setB(g, 0, 1, 0, lB, 0, 0);
            setC(g, 0, lA, 0, 1);
            ops_rc(g, c->KxBA, c->TAB, nB, c->WAA, nA);
            g.alpha = 0.5;
            run(c, g);
        }
        {
            TcGemm g = G0(oa * oa, vb * vb, NQ);
            setA(g, n, 1, oa, 0, nn, 0, 0);
            setB(g, 0, nn, n, 1, vb, 1);
            setC(g, vb * lA, vb, 1, lA);
            ops_cc(g, c->Lt[0], plane, c->Lt[1] + (long long)ob * n + ob, plane, c->WAA, nA);
            g.beta = 1.0;
            run(c, g);
        }
        EW(c, k_add_Fd, (long long)oa * vb * vb + (long long)oa * oa * vb, oa, vb, n, c->Ft[0], oa, c->Ft[1], ob, c->WAA, lA, (long long)nA, 0LL, 0LL, 0, oa);
        if (c->ring3m) {                                   // left operand T_AB^T: k-fast = 0, rows stride 1
            EW(c, k_r3m_W, (long long)nA * nA, (long long)nA, (long long)nA, c->WAA, c->Wd_AA);
            cplx3m(c, nB, nA, nA, c->Ts_AB, 1, 1, nB, c->TAB, 1, 1, lB, nB, c->WAA, lA, nA, c->Wd_AA, nA, c->ZBA, lA, nA, -1.0, 0.0);
        } else {
            TcGemm g = G0(nB, nA, nA);
            setA(g, 0, 1, 0, 0, lB, 0, 0);
            setB(g, 0, lA, 0, 1, 0, 1);
            setC(g, 0, lA, 0, 1);
            ops_cc(g, c->TAB, nB, c->WAA, nA, c->ZBA, nA);
            g.alpha = -1.0;
            run(c, g);
        }
    }

    // ---- 11. ladders (pp with all-orbital rows; hh and the T1 corrections from the occupied rows)
    c->sec = 11;
    BR(3);
    WAITEV(3, 0);
    // same-spin ladder outputs: only row tiles with p-tile <= q-tile are written by the kernel, while the o^4 corrections below
    // accumulate into every (a,b) row -- clear the buffers so that the rows nobody reads do not grow from evaluation to evaluation
    for (int s = 0; s < 2; ++s)
        if (d.po[s] > 0) CK(cudaMemsetAsync(c->Yss[s], 0, (size_t)(nn * 2 * d.po[s]) * 8, ST));
    if (c->timing && !c->capturing) CK(cudaEventRecord(c->ev[0], ST));
    c->launches += ladder_launch(c->lb, ST, c->num_sms, c->lad_side, c->lad_ev[0], c->lad_ev[1], c->opt.lad.overlap);
    c->flops += ladder_flops(c->lb);
    c->lad_flops = ladder_flops(c->lb);
    if (c->timing && !c->capturing) CK(cudaEventRecord(c->ev[1], ST));
    if (par) CK(cudaEventRecord(c->evs[9], c->S[3]));     // evs[9]: ladder output ready

    if (d.oo > 0) {
        const int oa = d.o[0], ob = d.o[1], va = d.v[0], vb = d.v[1], oo = d.oo;
        const long long lY = 2LL * oo;
        double* Yvv = c->Yab + ((long long)oa * n + ob) * lY;
        BR(7);
        WAITEV(7, 1);
        {   // <mN||iJ>~ = sum_Q L~_mi L~_NJ   (independent of the ladder: own branch)
            TcGemm g = G0(oa * oa, ob * ob, NQ);
            setA(g, n, 1, oa, 0, nn, 0, 0);
            setB(g, 0, nn, n, 1, ob, 1);
            setC(g, ob * lY, ob, lY, 1);
            ops_cc(g, c->Lt[0], plane, c->Lt[1], plane, c->Wooab, oo);
            run(c, g);
        }
        if (par) CK(cudaEventRecord(c->evs[8], c->S[7]));
        BR(3);
        WAITEV(3, 8);
        {   // + t_mN^aB <mN||iJ>~
            TcGemm g = G0(va * vb, oo, oo);
            setA(g, vb * lY, lY, vb, 0, 1, 0, 1);
            setB(g, 0, lY, 0, 1, 0, 1);
            setC(g, n * lY, lY, 0, 1);
            ops_cc(g, c->Xab, oo, c->Wooab, oo, Yvv, oo);
            g.beta = 1.0;
            run(c, g);
        }
        {   // + tau_mN^aB Y_iJ^mN
            TcGemm g = G0(va * vb, oo, oo);
            setA(g, vb * lY, lY, vb, ob, 1, ob, 1);
            setB(g, n * lY, lY, 0, 1, 0, 1);
            setC(g, n * lY, lY, 0, 1);
            ops_cc(g, c->tauab, oo, c->Yab, oo, Yvv, oo);
            g.beta = 1.0;
            run(c, g);
        }
        {   // - sum_m t_m^a Y_iJ^mB
            TcGemm g = G0(va, vb * oo, oa);
            setA(g, 0, 1, 0, 0, va, 0, 0);
            setB(g, 0, n * lY, lY, 1, oo, 1);
            setC(g, 0, n * lY, lY, 1);
            ops_cc(g, c->t1r, n1, c->Yab + (long long)ob * lY, oo, Yvv, oo);
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
        {   // - sum_N t_N^B Y_iJ^aN   (batched over a)
            TcGemm g = G0(vb, oo, ob);
            setA(g, 0, 1, 0, 0, vb, 0, 0);
            setB(g, 0, lY, 0, 1, 0, 1);
            setC(g, 0, lY, 0, 1);
            ops_cc(g, c->t1r + d.n1a, n1, c->Yab + (long long)oa * n * lY, oo, Yvv, oo);
            g.nsb = va; g.sbA = 0; g.sbB = n * lY; g.sbC = n * lY;
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
    }
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s], po = d.po[s];
        const long long off1 = s ? d.n1a : 0;
        if (po == 0) continue;
        const long long lP = 2LL * po, o2 = (long long)o * o;
        double* Yvv = c->Yss[s] + ((long long)o * n + o) * lP;
        BR(7);
        WAITEV(7, 1);
        {
            TcGemm g = G0(o * o, o * o, NQ);
            setA(g, n, 1, o, 0, nn, 0, 0);
            setB(g, 0, nn, n, 1, o, 1);
            setC(g, o * 2 * o2, o, 2 * o2, 1);
            ops_cc(g, c->Lt[s], plane, c->Lt[s], plane, c->W4[s], o2);
            run(c, g);
        }
        if (par) CK(cudaEventRecord(c->evs[13 + s], c->S[7]));
        BR(5 + s);
        WAITEV(5 + s, 9);
        WAITEV(5 + s, 13 + s);
        EW(c, k_ss_prep, (long long)po * po, o, po, n, c->opairs[s], c->W4[s], c->Yss[s], c->Wp[s], c->Yoop[s]);
        {
            TcGemm g = G0(v * v, po, po);
            setA(g, v * lP, lP, v, 0, 1, 0, 1);
            setB(g, 0, lP, 0, 1, 0, 1);
            setC(g, n * lP, lP, 0, 1);
            ops_cc(g, c->Xss[s], po, c->Wp[s], po, Yvv, po);
            g.beta = 1.0;
            run(c, g);
        }
        {
            TcGemm g = G0(v * v, po, po);
            setA(g, v * lP, lP, v, 0, 1, 0, 1);
            setB(g, 0, lP, 0, 1, 0, 1);
            setC(g, n * lP, lP, 0, 1);
            ops_cc(g, c->tauss[s], po, c->Yoop[s], po, Yvv, po);
            g.beta = 1.0;
            run(c, g);
        }
        {   // Zv[a][b] = sum_m t_m^a Y^{mb}
            TcGemm g = G0(v, v * po, o);
            setA(g, 0, 1, 0, 0, v, 0, 0);
            setB(g, 0, n * lP, lP, 1, po, 1);
            setC(g, 0, v * lP, lP, 1);
            ops_cc(g, c->t1r + off1, n1, c->Yss[s] + (long long)o * lP, po, c->Zv[s], po);
            run(c, g);
        }
    }

    LINK(2, 0, 4);
    LINK(3, 0, 5);
    LINK(4, 0, 10);
    if (d.po[0] > 0) LINK(5, 0, 11);
    if (d.po[1] > 0) LINK(6, 0, 12);
    BR(0);

    // ---- 12. antisymmetrise and write the packed residual
    c->sec = 12;
    {
        AsmArgs A;
        A.Zsc = c->Zsc; A.ZAB = c->ZAB; A.ZBA = c->ZBA; A.Yab = c->Yab; A.r1buf = c->r1buf;
        for (int s = 0; s < 2; ++s) {
            A.Yss[s] = c->Yss[s]; A.Zv[s] = c->Zv[s]; A.Ft[s] = c->Ft[s];
            A.opairs[s] = c->opairs[s]; A.vpairs[s] = c->vpairs[s];
        }
        A.r1p = r; A.r2p = r + 2 * d.n_t1;
        // tiled, shared-memory-staged assembly once the blocks are large enough to fill tiles; the element-per-thread
        // gather below that (Tiny-sized blocks)
        const bool tiled = d.v[0] >= 16 && d.v[1] >= 16;
        if (tiled) {
            if (d.oo > 0) {
                const long long nt = (long long)d.o[0] * ((d.o[1] + AS_TJ - 1) / AS_TJ) * ((d.v[0] + AS_TA - 1) / AS_TA) * ((d.v[1] + AS_TB - 1) / AS_TB);
                k_assemble_ab<<<(unsigned)(nt < c->num_sms * 8LL ? nt : c->num_sms * 8LL), 256, 0, c->S[c->si]>>>(d, A);
                c->launches++;
            }
            for (int s = 0; s < 2; ++s)
                if (d.po[s] > 0 && d.pv[s] > 0) {
                    const long long nt = (long long)((d.po[s] + AS_TJ - 1) / AS_TJ) * ((d.v[s] + AS_TA - 1) / AS_TA) * ((d.v[s] + AS_TB - 1) / AS_TB);
                    k_assemble_ss<<<(unsigned)(nt < c->num_sms * 8LL ? nt : c->num_sms * 8LL), 256, 0, c->S[c->si]>>>(d, s, A);
                    c->launches++;
                }
            EW(c, k_assemble_r1, d.n_t1, d, A);
        } else EW(c, k_assemble, d.n_t1 + d.n_t2, d, A);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { c->cuda_err = (int)e; return RTCC_ECUDA; }
    return RTCC_OK;
}

}  // namespace

namespace {

// ---------------------------------------------------------------------------------------------
// Low-memory evaluation of the same working equations (DESIGN.md sections 4 and 5).  Differences from residual_pipeline:
// one stream (the phases reuse one arena); the alpha-beta amplitudes are read in place from the packed input through
// two-level strides (interleaved complex: plane offset 1); the same-spin pair-space blocks are the only unpacked
// amplitudes; W and Z of the spin-conserving ring sector live in column slabs (a range of occupied indices j of one spin)
// that k_fold_slab adds into the packed residual; the spin-flip sector reuses the same memory; the ladder's buffers
// overlay the ring phase's; tau is never formed (tau = t + t1 t1 is applied as two contractions) and the T1 corrections
// are accumulated into the ladder output instead of a separate buffer.
// ---------------------------------------------------------------------------------------------
struct TOp { const double* p; long long pim, r_hi, r_lo, c_hi, c_lo; int Rlo, Clo; };

// T[(row pair of spin sr), (column pair of spin sc)] = t_{im}^{ae} as a strided operand (strides in doubles)
TOp t_block(const rtcc_ctx* c, const double* x, int sr, int sc)
{
    const Dims& d = c->d;
    TOp t{};
    if (sr == sc) {
        const long long n1s = (long long)d.o[sr] * d.v[sr];
        t.p = c->Tss[sr]; t.pim = n1s; t.r_hi = 0; t.r_lo = 2 * n1s; t.Rlo = 0; t.c_hi = 0; t.c_lo = 1; t.Clo = 0;
    } else {
        const long long va = d.v[0], vb = d.v[1], ob = d.o[1];
        t.p = x + 2 * d.n_t1 + 2 * d.off_t2[2]; t.pim = 1;
        if (sr == 0) { t.Rlo = (int)va; t.r_hi = 2 * ob * va * vb; t.r_lo = 2 * vb; t.Clo = (int)vb; t.c_hi = 2 * va * vb; t.c_lo = 2; }
        else         { t.Rlo = (int)vb; t.r_hi = 2 * va * vb; t.r_lo = 2; t.Clo = (int)va; t.c_hi = 2 * ob * va * vb; t.c_lo = 2 * vb; }
    }
    return t;
}

int residual_pipeline_lean(rtcc_ctx* c, const double* x, double* r)
{
    const Dims& d = c->d;
    const int n = d.n, NQ = d.NQ, n1 = d.n1;
    const long long nn = (long long)n * n, plane = (long long)NQ * nn, ld1 = 2LL * n1;
    const double* t1p = x;
    const double* t2p = x + 2 * d.n_t1;
    for (int i = 0; i < 8; ++i) c->S[i] = c->st;
    c->si = 0;
#define STL (c->st)
    const long long rowoff[2] = {0, d.n1a};
    const long long n1s_[2] = {d.n1a, d.n1b};

    // ---- 1. t1 planar; same-spin pair-space blocks; residual accumulator cleared
    c->sec = 1;
    EW(c, k_unpack_t1, n1, d, t1p, c->t1r);
    for (int s = 0; s < 2; ++s)
        if (n1s_[s] > 0) EW(c, k_build_Tss, n1s_[s] * n1s_[s], d, s, t2p, c->Tss[s]);
    CK(cudaMemsetAsync(r, 0, (size_t)c->namp * 16, STL));

    // ---- 2. T1-dressed Cholesky vectors (general path) and gamma
    c->sec = 2;
    if (c->fused_dress) {
        DressArgs da;
        for (int s = 0; s < 2; ++s) { da.L[s] = c->L[s]; da.Lt[s] = c->Lt[s]; }
        da.t1r = c->t1r; da.gam = c->gam;
        k_dress<<<NQ, 256, dress_smem(d), STL>>>(d, da);
        c->launches++;
    } else {
        for (int s = 0; s < 2; ++s) {
            const int o = d.o[s], v = d.v[s];
            const long long off1 = rowoff[s];
            CK(cudaMemcpyAsync(c->Lt[s], c->L[s], plane * 8, cudaMemcpyDeviceToDevice, STL));
            CK(cudaMemsetAsync(c->Lt[s] + plane, 0, plane * 8, STL));
            if (o == 0) continue;
            {
                TcGemm g = G0(NQ * n, o, v);
                setA(g, 0, n, 0, 0, 1, 0, 1);
                setB(g, 0, 1, 0, v, 0, 0);
                setC(g, 0, n, 0, 1);
                ops_rc(g, c->L[s] + o, c->t1r + off1, n1, c->Lt[s], plane);
                g.beta = 1.0;
                run(c, g);
            }
            {
                TcGemm g = G0(v, NQ * n, o);
                setA(g, 0, 1, 0, 0, v, 0, 0);
                setB(g, 0, n, nn, 1, n, 1);
                setC(g, 0, n, nn, 1);
                ops_cc(g, c->t1r + off1, n1, c->Lt[s], plane, c->Lt[s] + (long long)o * n, plane);
                g.alpha = -1.0; g.beta = 1.0;
                run(c, g);
            }
        }
        for (int s = 0; s < 2; ++s) {
            const int o = d.o[s], v = d.v[s];
            TcGemm g = G0(NQ, 1, o * v);
            setA(g, 0, nn, 0, n, 1, v, 1);
            setB(g, v, 1, 0, 0, 0, 0);
            setC(g, 0, 1, 0, 0);
            ops_rc(g, c->L[s] + o, c->t1r + rowoff[s], n1, c->gam, NQ);
            g.beta = s ? 1.0 : 0.0;
            run(c, g);
        }
    }

    // ---- 4. M^Q_(col) = sum_(me) L^Q_me T[(me),(col)]: per column spin, the same-spin block then the alpha-beta block
    c->sec = 4;
    for (int sc = 0; sc < 2; ++sc) {
        if (n1s_[sc] == 0) continue;
        bool first = true;
        for (int k = 0; k < 2; ++k) {
            const int sr = k == 0 ? sc : 1 - sc;
            const int o = d.o[sr], v = d.v[sr];
            if (n1s_[sr] == 0) continue;
            const TOp t = t_block(c, x, sr, sc);
            if (sr == sc) {          // planar block: one real GEMM over the stacked Re|Im columns
                TcGemm g = G0(NQ, 2 * (int)n1s_[sc], o * v);
                setA(g, 0, nn, 0, n, 1, v, 1);
                setB(g, (long long)v * t.r_lo, t.r_lo, n1s_[sc], 1, (int)n1s_[sc], 1);
                setC(g, 0, ld1, n1, 1);
                ops_rr(g, c->L[sr] + o, t.p, c->Mq + rowoff[sc]);
                g.beta = first ? 0.0 : 1.0;
                run(c, g);
            } else {
                TcGemm g = G0(NQ, (int)n1s_[sc], o * v);
                setA(g, 0, nn, 0, n, 1, v, 1);
                setB(g, t.r_hi, t.r_lo, t.c_hi, t.c_lo, t.Clo, t.c_lo < t.r_lo);
                setC(g, 0, ld1, t.Clo, 1);                 // the column index of C is split like B's (shared Nlo)
                ops_rc(g, c->L[sr] + o, t.p, t.pim, c->Mq + rowoff[sc], n1);
                g.beta = first ? 0.0 : 1.0;
                run(c, g);
            }
            first = false;
        }
    }

    // ---- 5. E
    c->sec = 5;
    {
        EnergyArgs ea;
        for (int s = 0; s < 2; ++s) { ea.L[s] = c->L[s]; ea.Lt[s] = c->Lt[s]; ea.fock[s] = c->fockd[s]; }
        ea.t1r = c->t1r; ea.Mq = c->Mq; ea.gam = c->gam; ea.partial = c->partial;
        ea.counter = c->counters; ea.out = c->scal;
        k_energy<<<RED_BLOCKS, RED_THREADS, 0, STL>>>(d, ea);
        c->launches += 1;
    }

    // ---- 6. dressed Fock, F_ae, F_mi (as residual_pipeline, general path)
    c->sec = 6;
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = rowoff[s];
        double* F = c->Ft[s];
        CK(cudaMemcpyAsync(F, c->Fb[s], nn * 8, cudaMemcpyDeviceToDevice, STL));
        CK(cudaMemsetAsync(F + nn, 0, nn * 8, STL));
        {
            TcGemm g = G0((int)nn, 1, NQ);
            setA(g, 0, 1, 0, 0, nn, 0, 0);
            setB(g, 0, 1, 0, 0, 0, 0);
            setC(g, 0, 1, 0, 0);
            ops_rc(g, c->L[s], c->gam, NQ, F, nn);
            g.beta = 1.0;
            run(c, g);
        }
        if (o > 0) {
            {
                TcGemm g = G0(n, o, v);
                setA(g, 0, n, 0, 0, 1, 0, 1);
                setB(g, 0, 1, 0, v, 0, 0);
                setC(g, 0, n, 0, 1);
                ops_cc(g, F + o, nn, c->t1r + off1, n1, F, nn);
                g.beta = 1.0;
                run(c, g);
            }
            {
                TcGemm g = G0(v, n, o);
                setA(g, 0, 1, 0, 0, v, 0, 0);
                setB(g, 0, n, 0, 1, 0, 1);
                setC(g, 0, n, 0, 1);
                ops_cc(g, c->t1r + off1, n1, F, nn, F + (long long)o * n, nn);
                g.alpha = -1.0; g.beta = 1.0;
                run(c, g);
            }
            {
                TcGemm g = G0(n, n, NQ * o);
                setA(g, 0, n, 0, nn, 1, o, 1);
                setB(g, nn, n, 0, 1, 0, 1);
                setC(g, 0, n, 0, 1);
                ops_cc(g, c->Lt[s], plane, c->Lt[s], plane, F, nn);
                g.alpha = -1.0; g.beta = 1.0;
                run(c, g);
            }
            {
                TcGemm g = G0(v, v, NQ * o);
                setA(g, 0, 1, 0, ld1, v, o, 0);
                setB(g, nn, n, 0, 1, 0, 1);
                setC(g, 0, n, 0, 1);
                ops_cr(g, c->Mq + off1, n1, c->L[s] + o, F + (long long)o * n + o, nn);
                g.alpha = -1.0; g.beta = 1.0;
                run(c, g);
            }
            {
                TcGemm g = G0(o, o, NQ * v);
                setA(g, 0, n, 0, nn, 1, v, 1);
                setB(g, ld1, 1, 0, v, 0, 0);
                setC(g, 0, n, 0, 1);
                ops_rc(g, c->L[s] + o, c->Mq + off1, n1, F, nn);
                g.beta = 1.0;
                run(c, g);
            }
        }
    }

    // ---- 7. singles: r1 = sum_me T[(ia),(me)] f~_me (block by block) - sum_Q,n M_na L~_ni + sum_Q,f M_if L~_af
    c->sec = 7;
    for (int sr = 0; sr < 2; ++sr) {
        if (n1s_[sr] == 0) continue;
        bool first = true;
        for (int sk = 0; sk < 2; ++sk) {
            const int o = d.o[sk], v = d.v[sk];
            if (n1s_[sk] == 0) continue;
            const TOp t = t_block(c, x, sr, sk);
            TcGemm g = G0((int)n1s_[sr], 1, o * v);
            if (sr == sk) setA(g, 0, t.r_lo, 0, v, 1, v, 1);
            else setA(g, t.r_hi, t.r_lo, t.Rlo, t.c_hi, t.c_lo, t.Clo, t.c_lo < t.r_lo);
            setB(g, n, 1, 0, 0, 0, 0);
            setC(g, sr == sk ? 0 : t.Rlo, 1, 0, 0);      // row index of C split like A's (shared Mlo)
            ops_cc(g, t.p, t.pim, c->Ft[sk] + o, nn, c->r1buf + rowoff[sr], n1);
            g.beta = first ? 0.0 : 1.0;
            run(c, g);
            first = false;
        }
        if (first) CK(cudaMemsetAsync(c->r1buf + rowoff[sr], 0, 0, STL));
    }
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s];
        const long long off1 = rowoff[s];
        if (o == 0) continue;
        {
            TcGemm g = G0(o, v, NQ * o);
            setA(g, 0, 1, 0, nn, n, o, 0);
            setB(g, ld1, v, 0, 1, 0, 1);
            setC(g, 0, v, 0, 1);
            ops_cc(g, c->Lt[s], plane, c->Mq + off1, n1, c->r1buf + off1, n1);
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
        {
            TcGemm g = G0(o, v, NQ * v);
            setA(g, 0, v, 0, ld1, 1, v, 1);
            setB(g, nn, 1, 0, n, 0, 0);
            setC(g, 0, v, 0, 1);
            ops_cc(g, c->Mq + off1, n1, c->Lt[s] + (long long)o * n + o, plane, c->r1buf + off1, n1);
            g.beta = 1.0;
            run(c, g);
        }
    }

    // ---- 8. N^Q_ia = L~^Q_ai + M^Q_ia; o^4 integrals <mn||ij>~ (the dressed vectors are dead once the ring is done)
    c->sec = 8;
    EW(c, k_add_Lvo, (long long)NQ * 2 * n1, d, c->Lt[0], c->Lt[1], c->Mq, c->Nq);
    if (d.oo > 0) {
        const int oa = d.o[0], ob = d.o[1];
        const long long lY = 2LL * d.oo;
        TcGemm g = G0(oa * oa, ob * ob, NQ);
        setA(g, n, 1, oa, 0, nn, 0, 0);
        setB(g, 0, nn, n, 1, ob, 1);
        setC(g, ob * lY, ob, lY, 1);
        ops_cc(g, c->Lt[0], plane, c->Lt[1], plane, c->Wooab, d.oo);
        run(c, g);
    }
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s];
        if (d.po[s] == 0) continue;
        const long long o2 = (long long)o * o;
        TcGemm g = G0(o * o, o * o, NQ);
        setA(g, n, 1, o, 0, nn, 0, 0);
        setB(g, 0, nn, n, 1, o, 1);
        setC(g, o * 2 * o2, o, 2 * o2, 1);
        ops_cc(g, c->Lt[s], plane, c->Lt[s], plane, c->W4[s], o2);
        run(c, g);
    }

    // ---- 9. spin-conserving ring sector, one column slab (occupied indices j0..j1 of spin sc) at a time:
    //         W[:, slab] = 1/2 Kx T[:, slab] + Xd + Fd ;   Z[:, slab] = 1/2 N^T N[:, slab] - T W[:, slab] ;   r2 += fold(Z slab)
    c->sec = 9;
    for (int sc = 0; sc < 2; ++sc) {
        const int osc = d.o[sc], vsc = d.v[sc];
        if (n1s_[sc] == 0) continue;
        for (int j0 = 0; j0 < osc; j0 += c->slab_j[sc]) {
            const int j1 = j0 + c->slab_j[sc] < osc ? j0 + c->slab_j[sc] : osc;
            const long long wc = (long long)(j1 - j0) * vsc, ldW = 2 * wc, c0 = (long long)j0 * vsc;
            for (int sr = 0; sr < 2; ++sr) {
                const int o = d.o[sr], v = d.v[sr];
                if (n1s_[sr] == 0) continue;
                const TOp t = t_block(c, x, sr, sc);
                double* Wr = c->Wslab + rowoff[sr] * ldW;
                if (sr == sc) {
                    TcGemm g = G0((int)n1s_[sr], (int)(2 * wc), (int)n1s_[sr]);
                    setA(g, 0, n1s_[sr], 0, 0, 1, 0, 1);
                    setB(g, 0, t.r_lo, n1s_[sc], 1, (int)wc, 1);
                    setC(g, 0, ldW, wc, 1);
                    ops_rr(g, c->Kx[sr], t.p + c0, Wr);
                    g.alpha = 0.5;
                    run(c, g);
                    {   // + Xd[(m,e),(j,b)] = sum_Q L~_mj L~_be, j in the slab
                        TcGemm h = G0(o * (j1 - j0), v * v, NQ);
                        setA(h, n, 1, j1 - j0, 0, nn, 0, 0);
                        setB(h, 0, nn, n, 1, v, 1);
                        setC(h, (long long)v * ldW, v, 1, ldW);
                        ops_cc(h, c->Lt[sr] + j0, plane, c->Lt[sr] + (long long)o * n + o, plane, Wr, wc);
                        h.beta = 1.0;
                        run(c, h);
                    }
                    EW(c, k_add_Fd, (long long)o * v * v + (long long)o * o * v, o, v, n, c->Ft[sr], o, c->Ft[sr], o, c->Wslab, ldW, wc,
                       rowoff[sr], -c0, j0, j1);
                } else {
                    TcGemm g = G0((int)n1s_[sr], (int)wc, (int)n1s_[sr]);
                    setA(g, 0, n1s_[sr], 0, (long long)t.Rlo, 1, t.Rlo, 1);
                    setB(g, t.r_hi, t.r_lo, t.c_hi, t.c_lo, t.Clo, t.c_lo < t.r_lo);
                    setC(g, 0, ldW, t.Clo, 1);
                    ops_rc(g, c->Kx[sr], t.p + (long long)j0 * t.c_hi, t.pim, Wr, wc);
                    g.alpha = 0.5;
                    run(c, g);
                }
            }
            {   // Z slab = 1/2 N^T N[:, slab]
                TcGemm g = G0(n1, (int)wc, NQ);
                setA(g, 0, 1, 0, 0, ld1, 0, 0);
                setB(g, 0, ld1, 0, 1, 0, 1);
                setC(g, 0, ldW, 0, 1);
                ops_cc(g, c->Nq, n1, c->Nq + rowoff[sc] + c0, n1, c->Zslab, wc);
                g.alpha = 0.5;
                run(c, g);
            }
            for (int sr = 0; sr < 2; ++sr) {
                if (n1s_[sr] == 0) continue;
                for (int sk = 0; sk < 2; ++sk) {
                    if (n1s_[sk] == 0) continue;
                    const TOp t = t_block(c, x, sr, sk);
                    TcGemm g = G0((int)n1s_[sr], (int)wc, (int)n1s_[sk]);
                    if (sr == sk) { setA(g, 0, t.r_lo, 0, 0, 1, 0, 1); setB(g, 0, ldW, 0, 1, 0, 1); }
                    else { setA(g, t.r_hi, t.r_lo, t.Rlo, t.c_hi, t.c_lo, t.Clo, t.c_lo < t.r_lo); setB(g, (long long)t.Clo * ldW, ldW, 0, 1, 0, 1); }
                    setC(g, sr == sk ? 0 : (long long)t.Rlo * ldW, ldW, 0, 1);
                    ops_cc(g, t.p, t.pim, c->Wslab + rowoff[sk] * ldW, wc, c->Zslab + rowoff[sr] * ldW, wc);
                    g.alpha = -1.0; g.beta = 1.0;
                    run(c, g);
                }
            }
            EW(c, k_fold_slab, d.n_t2, d, sc, j0, j1, c->Zslab, wc, c->opairs[sc], c->vpairs[sc], r + 2 * d.n_t1);
        }
    }

    // ---- 10. spin-flip sector with T_AB[(i,B),(M,e)] = -t_iM^eB read from the packed block (sign folded into alpha)
    c->sec = 10;
    if (d.nA > 0 && d.nB > 0) {
        const int oa = d.o[0], ob = d.o[1], va = d.v[0], vb = d.v[1], nA = d.nA, nB = d.nB;
        const long long lA = 2LL * nA, lB = 2LL * nB;
        const double* tp = x + 2 * d.n_t1 + 2 * d.off_t2[2];
        const long long rI = 2LL * ob * va * vb, rB = 2, cM = 2LL * va * vb, cE = 2LL * vb;      // strides of i, B, M, e
        double *W = c->Wsf, *Z = c->Zsf;
        {   // W_BB = 1/2 Kx_BA T_AB
            TcGemm g = G0(nB, nB, nA);
            setA(g, 0, nA, 0, vb, 1, vb, 1);
            setB(g, rI, rB, cM, cE, va, 0);
            setC(g, 0, lB, va, 1);
            ops_rc(g, c->KxBA, tp, 1, W, nB);
            g.alpha = -0.5;
            run(c, g);
        }
        {
            TcGemm g = G0(ob * ob, va * va, NQ);
            setA(g, n, 1, ob, 0, nn, 0, 0);
            setB(g, 0, nn, n, 1, va, 1);
            setC(g, va * lB, va, 1, lB);
            ops_cc(g, c->Lt[1], plane, c->Lt[0] + (long long)oa * n + oa, plane, W, nB);
            g.beta = 1.0;
            run(c, g);
        }
        EW(c, k_add_Fd, (long long)ob * va * va + (long long)ob * ob * va, ob, va, n, c->Ft[1], ob, c->Ft[0], oa, W, lB, (long long)nB, 0LL, 0LL, 0, ob);
        {   // Z_AB = -T_AB W_BB
            TcGemm g = G0(nA, nB, nB);
            setA(g, rI, rB, vb, cM, cE, va, 0);
            setB(g, (long long)va * lB, lB, 0, 1, 0, 1);
            setC(g, (long long)vb * lB, lB, 0, 1);
            ops_cc(g, tp, 1, W, nB, Z, nB);
            g.alpha = 1.0;
            run(c, g);
        }
        EW(c, k_fold_slab, d.n_t2, d, 2, 0, 0, Z, (long long)nB, c->opairs[0], c->vpairs[0], r + 2 * d.n_t1);
        {   // W_AA = 1/2 Kx_BA^T T_AB^T
            TcGemm g = G0(nA, nA, nB);
            setA(g, 0, 1, 0, (long long)va * nA, nA, va, 0);
            setB(g, cM, cE, rI, rB, vb, 1);
            setC(g, 0, lA, vb, 1);
            ops_rc(g, c->KxBA, tp, 1, W, nA);
            g.alpha = -0.5;
            run(c, g);
        }
        {
            TcGemm g = G0(oa * oa, vb * vb, NQ);
            setA(g, n, 1, oa, 0, nn, 0, 0);
            setB(g, 0, nn, n, 1, vb, 1);
            setC(g, vb * lA, vb, 1, lA);
            ops_cc(g, c->Lt[0], plane, c->Lt[1] + (long long)ob * n + ob, plane, W, nA);
            g.beta = 1.0;
            run(c, g);
        }
        EW(c, k_add_Fd, (long long)oa * vb * vb + (long long)oa * oa * vb, oa, vb, n, c->Ft[0], oa, c->Ft[1], ob, W, lA, (long long)nA, 0LL, 0LL, 0, oa);
        {   // Z_BA = -T_AB^T W_AA
            TcGemm g = G0(nB, nA, nA);
            setA(g, cM, cE, va, rI, rB, vb, 1);
            setB(g, (long long)vb * lA, lA, 0, 1, 0, 1);
            setC(g, (long long)va * lA, lA, 0, 1);
            ops_cc(g, tp, 1, W, nA, Z, nA);
            g.alpha = 1.0;
            run(c, g);
        }
        EW(c, k_fold_slab, d.n_t2, d, 3, 0, 0, Z, (long long)nA, c->opairs[0], c->vpairs[0], r + 2 * d.n_t1);
    }

    // ---- 11. ladder phase: the arena now holds the tile-major amplitudes and the ladder outputs
    c->sec = 11;
    if (d.oo > 0) {
        CK(cudaMemsetAsync(c->Xt_ab, 0, (size_t)c->xt_ab_cnt * 8, STL));
        EW(c, k_build_Xt_ab, (long long)d.v[0] * d.v[1] * d.oo, d, t2p, c->Xt_ab, (d.v[1] + 7) / 8, (2 * d.oo + c->nt2_ab - 1) / c->nt2_ab, c->nt2_ab);
    }
    for (int s = 0; s < 2; ++s)
        if (d.po[s] > 0) {
            CK(cudaMemsetAsync(c->Xt_ss[s], 0, (size_t)c->xt_ss_cnt[s] * 8, STL));
            EW(c, k_build_Xt_ss, (long long)d.v[s] * d.v[s] * d.po[s], d, s, t2p, c->opairs[s], c->Xt_ss[s], (d.v[s] + 7) / 8,
               (2 * d.po[s] + c->nt2_ss[s] - 1) / c->nt2_ss[s], c->nt2_ss[s], c->anti_ss[s]);
        }
    if (c->timing && !c->capturing) CK(cudaEventRecord(c->ev[0], STL));
    c->launches += ladder_launch(c->lb, STL, c->num_sms, c->lad_side, c->lad_ev[0], c->lad_ev[1], c->opt.lad.overlap);
    c->flops += ladder_flops(c->lb);
    c->lad_flops = ladder_flops(c->lb);
    if (c->timing && !c->capturing) CK(cudaEventRecord(c->ev[1], STL));

    if (d.oo > 0) {
        const int oa = d.o[0], ob = d.o[1], va = d.v[0], vb = d.v[1], oo = d.oo;
        const long long lY = 2LL * oo;
        const double* tp = x + 2 * d.n_t1 + 2 * d.off_t2[2];
        double* Yvv = c->Yab + ((long long)oa * n + ob) * lY;
        EW(c, k_add_oo_rows, (long long)oo * lY, oa, ob, n, (long long)oo, c->Wooab, c->Yab, c->Voo);
        {   // + t_mN^aB ( <mN||iJ>~ + Y_iJ^mN )      (the t1 t1 part of tau goes through the rows (m,B) below)
            TcGemm g = G0(va * vb, oo, oo);
            setA(g, 2LL * vb, 2, vb, 0, 2LL * va * vb, 0, 0);
            setB(g, 0, lY, 0, 1, 0, 1);
            setC(g, n * lY, lY, 0, 1);
            ops_cc(g, tp, 1, c->Voo, oo, Yvv, oo);
            g.beta = 1.0;
            run(c, g);
        }
        {   // rows (m,B): Y^{mB} -= sum_N t_N^B Y^{mN}   (batched over m)
            TcGemm g = G0(vb, oo, ob);
            setA(g, 0, 1, 0, 0, vb, 0, 0);
            setB(g, 0, lY, 0, 1, 0, 1);
            setC(g, 0, lY, 0, 1);
            ops_cc(g, c->t1r + d.n1a, n1, c->Yab, oo, c->Yab + (long long)ob * lY, oo);
            g.nsb = oa; g.sbA = 0; g.sbB = n * lY; g.sbC = n * lY;
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
        {   // - sum_m t_m^a Y_iJ^mB
            TcGemm g = G0(va, vb * oo, oa);
            setA(g, 0, 1, 0, 0, va, 0, 0);
            setB(g, 0, n * lY, lY, 1, oo, 1);
            setC(g, 0, n * lY, lY, 1);
            ops_cc(g, c->t1r, n1, c->Yab + (long long)ob * lY, oo, Yvv, oo);
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
        {   // - sum_N t_N^B Y_iJ^aN   (batched over a)
            TcGemm g = G0(vb, oo, ob);
            setA(g, 0, 1, 0, 0, vb, 0, 0);
            setB(g, 0, lY, 0, 1, 0, 1);
            setC(g, 0, lY, 0, 1);
            ops_cc(g, c->t1r + d.n1a, n1, c->Yab + (long long)oa * n * lY, oo, Yvv, oo);
            g.nsb = va; g.sbA = 0; g.sbB = n * lY; g.sbC = n * lY;
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
    }
    for (int s = 0; s < 2; ++s) {
        const int o = d.o[s], v = d.v[s], po = d.po[s], pv = d.pv[s];
        const long long off1 = rowoff[s];
        if (po == 0 || pv == 0) continue;
        const long long lP = 2LL * po;
        const double* tss = t2p + 2 * d.off_t2[s];
        EW(c, k_ss_prep_lean, (long long)po * po, o, po, n, c->opairs[s], c->W4[s], c->Yss[s], c->Vp[s], c->Yoo[s]);
        {   // rows (a<b): + t_mn^ab ( <mn||ij>~ + Y_ij^mn ), m<n, straight from the packed block
            TcGemm g = G0(pv, po, po);
            setA(g, 0, 2, 0, 0, 2LL * pv, 0, 0);
            setB(g, 0, lP, 0, 1, 0, 1);
            setC(g, 0, 0, 0, 1);
            ops_cc(g, tss, 1, c->Vp[s], po, c->Yss[s], po);
            g.cm_table = c->cmp[s];
            g.beta = 1.0;
            run(c, g);
        }
        {   // rows (m,b): Y^{mb} -= 1/2 sum_n t_n^b Y^{mn}   (batched over m; supplies the t1 t1 part of tau)
            TcGemm g = G0(v, po, o);
            setA(g, 0, 1, 0, 0, v, 0, 0);
            setB(g, 0, lP, 0, 1, 0, 1);
            setC(g, 0, lP, 0, 1);
            ops_cc(g, c->t1r + off1, n1, c->Yoo[s], po, c->Yss[s] + (long long)o * lP, po);
            g.nsb = o; g.sbA = 0; g.sbB = (long long)o * lP; g.sbC = n * lP;
            g.alpha = -0.5; g.beta = 1.0;
            run(c, g);
        }
        double* Yvv = c->Yss[s] + ((long long)o * n + o) * lP;
        {   // Y^{ab} -= sum_m t_m^a Y^{mb}
            TcGemm g = G0(v, v * po, o);
            setA(g, 0, 1, 0, 0, v, 0, 0);
            setB(g, 0, n * lP, lP, 1, po, 1);
            setC(g, 0, n * lP, lP, 1);
            ops_cc(g, c->t1r + off1, n1, c->Yss[s] + (long long)o * lP, po, Yvv, po);
            g.alpha = -1.0; g.beta = 1.0;
            run(c, g);
        }
        {   // Y^{ab} += sum_m t_m^b Y^{ma}
            TcGemm g = G0(v, v * po, o);
            setA(g, 0, 1, 0, 0, v, 0, 0);
            setB(g, 0, n * lP, lP, 1, po, 1);
            setC(g, 0, lP, n * lP, 1);
            ops_cc(g, c->t1r + off1, n1, c->Yss[s] + (long long)o * lP, po, Yvv, po);
            g.beta = 1.0;
            run(c, g);
        }
    }

    // ---- 12. ladder pieces and singles into the packed residual
    c->sec = 12;
    {
        AsmArgs A;
        memset(&A, 0, sizeof(A));
        A.Yab = c->Yab; A.r1buf = c->r1buf;
        for (int s = 0; s < 2; ++s) { A.Yss[s] = c->Yss[s]; A.Ft[s] = c->Ft[s]; A.opairs[s] = c->opairs[s]; A.vpairs[s] = c->vpairs[s]; }
        A.r1p = r; A.r2p = r + 2 * d.n_t1;
        EW(c, k_fold_ladder, d.n_t1 + d.n_t2, d, A);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { c->cuda_err = (int)e; return RTCC_ECUDA; }
    return RTCC_OK;
#undef STL
}

int run_pipeline(rtcc_ctx* c, const double* x, double* r)
{ return c->lean ? residual_pipeline_lean(c, x, r) : residual_pipeline(c, x, r); }

}  // namespace

namespace {

int copy_in(rtcc_ctx* c, double* dst, const double* src, long long ndoubles)
{
    if (ndoubles <= 0) return 0;
    CK(cudaMemcpyAsync(dst, src, ndoubles * 8, (c->flags & RTCC_HOST_PTRS) ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, c->st));
    return 0;
}
int copy_out(const rtcc_ctx* cc, double* dst, const double* src, long long ndoubles)
{
    rtcc_ctx* c = const_cast<rtcc_ctx*>(cc);
    if (ndoubles <= 0) return 0;
    CK(cudaMemcpyAsync(dst, src, ndoubles * 8, (c->flags & RTCC_HOST_PTRS) ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, c->st));
    return 0;
}

// gr = R(gx), scal[0..1] = E; graph replay unless timing is on
int eval_gx(rtcc_ctx* c)
{
    if (c->graph && !c->timing) {
        CK(cudaGraphLaunch(c->graph, c->st));
        c->launches += c->res_launches;
        c->flops += c->res_flops;
        return 0;
    }
    int rc = run_pipeline(c, c->gx, c->gr);
    return rc;
}

int read_scal(rtcc_ctx* c)
{
    CK(cudaMemcpyAsync(c->h_scal, c->scal, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CK(cudaStreamSynchronize(c->st));
    return 0;
}

// R(t(tau)) and E(t(tau)) of the current propagation state, evaluated on first use
int ensure_state(rtcc_ctx* c)
{
    if (c->state_valid) return RTCC_OK;
    CK(cudaMemcpyAsync(c->gx, c->t_cur, (size_t)c->namp * 16, cudaMemcpyDeviceToDevice, c->st));
    int rc = eval_gx(c);
    if (rc) return rc;
    CK(cudaMemcpyAsync(c->r_cur, c->gr, (size_t)c->namp * 16, cudaMemcpyDeviceToDevice, c->st));
    if (read_scal(c)) return RTCC_ECUDA;
    c->E[0] = c->h_scal[0]; c->E[1] = c->h_scal[1];
    c->state_valid = true;
    return RTCC_OK;
}

void model_ladder_flops(rtcc_ctx* c)
{
    // pp apply = 4[P(va)^2 P(oa) + P(vb)^2 P(ob) + (va vb)^2 oa ob],
    //                 pp W-build = 2K[2P(va)^2 + 2P(vb)^2 + (va vb)^2]
    const Dims& d = c->d;
    double pva = d.pv[0], pvb = d.pv[1], vab = (double)d.v[0] * d.v[1];
    c->lad_model = 4.0 * (pva * pva * d.po[0] + pvb * pvb * d.po[1] + vab * vab * d.oo)
                 + 2.0 * d.NQ * (2.0 * pva * pva + 2.0 * pvb * pvb + vab * vab);
}

}  // namespace


namespace {

struct SizePlan {
    long long persistent = 0, arena = 0;       // doubles
    long long a_lt[2]{}, a_tss[2]{}, a_wslab = 0, a_zslab = 0, a_wsf = 0, a_zsf = 0;      // arena offsets, ring phase
    long long a_xt_ab = 0, a_xt_ss[2]{}, a_yab = 0, a_yss[2]{};                           // arena offsets, ladder phase
    long long xt_ab = 0, xt_ss[2]{};
    int slab_j[2]{1, 1};
};

// Device memory of a context in doubles, in closed form (tested against rtcc_sizes).  standard: everything resident;
// lean: persistent part + one arena shared by the ring phase (dressed vectors, same-spin pair-space blocks, one column
// slab of W and Z, or the spin-flip W and Z) and the ladder phase (tile-major amplitudes and the ladder outputs).
// ring products large enough for the three-multiplication form (below this the two extra launches cost more than they save)
inline bool ring3m_default(const Dims& d) { return d.n1 >= 1536; }

long long size_plan(const Dims& d, bool lean, int want_slab_j, SizePlan* out, bool ring3m = false)
{
    const long long n = d.n, nn = n * n, NQ = d.NQ, plane = NQ * nn, n1 = d.n1, nA = d.nA, nB = d.nB, oo = d.oo;
    const long long namp = d.n_t1 + d.n_t2;
    const long long nQt = (NQ + 15) / 16, nPt = (n + 7) / 8;
    auto al = [](long long x) { return (x + 31) / 32 * 32; };             // cudaMalloc granularity is far coarser; 256 B here
    SizePlan sp;
    long long P = 0;
    long long xt_ss[2], yss[2], tss[2];
    for (int s = 0; s < 2; ++s) {
        const long long o = d.o[s], v = d.v[s], po = d.po[s];
        const long long nt2 = 2 * po <= 64 ? 64 : 128, ncol = (2 * po + nt2 - 1) / nt2;
        xt_ss[s] = ((v + 15) / 16) * ((v + 7) / 8) * ncol * 128 * (nt2 + 4);
        yss[s] = nn * 2 * po;
        tss[s] = 2 * (o * v) * (o * v);
        P += plane + nn + nn + 2 * nn + (o * v) * (o * v);                  // L, fockd, Fb, Ft, Kx
        P += nPt * ((v + 15) / 16) * nQt * 16 * LD_LDA1 + nPt * ((v + 7) / 8) * nQt * 16 * LD_LDB1;      // LtA, LtB
        P += o * o * 2 * o * o + 2 * (po * 2 * po);                        // W4, Wp/Vp, Yoop
        if (lean) P += o * o * 2 * po + d.pv[s];                           // Yoo, row table
        else P += 2 * plane + 3 * (v * v * 2 * po) + xt_ss[s] + yss[s];    // Lt, Xss, tauss, Zv, Xt_ss, Yss
    }
    const long long nt2ab = 2 * oo <= 64 ? 64 : 128, ncolab = (2 * oo + nt2ab - 1) / nt2ab;
    const long long xt_ab = ((d.v[0] + 15) / 16) * ((d.v[1] + 7) / 8) * ncolab * 128 * (nt2ab + 4), yab = nn * 2 * oo;
    P += nB * nA + 2 * n1 + 2 * (2 * NQ * n1) + 2 * NQ + 2 * n1 + oo * 2 * oo;          // KxBA, t1r, Mq, Nq, gam, r1buf, Wooab
    P += (32LL << 20) + 4 * 2 * namp;                                                    // GEMM workspace, gx, gr, t_cur, r_cur
    if (lean) P += oo * 2 * oo;                                                           // Voo
    else P += 3 * (2 * n1 * n1) + 3 * (2 * nA * nB) + 2 * nB * nB + 2 * nA * nA + 2 * ((long long)d.v[0] * d.v[1] * 2 * oo) + xt_ab + yab;
    if (!lean && ring3m) P += 2 * n1 * n1 + nA * nB + nB * nB + nA * nA;                // Ts_sc, Wd_sc, Ts_AB, Wd_BB, Wd_AA
    sp.persistent = P;
    sp.xt_ab = xt_ab; sp.xt_ss[0] = xt_ss[0]; sp.xt_ss[1] = xt_ss[1];
    if (lean) {
        long long a = 0;
        for (int s = 0; s < 2; ++s) { sp.a_lt[s] = a; a += al(2 * plane); }
        const long long after_lt = a;
        for (int s = 0; s < 2; ++s) { sp.a_tss[s] = a; a += al(tss[s]); }
        const long long ring_fixed = a;
        long long c = 0;
        sp.a_xt_ab = c; c += al(xt_ab);
        for (int s = 0; s < 2; ++s) { sp.a_xt_ss[s] = c; c += al(xt_ss[s]); }
        sp.a_yab = c; c += al(yab);
        for (int s = 0; s < 2; ++s) { sp.a_yss[s] = c; c += al(yss[s]); }
        const long long ladder_total = c;
        const long long sf = al(2 * (nB > nA ? nB * nB : nA * nA)) + al(2 * nA * nB);
        // column slabs: as many occupied indices j per slab as fit beside the fixed part without growing the arena beyond the
        // ladder phase (at least one)
        for (int s = 0; s < 2; ++s) {
            const long long per_j = 2 * (n1 * 2 * d.v[s]);                   // W and Z columns of one j
            long long room = ladder_total - ring_fixed;
            long long nj = per_j > 0 ? room / (per_j + 64) : d.o[s];
            if (nj < 1) nj = 1;
            if (nj > d.o[s]) nj = d.o[s];
            if (want_slab_j > 0 && want_slab_j < nj) nj = want_slab_j;
            if (nj < 1) nj = 1;
            sp.slab_j[s] = (int)nj;
        }
        long long wc = 0;
        for (int s = 0; s < 2; ++s) { const long long w = (long long)sp.slab_j[s] * d.v[s]; if (w > wc) wc = w; }
        sp.a_wslab = ring_fixed; sp.a_zslab = ring_fixed + al(n1 * 2 * wc);
        const long long ring_total = sp.a_zslab + al(n1 * 2 * wc);
        sp.a_wsf = after_lt; sp.a_zsf = after_lt + al(2 * (nB > nA ? nB * nB : nA * nA));
        const long long sf_total = after_lt + sf;
        sp.arena = ring_total > ladder_total ? ring_total : ladder_total;
        if (sf_total > sp.arena) sp.arena = sf_total;
    }
    if (out) *out = sp;
    return sp.persistent + sp.arena;
}

}  // namespace

extern "C" {

const char* rtcc_strerror(int code)
{
    switch (code) {
        case RTCC_OK: return "ok";
        case RTCC_EINVAL: return "invalid argument";
        case RTCC_ENOMEM: return "out of memory";
        case RTCC_ECUDA: return "CUDA error";
        case RTCC_ENOCONV: return "micro-iterations did not converge";
        case RTCC_ENONFINITE: return "non-finite amplitudes";
        case RTCC_EIO: return "checkpoint file: I/O error or wrong format";
        default: return "unknown error";
    }
}

int rtcc_last_cuda_error(const rtcc_ctx* c) { return c ? c->cuda_err : g_create_cuda_err; }

int rtcc_set_default_option(const char* name, int value)
{
    if (!name) return RTCC_EINVAL;
    const std::string k(name);
    if (k == "fused") g_opt.fused = value != 0;
    else if (k == "fused_fock") g_opt.fused_fock = value != 0;
    else if (k == "graph") g_opt.graph = value != 0;
    else if (k == "stream_priorities") g_opt.prio = value != 0;
    else if (k == "gemm_tile") { if (value != 0 && value != 64 && value != 128) return RTCC_EINVAL; g_opt.tile = value; }
    else if (k == "ladder_split") { if (value < 0 || value > 64) return RTCC_EINVAL; g_opt.lad.force_split = value; }
    else if (k == "max_cluster") { if (value < 1 || value > 16) return RTCC_EINVAL; g_opt.lad.max_cluster = value; }
    else if (k == "ladder_cluster") { if (value < 0 || value > 16) return RTCC_EINVAL; g_opt.lad.force_cluster = value; }
    else if (k == "ladder_antisym") g_opt.lad.anti = value != 0;
    else if (k == "ladder_overlap") { if (value < 0 || value > 2) return RTCC_EINVAL; g_opt.lad.overlap = value; }
    else if (k == "ladder_tiles") { if (value < 1 || value > LW_MAXC) return RTCC_EINVAL; g_opt.lad.max_tiles = value; }
    else if (k == "lean") { if (value < -1 || value > 1) return RTCC_EINVAL; g_opt.lean = value; }
    else if (k == "ring_3m") { if (value < -1 || value > 1) return RTCC_EINVAL; g_opt.ring3m = value; }
    else if (k == "lean_slab") { if (value < 0) return RTCC_EINVAL; g_opt.lean_slab_j = value; }
    else if (k == "reset") g_opt = RtccOptions();
    else return RTCC_EINVAL;
    return RTCC_OK;
}

void rtcc_destroy(rtcc_ctx* c)
{
    if (!c) return;
    if (c->graph) cudaGraphExecDestroy(c->graph);
    if (c->ev[0]) cudaEventDestroy(c->ev[0]);
    if (c->ev[1]) cudaEventDestroy(c->ev[1]);
    if (c->ev_delta) cudaEventDestroy(c->ev_delta);
    for (int i = 0; i < 7; ++i) if (c->aux[i]) cudaStreamDestroy(c->aux[i]);
    if (c->lad_side) cudaStreamDestroy(c->lad_side);
    for (int i = 0; i < 2; ++i) if (c->lad_ev[i]) cudaEventDestroy(c->lad_ev[i]);
    for (int i = 0; i < 16; ++i) if (c->evs[i]) cudaEventDestroy(c->evs[i]);
    for (void* p : c->allocs) cudaFree(p);
    if (c->h_scal) cudaFreeHost(c->h_scal);
    delete c;
}

int rtcc_create(rtcc_ctx** out, int oa, int ob, int va, int vb, int NQ, const double* L, const double* fock,
                unsigned flags, void* cuda_stream)
{
    if (!out) return RTCC_EINVAL;
    *out = nullptr;
    if (!L || !fock || oa < 0 || ob < 0 || va < 1 || vb < 1 || NQ < 1 || oa + va != ob + vb || oa + ob < 1) return RTCC_EINVAL;
    if ((long long)(oa + va) * (oa + va) * (long long)NQ >= (1LL << 40)) return RTCC_EINVAL;
    rtcc_ctx* c = new (std::nothrow) rtcc_ctx();
    if (!c) return RTCC_ENOMEM;
    c->flags = flags;
    c->st = (cudaStream_t)cuda_stream;
    c->opt = g_opt;
    int rc = RTCC_OK;
#define FAIL(code) do { rc = (code); goto fail; } while (0)
#define CKC(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { c->cuda_err = (int)e_; rc = RTCC_ECUDA; goto fail; } } while (0)
#define DA(p, cnt, name) do { int r_ = dalloc(c, &(p), (long long)(cnt), name); if (r_) { rc = r_; goto fail; } } while (0)
    {
        Dims& d = c->d;
        d.o[0] = oa; d.o[1] = ob; d.v[0] = va; d.v[1] = vb; d.n = oa + va; d.NQ = NQ;
        d.n1a = oa * va; d.n1b = ob * vb; d.n1 = d.n1a + d.n1b;
        d.nA = oa * vb; d.nB = ob * va;
        for (int s = 0; s < 2; ++s) { d.po[s] = d.o[s] * (d.o[s] - 1) / 2; d.pv[s] = d.v[s] * (d.v[s] - 1) / 2; }
        d.oo = oa * ob;
        d.off_t1[0] = 0; d.off_t1[1] = d.n1a;
        d.off_t2[0] = 0; d.off_t2[1] = (long long)d.po[0] * d.pv[0];
        d.off_t2[2] = d.off_t2[1] + (long long)d.po[1] * d.pv[1];
        d.n_t1 = d.n1;
        d.n_t2 = d.off_t2[2] + (long long)d.oo * va * vb;
        c->namp = d.n_t1 + d.n_t2;
        const int n = d.n, n1 = d.n1;
        const long long nn = (long long)n * n, plane = (long long)NQ * nn;

        int dev = 0;
        CKC(cudaGetDevice(&dev));
        CKC(cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev));
        CKC(tcgemm_init());
        CKC(ladder_init());
        if (dress_smem(d) <= 200 * 1024 && c->opt.fused) {
            CKC(cudaFuncSetAttribute(k_dress, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dress_smem(d)));
            c->fused_dress = true;
            // dressed Fock / F / singles fused kernels: per-thread element counts and shared memory must fit
            const int om = d.o[0] > d.o[1] ? d.o[0] : d.o[1], vm = d.v[0] > d.v[1] ? d.v[0] : d.v[1];
            c->smem_fockp = sizeof(double) * 4 * (size_t)n * om;
            c->smem_fockf = sizeof(double) * (2 * (size_t)nn + 2 * (size_t)om * vm + 2 * (size_t)n * om);
            c->smem_postp = sizeof(double) * (3 * (size_t)om * vm + 2 * (size_t)om * om + 2 * (size_t)vm * vm);
            if (nn <= FUSE_MAXE * FUSE_T && (long long)vm * vm <= FUSE_MAXE * FUSE_T && om * om <= FUSE_T && om * vm <= 2 * FUSE_T &&
                c->smem_fockf <= 200 * 1024 && c->smem_postp <= 200 * 1024) {
                CKC(cudaFuncSetAttribute(k_fock_partial, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_fockp));
                CKC(cudaFuncSetAttribute(k_fock_finish, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_fockf));
                CKC(cudaFuncSetAttribute(k_postm_partial, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_postp));
                c->fuse_nch = NQ < 74 ? NQ : 74;
                c->fuse_sz = (long long)vm * vm + (long long)om * om + (long long)om * vm;
                c->fused_fock = c->opt.fused_fock != 0;
            }
        }
        CKC(cudaEventCreate(&c->ev[0]));
        CKC(cudaEventCreate(&c->ev[1]));
        CKC(cudaEventCreateWithFlags(&c->ev_delta, cudaEventDisableTiming));
        {   // helper branches: everything latency-bound outranks the SM-filling ladder branch (aux[2] = S[3])
            int lo = 0, hi = 0;
            CKC(cudaDeviceGetStreamPriorityRange(&lo, &hi));
            const bool prio = c->opt.prio != 0;
            for (int i = 0; i < 7; ++i)
                CKC(cudaStreamCreateWithPriority(&c->aux[i], cudaStreamNonBlocking, (prio && i != 2) ? hi : lo));
            CKC(cudaStreamCreateWithPriority(&c->lad_side, cudaStreamNonBlocking, lo));
        }
        for (int i = 0; i < 16; ++i) CKC(cudaEventCreateWithFlags(&c->evs[i], cudaEventDisableTiming));
        for (int i = 0; i < 2; ++i) CKC(cudaEventCreateWithFlags(&c->lad_ev[i], cudaEventDisableTiming));
        for (int i = 0; i < 8; ++i) c->S[i] = c->st;
        c->si = 0;
#ifdef RTCC_DEBUG_KNOBS
        if (const char* e = getenv("RTCC_SKIP_MASK")) c->skipmask = (unsigned)strtoul(e, nullptr, 0);
#endif
        CKC(cudaMallocHost((void**)&c->h_scal, 8 * sizeof(double)));

        // lean or standard layout?
        {
            SizePlan sp;
            // three-multiplication ring products: worth two extra launches and 2 n1^2 + ... doubles once the products are large
            bool r3m = c->opt.ring3m == 1 || (c->opt.ring3m == -1 && ring3m_default(d));
            const long long std_doubles = size_plan(d, false, 0, nullptr, false);
            const long long std3_doubles = size_plan(d, false, 0, nullptr, true);
            bool lean = c->opt.lean == 1;
            if (c->opt.lean == -1) {
                size_t fr = 0, tot = 0;
                CKC(cudaMemGetInfo(&fr, &tot));
                if (r3m && (double)std3_doubles * 8.0 > 0.94 * (double)fr) r3m = false;
                lean = (double)std_doubles * 8.0 > 0.94 * (double)fr;
            }
            c->lean = lean;
            c->ring3m = r3m && !lean;
            if (lean) {
                size_plan(d, true, c->opt.lean_slab_j, &sp);
                c->arena_cap = sp.arena;
                DA(c->arena, sp.arena, nullptr);
                c->slab_j[0] = sp.slab_j[0]; c->slab_j[1] = sp.slab_j[1];
                for (int s = 0; s < 2; ++s) {
                    c->Lt[s] = c->arena + sp.a_lt[s]; c->Tss[s] = c->arena + sp.a_tss[s];
                    c->Xt_ss[s] = c->arena + sp.a_xt_ss[s]; c->Yss[s] = c->arena + sp.a_yss[s];
                    c->xt_ss_cnt[s] = sp.xt_ss[s];
                }
                c->Wslab = c->arena + sp.a_wslab; c->Zslab = c->arena + sp.a_zslab;
                c->Wsf = c->arena + sp.a_wsf; c->Zsf = c->arena + sp.a_zsf;
                c->Xt_ab = c->arena + sp.a_xt_ab; c->Yab = c->arena + sp.a_yab;
                c->xt_ab_cnt = sp.xt_ab;
                c->fused_fock = false;                       // the fused singles kernel reads the whole pair-space matrix
                c->named.push_back({"Yab", {c->Yab, (long long)nn * 2 * d.oo}});
            }
        }
        for (int s = 0; s < 2; ++s) {
            DA(c->L[s], plane, s ? "L1" : "L0");
            if (!c->lean) DA(c->Lt[s], 2 * plane, s ? "Lt1" : "Lt0");
            DA(c->fockd[s], nn, nullptr);
            DA(c->Fb[s], nn, s ? "Fb1" : "Fb0");
            DA(c->Ft[s], 2 * nn, s ? "Ft1" : "Ft0");
            DA(c->Kx[s], (long long)d.o[s] * d.v[s] * d.o[s] * d.v[s], s ? "Kx1" : "Kx0");
            const int po = d.po[s], v = d.v[s], o = d.o[s];
            if (!c->lean) {
                DA(c->Xss[s], (long long)v * v * 2 * po, s ? "Xss1" : "Xss0");
                CKC(cudaMemsetAsync(c->Xss[s], 0, (size_t)std::max<long long>((long long)v * v * 2 * po, 1) * 8, c->st));   // rows e == f stay zero
            }
            {
                const int nt2 = 2 * po <= 64 ? 64 : 128;
                c->nt2_ss[s] = nt2;
                const long long ncol = (2 * po + nt2 - 1) / nt2;
                const long long cx = (long long)((v + 15) / 16) * ((v + 7) / 8) * ncol * 128 * (nt2 + 4);
                if (!c->lean) {
                    DA(c->Xt_ss[s], cx, nullptr);
                    CKC(cudaMemsetAsync(c->Xt_ss[s], 0, (size_t)(cx > 0 ? cx : 1) * 8, c->st));
                }
                const long long nQt = (NQ + 15) / 16, nPt = (n + 7) / 8;
                const long long ca = nPt * ((v + 15) / 16) * nQt * 16 * LD_LDA1, cb = nPt * ((v + 7) / 8) * nQt * 16 * LD_LDB1;
                DA(c->LtA[s], ca, nullptr);
                DA(c->LtB[s], cb, nullptr);
                CKC(cudaMemsetAsync(c->LtA[s], 0, (size_t)ca * 8, c->st));
                CKC(cudaMemsetAsync(c->LtB[s], 0, (size_t)cb * 8, c->st));
            }
            DA(c->W4[s], (long long)o * o * 2 * o * o, nullptr);
            DA(c->Wp[s], (long long)po * 2 * po, nullptr);
            DA(c->Yoop[s], (long long)po * 2 * po, nullptr);
            if (c->lean) {
                c->Vp[s] = c->Wp[s];
                DA(c->Yoo[s], (long long)o * o * 2 * po, nullptr);
                DA(c->cmp[s], d.pv[s], nullptr);
            } else {
                DA(c->tauss[s], (long long)v * v * 2 * po, nullptr);
                CKC(cudaMemsetAsync(c->tauss[s], 0, (size_t)std::max<long long>((long long)v * v * 2 * po, 1) * 8, c->st));
                DA(c->Yss[s], nn * 2 * po, s ? "Yss1" : "Yss0");
                DA(c->Zv[s], (long long)v * v * 2 * po, s ? "Zv1" : "Zv0");
                CKC(cudaMemsetAsync(c->Yss[s], 0, (size_t)(nn * 2 * po > 0 ? nn * 2 * po : 1) * 8, c->st));
            }
        }
        DA(c->KxBA, (long long)d.nB * d.nA, "KxBA");
        DA(c->t1r, 2LL * n1, "t1r");
        if (!c->lean) {
            DA(c->Tsc, 2LL * n1 * n1, "Tsc");
            CKC(cudaMemsetAsync(c->Tsc, 0, (size_t)(2LL * n1 * n1 > 0 ? 2LL * n1 * n1 : 1) * 8, c->st));   // i == m / a == e places stay zero
            DA(c->Wsc, 2LL * n1 * n1, "Wsc");
            DA(c->Zsc, 2LL * n1 * n1, "Zsc");
            DA(c->TAB, 2LL * d.nA * d.nB, "TAB");
            DA(c->WBB, 2LL * d.nB * d.nB, "WBB");
            DA(c->WAA, 2LL * d.nA * d.nA, "WAA");
            DA(c->ZAB, 2LL * d.nA * d.nB, "ZAB");
            DA(c->ZBA, 2LL * d.nB * d.nA, "ZBA");
            if (c->ring3m) {
                DA(c->Ts_sc, (long long)n1 * n1, nullptr);
                CKC(cudaMemsetAsync(c->Ts_sc, 0, (size_t)((long long)n1 * n1 > 0 ? (long long)n1 * n1 : 1) * 8, c->st));
                DA(c->Wd_sc, (long long)n1 * n1, nullptr);
                DA(c->Ts_AB, (long long)d.nA * d.nB, nullptr);
                DA(c->Wd_BB, (long long)d.nB * d.nB, nullptr);
                DA(c->Wd_AA, (long long)d.nA * d.nA, nullptr);
            }
        }
        DA(c->Mq, 2LL * NQ * n1, "Mq");
        if (c->fused_fock) {
            DA(c->fockPart, (long long)c->fuse_nch * 8 * nn, nullptr);
            DA(c->fockRed, 8 * nn, nullptr);
            DA(c->postPart, (long long)c->fuse_nch * 4 * c->fuse_sz, nullptr);
            DA(c->postRed, 4 * c->fuse_sz, nullptr);
        }
        DA(c->Nq, 2LL * NQ * n1, "Nq");
        DA(c->gam, 2LL * NQ, "gam");
        DA(c->r1buf, 2LL * n1, "r1buf");
        {
            const int nt2 = 2 * d.oo <= 64 ? 64 : 128;
            c->nt2_ab = nt2;
            const long long ncol = (2 * d.oo + nt2 - 1) / nt2;
            const long long cx = (long long)((va + 15) / 16) * ((vb + 7) / 8) * ncol * 128 * (nt2 + 4);
            if (!c->lean) {
                DA(c->Xt_ab, cx, nullptr);
                CKC(cudaMemsetAsync(c->Xt_ab, 0, (size_t)(cx > 0 ? cx : 1) * 8, c->st));
            }
        }
        if (!c->lean) {
            DA(c->Xab, (long long)va * vb * 2 * d.oo, "Xab");
            DA(c->tauab, (long long)va * vb * 2 * d.oo, nullptr);
            DA(c->Yab, nn * 2 * d.oo, "Yab");
        } else DA(c->Voo, (long long)d.oo * 2 * d.oo, nullptr);
        DA(c->Wooab, (long long)d.oo * 2 * d.oo, nullptr);
        c->ws_cap = 32LL << 20;
        DA(c->ws, c->ws_cap, nullptr);
        DA(c->partial, 2 * RED_BLOCKS, nullptr);
        DA(c->bmax, RED_BLOCKS, nullptr);
        DA(c->scal, 8, nullptr);
        DA(c->gx, 2 * c->namp, "gx");
        DA(c->gr, 2 * c->namp, "gr");
        DA(c->t_cur, 2 * c->namp, nullptr);
        DA(c->r_cur, 2 * c->namp, nullptr);
        DA(c->counters, 4, nullptr);
        CKC(cudaMemsetAsync(c->counters, 0, 4 * sizeof(unsigned), c->st));

        // inputs
        const cudaMemcpyKind kin = (flags & RTCC_HOST_PTRS) ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
        for (int s = 0; s < 2; ++s) {
            CKC(cudaMemcpyAsync(c->L[s], L + s * plane, plane * 8, kin, c->st));
            CKC(cudaMemcpyAsync(c->fockd[s], fock + s * nn, nn * 8, kin, c->st));
        }
        // pair tables and ladder row tiles
        for (int s = 0; s < 2; ++s) {
            std::vector<int2> op((size_t)(d.po[s] > 0 ? d.po[s] : 1)), vp((size_t)(d.pv[s] > 0 ? d.pv[s] : 1));
            for (int j = 0; j < d.o[s]; ++j) for (int i = 0; i < j; ++i) op[(size_t)pair_index(i, j)] = make_int2(i, j);
            for (int b = 0; b < d.v[s]; ++b) for (int a = 0; a < b; ++a) vp[(size_t)pair_index(a, b)] = make_int2(a, b);
            DA(c->opairs[s], op.size(), nullptr);
            DA(c->vpairs[s], vp.size(), nullptr);
            CKC(cudaMemcpy(c->opairs[s], op.data(), op.size() * sizeof(int2), cudaMemcpyHostToDevice));
            CKC(cudaMemcpy(c->vpairs[s], vp.data(), vp.size() * sizeof(int2), cudaMemcpyHostToDevice));
            if (c->lean && d.pv[s] > 0)
                k_pair_row_table<<<nblk(d.pv[s], 1024), 256, 0, c->st>>>(d.o[s], n, d.pv[s], 2LL * d.po[s], c->vpairs[s], c->cmp[s]);
        }
        {
            std::vector<int2> tab, tss;
            for (int p0 = 0; p0 < n; p0 += LD_PP)
                for (int q0 = 0; q0 < n; q0 += LD_PQ) {
                    tab.push_back(make_int2(p0, q0));
                    if (p0 <= q0) tss.push_back(make_int2(p0, q0));
                }
            DA(c->tiles_ab, tab.size(), nullptr);
            CKC(cudaMemcpy(c->tiles_ab, tab.data(), tab.size() * sizeof(int2), cudaMemcpyHostToDevice));
            c->ntiles_ab = (int)tab.size();
            for (int s = 0; s < 2; ++s) {
                DA(c->tiles_ss[s], tss.size(), nullptr);
                CKC(cudaMemcpy(c->tiles_ss[s], tss.data(), tss.size() * sizeof(int2), cudaMemcpyHostToDevice));
                c->ntiles_ss[s] = (int)tss.size();
            }
        }
        {   // ladder work plan: one launch for the ab, aa, bb cases
            LadderBatch& B = c->lb;
            B.ncase = 0;
            B.NQ = (NQ + 15) / 16 * 16;
            for (int s = 0; s < 2; ++s) {
                const int v = d.v[s], nQt = (NQ + 15) / 16;
                EW(c, k_tile_L, (long long)NQ * n * v, NQ, n, d.o[s], v, LD_PP, LD_PE, (v + 15) / 16, nQt, c->L[s], c->LtA[s]);
                EW(c, k_tile_L, (long long)NQ * n * v, NQ, n, d.o[s], v, LD_PQ, LD_PF, (v + 7) / 8, nQt, c->L[s], c->LtB[s]);
            }
            auto add = [&](int sa, int sb, const double* Xt, int cols, double* Y, const int2* tiles, int ntiles) {
                if (cols <= 0 || ntiles <= 0) return;
                LadderCase& g = B.c[B.ncase++];
                g.LA = c->LtA[sa]; g.LB = c->LtB[sb];
                g.nA = g.nB = n; g.vA = d.v[sa]; g.vB = d.v[sb];
                g.X = Xt; g.N2 = 2 * cols; g.Y = Y; g.ldY = 2LL * cols; g.Ypart = nullptr;
                g.tiles = tiles; g.ntiles = ntiles;
                g.same = sa == sb; g.anti = 0;
            };
            add(0, 1, c->Xt_ab, d.oo, c->Yab, c->tiles_ab, c->ntiles_ab);
            add(0, 0, c->Xt_ss[0], d.po[0], c->Yss[0], c->tiles_ss[0], c->ntiles_ss[0]);
            add(1, 1, c->Xt_ss[1], d.po[1], c->Yss[1], c->tiles_ss[1], c->ntiles_ss[1]);
            ladder_probe_occupancy(c->locc, c->num_sms);
            ladder_plan(B, c->num_sms, 8, c->locc, c->opt.lad);
            for (int i = 0; i < B.ncase; ++i)
                for (int s = 0; s < 2; ++s)
                    if (B.c[i].same && B.c[i].X == c->Xt_ss[s]) c->anti_ss[s] = B.c[i].anti;
            for (int i = 0; i < B.ncase; ++i)
                if (B.c[i].nsplit > 1) {
                    const long long cnt = (long long)B.c[i].nsplit * nn * B.c[i].ldY;
                    DA(B.c[i].Ypart, cnt, nullptr);
                    CKC(cudaMemsetAsync(B.c[i].Ypart, 0, (size_t)cnt * 8, c->st));
                }
        }
        // constant integral blocks: Kx (exchange-type oovv), K_bare added to the Fock matrix
        for (int s = 0; s < 2; ++s) {
            const int o = d.o[s], v = d.v[s], n1s = o * v;
            CKC(cudaMemcpyAsync(c->Fb[s], c->fockd[s], nn * 8, cudaMemcpyDeviceToDevice, c->st));
            if (o == 0) continue;
            {
                TcGemm g = G0(n1s, n1s, NQ);
                setA(g, n, 1, v, 0, nn, 0, 0);
                setB(g, 0, nn, n, 1, v, 1);
                setC(g, (long long)v * n1s, 1, v, n1s);
                ops_rr(g, c->L[s] + o, c->L[s] + o, c->Kx[s]);
                run(c, g);
            }
            {
                TcGemm g = G0(n, n, NQ * o);
                setA(g, 0, n, 0, nn, 1, o, 1);
                setB(g, nn, n, 0, 1, 0, 1);
                setC(g, 0, n, 0, 1);
                ops_rr(g, c->L[s], c->L[s], c->Fb[s]);
                g.beta = 1.0;
                run(c, g);
            }
        }
        if (d.nA > 0 && d.nB > 0) {
            TcGemm g = G0(ob * vb, oa * va, NQ);
            setA(g, n, 1, vb, 0, nn, 0, 0);
            setB(g, 0, nn, n, 1, va, 1);
            setC(g, (long long)va * d.nA, 1, vb, d.nA);
            ops_rr(g, c->L[1] + ob, c->L[0] + oa, c->KxBA);
            run(c, g);
        }
        {   // orbital-energy tables of the five segments of the packed amplitude vector (denominators formed on the fly)
            const long long cnt[10] = {oa, ob, d.po[0], d.po[1], d.oo, va, vb, d.pv[0], d.pv[1], (long long)va * vb};
            long long tot = 0, offs[10];
            for (int k = 0; k < 10; ++k) { offs[k] = tot; tot += cnt[k]; }
            DA(c->dtab, tot, nullptr);
            EW(c, k_build_denominator_tables, tot, d, c->fockd[0], c->fockd[1], c->opairs[0], c->opairs[1], c->vpairs[0], c->vpairs[1], c->dtab);
            AmpSegs& sg = c->segs;
            const long long len[5] = {(long long)oa * va, (long long)ob * vb, (long long)d.po[0] * d.pv[0], (long long)d.po[1] * d.pv[1], (long long)d.oo * va * vb};
            const int ncol[5] = {va, vb, d.pv[0], d.pv[1], va * vb};
            sg.off[0] = 0;
            for (int k = 0; k < 5; ++k) {
                sg.off[k + 1] = sg.off[k] + len[k];
                sg.ncol[k] = ncol[k] > 0 ? ncol[k] : 1;
                sg.rowE[k] = c->dtab + offs[k];
                sg.colE[k] = c->dtab + offs[5 + k];
            }
        }
        CKC(cudaMemsetAsync(c->t_cur, 0, (size_t)c->namp * 16, c->st));
        CKC(cudaMemsetAsync(c->gx, 0, (size_t)c->namp * 16, c->st));
        model_ladder_flops(c);

        // One evaluation is captured as a CUDA graph (the capture pass also counts its launches / flops).  R(T=0), E(T=0) are
        // evaluated by the first call that needs them (ensure_state): a residual costs minutes at the largest sizes.
        c->state_valid = false;
        if (c->opt.graph) {
            cudaStream_t cs = nullptr;
            cudaStream_t user = c->st;
            CKC(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
            long long l0 = c->launches; double f0 = c->flops;
            c->st = cs; c->capturing = true;
            cudaGraph_t gph = nullptr;
            cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
            int prc = RTCC_OK;
            if (e == cudaSuccess) {
                prc = run_pipeline(c, c->gx, c->gr);
                e = cudaStreamEndCapture(cs, &gph);
            }
            c->st = user; c->capturing = false;
            c->res_launches = c->launches - l0; c->res_flops = c->flops - f0;
            c->launches = l0; c->flops = f0;
            if (e == cudaSuccess && prc == RTCC_OK && gph) e = cudaGraphInstantiate(&c->graph, gph, 0);
            if (gph) cudaGraphDestroy(gph);
            cudaStreamDestroy(cs);
            if (e != cudaSuccess || prc != RTCC_OK) { c->cuda_err = (int)e; rc = RTCC_ECUDA; goto fail; }
        }
        CKC(cudaStreamSynchronize(c->st));
    }
    *out = c;
    return RTCC_OK;
fail:
    g_create_cuda_err = c->cuda_err;
    cudaGetLastError();
    rtcc_destroy(c);
    return rc;
#undef FAIL
#undef CKC
#undef DA
}

int rtcc_sizes(const rtcc_ctx* c, long long* n_t1, long long* n_t2, long long* workspace_bytes)
{
    if (!c) return RTCC_EINVAL;
    if (n_t1) *n_t1 = c->d.n_t1;
    if (n_t2) *n_t2 = c->d.n_t2;
    if (workspace_bytes) *workspace_bytes = c->bytes;
    return RTCC_OK;
}

int rtcc_problem_sizes(int oa, int ob, int va, int vb, int NQ, long long out[6])
{
    if (!out || oa < 0 || ob < 0 || va < 1 || vb < 1 || NQ < 1 || oa + va != ob + vb) return RTCC_EINVAL;
    Dims d{};
    d.o[0] = oa; d.o[1] = ob; d.v[0] = va; d.v[1] = vb; d.n = oa + va; d.NQ = NQ;
    d.n1a = oa * va; d.n1b = ob * vb; d.n1 = d.n1a + d.n1b; d.nA = oa * vb; d.nB = ob * va;
    for (int s = 0; s < 2; ++s) { d.po[s] = d.o[s] * (d.o[s] - 1) / 2; d.pv[s] = d.v[s] * (d.v[s] - 1) / 2; }
    d.oo = oa * ob;
    d.off_t2[0] = 0; d.off_t2[1] = (long long)d.po[0] * d.pv[0]; d.off_t2[2] = d.off_t2[1] + (long long)d.po[1] * d.pv[1];
    d.n_t1 = d.n1; d.n_t2 = d.off_t2[2] + (long long)d.oo * va * vb;
    out[0] = d.n_t1;
    out[1] = d.n_t2;
    out[2] = (long long)oa * oa * va * va + (long long)ob * ob * vb * vb + (long long)oa * ob * va * vb;     // the paper's unpacked spin blocks
    out[3] = 2LL * NQ * d.n * d.n;
    out[4] = 8 * size_plan(d, false, 0, nullptr, ring3m_default(d));
    out[5] = 8 * size_plan(d, true, 0, nullptr);
    return RTCC_OK;
}

int rtcc_residual(rtcc_ctx* c, const double* t1, const double* t2, double* r1, double* r2)
{
    if (!c || !t1 || !t2 || !r1 || !r2) return RTCC_EINVAL;
    const Dims& d = c->d;
    if (copy_in(c, c->gx, t1, 2 * d.n_t1)) return RTCC_ECUDA;
    if (copy_in(c, c->gx + 2 * d.n_t1, t2, 2 * d.n_t2)) return RTCC_ECUDA;
    int rc = eval_gx(c);
    if (rc) return rc;
    if (copy_out(c, r1, c->gr, 2 * d.n_t1)) return RTCC_ECUDA;
    if (copy_out(c, r2, c->gr + 2 * d.n_t1, 2 * d.n_t2)) return RTCC_ECUDA;
    if (read_scal(c)) return RTCC_ECUDA;
    c->E_res[0] = c->h_scal[0]; c->E_res[1] = c->h_scal[1];
    if (c->timing) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]));
        c->lad_ms = ms;
    }
    return RTCC_OK;
}

int rtcc_residual_energy(const rtcc_ctx* c, double out[2])
{
    if (!c || !out) return RTCC_EINVAL;
    out[0] = c->E_res[0]; out[1] = c->E_res[1];
    return RTCC_OK;
}

int rtcc_set_amplitudes(rtcc_ctx* c, const double* t1, const double* t2, double time, const double cc[2])
{
    if (!c || !t1 || !t2 || !cc || !std::isfinite(time)) return RTCC_EINVAL;
    const Dims& d = c->d;
    if (copy_in(c, c->gx, t1, 2 * d.n_t1)) return RTCC_ECUDA;
    if (copy_in(c, c->gx + 2 * d.n_t1, t2, 2 * d.n_t2)) return RTCC_ECUDA;
    int rc = eval_gx(c);
    if (rc) return rc;
    CK(cudaMemcpyAsync(c->t_cur, c->gx, (size_t)c->namp * 16, cudaMemcpyDeviceToDevice, c->st));
    CK(cudaMemcpyAsync(c->r_cur, c->gr, (size_t)c->namp * 16, cudaMemcpyDeviceToDevice, c->st));
    if (read_scal(c)) return RTCC_ECUDA;
    c->E[0] = c->h_scal[0]; c->E[1] = c->h_scal[1];
    c->time = time; c->C[0] = cc[0]; c->C[1] = cc[1];
    c->state_valid = true;
    return RTCC_OK;
}

int rtcc_get_amplitudes(const rtcc_ctx* c, double* t1, double* t2)
{
    if (!c || !t1 || !t2) return RTCC_EINVAL;
    const Dims& d = c->d;
    if (copy_out(c, t1, c->t_cur, 2 * d.n_t1)) return RTCC_ECUDA;
    if (copy_out(c, t2, c->t_cur + 2 * d.n_t1, 2 * d.n_t2)) return RTCC_ECUDA;
    if (cudaStreamSynchronize(c->st) != cudaSuccess) return RTCC_ECUDA;
    return RTCC_OK;
}

// ---- checkpoint / restart.  File: header, then t(tau) and R(t(tau)) as packed interleaved complex128.
namespace {
struct CkptHeader {
    char magic[8];                 // "RTCCCKP1"
    int oa, ob, va, vb, nchol, mode, max_micro, fixed_micro;
    long long n_t1, n_t2;
    double tol, time, C[2], E[2];
};
int stream_file(rtcc_ctx* c, FILE* f, double* dev, long long ndoubles, bool write)
{
    const long long chunk = 1LL << 23;                          // 64 MiB of doubles per hop through pinned memory
    double* h = nullptr;
    if (cudaMallocHost((void**)&h, (size_t)chunk * 8) != cudaSuccess) { cudaGetLastError(); return RTCC_ENOMEM; }
    int rc = RTCC_OK;
    for (long long o = 0; o < ndoubles && !rc; o += chunk) {
        const long long m = ndoubles - o < chunk ? ndoubles - o : chunk;
        if (write) {
            if (cudaMemcpyAsync(h, dev + o, (size_t)m * 8, cudaMemcpyDeviceToHost, c->st) != cudaSuccess || cudaStreamSynchronize(c->st) != cudaSuccess) rc = RTCC_ECUDA;
            else if (fwrite(h, 8, (size_t)m, f) != (size_t)m) rc = RTCC_EIO;
        } else {
            if (fread(h, 8, (size_t)m, f) != (size_t)m) rc = RTCC_EIO;
            else if (cudaMemcpyAsync(dev + o, h, (size_t)m * 8, cudaMemcpyHostToDevice, c->st) != cudaSuccess || cudaStreamSynchronize(c->st) != cudaSuccess) rc = RTCC_ECUDA;
        }
    }
    cudaFreeHost(h);
    return rc;
}
}  // namespace

int rtcc_save(const rtcc_ctx* cc, const char* path)
{
    rtcc_ctx* c = const_cast<rtcc_ctx*>(cc);
    if (!c || !path) return RTCC_EINVAL;
    { int rc0 = ensure_state(c); if (rc0) return rc0; }
    FILE* f = fopen(path, "wb");
    if (!f) return RTCC_EIO;
    CkptHeader h;
    memset(&h, 0, sizeof(h));
    memcpy(h.magic, "RTCCCKP1", 8);
    const Dims& d = c->d;
    h.oa = d.o[0]; h.ob = d.o[1]; h.va = d.v[0]; h.vb = d.v[1]; h.nchol = d.NQ;
    h.mode = c->mode; h.max_micro = c->max_micro; h.fixed_micro = c->fixed_micro; h.tol = c->tol;
    h.n_t1 = d.n_t1; h.n_t2 = d.n_t2; h.time = c->time;
    h.C[0] = c->C[0]; h.C[1] = c->C[1]; h.E[0] = c->E[0]; h.E[1] = c->E[1];
    int rc = fwrite(&h, sizeof(h), 1, f) == 1 ? RTCC_OK : RTCC_EIO;
    if (!rc) rc = stream_file(c, f, c->t_cur, 2 * c->namp, true);
    if (!rc) rc = stream_file(c, f, c->r_cur, 2 * c->namp, true);
    if (fclose(f) != 0 && !rc) rc = RTCC_EIO;
    return rc;
}

int rtcc_load(rtcc_ctx* c, const char* path)
{
    if (!c || !path) return RTCC_EINVAL;
    FILE* f = fopen(path, "rb");
    if (!f) return RTCC_EIO;
    CkptHeader h;
    const Dims& d = c->d;
    int rc = RTCC_OK;
    if (fread(&h, sizeof(h), 1, f) != 1 || memcmp(h.magic, "RTCCCKP1", 8) != 0) rc = RTCC_EIO;
    else if (h.oa != d.o[0] || h.ob != d.o[1] || h.va != d.v[0] || h.vb != d.v[1] || h.nchol != d.NQ || h.n_t1 != d.n_t1 || h.n_t2 != d.n_t2)
        rc = RTCC_EINVAL;                          // written for another problem
    if (!rc) {
        // read into the iterate buffers first so that a short file leaves the propagation state untouched
        rc = stream_file(c, f, c->gx, 2 * c->namp, false);
        if (!rc) rc = stream_file(c, f, c->gr, 2 * c->namp, false);
        if (!rc && fgetc(f) != EOF) rc = RTCC_EIO;
    }
    fclose(f);
    if (rc) return rc;
    CK(cudaMemcpyAsync(c->t_cur, c->gx, (size_t)c->namp * 16, cudaMemcpyDeviceToDevice, c->st));
    CK(cudaMemcpyAsync(c->r_cur, c->gr, (size_t)c->namp * 16, cudaMemcpyDeviceToDevice, c->st));
    CK(cudaStreamSynchronize(c->st));
    c->mode = h.mode; c->max_micro = h.max_micro; c->fixed_micro = h.fixed_micro; c->tol = h.tol;
    c->time = h.time; c->C[0] = h.C[0]; c->C[1] = h.C[1]; c->E[0] = h.E[0]; c->E[1] = h.E[1];
    c->state_valid = true;
    return RTCC_OK;
}

int rtcc_get_state(const rtcc_ctx* cc, double* t1, double* t2, double* r1, double* r2, double scal[5])
{
    rtcc_ctx* c = const_cast<rtcc_ctx*>(cc);
    if (!c || !t1 || !t2 || !r1 || !r2 || !scal) return RTCC_EINVAL;
    { int rc0 = ensure_state(c); if (rc0) return rc0; }
    const Dims& d = c->d;
    if (copy_out(c, t1, c->t_cur, 2 * d.n_t1) || copy_out(c, t2, c->t_cur + 2 * d.n_t1, 2 * d.n_t2)) return RTCC_ECUDA;
    if (copy_out(c, r1, c->r_cur, 2 * d.n_t1) || copy_out(c, r2, c->r_cur + 2 * d.n_t1, 2 * d.n_t2)) return RTCC_ECUDA;
    if (cudaStreamSynchronize(c->st) != cudaSuccess) return RTCC_ECUDA;
    scal[0] = c->time; scal[1] = c->C[0]; scal[2] = c->C[1]; scal[3] = c->E[0]; scal[4] = c->E[1];
    return RTCC_OK;
}

int rtcc_set_state(rtcc_ctx* c, const double* t1, const double* t2, const double* r1, const double* r2, const double scal[5])
{
    if (!c || !t1 || !t2 || !r1 || !r2 || !scal) return RTCC_EINVAL;
    for (int i = 0; i < 5; ++i) if (!std::isfinite(scal[i])) return RTCC_EINVAL;
    const Dims& d = c->d;
    // no residual evaluation: R(T(tau)) and E(tau) are part of the state the caller hands back
    if (copy_in(c, c->t_cur, t1, 2 * d.n_t1) || copy_in(c, c->t_cur + 2 * d.n_t1, t2, 2 * d.n_t2)) return RTCC_ECUDA;
    if (copy_in(c, c->r_cur, r1, 2 * d.n_t1) || copy_in(c, c->r_cur + 2 * d.n_t1, r2, 2 * d.n_t2)) return RTCC_ECUDA;
    if (c->flags & RTCC_HOST_PTRS) CK(cudaStreamSynchronize(c->st));      // the caller may reuse its host arrays on return
    c->time = scal[0]; c->C[0] = scal[1]; c->C[1] = scal[2]; c->E[0] = scal[3]; c->E[1] = scal[4];
    c->state_valid = true;
    return RTCC_OK;
}

int rtcc_set_solver(rtcc_ctx* c, int mode, double tol, int max_micro, int fixed_micro)
{
    if (!c || (mode != 0 && mode != 1) || !(tol > 0.0) || max_micro < 1 || fixed_micro < 0) return RTCC_EINVAL;
    c->mode = mode; c->tol = tol; c->max_micro = max_micro; c->fixed_micro = fixed_micro;
    return RTCC_OK;
}

// restores R(t(tau)) after a failed step (its storage held B): one residual evaluation at the unchanged amplitudes
static int restore_r_cur(rtcc_ctx* c)
{
    c->state_valid = false;
    return ensure_state(c);
}
int rtcc_step(rtcc_ctx* c, double dt)
{
    if (!c || !std::isfinite(dt)) return RTCC_EINVAL;
    { int rc0 = ensure_state(c); if (rc0) return rc0; }
    const long long N = c->namp;
    const double hh = 0.5 * dt;
    int k = 0;
    double E_new[2] = {0, 0};
    int fail = RTCC_OK;
    for (;;) {
        // first micro-iteration: B = t + (i dt/2) R(t) is formed inside the update and stored over R(t); later ones update the
        // iterate in place.  Three amplitude-sized vectors (t, B, iterate) + the residual of the iterate.
        const double* xin = k == 0 ? c->t_cur : c->gx;
        const double* rin = k == 0 ? c->r_cur : c->gr;
        k_am_update<<<RED_BLOCKS, RED_THREADS, 0, c->st>>>(N, c->segs, c->r_cur, rin, xin, c->mode, k == 0 ? 1 : 0, hh, c->gx, c->bmax,
                                                           c->counters + 1, c->scal + 2);
        c->launches += 1;
        if (cudaGetLastError() != cudaSuccess) { fail = RTCC_ECUDA; break; }
        ++k;
        const bool last_fixed = c->fixed_micro > 0 && k >= c->fixed_micro;
        // The convergence measure is copied back behind the update and the residual R(x_k) -- needed whether or not the
        // iteration stops here -- is launched at once; the host then waits only for the small copy, so the GPU never idles
        // on the host's decision.
        if (c->fixed_micro == 0) {
            CK(cudaMemcpyAsync(c->h_scal + 2, c->scal + 2, sizeof(double), cudaMemcpyDeviceToHost, c->st));
            CK(cudaEventRecord(c->ev_delta, c->st));
        }
        int rc = eval_gx(c);
        if (rc) { fail = rc; break; }
        if (c->fixed_micro > 0) {
            if (last_fixed) break;
            continue;
        }
        CK(cudaEventSynchronize(c->ev_delta));
        if (!std::isfinite(c->h_scal[2])) { fail = RTCC_ENONFINITE; break; }
        if (c->h_scal[2] < c->tol) break;
        if (k >= c->max_micro) { fail = RTCC_ENOCONV; break; }
    }
    if (!fail) {
        if (read_scal(c)) fail = RTCC_ECUDA;
        else if (!std::isfinite(c->h_scal[2]) || !std::isfinite(c->h_scal[0]) || !std::isfinite(c->h_scal[1])) fail = RTCC_ENONFINITE;
    }
    if (fail) {                                   // state not advanced: t(tau) is untouched, R(t(tau)) is evaluated again
        cudaStreamSynchronize(c->st);
        cudaGetLastError();
        if (k > 0) { int rc = restore_r_cur(c); if (rc && fail != RTCC_ECUDA) return rc; }
        return fail;
    }
    E_new[0] = c->h_scal[0]; E_new[1] = c->h_scal[1];
    // C += (i dt/2) (E_old + E_new)
    const double sr = c->E[0] + E_new[0], si = c->E[1] + E_new[1];
    c->C[0] += -hh * si;
    c->C[1] += hh * sr;
    CK(cudaMemcpyAsync(c->t_cur, c->gx, (size_t)N * 16, cudaMemcpyDeviceToDevice, c->st));
    CK(cudaMemcpyAsync(c->r_cur, c->gr, (size_t)N * 16, cudaMemcpyDeviceToDevice, c->st));
    c->E[0] = E_new[0]; c->E[1] = E_new[1];
    c->time += dt;
    c->last_micro = k;
    if (c->timing) {                      // ladder time of the step's last residual evaluation (the stream is idle: read_scal waited)
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]) == cudaSuccess) c->lad_ms = ms; else cudaGetLastError();
    }
    return RTCC_OK;
}

int rtcc_cumulant(const rtcc_ctx* cc, double out[4])
{
    rtcc_ctx* c = const_cast<rtcc_ctx*>(cc);
    if (!c || !out) return RTCC_EINVAL;
    { int rc0 = ensure_state(c); if (rc0) return rc0; }
    out[0] = c->C[0]; out[1] = c->C[1]; out[2] = c->E[0]; out[3] = c->E[1];
    return RTCC_OK;
}

int rtcc_last_micro_iterations(const rtcc_ctx* c) { return c ? c->last_micro : RTCC_EINVAL; }
double rtcc_time(const rtcc_ctx* c) { return c ? c->time : 0.0; }

int rtcc_counters(const rtcc_ctx* c, long long* launches, double* flops)
{
    if (!c) return RTCC_EINVAL;
    if (launches) *launches = c->launches;
    if (flops) *flops = c->flops;
    return RTCC_OK;
}
int rtcc_reset_counters(rtcc_ctx* c)
{
    if (!c) return RTCC_EINVAL;
    c->launches = 0; c->flops = 0.0;
    return RTCC_OK;
}
int rtcc_set_timing(rtcc_ctx* c, int on)
{
    if (!c) return RTCC_EINVAL;
    c->timing = on ? 1 : 0;
    return RTCC_OK;
}
int rtcc_ladder_timing(const rtcc_ctx* c, double* ms, double* flops, double* model_flops)
{
    if (!c) return RTCC_EINVAL;
    if (ms) *ms = c->lad_ms;
    if (flops) *flops = c->lad_flops;
    if (model_flops) *model_flops = c->lad_model;
    return RTCC_OK;
}

int rtcc_ladder_plan(const rtcc_ctx* c, int spin_case, int out[8])
{
    if (!c || !out || spin_case < 0 || spin_case >= c->lb.ncase) return RTCC_EINVAL;
    const LadderCase& g = c->lb.c[spin_case];
    out[0] = g.N2; out[1] = g.nt2; out[2] = g.ncol; out[3] = g.cl; out[4] = g.ngrp; out[5] = g.nsplit; out[6] = g.ntiles;
    out[7] = g.cl > 0 ? c->locc.act[g.cl] : c->num_sms;
    return RTCC_OK;
}

int rtcc_ladder_occupancy(const rtcc_ctx* c, int out[17])
{
    if (!c || !out) return RTCC_EINVAL;
    for (int i = 0; i <= 16; ++i) out[i] = c->locc.act[i];
    return RTCC_OK;
}

int rtcc_build_fock(int n, int NQ, const double* L, const double* eps, int cs, int ci, double* fock, unsigned flags, void* stream)
{
    if (n < 1 || NQ < 1 || !L || !eps || !fock || (cs != 0 && cs != 1) || ci < 0 || ci >= n) return RTCC_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const long long nn = (long long)n * n, nL = 2LL * NQ * nn;
    const double *dL = L, *de = eps; double* df = fock;
    double* buf = nullptr;
    cudaError_t e = cudaSuccess;
    if (flags & RTCC_HOST_PTRS) {
        if (cudaMalloc(&buf, (size_t)(nL + 2 * n + 2 * nn) * 8) != cudaSuccess) { cudaGetLastError(); return RTCC_ENOMEM; }
        e = cudaMemcpyAsync(buf, L, (size_t)nL * 8, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(buf + nL, eps, (size_t)2 * n * 8, cudaMemcpyHostToDevice, st);
        dL = buf; de = buf + nL; df = buf + nL + 2 * n;
    }
    if (e == cudaSuccess) {
        k_build_fock<<<nblk(2 * nn, 148 * 8), 256, 0, st>>>(n, NQ, dL, de, cs, ci, df);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess && (flags & RTCC_HOST_PTRS)) e = cudaMemcpyAsync(fock, df, (size_t)2 * nn * 8, cudaMemcpyDeviceToHost, st);
    const cudaError_t es = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = es;
    if (buf) cudaFree(buf);
    if (e != cudaSuccess) cudaGetLastError();
    return e == cudaSuccess ? RTCC_OK : RTCC_ECUDA;
}

int rtcc_spectral_function(int nt, double dt, const double* C, double eps_c, double e_corr, double eta, int nw,
                           const double* omega, double* G, double* A)
{
    if (nt < 2 || nw < 1 || !C || !omega || !A || !(dt > 0.0) || !(eta >= 0.0) || !std::isfinite(eps_c + e_corr)) return RTCC_EINVAL;
    double* buf = nullptr;
    const size_t cnt = (size_t)4 * nt + 2 * (size_t)nw;
    if (cudaMalloc(&buf, cnt * 8) != cudaSuccess) { cudaGetLastError(); return RTCC_ENOMEM; }
    double *dC = buf, *dG = buf + 2 * (size_t)nt, *dW = dG + 2 * (size_t)nt, *dA = dW + nw;
    cudaMemcpy(dC, C, (size_t)2 * nt * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dW, omega, (size_t)nw * 8, cudaMemcpyHostToDevice);
    k_green<<<nblk(nt, 1024), 256>>>(nt, dt, dC, eps_c + e_corr, dG);
    k_spectral<<<nw, RED_THREADS>>>(nt, dt, dG, eta, nw, dW, dA);
    cudaError_t e = cudaMemcpy(A, dA, (size_t)nw * 8, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && G) e = cudaMemcpy(G, dG, (size_t)2 * nt * 8, cudaMemcpyDeviceToHost);
    cudaFree(buf);
    return e == cudaSuccess ? RTCC_OK : RTCC_ECUDA;
}

int rtcc_fp64_peak(double* tflops)
{
    if (!tflops) return RTCC_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return RTCC_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return RTCC_ECUDA;
    double* buf = nullptr;
    const int grid = sms * 2, iters = 4000;
    if (cudaMalloc(&buf, (size_t)grid * 256 * 8) != cudaSuccess) { cudaGetLastError(); return RTCC_ENOMEM; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        k_dmma_peak<<<grid, 256>>>(buf, iters, 1e-9);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf);
    if (cudaGetLastError() != cudaSuccess) return RTCC_ECUDA;
    const double fl = 16.0 * 2.0 * 8 * 8 * 4 * (double)iters * 8.0 * grid;
    *tflops = fl / (best * 1e-3) * 1e-12;
    return RTCC_OK;
}

long long rtcc_debug_buffer(const rtcc_ctx* c, const char* name, double* out, long long max_doubles)
{
    if (!c || !name) return RTCC_EINVAL;
    for (auto& kv : c->named)
        if (kv.first == name) {
            long long cnt = kv.second.second;
            if (out && max_doubles > 0) {
                long long m = cnt < max_doubles ? cnt : max_doubles;
                if (cudaMemcpy(out, kv.second.first, (size_t)m * 8, cudaMemcpyDeviceToHost) != cudaSuccess) return RTCC_ECUDA;
            }
            return cnt;
        }
    return RTCC_EINVAL;
}

int rtcc_debug_gemm(int M, int N, int K, const double* A, const double* B, double* C, double alpha, double beta, int cplx)
{
    if (M < 1 || N < 1 || K < 0 || !A || !B || !C) return RTCC_EINVAL;
    const int np = cplx ? 2 : 1;
    double *dA = nullptr, *dB = nullptr, *dC = nullptr, *ws = nullptr;
    int sms = 148, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long wscap = 4LL << 20;
    if (cudaMalloc(&dA, (size_t)np * M * (K > 0 ? K : 1) * 8) != cudaSuccess || cudaMalloc(&dB, (size_t)np * (K > 0 ? K : 1) * N * 8) != cudaSuccess ||
        cudaMalloc(&dC, (size_t)np * M * N * 8) != cudaSuccess || cudaMalloc(&ws, wscap * 8) != cudaSuccess) {
        cudaFree(dA); cudaFree(dB); cudaFree(dC); cudaFree(ws);
        return RTCC_ENOMEM;
    }
    cudaMemcpy(dA, A, (size_t)np * M * K * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dB, B, (size_t)np * K * N * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dC, C, (size_t)np * M * N * 8, cudaMemcpyHostToDevice);
    tcgemm_init();
    TcGemm g = G0(M, N, K);
    setA(g, 0, K, 0, 0, 1, 0, 1);
    setB(g, 0, N, 0, 1, 0, 1);
    setC(g, 0, N, 0, 1);
    if (cplx) ops_cc(g, dA, (long long)M * K, dB, (long long)K * N, dC, (long long)M * N);
    else ops_rr(g, dA, dB, dC);
    g.alpha = alpha; g.beta = beta; g.ws = ws;
    tcgemm_launch(g, nullptr, wscap, sms, nullptr);
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(C, dC, (size_t)np * M * N * 8, cudaMemcpyDeviceToHost);
    cudaFree(dA); cudaFree(dB); cudaFree(dC); cudaFree(ws);
    return e == cudaSuccess ? RTCC_OK : RTCC_ECUDA;
}

}  // extern "C"
