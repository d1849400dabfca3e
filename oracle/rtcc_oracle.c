/*
 * rtcc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU oracle for the RT-EOM-CCSD right-hand side
 * (arXiv:2301.04249; /root/reference/PAPER.md).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may call it.  It shares no code
 * with the CUDA path under paper_2301_04249_b200/.
 *
 * What it computes (spin-orbital form, fp64, complex128 amplitudes):
 *   - the full antisymmetrised two-electron integrals <pq||rs> = (pr|qs) - (ps|qr) with
 *     (pq|rs) = sum_Q L^Q_pq L^Q_rs                 ("v^{rs}_{pq} = <pq||rs>";
 *                                                     PAPER.md:31,:129-131 Cholesky vectors)
 *   - R1_i^a  = <Phi_i^a |(H_N e^{T1+T2})_C|Phi>      (Eq. 7)
 *   - R2_ij^ab= <Phi_ij^ab|(H_N e^{T1+T2})_C|Phi>     (Eq. 8)
 *   - E       = <Phi|(H_N e^{T})_C|Phi>               (Eq. 5 integrand; Eq. 6
 *                                                     plus the f_ia t_i^a term, reading R4)
 * The paper prints only the formal projections; the expansion used here is the standard
 * spin-orbital CCSD one in intermediates F, W (reading R1), with
 * the FULL Fock blocks inside F_ae / F_mi so that the result is the complete projection
 * (no denominators).  Naive loops, no blocking, no BLAS; OpenMP only over the outermost loop.
 *
 * Parity pins (tests/test_oracle_pins.py): determinant-space brute force (P-0), Cholesky
 * reconstruction (P-1), exact two-electron dynamics (P-2), stationary limit = FCI (P-3),
 * t=0 / short time (P-4), weak-coupling closed form (P-5), invariants (P-6), separability (P-7).
 *
 * Index conventions: spin-orbitals ordered [alpha occ | beta occ | alpha virt | beta virt];
 * no = number of occupied, nv = number of virtual spin-orbitals, N = no+nv.
 * i,j,m,n occupied (0..no-1); a,b,e,f virtual (stored 0..nv-1, spin-orbital index no+a).
 * t1[i][a], t2[i][j][a][b], r1, r2 likewise; g[p][q][r][s] = <pq||rs> real; f[p][q] real.
 */
#include <complex.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Spin-orbital Cholesky vectors and Fock matrix from the per-spin inputs of the boundary
 * (include/rtcc.h): L[2][K][n][n], fock[2][n][n], each spin in its own [occ|virt] order.
 * L^Q_pq(spin-orbital) = 0 unless spin(p) == spin(q). */
static int so_index(int spin, int p, int oa, int ob, int va, int vb)
{
    int o = spin ? ob : oa;
    int no = oa + ob;
    if (p < o) return spin ? oa + p : p;
    return spin ? no + va + (p - o) : no + (p - o);
}

void orc_build_so(int oa, int ob, int va, int vb, int K, const double *L, const double *fock,
                  double *Lso /* [K][N][N] */, double *fso /* [N][N] */)
{
    int n = oa + va;            /* == ob + vb */
    int N = 2 * n;
    memset(Lso, 0, sizeof(double) * (size_t)K * N * N);
    memset(fso, 0, sizeof(double) * (size_t)N * N);
    for (int s = 0; s < 2; ++s)
        for (int p = 0; p < n; ++p)
            for (int q = 0; q < n; ++q) {
                int P = so_index(s, p, oa, ob, va, vb), Q_ = so_index(s, q, oa, ob, va, vb);
                fso[(size_t)P * N + Q_] = fock[((size_t)s * n + p) * n + q];
                for (int Q = 0; Q < K; ++Q)
                    Lso[((size_t)Q * N + P) * N + Q_] = L[(((size_t)s * K + Q) * n + p) * n + q];
            }
}

/* (pq|rs) = sum_Q L^Q_pq L^Q_rs  -- one element, direct Q-sum. */
double orc_eri_chem(int N, int K, const double *Lso, int p, int q, int r, int s)
{
    double acc = 0.0;
    for (int Q = 0; Q < K; ++Q)
        acc += Lso[((size_t)Q * N + p) * N + q] * Lso[((size_t)Q * N + r) * N + s];
    return acc;
}

/* g[p][q][r][s] = <pq||rs> = (pr|qs) - (ps|qr). */
void orc_eri_antisym(int N, int K, const double *Lso, double *g)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int p = 0; p < N; ++p)
        for (int q = 0; q < N; ++q)
            for (int r = 0; r < N; ++r)
                for (int s = 0; s < N; ++s) {
                    double d = 0.0, x = 0.0;
                    for (int Q = 0; Q < K; ++Q) {
                        const double *LQ = Lso + (size_t)Q * N * N;
                        d += LQ[(size_t)p * N + r] * LQ[(size_t)q * N + s];
                        x += LQ[(size_t)p * N + s] * LQ[(size_t)q * N + r];
                    }
                    g[(((size_t)p * N + q) * N + r) * N + s] = d - x;
                }
}

#define G(p, q, r, s) g[((((size_t)(p)) * N + (q)) * N + (r)) * N + (s)]
#define F(p, q) f[(size_t)(p) * N + (q)]
#define T1(i, a) t1[(size_t)(i) * nv + (a)]
#define T2(i, j, a, b) t2[((((size_t)(i)) * no + (j)) * nv + (a)) * nv + (b)]
#define R1(i, a) r1[(size_t)(i) * nv + (a)]
#define R2(i, j, a, b) r2[((((size_t)(i)) * no + (j)) * nv + (a)) * nv + (b)]
#define V(a) (no + (a)) /* spin-orbital index of virtual a */

/* tau~_ij^ab = t_ij^ab + 1/2 (t_i^a t_j^b - t_i^b t_j^a);  tau_ij^ab = t_ij^ab + t_i^a t_j^b - t_i^b t_j^a */
static inline cplx tau_t(const cplx *t1, const cplx *t2, int no, int nv, int i, int j, int a, int b)
{
    return T2(i, j, a, b) + 0.5 * (T1(i, a) * T1(j, b) - T1(i, b) * T1(j, a));
}
static inline cplx tau_f(const cplx *t1, const cplx *t2, int no, int nv, int i, int j, int a, int b)
{
    return T2(i, j, a, b) + T1(i, a) * T1(j, b) - T1(i, b) * T1(j, a);
}

/*
 * Residuals R1, R2 and E.  Returns 0, or -1 if scratch allocation fails.
 * E = sum_ia f_ia t_i^a + 1/4 sum <ij||ab> t_ij^ab + 1/2 sum <ij||ab> t_i^a t_j^b.
 */
int orc_residual(int no, int nv, const double *f, const double *g, const cplx *t1, const cplx *t2,
                 cplx *r1, cplx *r2, cplx *E_out)
{
    const int N = no + nv;
    cplx *Fae = malloc(sizeof(cplx) * (size_t)nv * nv);
    cplx *Fmi = malloc(sizeof(cplx) * (size_t)no * no);
    cplx *Fme = malloc(sizeof(cplx) * (size_t)no * nv);
    cplx *Wmnij = malloc(sizeof(cplx) * (size_t)no * no * no * no);
    cplx *Wmbej = malloc(sizeof(cplx) * (size_t)no * nv * nv * no);
    if (!Fae || !Fmi || !Fme || !Wmnij || !Wmbej) {
        free(Fae); free(Fmi); free(Fme); free(Wmnij); free(Wmbej);
        return -1;
    }
#define FAE(a, e) Fae[(size_t)(a) * nv + (e)]
#define FMI(m, i) Fmi[(size_t)(m) * no + (i)]
#define FME(m, e) Fme[(size_t)(m) * nv + (e)]
#define WMNIJ(m, n, i, j) Wmnij[((((size_t)(m)) * no + (n)) * no + (i)) * no + (j)]
#define WMBEJ(m, b, e, j) Wmbej[((((size_t)(m)) * nv + (b)) * nv + (e)) * no + (j)]

    /* F_ae = f_ae - 1/2 S_m f_me t_m^a + S_mf t_m^f <ma||fe> - 1/2 S_mnf tau~_mn^af <mn||ef> */
#pragma omp parallel for schedule(static)
    for (int a = 0; a < nv; ++a)
        for (int e = 0; e < nv; ++e) {
            cplx x = F(V(a), V(e));
            for (int m = 0; m < no; ++m) x -= 0.5 * F(m, V(e)) * T1(m, a);
            for (int m = 0; m < no; ++m)
                for (int ff = 0; ff < nv; ++ff) x += T1(m, ff) * G(m, V(a), V(ff), V(e));
            for (int m = 0; m < no; ++m)
                for (int n = 0; n < no; ++n)
                    for (int ff = 0; ff < nv; ++ff)
                        x -= 0.5 * tau_t(t1, t2, no, nv, m, n, a, ff) * G(m, n, V(e), V(ff));
            FAE(a, e) = x;
        }
    /* F_mi = f_mi + 1/2 S_e t_i^e f_me + S_ne t_n^e <mn||ie> + 1/2 S_nef tau~_in^ef <mn||ef> */
#pragma omp parallel for schedule(static)
    for (int m = 0; m < no; ++m)
        for (int i = 0; i < no; ++i) {
            cplx x = F(m, i);
            for (int e = 0; e < nv; ++e) x += 0.5 * T1(i, e) * F(m, V(e));
            for (int n = 0; n < no; ++n)
                for (int e = 0; e < nv; ++e) x += T1(n, e) * G(m, n, i, V(e));
            for (int n = 0; n < no; ++n)
                for (int e = 0; e < nv; ++e)
                    for (int ff = 0; ff < nv; ++ff)
                        x += 0.5 * tau_t(t1, t2, no, nv, i, n, e, ff) * G(m, n, V(e), V(ff));
            FMI(m, i) = x;
        }
    /* F_me = f_me + S_nf t_n^f <mn||ef> */
#pragma omp parallel for schedule(static)
    for (int m = 0; m < no; ++m)
        for (int e = 0; e < nv; ++e) {
            cplx x = F(m, V(e));
            for (int n = 0; n < no; ++n)
                for (int ff = 0; ff < nv; ++ff) x += T1(n, ff) * G(m, n, V(e), V(ff));
            FME(m, e) = x;
        }
    /* W_mnij = <mn||ij> + S_e (t_j^e <mn||ie> - t_i^e <mn||je>) + 1/4 S_ef tau_ij^ef <mn||ef> */
#pragma omp parallel for collapse(2) schedule(static)
    for (int m = 0; m < no; ++m)
        for (int n = 0; n < no; ++n)
            for (int i = 0; i < no; ++i)
                for (int j = 0; j < no; ++j) {
                    cplx x = G(m, n, i, j);
                    for (int e = 0; e < nv; ++e)
                        x += T1(j, e) * G(m, n, i, V(e)) - T1(i, e) * G(m, n, j, V(e));
                    for (int e = 0; e < nv; ++e)
                        for (int ff = 0; ff < nv; ++ff)
                            x += 0.25 * tau_f(t1, t2, no, nv, i, j, e, ff) * G(m, n, V(e), V(ff));
                    WMNIJ(m, n, i, j) = x;
                }
    /* W_mbej = <mb||ej> + S_f t_j^f <mb||ef> - S_n t_n^b <mn||ej>
     *          - S_nf (1/2 t_jn^fb + t_j^f t_n^b) <mn||ef> */
#pragma omp parallel for collapse(2) schedule(static)
    for (int m = 0; m < no; ++m)
        for (int b = 0; b < nv; ++b)
            for (int e = 0; e < nv; ++e)
                for (int j = 0; j < no; ++j) {
                    cplx x = G(m, V(b), V(e), j);
                    for (int ff = 0; ff < nv; ++ff) x += T1(j, ff) * G(m, V(b), V(e), V(ff));
                    for (int n = 0; n < no; ++n) x -= T1(n, b) * G(m, n, V(e), j);
                    for (int n = 0; n < no; ++n)
                        for (int ff = 0; ff < nv; ++ff)
                            x -= (0.5 * T2(j, n, ff, b) + T1(j, ff) * T1(n, b)) * G(m, n, V(e), V(ff));
                    WMBEJ(m, b, e, j) = x;
                }

    /* R1_i^a = f_ia + S_e t_i^e F_ae - S_m t_m^a F_mi + S_me t_im^ae F_me - S_nf t_n^f <na||if>
     *          - 1/2 S_mef t_im^ef <ma||ef> - 1/2 S_men t_mn^ae <nm||ei> */
#pragma omp parallel for schedule(static)
    for (int i = 0; i < no; ++i)
        for (int a = 0; a < nv; ++a) {
            cplx x = F(i, V(a));
            for (int e = 0; e < nv; ++e) x += T1(i, e) * FAE(a, e);
            for (int m = 0; m < no; ++m) x -= T1(m, a) * FMI(m, i);
            for (int m = 0; m < no; ++m)
                for (int e = 0; e < nv; ++e) x += T2(i, m, a, e) * FME(m, e);
            for (int n = 0; n < no; ++n)
                for (int ff = 0; ff < nv; ++ff) x -= T1(n, ff) * G(n, V(a), i, V(ff));
            for (int m = 0; m < no; ++m)
                for (int e = 0; e < nv; ++e)
                    for (int ff = 0; ff < nv; ++ff)
                        x -= 0.5 * T2(i, m, e, ff) * G(m, V(a), V(e), V(ff));
            for (int m = 0; m < no; ++m)
                for (int e = 0; e < nv; ++e)
                    for (int n = 0; n < no; ++n) x -= 0.5 * T2(m, n, a, e) * G(n, m, V(e), i);
            R1(i, a) = x;
        }

    /* R2_ij^ab, all terms except the W_abef one (added below, (a,b) slice by (a,b) slice). */
#pragma omp parallel for collapse(2) schedule(static)
    for (int i = 0; i < no; ++i)
        for (int j = 0; j < no; ++j)
            for (int a = 0; a < nv; ++a)
                for (int b = 0; b < nv; ++b) {
                    cplx x = G(i, j, V(a), V(b));
                    /* P(ab) S_e t_ij^ae (F_be - 1/2 S_m t_m^b F_me) */
                    for (int e = 0; e < nv; ++e) {
                        cplx fb = FAE(b, e), fa = FAE(a, e);
                        for (int m = 0; m < no; ++m) {
                            fb -= 0.5 * T1(m, b) * FME(m, e);
                            fa -= 0.5 * T1(m, a) * FME(m, e);
                        }
                        x += T2(i, j, a, e) * fb - T2(i, j, b, e) * fa;
                    }
                    /* - P(ij) S_m t_im^ab (F_mj + 1/2 S_e t_j^e F_me) */
                    for (int m = 0; m < no; ++m) {
                        cplx fj = FMI(m, j), fi = FMI(m, i);
                        for (int e = 0; e < nv; ++e) {
                            fj += 0.5 * T1(j, e) * FME(m, e);
                            fi += 0.5 * T1(i, e) * FME(m, e);
                        }
                        x -= T2(i, m, a, b) * fj - T2(j, m, a, b) * fi;
                    }
                    /* 1/2 S_mn tau_mn^ab W_mnij */
                    for (int m = 0; m < no; ++m)
                        for (int n = 0; n < no; ++n)
                            x += 0.5 * tau_f(t1, t2, no, nv, m, n, a, b) * WMNIJ(m, n, i, j);
                    /* P(ij)P(ab) S_me ( t_im^ae W_mbej - t_i^e t_m^a <mb||ej> ) */
                    for (int m = 0; m < no; ++m)
                        for (int e = 0; e < nv; ++e) {
                            x += T2(i, m, a, e) * WMBEJ(m, b, e, j) - T1(i, e) * T1(m, a) * G(m, V(b), V(e), j);
                            x -= T2(j, m, a, e) * WMBEJ(m, b, e, i) - T1(j, e) * T1(m, a) * G(m, V(b), V(e), i);
                            x -= T2(i, m, b, e) * WMBEJ(m, a, e, j) - T1(i, e) * T1(m, b) * G(m, V(a), V(e), j);
                            x += T2(j, m, b, e) * WMBEJ(m, a, e, i) - T1(j, e) * T1(m, b) * G(m, V(a), V(e), i);
                        }
                    /* P(ij) S_e t_i^e <ab||ej> */
                    for (int e = 0; e < nv; ++e)
                        x += T1(i, e) * G(V(a), V(b), V(e), j) - T1(j, e) * G(V(a), V(b), V(e), i);
                    /* - P(ab) S_m t_m^a <mb||ij> */
                    for (int m = 0; m < no; ++m)
                        x -= T1(m, a) * G(m, V(b), i, j) - T1(m, b) * G(m, V(a), i, j);
                    R2(i, j, a, b) = x;
                }

    /* + 1/2 S_ef tau_ij^ef W_abef with
     * W_abef = <ab||ef> + S_m (t_m^b <ma||ef> - t_m^a <mb||ef>) + 1/4 S_mn tau_mn^ab <mn||ef>.
     * W_abef is formed per (a,b) for all (e,f) exactly as defined and used at once, so that the
     * v^4 tensor is never held in memory (same arithmetic as storing it). */
    int fail = 0;
#pragma omp parallel
    {
        cplx *Wab = malloc(sizeof(cplx) * (size_t)nv * nv);
        if (!Wab) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for collapse(2) schedule(static)
            for (int a = 0; a < nv; ++a)
                for (int b = 0; b < nv; ++b) {
                    for (int e = 0; e < nv; ++e)
                        for (int ff = 0; ff < nv; ++ff) {
                            cplx w = G(V(a), V(b), V(e), V(ff));
                            for (int m = 0; m < no; ++m)
                                w += T1(m, b) * G(m, V(a), V(e), V(ff)) - T1(m, a) * G(m, V(b), V(e), V(ff));
                            for (int m = 0; m < no; ++m)
                                for (int n = 0; n < no; ++n)
                                    w += 0.25 * tau_f(t1, t2, no, nv, m, n, a, b) * G(m, n, V(e), V(ff));
                            Wab[(size_t)e * nv + ff] = w;
                        }
                    for (int i = 0; i < no; ++i)
                        for (int j = 0; j < no; ++j) {
                            cplx x = 0.0;
                            for (int e = 0; e < nv; ++e)
                                for (int ff = 0; ff < nv; ++ff)
                                    x += 0.5 * tau_f(t1, t2, no, nv, i, j, e, ff) * Wab[(size_t)e * nv + ff];
                            R2(i, j, a, b) += x;
                        }
                }
        }
        free(Wab);
    }

    /* E = S_ia f_ia t_i^a + 1/4 S_ijab <ij||ab> t_ij^ab + 1/2 S_ijab <ij||ab> t_i^a t_j^b */
    cplx E = 0.0;
    for (int i = 0; i < no; ++i)
        for (int a = 0; a < nv; ++a) E += F(i, V(a)) * T1(i, a);
    for (int i = 0; i < no; ++i)
        for (int j = 0; j < no; ++j)
            for (int a = 0; a < nv; ++a)
                for (int b = 0; b < nv; ++b)
                    E += G(i, j, V(a), V(b)) * (0.25 * T2(i, j, a, b) + 0.5 * T1(i, a) * T1(j, b));
    *E_out = E;

    free(Fae); free(Fmi); free(Fme); free(Wmnij); free(Wmbej);
    return fail ? -1 : 0;
}
