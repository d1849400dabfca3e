/*
 * rtcc_sampled.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Sampled-element CPU oracle (tier B of SURVEY.md 8(c)) for the problem sizes where the full
 * 4-index tensor of rtcc_oracle.c does not fit (BASELINE.json configs 3-5).  It evaluates the SAME
 * spin-orbital working equations (Eqs. 7-8; Eq. 5)
 * for ONE output element R2[i,j,a,b] / R1[i,a] at a time.  Every integral is a direct sum over the
 * Cholesky vectors, (pq|rs) = sum_Q L^Q_pq L^Q_rs, <pq||rs> = (pr|qs) - (ps|qr) (PAPER.md:41,
 * :129-131); L^Q_pq = 0 unless spin(p) = spin(q) (O-1).  Amplitudes are read from the packed boundary
 * blocks through accessors that apply the antisymmetry and spin rules of O-1.  Naive loops; OpenMP
 * over an outer loop only.  What is kept between samples is only (a) the o^2 v^2 table
 * (me|nf) from which <mn||ef> = (me|nf) - (mf|ne) is read, and (b) index slices an element needs
 * (<ma||ef> for one a, <mn||ie> for one i, F_ae for one a, F_mi for one i, W_mbej for one (b,j)),
 * each exactly as O-2 defines it, cached because several samples share indices.
 *
 * Only tests/ and bench.py's cpu_baseline leg may call this.  It shares no code with the CUDA path.
 * Pinned by tests/test_oracle_pins.py::test_sampled_c_oracle_matches_full_oracle (every packed element
 * against the determinant-pinned tier-A oracle, complex amplitudes, general Fock matrix).
 *
 * Index conventions (as rtcc_oracle.c): spin-orbitals [alpha occ | beta occ | alpha virt | beta virt];
 * occupied i in [0,no), virtual a in [0,nv) (spin-orbital index no+a).
 */
#include <complex.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

typedef struct {
    int oa, ob, va, vb, K, n, no, nv, n1a, n1;
    double *LT[2];            /* per spin [n][n][K]: the K-vector of an orbital pair is contiguous */
    double *fock;             /* [2][n][n] */
    cplx *t1p, *t2p;          /* packed boundary amplitudes (copies) */
    long long off_bb, off_ab, n_t1, n_t2;
    double *ovov;             /* (me|nf), same-spin pairs (m,e),(n,f): [n1][n1] */
    cplx *Fme;                /* [no][nv] */
    cplx **Fae_row;           /* [nv] -> F_ae for all e */
    cplx **Fmi_col;           /* [no] -> F_mi for all m */
    double **Gmaef;           /* [nv] -> <ma||ef> [no][nv][nv] */
    double **Gmnie;           /* [no] -> <mn||ie> [no][no][nv] */
    cplx **Wmbej;             /* [nv*no] -> W_mbej [no][nv] for (b,j) */
    double **gmbej;           /* [nv*no] -> <mb||ej> [no][nv] */
} sctx;

static long long npair(long long n) { return n * (n - 1) / 2; }
static long long pairidx(long long x, long long y) { return y * (y - 1) / 2 + x; }   /* x < y */

/* ---- spin-orbital bookkeeping (O-1) */
static inline int occ_spin(const sctx *c, int i) { return i < c->oa ? 0 : 1; }
static inline int vir_spin(const sctx *c, int a) { return a < c->va ? 0 : 1; }
static inline int occ_orb(const sctx *c, int i) { return i < c->oa ? i : i - c->oa; }
static inline int vir_orb(const sctx *c, int a) { return a < c->va ? c->oa + a : c->ob + (a - c->va); }
/* general spin-orbital P in [0, no+nv) */
static inline int so_spin(const sctx *c, int P) { return P < c->no ? occ_spin(c, P) : vir_spin(c, P - c->no); }
static inline int so_orb(const sctx *c, int P) { return P < c->no ? occ_orb(c, P) : vir_orb(c, P - c->no); }
#define VV(a) (c->no + (a))

static inline double fso(const sctx *c, int P, int Q)
{
    int s = so_spin(c, P);
    if (s != so_spin(c, Q)) return 0.0;
    return c->fock[((size_t)s * c->n + so_orb(c, P)) * c->n + so_orb(c, Q)];
}

/* (PR|QS) = sum_Q L_PR L_QS */
static double coul(const sctx *c, int P, int R, int Q, int S)
{
    int s1 = so_spin(c, P), s2 = so_spin(c, Q);
    if (s1 != so_spin(c, R) || s2 != so_spin(c, S)) return 0.0;
    const double *x = c->LT[s1] + ((size_t)so_orb(c, P) * c->n + so_orb(c, R)) * c->K;
    const double *y = c->LT[s2] + ((size_t)so_orb(c, Q) * c->n + so_orb(c, S)) * c->K;
    double acc = 0.0;
#pragma omp simd reduction(+ : acc)
    for (int k = 0; k < c->K; ++k) acc += x[k] * y[k];
    return acc;
}
/* <PQ||RS> = (PR|QS) - (PS|QR) */
static double anti(const sctx *c, int P, int Q, int R, int S) { return coul(c, P, R, Q, S) - coul(c, P, S, Q, R); }

/* ---- amplitudes from the packed blocks (include/rtcc.h layout; antisymmetry and spin rules of O-1) */
static cplx T1(const sctx *c, int i, int a)
{
    int s = occ_spin(c, i);
    if (s != vir_spin(c, a)) return 0.0;
    if (s == 0) return c->t1p[(size_t)i * c->va + a];
    return c->t1p[(size_t)c->oa * c->va + (size_t)(i - c->oa) * c->vb + (a - c->va)];
}
static cplx T2(const sctx *c, int i, int j, int a, int b)
{
    if (i == j || a == b) return 0.0;
    int si = occ_spin(c, i), sj = occ_spin(c, j), sa = vir_spin(c, a), sb = vir_spin(c, b);
    double sign = 1.0;
    if (si == sj) {
        if (sa != si || sb != si) return 0.0;
        int ii = occ_orb(c, i), jj = occ_orb(c, j);
        int aa = si ? a - c->va : a, bb = si ? b - c->va : b;
        if (ii > jj) { int t = ii; ii = jj; jj = t; sign = -sign; }
        if (aa > bb) { int t = aa; aa = bb; bb = t; sign = -sign; }
        long long off = si ? c->off_bb : 0, pv = npair(si ? c->vb : c->va);
        return sign * c->t2p[off + pairidx(ii, jj) * pv + pairidx(aa, bb)];
    }
    if (sa == sb) return 0.0;
    if (si == 1) { int t = i; i = j; j = t; sign = -sign; }      /* now i alpha, j beta */
    if (sa == 1) { int t = a; a = b; b = t; sign = -sign; }      /* now a alpha, b beta */
    return sign * c->t2p[c->off_ab + (((size_t)i * c->ob + (j - c->oa)) * c->va + a) * c->vb + (b - c->va)];
}
static cplx tau(const sctx *c, int i, int j, int a, int b)
{ return T2(c, i, j, a, b) + T1(c, i, a) * T1(c, j, b) - T1(c, i, b) * T1(c, j, a); }
static cplx taut(const sctx *c, int i, int j, int a, int b)
{ return T2(c, i, j, a, b) + 0.5 * (T1(c, i, a) * T1(c, j, b) - T1(c, i, b) * T1(c, j, a)); }

/* ---- the o^2 v^2 block: index of the same-spin pair (m,e) in the (me|nf) table */
static inline long long ovpair(const sctx *c, int m, int e)
{
    if (occ_spin(c, m) == 0) return (long long)m * c->va + e;
    return c->n1a + (long long)(m - c->oa) * c->vb + (e - c->va);
}
/* out[f] = <mn||ef> = (me|nf) - (mf|ne) for all virtual f */
static void oovv_row(const sctx *c, int m, int n, int e, double *out)
{
    int sm = occ_spin(c, m), sn = occ_spin(c, n), se = vir_spin(c, e);
    for (int f = 0; f < c->nv; ++f) out[f] = 0.0;
    if (sm == se) {                    /* (me|nf): f has the spin of n */
        int f0 = sn ? c->va : 0, nf = sn ? c->vb : c->va;
        const double *row = c->ovov + (size_t)ovpair(c, m, e) * c->n1 + ovpair(c, n, f0);
        for (int x = 0; x < nf; ++x) out[f0 + x] += row[x];
    }
    if (sn == se) {                    /* (mf|ne) = (ne|mf): f has the spin of m */
        int f0 = sm ? c->va : 0, nf = sm ? c->vb : c->va;
        const double *row = c->ovov + (size_t)ovpair(c, n, e) * c->n1 + ovpair(c, m, f0);
        for (int x = 0; x < nf; ++x) out[f0 + x] -= row[x];
    }
}

int sorc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void sorc_destroy(sctx *c)
{
    if (!c) return;
    for (int s = 0; s < 2; ++s) free(c->LT[s]);
    free(c->fock); free(c->t1p); free(c->t2p); free(c->ovov); free(c->Fme);
    if (c->Fae_row) for (int a = 0; a < c->nv; ++a) free(c->Fae_row[a]);
    if (c->Gmaef) for (int a = 0; a < c->nv; ++a) free(c->Gmaef[a]);
    if (c->Fmi_col) for (int i = 0; i < c->no; ++i) free(c->Fmi_col[i]);
    if (c->Gmnie) for (int i = 0; i < c->no; ++i) free(c->Gmnie[i]);
    if (c->Wmbej) for (long long x = 0; x < (long long)c->nv * c->no; ++x) { free(c->Wmbej[x]); free(c->gmbej[x]); }
    free(c->Fae_row); free(c->Gmaef); free(c->Fmi_col); free(c->Gmnie); free(c->Wmbej); free(c->gmbej);
    free(c);
}

/* frees the per-index slices (the big ones are <ma||ef>: no*nv*nv doubles each) */
void sorc_drop_slices(sctx *c)
{
    for (int a = 0; a < c->nv; ++a) { free(c->Gmaef[a]); c->Gmaef[a] = NULL; }
}

/* L [2][K][n][n], fock [2][n][n], t1p/t2p packed complex (interleaved).  Returns NULL when out of memory. */
sctx *sorc_create(int oa, int ob, int va, int vb, int K, const double *L, const double *fock, const double *t1p, const double *t2p)
{
    sctx *c = (sctx *)calloc(1, sizeof(sctx));
    if (!c) return NULL;
    c->oa = oa; c->ob = ob; c->va = va; c->vb = vb; c->K = K;
    c->n = oa + va; c->no = oa + ob; c->nv = va + vb;
    c->n1a = oa * va; c->n1 = oa * va + ob * vb;
    c->off_bb = npair(oa) * npair(va);
    c->off_ab = c->off_bb + npair(ob) * npair(vb);
    c->n_t1 = c->n1;
    c->n_t2 = c->off_ab + (long long)oa * ob * va * vb;
    const int n = c->n, no = c->no, nv = c->nv;
    const size_t nn = (size_t)n * n;
    int ok = 1;
    for (int s = 0; s < 2; ++s) ok &= (c->LT[s] = (double *)malloc(sizeof(double) * nn * K)) != NULL;
    ok &= (c->fock = (double *)malloc(sizeof(double) * 2 * nn)) != NULL;
    ok &= (c->t1p = (cplx *)malloc(sizeof(cplx) * (size_t)(c->n_t1 > 0 ? c->n_t1 : 1))) != NULL;
    ok &= (c->t2p = (cplx *)malloc(sizeof(cplx) * (size_t)(c->n_t2 > 0 ? c->n_t2 : 1))) != NULL;
    ok &= (c->ovov = (double *)malloc(sizeof(double) * (size_t)(c->n1 > 0 ? c->n1 : 1) * (size_t)(c->n1 > 0 ? c->n1 : 1))) != NULL;
    ok &= (c->Fme = (cplx *)malloc(sizeof(cplx) * (size_t)(no > 0 ? no : 1) * nv)) != NULL;
    ok &= (c->Fae_row = (cplx **)calloc((size_t)nv, sizeof(cplx *))) != NULL;
    ok &= (c->Gmaef = (double **)calloc((size_t)nv, sizeof(double *))) != NULL;
    ok &= (c->Fmi_col = (cplx **)calloc((size_t)(no > 0 ? no : 1), sizeof(cplx *))) != NULL;
    ok &= (c->Gmnie = (double **)calloc((size_t)(no > 0 ? no : 1), sizeof(double *))) != NULL;
    ok &= (c->Wmbej = (cplx **)calloc((size_t)nv * (no > 0 ? no : 1), sizeof(cplx *))) != NULL;
    ok &= (c->gmbej = (double **)calloc((size_t)nv * (no > 0 ? no : 1), sizeof(double *))) != NULL;
    if (!ok) { sorc_destroy(c); return NULL; }
    memcpy(c->fock, fock, sizeof(double) * 2 * nn);
    memcpy(c->t1p, t1p, sizeof(cplx) * (size_t)c->n_t1);
    memcpy(c->t2p, t2p, sizeof(cplx) * (size_t)c->n_t2);
    for (int s = 0; s < 2; ++s) {
#pragma omp parallel for schedule(static)
        for (long long pq = 0; pq < (long long)nn; ++pq)
            for (int Q = 0; Q < K; ++Q) c->LT[s][(size_t)pq * K + Q] = L[((size_t)s * K + Q) * nn + pq];
    }
    /* (me|nf) for same-spin pairs; symmetric, so the lower triangle is mirrored.  Every element is the plain sum over Q of
     * L_me L_nf; four rows X are taken against one row Y at a time only so that the K-vector of Y is read once for the four
     * (the table is 1.4e9 dot products of length 2200 at config 5). */
    {
        const long long n1 = c->n1;
        double *ov = (double *)malloc(sizeof(double) * (size_t)(n1 > 0 ? n1 : 1) * K);          /* L_me by pair index, K contiguous */
        if (!ov) { sorc_destroy(c); return NULL; }
#pragma omp parallel for schedule(static)
        for (long long X = 0; X < n1; ++X) {
            int m, e, sp;
            if (X < c->n1a) { sp = 0; m = (int)(X / va); e = oa + (int)(X % va); }
            else { long long y = X - c->n1a; sp = 1; m = (int)(y / vb); e = ob + (int)(y % vb); }
            memcpy(ov + (size_t)X * K, c->LT[sp] + ((size_t)m * n + e) * K, sizeof(double) * K);
        }
#pragma omp parallel for schedule(dynamic, 4)
        for (long long X0 = 0; X0 < n1; X0 += 4) {
            const int nx = (int)(n1 - X0 < 4 ? n1 - X0 : 4);
            for (long long Y = X0; Y < n1; ++Y) {
                const double *y = ov + (size_t)Y * K;
                double acc[4] = {0.0, 0.0, 0.0, 0.0};
                for (int r = 0; r < nx; ++r) {
                    const double *x = ov + (size_t)(X0 + r) * K;
                    double a = 0.0;
#pragma omp simd reduction(+ : a)
                    for (int k = 0; k < K; ++k) a += x[k] * y[k];
                    acc[r] = a;
                }
                for (int r = 0; r < nx; ++r) c->ovov[(size_t)(X0 + r) * n1 + Y] = acc[r];
            }
        }
        free(ov);
#pragma omp parallel for schedule(static)
        for (long long X = 0; X < n1; ++X)
            for (long long Y = 0; Y < X; ++Y) c->ovov[(size_t)X * n1 + Y] = c->ovov[(size_t)Y * n1 + X];
    }
    /* F_me = f_me + sum_nf t_n^f <mn||ef> */
#pragma omp parallel
    {
        double *row = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
        for (long long me = 0; me < (long long)no * nv; ++me) {
            int m = (int)(me / nv), e = (int)(me % nv);
            cplx acc = fso(c, m, VV(e));
            for (int nn_ = 0; nn_ < no; ++nn_) {
                oovv_row(c, m, nn_, e, row);
                for (int f = 0; f < nv; ++f) acc += T1(c, nn_, f) * row[f];
            }
            c->Fme[me] = acc;
        }
        free(row);
    }
    return c;
}

/* <ma||ef> for all m, e, f  (a fixed):  [no][nv][nv] */
static const double *get_Gmaef(sctx *c, int a)
{
    if (c->Gmaef[a]) return c->Gmaef[a];
    const int no = c->no, nv = c->nv;
    double *G = (double *)malloc(sizeof(double) * (size_t)no * nv * nv);
    if (!G) return NULL;
#pragma omp parallel for schedule(static)
    for (long long me = 0; me < (long long)no * nv; ++me) {
        int m = (int)(me / nv), e = (int)(me % nv);
        for (int f = 0; f < nv; ++f) G[(size_t)me * nv + f] = anti(c, m, VV(a), VV(e), VV(f));
    }
    return c->Gmaef[a] = G;
}
/* <mn||ie> for all m, n, e  (i fixed):  [no][no][nv] */
static const double *get_Gmnie(sctx *c, int i)
{
    if (c->Gmnie[i]) return c->Gmnie[i];
    const int no = c->no, nv = c->nv;
    double *G = (double *)malloc(sizeof(double) * (size_t)no * no * nv);
    if (!G) return NULL;
#pragma omp parallel for schedule(static)
    for (long long mn = 0; mn < (long long)no * no; ++mn) {
        int m = (int)(mn / no), n = (int)(mn % no);
        for (int e = 0; e < nv; ++e) G[(size_t)mn * nv + e] = anti(c, m, n, i, VV(e));
    }
    return c->Gmnie[i] = G;
}

/* F_ae = f_ae - 1/2 sum_m f_me t_m^a + sum_mf t_m^f <ma||fe> - 1/2 sum_mnf tau~_mn^af <mn||ef>   (all e, a fixed) */
static const cplx *get_Fae_row(sctx *c, int a)
{
    if (c->Fae_row[a]) return c->Fae_row[a];
    const int no = c->no, nv = c->nv;
    const double *G = get_Gmaef(c, a);
    cplx *F = (cplx *)malloc(sizeof(cplx) * nv);
    cplx *tt = (cplx *)malloc(sizeof(cplx) * (size_t)(no > 0 ? no : 1) * no * nv);      /* tau~_mn^af, [m][n][f] */
    if (!G || !F || !tt) { free(F); free(tt); return NULL; }
    for (int m = 0; m < no; ++m)
        for (int n = 0; n < no; ++n)
            for (int f = 0; f < nv; ++f) tt[((size_t)m * no + n) * nv + f] = taut(c, m, n, a, f);
#pragma omp parallel
    {
        double *row = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
        for (int e = 0; e < nv; ++e) {
            cplx acc = fso(c, VV(a), VV(e));
            for (int m = 0; m < no; ++m) acc -= 0.5 * fso(c, m, VV(e)) * T1(c, m, a);
            for (int m = 0; m < no; ++m)
                for (int f = 0; f < nv; ++f) acc += T1(c, m, f) * G[((size_t)m * nv + f) * nv + e];     /* <ma||fe> */
            for (int m = 0; m < no; ++m)
                for (int n = 0; n < no; ++n) {
                    oovv_row(c, m, n, e, row);
                    const cplx *t = tt + ((size_t)m * no + n) * nv;
                    cplx s = 0.0;
                    for (int f = 0; f < nv; ++f) s += t[f] * row[f];
                    acc -= 0.5 * s;
                }
            F[e] = acc;
        }
        free(row);
    }
    free(tt);
    return c->Fae_row[a] = F;
}

/* F_mi = f_mi + 1/2 sum_e t_i^e f_me + sum_ne t_n^e <mn||ie> + 1/2 sum_nef tau~_in^ef <mn||ef>   (all m, i fixed) */
static const cplx *get_Fmi_col(sctx *c, int i)
{
    if (c->Fmi_col[i]) return c->Fmi_col[i];
    const int no = c->no, nv = c->nv;
    const double *G = get_Gmnie(c, i);
    cplx *F = (cplx *)malloc(sizeof(cplx) * (no > 0 ? no : 1));
    cplx *tt = (cplx *)malloc(sizeof(cplx) * (size_t)(no > 0 ? no : 1) * nv * nv);      /* tau~_in^ef, [n][e][f] */
    if (!G || !F || !tt) { free(F); free(tt); return NULL; }
#pragma omp parallel for schedule(static)
    for (long long ne = 0; ne < (long long)no * nv; ++ne)
        for (int f = 0; f < nv; ++f) tt[(size_t)ne * nv + f] = taut(c, i, (int)(ne / nv), (int)(ne % nv), f);
#pragma omp parallel
    {
        double *row = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
        for (int m = 0; m < no; ++m) {
            cplx acc = fso(c, m, i);
            for (int e = 0; e < nv; ++e) acc += 0.5 * T1(c, i, e) * fso(c, m, VV(e));
            for (int n = 0; n < no; ++n)
                for (int e = 0; e < nv; ++e) acc += T1(c, n, e) * G[((size_t)m * no + n) * nv + e];
            for (int n = 0; n < no; ++n)
                for (int e = 0; e < nv; ++e) {
                    oovv_row(c, m, n, e, row);
                    const cplx *t = tt + ((size_t)n * nv + e) * nv;
                    cplx s = 0.0;
                    for (int f = 0; f < nv; ++f) s += t[f] * row[f];
                    acc += 0.5 * s;
                }
            F[m] = acc;
        }
        free(row);
    }
    free(tt);
    return c->Fmi_col[i] = F;
}

/* W_mbej = <mb||ej> + sum_f t_j^f <mb||ef> - sum_n t_n^b <mn||ej> - sum_nf (1/2 t_jn^fb + t_j^f t_n^b) <mn||ef>
 * for all m, e  ((b,j) fixed); also keeps the bare <mb||ej>. */
static int get_Wmbej(sctx *c, int b, int j, const cplx **Wout, const double **gout)
{
    const int no = c->no, nv = c->nv;
    const size_t key = (size_t)b * no + j;
    if (!c->Wmbej[key]) {
        const double *Gb = get_Gmaef(c, b);          /* <mb||ef> */
        const double *Gj = get_Gmnie(c, j);          /* <mn||je> = -<mn||ej> */
        cplx *W = (cplx *)malloc(sizeof(cplx) * (size_t)no * nv);
        double *g = (double *)malloc(sizeof(double) * (size_t)no * nv);
        cplx *ss = (cplx *)malloc(sizeof(cplx) * (size_t)no * nv);                      /* 1/2 t_jn^fb + t_j^f t_n^b, [n][f] */
        if (!Gb || !Gj || !W || !g || !ss) { free(W); free(g); free(ss); return -1; }
        for (int n = 0; n < no; ++n)
            for (int f = 0; f < nv; ++f) ss[(size_t)n * nv + f] = 0.5 * T2(c, j, n, f, b) + T1(c, j, f) * T1(c, n, b);
#pragma omp parallel
        {
            double *row = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
            for (long long me = 0; me < (long long)no * nv; ++me) {
                int m = (int)(me / nv), e = (int)(me % nv);
                double g0 = anti(c, m, VV(b), VV(e), j);
                cplx acc = g0;
                for (int f = 0; f < nv; ++f) acc += T1(c, j, f) * Gb[((size_t)m * nv + e) * nv + f];
                for (int n = 0; n < no; ++n) acc -= T1(c, n, b) * (-Gj[((size_t)m * no + n) * nv + e]);
                for (int n = 0; n < no; ++n) {
                    oovv_row(c, m, n, e, row);
                    const cplx *t = ss + (size_t)n * nv;
                    cplx s = 0.0;
                    for (int f = 0; f < nv; ++f) s += t[f] * row[f];
                    acc -= s;
                }
                W[me] = acc; g[me] = g0;
            }
            free(row);
        }
        free(ss);
        c->Wmbej[key] = W; c->gmbej[key] = g;
    }
    *Wout = c->Wmbej[key]; *gout = c->gmbej[key];
    return 0;
}

/* R2_ij^ab (spin-orbital indices, a and b counted from the first virtual); out = (re, im).  Returns 0 or -1 (memory). */
int sorc_r2(sctx *c, int i, int j, int a, int b, double *out)
{
    const int no = c->no, nv = c->nv;
    cplx x = anti(c, i, j, VV(a), VV(b));
    const cplx *Fae_a = get_Fae_row(c, a), *Fae_b = get_Fae_row(c, b);
    const cplx *Fmi_i = get_Fmi_col(c, i), *Fmi_j = get_Fmi_col(c, j);
    if (!Fae_a || !Fae_b || !Fmi_i || !Fmi_j) return -1;
    /* P(ab) sum_e t_ij^ae (F_be - 1/2 sum_m t_m^b F_me) */
    for (int e = 0; e < nv; ++e) {
        cplx Fb = Fae_b[e], Fa = Fae_a[e];
        for (int m = 0; m < no; ++m) {
            Fb -= 0.5 * T1(c, m, b) * c->Fme[(size_t)m * nv + e];
            Fa -= 0.5 * T1(c, m, a) * c->Fme[(size_t)m * nv + e];
        }
        x += T2(c, i, j, a, e) * Fb - T2(c, i, j, b, e) * Fa;
    }
    /* - P(ij) sum_m t_im^ab (F_mj + 1/2 sum_e t_j^e F_me) */
    for (int m = 0; m < no; ++m) {
        cplx Fj = Fmi_j[m], Fi = Fmi_i[m];
        for (int e = 0; e < nv; ++e) {
            Fj += 0.5 * T1(c, j, e) * c->Fme[(size_t)m * nv + e];
            Fi += 0.5 * T1(c, i, e) * c->Fme[(size_t)m * nv + e];
        }
        x -= T2(c, i, m, a, b) * Fj - T2(c, j, m, a, b) * Fi;
    }
    cplx *tij = (cplx *)malloc(sizeof(cplx) * (size_t)nv * nv);       /* tau_ij^ef */
    cplx *tab = (cplx *)malloc(sizeof(cplx) * (size_t)(no > 0 ? no : 1) * no);   /* tau_mn^ab */
    cplx *Wef = (cplx *)malloc(sizeof(cplx) * (size_t)nv * nv);
    if (!tij || !tab || !Wef) { free(tij); free(tab); free(Wef); return -1; }
    for (int e = 0; e < nv; ++e) for (int f = 0; f < nv; ++f) tij[(size_t)e * nv + f] = tau(c, i, j, e, f);
    for (int m = 0; m < no; ++m) for (int n = 0; n < no; ++n) tab[(size_t)m * no + n] = tau(c, m, n, a, b);
    /* 1/2 sum_mn tau_mn^ab W_mnij,  W_mnij = <mn||ij> + sum_e (t_j^e <mn||ie> - t_i^e <mn||je>) + 1/4 sum_ef tau_ij^ef <mn||ef> */
    {
        const double *Gi = get_Gmnie(c, i), *Gj = get_Gmnie(c, j);
        if (!Gi || !Gj) { free(tij); free(tab); free(Wef); return -1; }
        double sr = 0.0, si = 0.0;
#pragma omp parallel reduction(+ : sr, si)
        {
            double *row = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
            for (long long mn = 0; mn < (long long)no * no; ++mn) {
                int m = (int)(mn / no), n = (int)(mn % no);
                cplx W = anti(c, m, n, i, j);
                for (int e = 0; e < nv; ++e) W += T1(c, j, e) * Gi[(size_t)mn * nv + e] - T1(c, i, e) * Gj[(size_t)mn * nv + e];
                cplx q = 0.0;
                for (int e = 0; e < nv; ++e) {
                    oovv_row(c, m, n, e, row);
                    const cplx *t = tij + (size_t)e * nv;
                    for (int f = 0; f < nv; ++f) q += t[f] * row[f];
                }
                W += 0.25 * q;
                cplx term = 0.5 * tab[mn] * W;
                sr += creal(term); si += cimag(term);
            }
            free(row);
        }
        x += sr + si * I;
    }
    /* 1/2 sum_ef tau_ij^ef W_abef,  W_abef = <ab||ef> + sum_m (t_m^b <ma||ef> - t_m^a <mb||ef>) + 1/4 sum_mn tau_mn^ab <mn||ef> */
    {
        const double *Ga = get_Gmaef(c, a), *Gb = get_Gmaef(c, b);
        if (!Ga || !Gb) { free(tij); free(tab); free(Wef); return -1; }
#pragma omp parallel
        {
            double *row = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
            for (int e = 0; e < nv; ++e) {
                cplx *W = Wef + (size_t)e * nv;
                for (int f = 0; f < nv; ++f) W[f] = anti(c, VV(a), VV(b), VV(e), VV(f));
                for (int m = 0; m < no; ++m) {
                    const cplx tb = T1(c, m, b), ta = T1(c, m, a);
                    const double *ga = Ga + ((size_t)m * nv + e) * nv, *gb = Gb + ((size_t)m * nv + e) * nv;
                    for (int f = 0; f < nv; ++f) W[f] += tb * ga[f] - ta * gb[f];
                }
                for (int m = 0; m < no; ++m)
                    for (int n = 0; n < no; ++n) {
                        oovv_row(c, m, n, e, row);
                        const cplx t = 0.25 * tab[(size_t)m * no + n];
                        for (int f = 0; f < nv; ++f) W[f] += t * row[f];
                    }
            }
            free(row);
        }
        cplx s = 0.0;
        for (size_t ef = 0; ef < (size_t)nv * nv; ++ef) s += tij[ef] * Wef[ef];
        x += 0.5 * s;
    }
    free(tij); free(tab); free(Wef);
    /* P(ij)P(ab) sum_me ( t_im^ae W_mbej - t_i^e t_m^a <mb||ej> ) */
    {
        const int perm[4][4] = {{i, j, a, b}, {j, i, a, b}, {i, j, b, a}, {j, i, b, a}};
        const double sg[4] = {1.0, -1.0, -1.0, 1.0};
        for (int k = 0; k < 4; ++k) {
            const int ii = perm[k][0], jj = perm[k][1], aa = perm[k][2], bb = perm[k][3];
            const cplx *W; const double *g;
            if (get_Wmbej(c, bb, jj, &W, &g)) return -1;
            cplx s = 0.0;
            for (int m = 0; m < no; ++m)
                for (int e = 0; e < nv; ++e)
                    s += T2(c, ii, m, aa, e) * W[(size_t)m * nv + e] - T1(c, ii, e) * T1(c, m, aa) * g[(size_t)m * nv + e];
            x += sg[k] * s;
        }
    }
    /* P(ij) sum_e t_i^e <ab||ej> - P(ab) sum_m t_m^a <mb||ij> */
    for (int e = 0; e < nv; ++e)
        x += T1(c, i, e) * anti(c, VV(a), VV(b), VV(e), j) - T1(c, j, e) * anti(c, VV(a), VV(b), VV(e), i);
    for (int m = 0; m < no; ++m)
        x -= T1(c, m, a) * anti(c, m, VV(b), i, j) - T1(c, m, b) * anti(c, m, VV(a), i, j);
    out[0] = creal(x); out[1] = cimag(x);
    return 0;
}

/* R1_i^a = f_ia + sum_e t_i^e F_ae - sum_m t_m^a F_mi + sum_me t_im^ae F_me - sum_nf t_n^f <na||if>
 *          - 1/2 sum_mef t_im^ef <ma||ef> - 1/2 sum_men t_mn^ae <nm||ei> */
int sorc_r1(sctx *c, int i, int a, double *out)
{
    const int no = c->no, nv = c->nv;
    const cplx *Fae = get_Fae_row(c, a), *Fmi = get_Fmi_col(c, i);
    const double *Ga = get_Gmaef(c, a), *Gi = get_Gmnie(c, i);
    if (!Fae || !Fmi || !Ga || !Gi) return -1;
    cplx x = fso(c, i, VV(a));
    for (int e = 0; e < nv; ++e) x += T1(c, i, e) * Fae[e];
    for (int m = 0; m < no; ++m) x -= T1(c, m, a) * Fmi[m];
    for (int m = 0; m < no; ++m)
        for (int e = 0; e < nv; ++e) x += T2(c, i, m, a, e) * c->Fme[(size_t)m * nv + e];
    for (int n = 0; n < no; ++n)
        for (int f = 0; f < nv; ++f) x -= T1(c, n, f) * anti(c, n, VV(a), i, VV(f));
    for (int m = 0; m < no; ++m)
        for (int e = 0; e < nv; ++e)
            for (int f = 0; f < nv; ++f) x -= 0.5 * T2(c, i, m, e, f) * Ga[((size_t)m * nv + e) * nv + f];
    for (int m = 0; m < no; ++m)
        for (int e = 0; e < nv; ++e)
            for (int n = 0; n < no; ++n) x -= 0.5 * T2(c, m, n, a, e) * (-Gi[((size_t)n * no + m) * nv + e]);   /* <nm||ei> = -<nm||ie> */
    out[0] = creal(x); out[1] = cimag(x);
    return 0;
}

/* E = sum_ia f_ia t_i^a + 1/4 sum <ij||ab> t_ij^ab + 1/2 sum <ij||ab> t_i^a t_j^b */
void sorc_energy(sctx *c, double *out)
{
    const int no = c->no, nv = c->nv;
    double sr = 0.0, si = 0.0;
#pragma omp parallel reduction(+ : sr, si)
    {
        double *row = (double *)malloc(sizeof(double) * nv);
#pragma omp for schedule(static)
        for (int i = 0; i < no; ++i) {
            cplx acc = 0.0;
            for (int a = 0; a < nv; ++a) acc += fso(c, i, VV(a)) * T1(c, i, a);
            for (int j = 0; j < no; ++j)
                for (int a = 0; a < nv; ++a) {
                    oovv_row(c, i, j, a, row);
                    for (int b = 0; b < nv; ++b)
                        acc += row[b] * (0.25 * T2(c, i, j, a, b) + 0.5 * T1(c, i, a) * T1(c, j, b));
                }
            sr += creal(acc); si += cimag(acc);
        }
        free(row);
    }
    out[0] = sr; out[1] = si;
}
