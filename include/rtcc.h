/*
 * rtcc.h -- C ABI of librtcc: the per-time-step hot path of the RT-EOM-CCSD cumulant Green's function
 * method (arXiv:2301.04249; /root/reference/PAPER.md) on one NVIDIA B200 (sm_100a).
 *
 * What the library computes (spin-explicit alpha-alpha / beta-beta / alpha-beta blocks, fp64, complex128
 * amplitudes, real Cholesky vectors L^Q_pq with (pq|rs) = sum_Q L^Q_pq L^Q_rs):
 *   R1_i^a   = <Phi_i^a  |(H_N e^{T1+T2})_C|Phi>     PAPER.md:76  Eq. 7
 *   R2_ij^ab = <Phi_ij^ab|(H_N e^{T1+T2})_C|Phi>     PAPER.md:79  Eq. 8
 *   E        = <Phi|(H_N e^{T})_C|Phi>               PAPER.md:58  Eq. 5 (integrand), :63 Eq. 6
 *   i dt/dtau = -R  i.e. dt/dtau = +i R              PAPER.md:46  Eq. 2
 *   t(tau+dt) = t(tau) + (i dt/2) [R(t(tau)) + R(t(tau+dt))]   PAPER.md:93 Eq. 9, fixed-point solved (:103)
 *   C(tau)   = i int_0^tau E dtau'  by the trapezoid rule       PAPER.md:58 Eq. 5, :89
 * with T1 = T2 = 0 and C = 0 at tau = 0.
 *
 * Conventions common to all calls
 *   - Return value: 0 (RTCC_OK) or a negative error code; no exceptions, no aborts, nothing is printed.
 *   - Array arguments are DEVICE pointers on the current CUDA device unless the context was created
 *     with RTCC_HOST_PTRS, in which case every array argument of every call is a HOST pointer and the
 *     library performs the copies (on its stream, synchronously).
 *   - Complex arrays are interleaved (re, im) doubles.
 *   - Packed amplitude layout (t1, r1: n_t1 complex; t2, r2: n_t2 complex):
 *       t1 = [ alpha (i,a) at i*v_alpha + a | beta (I,A) at I*v_beta + A ]
 *       t2 = [ alpha-alpha packed | beta-beta packed | alpha-beta full ]
 *       same-spin element (i<j, a<b) at pair(i,j)*P(v) + pair(a,b), pair(x,y) = y(y-1)/2 + x, P(n)=n(n-1)/2;
 *       alpha-beta element (i,J,a,B) at ((i*o_beta + J)*v_alpha + a)*v_beta + B.
 *   - The caller owns every buffer it passes; the context owns all internal state.
 *   - A context is not thread-safe; all work is issued on the stream given at creation.
 */
#ifndef RTCC_H
#define RTCC_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rtcc_ctx rtcc_ctx;

enum {
    RTCC_OK = 0,
    RTCC_EINVAL = -1,     /* null pointer, non-positive size, o_a+v_a != o_b+v_b, dt not finite, ... */
    RTCC_ENOMEM = -2,     /* device or host allocation failed */
    RTCC_ECUDA = -3,      /* a CUDA call failed; rtcc_last_cuda_error() has the cudaError_t value */
    RTCC_ENOCONV = -4,    /* micro-iterations reached max_micro; propagation state NOT advanced */
    RTCC_ENONFINITE = -5, /* NaN/Inf met in the amplitude update; propagation state NOT advanced */
    RTCC_EIO = -6         /* checkpoint file could not be opened / read / written, or is not a checkpoint */
};

enum { RTCC_HOST_PTRS = 1u };

/* Create a context for one (N-1)-electron problem.
 *   o_alpha, o_beta >= 0, v_alpha, v_beta >= 1, o_alpha+v_alpha == o_beta+v_beta =: n, n_chol >= 1.
 *   L    [2][n_chol][n][n] real, alpha then beta, each spin in its own [occupied | virtual] orbital order,
 *        symmetric in (p,q).
 *   fock [2][n][n] real symmetric Fock matrix of the (N-1)-electron reference (need not be diagonal).
 *   Both are copied.  cuda_stream: a cudaStream_t (NULL = default stream).
 * State after creation: T1 = T2 = 0, C = 0, tau = 0; R(T=0) and E(T=0) are evaluated by the first call that needs them
 * (rtcc_step, rtcc_cumulant, rtcc_save). */
int rtcc_create(rtcc_ctx** out, int o_alpha, int o_beta, int v_alpha, int v_beta, int n_chol,
                const double* L, const double* fock, unsigned flags, void* cuda_stream);
void rtcc_destroy(rtcc_ctx* ctx);

/* Process-wide tuning defaults read by rtcc_create (contexts already created are not affected; not thread-safe).  They
 * select between code paths that compute the same result (the tests use them to force each path):
 *   "fused" (1)             fused T1-dressing kernel when an n x n Cholesky slice fits in shared memory (0: GEMM path)
 *   "fused_fock" (1)        fused dressed-Fock / F / singles kernels for small n (0: GEMM path)
 *   "graph" (1)             replay one CUDA graph per residual evaluation (0: plain launches)
 *   "stream_priorities" (1) latency-bound branches of the graph outrank the ladder branch
 *   "gemm_tile" (0)         0: automatic, 64 or 128: force the contraction tile
 *   "ladder_split" (0)      0: automatic, k >= 1: force k slices of the (e,f) plane per ladder work item
 *   "max_cluster" (16)      largest thread-block cluster the wide ladder kernel may use (1..16)
 *   "ladder_cluster" (0)    0: automatic, k >= 1: force clusters of k CTAs in the wide ladder kernel
 *   "ladder_tiles" (5)      column tiles one CTA of the wide ladder kernel may hold (1..5; 4 of them parked in tensor memory)
 *   "ladder_antisym" (1)    wide ladder kernel, same-spin cases: visit only (e,f) chunks that hold an e < f, two W products per
 *                           chunk combined to (pe|qf) - (pf|qe), one application (0: every (e,f) chunk, one product each)
 *   "ladder_overlap" (1)    wide ladder launches of different cluster sizes: 0 one after the other on one stream; 1 side by side,
 *                           the launch with the longest CTAs first and the others on a helper stream, so that their CTAs fill
 *                           its last, partly empty wave; 2 side by side, shortest first (for comparison)
 *   "lean" (-1)             -1: low-memory layout only when the standard one does not fit, 0: never, 1: always
 *   "ring_3m" (-1)          complex x complex ring products T.W by three real multiplications instead of four (same result up to
 *                           rounding): -1 automatic (pair space >= 1536 and the two extra matrices fit), 0 never, 1 always
 *   "lean_slab" (0)         0: automatic, k >= 1: at most k occupied indices per column slab of the low-memory ring
 *   "reset"                 back to the defaults (value ignored)
 * Returns RTCC_EINVAL for an unknown name or a value out of range. */
int rtcc_set_default_option(const char* name, int value);

/* n_t1, n_t2: complex element counts of the packed arrays; workspace_bytes: device memory held. */
int rtcc_sizes(const rtcc_ctx* ctx, long long* n_t1, long long* n_t2, long long* workspace_bytes);

/* Size accounting without a context (Table 2; needs no GPU):
 *   out[0] n_t1, out[1] n_t2   complex elements of the packed boundary arrays
 *   out[2]  complex elements of ONE T2 in the paper's storage -- the three unpacked spin blocks
 *           o_a^2 v_a^2 + o_b^2 v_b^2 + o_a o_b v_a v_b (x 16 bytes reproduces the "T2" column of Table 2)
 *   out[3]  doubles of the Cholesky vectors L[2][n_chol][n][n]
 *   out[4]  bytes of device memory a context holds with every intermediate resident (the standard layout)
 *   out[5]  bytes with the low-memory layout (packed alpha-beta amplitudes read in place, ring intermediates in column slabs,
 *           one arena shared by the ring and ladder phases); rtcc_create picks it when out[4] exceeds the free memory. */
int rtcc_problem_sizes(int o_alpha, int o_beta, int v_alpha, int v_beta, int n_chol, long long out[6]);

/* Pure evaluation of Eqs. 7-8 at the given amplitudes; does not touch the propagation state.
 * r1/r2 receive R1/R2 in the packed layout. */
int rtcc_residual(rtcc_ctx* ctx, const double* t1, const double* t2, double* r1, double* r2);
/* Value of E = <Phi|(H_N e^T)_C|Phi> (Re, Im) computed by the most recent rtcc_residual call. */
int rtcc_residual_energy(const rtcc_ctx* ctx, double out[2]);

/* Restart support: set amplitudes, time and cumulant, re-evaluate R and E there. c is a HOST pointer. */
int rtcc_set_amplitudes(rtcc_ctx* ctx, const double* t1, const double* t2, double time, const double c[2]);
int rtcc_get_amplitudes(const rtcc_ctx* ctx, double* t1, double* t2);

/* Checkpoint / restart ("amplitudes of steps i-1 and i, Fock matrix, Cholesky vectors"): Eq. 9 is a one-step
 * method, so the propagation state is T(tau), R(T(tau)), tau, C(tau), E(tau) and the solver settings; the Fock matrix and the
 * Cholesky vectors are the caller's inputs to rtcc_create and are not duplicated.  rtcc_save writes them to `path` (host file
 * system; little-endian: a 104-byte header -- magic "RTCCCKP1", o_alpha, o_beta, v_alpha, v_beta, n_chol, solver mode,
 * max_micro, fixed_micro as int32, n_t1, n_t2 as int64, tol, tau, Re C, Im C, Re E, Im E as float64 -- then t1|t2 and r1|r2 as
 * packed interleaved complex128).  rtcc_load restores them into a context created for the same problem (RTCC_EINVAL if the
 * sizes differ, RTCC_EIO for a short or foreign file; the state is untouched on error).  A loaded run continues bit-identically. */
int rtcc_save(const rtcc_ctx* ctx, const char* path);
int rtcc_load(rtcc_ctx* ctx, const char* path);

/* The same state through memory instead of a file (pointer kind as chosen at rtcc_create; scal is a HOST array:
 * tau, Re C, Im C, Re E, Im E).  rtcc_get_state copies T(tau) -> t1|t2 and R(T(tau)) -> r1|r2 (packed layout);
 * rtcc_set_state installs them WITHOUT evaluating the residual -- the caller vouches that r1|r2 is R at t1|t2 (as returned
 * by rtcc_get_state or rtcc_residual); a run continued from a state taken with rtcc_get_state is bit-identical.  Solver
 * settings are not part of this call (rtcc_set_solver).  RTCC_EINVAL for a NULL pointer or a non-finite scalar. */
int rtcc_get_state(const rtcc_ctx* ctx, double* t1, double* t2, double* r1, double* r2, double scal[5]);
int rtcc_set_state(rtcc_ctx* ctx, const double* t1, const double* t2, const double* r1, const double* r2, const double scal[5]);

/* Solver of the implicit Eq. 9.  mode 0: plain fixed point t(k+1) = B + (i dt/2) R(t(k));
 * mode 1: orbital-energy-denominator preconditioned iteration with the same fixed point.
 * Converged when max |t(k+1)-t(k)| over all packed elements < tol; fixed_micro > 0 performs exactly that many
 * iterations instead.  Defaults: mode 0, tol 1e-4, max_micro 200, fixed_micro 0. */
int rtcc_set_solver(rtcc_ctx* ctx, int mode, double tol, int max_micro, int fixed_micro);

/* Advance tau -> tau + dt by Eq. 9 and update the cumulant by the trapezoid rule. */
int rtcc_step(rtcc_ctx* ctx, double dt);
/* out (HOST): Re C, Im C, Re E, Im E at the current time; E = -i dC/dtau. */
int rtcc_cumulant(const rtcc_ctx* ctx, double out[4]);
int rtcc_last_micro_iterations(const rtcc_ctx* ctx);
double rtcc_time(const rtcc_ctx* ctx);

/* Instrumentation: kernel launches and executed tensor-pipe flops since creation / since last reset. */
int rtcc_counters(const rtcc_ctx* ctx, long long* launches, double* dmma_flops);
int rtcc_reset_counters(rtcc_ctx* ctx);
/* Device time (ms) and executed flops of the pp-ladder kernels of the most recent residual evaluation
 * that ran with timing enabled (rtcc_set_timing(ctx, 1) brackets them with CUDA events). */
int rtcc_set_timing(rtcc_ctx* ctx, int on);
int rtcc_ladder_timing(const rtcc_ctx* ctx, double* ms, double* flops, double* model_flops);

/* Launch plan of the pp-ladder for spin case 0, 1, 2 (those with a non-empty block, in the order ab, aa, bb; RTCC_EINVAL past
 * the last): out = { stacked Re|Im columns, column tile width, column tiles, CTAs per cluster (0: narrow batched kernel),
 * column groups, (e,f) slices, row tiles, SMs the clusters can occupy }. */
int rtcc_ladder_plan(const rtcc_ctx* ctx, int spin_case, int out[8]);
/* out[k], k = 1..16: SMs that clusters of k CTAs of the wide ladder kernel can occupy at once on this device (0: not
 * schedulable), from cudaOccupancyMaxActiveClusters; the plan weighs cluster sizes with it. */
int rtcc_ladder_occupancy(const rtcc_ctx* ctx, int out[17]);

/* (N-1)-electron Fock matrix from the Cholesky vectors and the orbital energies of the N-electron reference
 * (f_pq = eps_p delta_pq - v_pc^qc, c = core-hole spin-orbital; v_pq^rs = <pq||rs>):
 *   fock[s][p][q] = eps[s][p] delta_pq - sum_Q L[s][Q][p][q] L[cs][Q][c][c] + delta(s,cs) sum_Q L[s][Q][p][c] L[s][Q][c][q]
 * L [2][n_chol][n][n], eps [2][n], fock [2][n][n] (out); core_spin in {0,1}, 0 <= core_index < n (position of the core
 * orbital in that spin's orbital order).  flags & RTCC_HOST_PTRS: arrays are host pointers, else device pointers. */
int rtcc_build_fock(int n, int n_chol, const double* L, const double* eps, int core_spin, int core_index, double* fock,
                    unsigned flags, void* cuda_stream);

/* Core-hole Green's function and spectral function from a recorded cumulant (PAPER.md:41, :52-56 Eqs. 3-4; :103):
 *   G(tau_k) = -i exp(-i (eps_c + e_corr) tau_k) exp(C(tau_k)),   tau_k = k dt, k = 0..nt-1
 *   A(omega) = -(1/pi) Im int_0^T G(tau) exp(i omega tau - eta tau) dtau      (trapezoid rule on the recorded grid;
 *   the paper does not state its broadening: eta >= 0 is the caller's Lorentzian half width, reading R14)
 * All pointers are HOST pointers: C [nt][2] (re, im), omega [nw], G [nt][2] out (may be NULL), A [nw] out. */
int rtcc_spectral_function(int nt, double dt, const double* C, double eps_c, double e_corr, double eta, int nw,
                           const double* omega, double* G, double* A);

/* Measured FP64 tensor-pipe peak (TFLOP/s) of the current device: register-resident DMMA loop. */
int rtcc_fp64_peak(double* tflops);

/* Test hook: copy a named internal buffer (e.g. "Zsc", "Yab", "Mq") to a HOST array; returns the number
 * of doubles the buffer holds (or a negative error), copying at most max_doubles. */
long long rtcc_debug_buffer(const rtcc_ctx* ctx, const char* name, double* out, long long max_doubles);

/* Test hook for the contraction primitive: C[M][N] = alpha * A[M][K] * B[K][N] + beta * C, all dense row-major
 * HOST arrays; cplx != 0 treats A, B, C as planar complex ([2][rows][cols]). */
int rtcc_debug_gemm(int M, int N, int K, const double* A, const double* B, double* C, double alpha, double beta, int cplx);

/* cudaError_t behind the most recent RTCC_ECUDA / RTCC_ENOMEM of this context; ctx == NULL: of the most recent failed rtcc_create. */
int rtcc_last_cuda_error(const rtcc_ctx* ctx);
const char* rtcc_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif
