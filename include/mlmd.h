/*
 * mlmd.h -- C ABI of libmlmd: the domain-batched real-time Kohn-Sham step on one B200 (sm_100a).
 *
 * One handle = a batch of `ndom` same-shaped, independent divide-and-conquer domains
 * (PAPER.md L126, L298).  Orbitals psi_n on a periodic real-space grid are advanced by
 *
 *     psi <- sum_{m=0..4} (-i dt H)^m / m!  psi,       H = 1/2 (-i grad + A)^2 + V_loc + V_NL
 *
 * (Eq. (2) L138 and Eq. (3); BASELINE.json north_star: 4th-order Taylor propagator,
 * 4th-order central finite differences, Kleinman-Bylander projectors
 * V_NL psi = sum_p beta_p D_p <beta_p|psi>, <a|b> = dv * sum_r conj(a) b), and every step ends
 * with rho(r) = sum_n f_n |psi_n(r)|^2.  Hartree atomic units; `A` means (e/c)A of Eq. (3).
 * The readings of the paper that fix the details (D1..D26) are listed in DESIGN.md.
 *
 * Conventions
 *   layout     psi[dom][ix][iy][iz][n] complex64 (re,im interleaved), orbital index n fastest
 *              (PAPER.md L170); grid point index r = (ix*ny + iy)*nz + iz; beta[dom][r][p];
 *              vloc[dom][r]; rho[dom][r]; D[dom][p]; occ[dom][n]; S[dom][m][n].
 *   where      every data pointer comes with MLMD_HOST or MLMD_DEVICE saying where it lives
 *              (device = the CUDA device current at mlmd_domain_create).
 *   ownership  the caller owns every buffer it passes, including the workspace, which must stay
 *              alive and untouched until mlmd_domain_destroy.  set_* calls copy their inputs
 *              into the workspace.  The library allocates no device memory after create.
 *   stream     all work is ordered on the stream given at create (small batches replay a CUDA graph of
 *              the step on an internal stream that is forked from and joined to that stream).  Calls are asynchronous
 *              w.r.t. the host except: any call with a MLMD_HOST pointer (synchronises the stream
 *              before returning), mlmd_set_vloc (reads back max|V|), and mlmd_propagate when the
 *              handle was created with MLMD_CHECK_FINITE.
 *   errors     every call returns a status; on error nothing is written to caller buffers and
 *              mlmd_last_error() describes the failure.  Nothing throws or aborts.
 *   threading  one handle is not re-entrant; distinct handles are independent.
 *   device     requires compute capability 10.x; anything else -> MLMD_ERR_CUDA.  There is no
 *              CPU fallback.
 */
#ifndef MLMD_H
#define MLMD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* The library is built with hidden visibility: these are its only exported symbols. */
#if defined(__GNUC__)
#define MLMD_API __attribute__((visibility("default")))
#else
#define MLMD_API
#endif

typedef struct mlmd_domain mlmd_domain_t;

enum {
    MLMD_OK = 0,
    MLMD_ERR_ARG = 1,       /* NULL pointer, bad enum, negative size */
    MLMD_ERR_SHAPE = 2,     /* grid axis < 5, nproj > nproj_max, workspace too small, ... */
    MLMD_ERR_STATE = 3,     /* e.g. propagate before set_orbitals / set_vloc */
    MLMD_ERR_CUDA = 4,      /* CUDA runtime error or unsupported device */
    MLMD_ERR_NOMEM = 5,
    MLMD_ERR_NONFINITE = 6, /* MLMD_CHECK_FINITE found NaN/Inf in psi after propagate */
    MLMD_WARN_UNSTABLE = 7  /* work done, but the a-priori Taylor-4 stability bound is exceeded */
};
enum { MLMD_HOST = 0, MLMD_DEVICE = 1 };
enum { MLMD_BETA_REAL32 = 0, MLMD_BETA_COMPLEX64 = 1 };
enum {
    MLMD_GEMM_FP32GRADE = 0, /* default: 3xTF32 on tcgen05 tensor cores, FP32 accumulate          */
    MLMD_GEMM_FP64 = 1,      /* FP64 accumulation of exact FP32 products (CUDA cores; slow, check) */
    MLMD_GEMM_LOWP_BF16 = 2, /* opt-in: BF16 operands, FP32 accumulate      */
    MLMD_GEMM_TF32X1 = 3,    /* optional rung: single TF32 product, FP32 accumulate               */
    MLMD_GEMM_FP32_SIMT = 4, /* plain FP32 FMA on CUDA cores (portable fallback, any shape)       */
    MLMD_GEMM_FP32GRADE_STAGED = 5 /* opt-in: mlmd_propagate's three inner Horner stages (whose V_NL terms reach
                                * the result with weights dt^4/24, dt^3/6, dt^2/2) use 1 product of
                                * nearest-rounded TF32 operands in the projection and 2 in the back-application
                                * (beta hi + lo, W hi); the outermost stage stays 3xTF32.  Same tolerances as
                                * mode 0.  Every other call behaves as mode 0. */
};
enum {
    MLMD_KEEP_PSI0 = 1u,    /* snapshot Psi(0) at mlmd_set_orbitals for mlmd_overlap(which=1)     */
    MLMD_CHECK_FINITE = 2u, /* scan psi for NaN/Inf at the end of every mlmd_propagate            */
    MLMD_BORROW_PSI = 4u    /* Psi lives in the CALLER's device buffer: mlmd_set_orbitals(where = MLMD_DEVICE)
                             * adopts the pointer instead of copying, every step updates that buffer in place and the
                             * workspace holds no Psi copy.  The buffer is complex64
                             * [ndom][nx][ny][nz][norb], 256-byte aligned, norb a multiple of 16 (rows need no padding),
                             * and must stay alive and untouched by the caller while a call is in flight.            */
};
/* Run-time options (mlmd_set_option); each is read when it is set, never from the environment. */
enum {
    MLMD_OPT_GRAPH = 0,     /* 1 (default): small, launch-bound batches replay a CUDA graph of the step; 0: eager launches */
    MLMD_OPT_STENCIL = 1,   /* 0 (default): TMA-staged kernel when ny, nz are multiples of 16, else the fallbacks;
                             * 1: register-marching kernel; 2: one-thread-per-output kernel (cross-checks)            */
    MLMD_OPT_GEMM_PATH = 2, /* 0 (default): tcgen05 kernels when ngrid is a multiple of 128; 1: CUDA-core kernels        */
    MLMD_OPT_KICK_NORM = 3, /* mlmd_propagate_split, norm after the second kick (and, with MLMD_OPT_LOCAL_SOLVER = 1, after
                             * the first): 0 (default) from the projector Gram matrix when it applies; 1: always by a pass
                             * over psi                                                                               */
    MLMD_OPT_FD_ORDER = 4,  /* order of the central finite differences of the kinetic and A.grad terms: 4 (default; north_star:
                             * 13-point star) or 2 (the paper's own "7-point star stencil" on "nearest-neighbor mesh points",
                             * PAPER.md L147, L283): c2 = [1, -2, 1] / h^2, c1 = [-1/2, 0, 1/2] / h.
                             * mlmd_propagate, mlmd_propagate_split and mlmd_current follow it; the stability bound of
                             * mlmd_propagate becomes dt [ 2 sum_d 1/h_d^2 + sum_d |A_d|/h_d + ... ]                    */
    MLMD_OPT_LOCAL_SOLVER = 5, /* how mlmd_propagate_split evaluates exp(-i dt h_loc) in Eq. (2): 0 (default) the 4th-order
                             * Taylor sum on the differences MLMD_OPT_FD_ORDER selects (reading D28); 1 the paper's own
                             * "block-diagonal split-operator solver" (ref. [41]; reading
                             * D33): space splitting of the 2nd-order (7-point) operator into 2 x 2 nearest-neighbour blocks,
                             * exp(-i dt/2 (V + 1/2|A|^2)) prod_d [even(dt/2) odd(dt) even(dt/2)] exp(-i dt/2 (V + 1/2|A|^2)):
                             * unitary for any dt, time-reversible, O(dt^3) per step.  Needs even nx, ny, nz (<= 256 each),
                             * else MLMD_ERR_SHAPE.  mlmd_propagate (Taylor-4 of the full H) ignores it.               */
    MLMD_OPT_COUNT = 6
};

/* Bytes of device workspace mlmd_domain_create needs for this shape (0 on invalid arguments).
 * Holds Psi, two Psi-sized stage buffers (Horner form of the Taylor sum), optional Psi(0),
 * V_loc, beta (and its split copies), D, occupations, rho, projection scratch. */
MLMD_API size_t mlmd_workspace_bytes(int ndom, int nx, int ny, int nz, int norb, int nproj_max, unsigned flags);

/* Create a batch of ndom periodic domains of nx*ny*nz points (each axis >= 5: the five radius-2
 * periodic neighbours must be distinct), spacings hx,hy,hz (bohr), norb orbitals, at most
 * nproj_max REAL projector rows (a complex64 projector counts twice: mlmd_set_projectors needs
 * nproj <= nproj_max for MLMD_BETA_REAL32 and 2*nproj <= nproj_max for MLMD_BETA_COMPLEX64).  workspace_dev: device memory, 256-byte
 * aligned, >= mlmd_workspace_bytes(...).  cuda_stream: a cudaStream_t passed as void*
 * (NULL = legacy default stream). */
MLMD_API int mlmd_domain_create(mlmd_domain_t **out, int ndom, int nx, int ny, int nz, double hx, double hy,
                       double hz, int norb, int nproj_max, void *workspace_dev, size_t workspace_bytes,
                       void *cuda_stream, unsigned flags);
MLMD_API int mlmd_domain_destroy(mlmd_domain_t *h);

/* Psi(t=0) and occupations f_n >= 0 (occ may be NULL = keep previous / all 2.0).
 * psi: complex64 [ndom][nx][ny][nz][norb] at `where`; occ: double [ndom][norb], HOST. */
MLMD_API int mlmd_set_orbitals(mlmd_domain_t *h, const void *psi_c64, const double *occ, int where);
MLMD_API int mlmd_get_orbitals(mlmd_domain_t *h, void *psi_c64, int where);

/* Local potential v_loc(r) of Eq. (3) in Hartree, float [ndom][nx][ny][nz]; frozen during a
 * propagate call (only Delta v_loc is passed once per MD step; reading D25). */
MLMD_API int mlmd_set_vloc(mlmd_domain_t *h, const float *vloc, int where);

/* Nonlocal operator V_NL = dv * B diag(D) B^H (north_star; Eq. (5) L199 is the case
 * B = Psi(0)).  beta: [ndom][ngrid][nproj], float (MLMD_BETA_REAL32) or complex64
 * (MLMD_BETA_COMPLEX64) at `where`; D: double [ndom][nproj] in Hartree, HOST.
 * nproj = 0 switches V_NL off (beta, D may be NULL). */
MLMD_API int mlmd_set_projectors(mlmd_domain_t *h, int nproj, const void *beta, int beta_dtype, const double *D,
                        int where);

MLMD_API int mlmd_set_gemm_mode(mlmd_domain_t *h, int mode);

/* Set one MLMD_OPT_* option (unknown key or value -> MLMD_ERR_ARG).  Takes effect from the next call on. */
MLMD_API int mlmd_set_option(mlmd_domain_t *h, int key, int value);

/* nsteps Taylor-4 steps of size dt.  A: double [nsteps][a_ndom][3], HOST; A[n] is the vector
 * potential at the step midpoint t_n + dt/2 (Eq. (2)), uniform inside a domain;
 * a_ndom = 1 (same field for every domain) or ndom.  The density of the final state is kept
 * for mlmd_density.  Returns MLMD_WARN_UNSTABLE (work still done) if
 * dt * [ (8/3) sum_d 1/h_d^2 + 1.3722 sum_d |A_d|/h_d + |A|^2/2 + max|V_loc| + max|D| ] > 2 sqrt(2). */
MLMD_API int mlmd_propagate(mlmd_domain_t *h, int nsteps, double dt, const double *A, int a_ndom);

/* nsteps steps of the paper's literal Eq. (2):
 *     psi <- K exp(-i dt h_loc(t_n + dt/2)) K psi,   K psi_n = (psi_n - i dt/2 V_NL psi_n) ||psi_n|| / ||psi_n - i dt/2 V_NL psi_n||
 * i.e. a normalised first-order nonlocal half-kick (the norm is taken per orbital on the state the kick
 * acts on, reading D27), the 4th-order Taylor sum of h_loc = 1/2(-i grad + A)^2 + V_loc alone (D28), and
 * a second half-kick.  With beta = Psi(0) (MLMD_BETA_COMPLEX64) and D_p = const this V_NL is the nonlocal
 * correction of Eq. (5) L199 with delta = -i dt/2 D dv.  Two V_NL applications per step instead of four.
 * Arguments, density and return values as mlmd_propagate; the stability bound leaves out max|D| (the
 * normalised kick is stable for any dt |D|).  With nproj = 0 it is the same map as mlmd_propagate.
 * With MLMD_OPT_LOCAL_SOLVER = 1 the middle factor is the paper's own block-diagonal split-operator solver on the
 * 7-point operator (reading D33) instead of the Taylor sum: unitary for any dt (no stability
 * warning), needs even nx, ny, nz (else MLMD_ERR_SHAPE). */
MLMD_API int mlmd_propagate_split(mlmd_domain_t *h, int nsteps, double dt, const double *A, int a_ndom);

/* rho(r) = sum_n f_n |psi_n(r)|^2 of the current state, float [ndom][nx][ny][nz] at `where`. */
MLMD_API int mlmd_density(mlmd_domain_t *h, float *rho, int where);

/* S[dom] = dv * Phi^H Psi(t), complex64 [ndom][norb][norb] at `where` (CGEMM(1)):
 * which = 0: Phi = Psi(t) (Gram matrix); which = 1: Phi = Psi(0) (needs MLMD_KEEP_PSI0).
 * Always evaluated in the FP32-grade (or FP64) GEMM mode: it is a measurement. */
MLMD_API int mlmd_overlap(mlmd_domain_t *h, int which, void *S_c64, int where);

/* Occupations of the t = 0 orbitals and number of excited electrons per domain (LFD hands the
 * occupation numbers f_s back to QXMD; L159: n_exc "is computed from f_s"; L283: overlap matrix between the
 * orbitals at time t and 0).  The paper gives no formula; reading D29:
 *     f_s(t) = sum_n f_n |S_sn|^2,  S = dv Psi(0)^H Psi(t) (mlmd_overlap which = 1; needs MLMD_KEEP_PSI0),
 *     n_exc  = sum_s max(f_s(0) - f_s(t), 0).
 * f: double [ndom][norb], n_exc: double [ndom], both at `where`. */
MLMD_API int mlmd_occupations(mlmd_domain_t *h, double *f, double *n_exc, int where);

/* Observables of the current state that feed the light-matter loop ("GEMMification is applied to
 * nonlocal correction in energy and electric current ... used in Maxwell's equations"; SURVEY.md 8(f) NEXT-2;
 * the paper gives no formulas: reading D30).
 * mlmd_energy_nl: E[dom] = sum_n f_n <psi_n|V_NL|psi_n> = dv^2 sum_n f_n sum_p D_p |sum_r conj(beta_rp) psi_rn|^2
 *   in Hartree (the projection GEMM of the step + a reduction); double [ndom] at `where`; 0 when nproj = 0.
 * mlmd_current: J[dom][d] = sum_n f_n Re<psi_n| -i D1_d + A_d |psi_n>, D1 the 4th-order first difference of H,
 *   A: double [a_ndom][3] HOST (a_ndom = 1 or ndom), J: double [ndom][3] at `where`.  This is the current of
 *   h_loc's velocity operator; the nonlocal-pseudopotential term -i[r, V_NL] is mlmd_current_nl. */
MLMD_API int mlmd_energy_nl(mlmd_domain_t *h, double *E, int where);
MLMD_API int mlmd_current(mlmd_domain_t *h, const double *A, int a_ndom, double *J, int where);

/* Nonlocal (pseudopotential) part of the current, the term PAPER.md L201 says is GEMMified (reading D31):
 *     J_nl[dom][d] = sum_n f_n <psi_n| -i [r_d, V_NL] |psi_n> = 2 dv^2 sum_n f_n sum_p D_p Im( conj(G_dpn) C_pn ),
 *     C_pn = sum_r conj(beta_p(r)) psi_n(r),  G_dpn = sum_r conj(rbeta_dp(r)) psi_n(r),  rbeta_dp(r) = (r - R_p)_d beta_p(r)
 * i.e. the projection GEMM of the step against beta and against the three caller-supplied arrays rbeta_d (the paper's
 * atom positions R_p are the caller's; a constant shift of r commutes with V_NL, so any centre per projector gives the
 * commutator with r itself).  rbeta: [3][ndom][ngrid][nproj], same dtype as the beta given to mlmd_set_projectors, at
 * `where_rbeta`; it is staged through a Psi-sized work buffer one direction at a time (nothing is kept).
 * J: double [ndom][3] at `where`.  The total TDCDFT current is mlmd_current + mlmd_current_nl.  0 when nproj = 0. */
MLMD_API int mlmd_current_nl(mlmd_domain_t *h, const void *rbeta, int where_rbeta, double *J, int where);

/* Per-kernel-class timing of mlmd_propagate with CUDA events on the handle's stream (bench.py's
 * roofline numbers).  mlmd_profile(h, 1) starts recording (and clears earlier records),
 * mlmd_profile(h, 0) stops.  mlmd_profile_read synchronises the stream and returns the summed
 * device time in milliseconds and the number of launches of class `kind` recorded so far. */
enum { MLMD_K_STENCIL = 0, MLMD_K_PROJ = 1, MLMD_K_BACK = 2, MLMD_K_GLUE = 3, MLMD_K_DENSITY = 4,
       MLMD_K_NLP = 5 /* fused back-application + projection */,
       MLMD_K_NORM = 6 /* per-orbital norms of the split step */, MLMD_K_COUNT = 7 };
MLMD_API int mlmd_profile(mlmd_domain_t *h, int enable);
MLMD_API int mlmd_profile_read(mlmd_domain_t *h, int kind, double *ms_total, long long *launches);

/* Which kernels run the nonlocal GEMMs for the current mode and shape: 0 = CUDA cores (SIMT),
 * 1 = tcgen05 tensor cores. */
MLMD_API int mlmd_gemm_path(const mlmd_domain_t *h);

/* Number of kernels the library launched on this handle since create (bench.py's gpu_launches). */
MLMD_API long long mlmd_launch_count(const mlmd_domain_t *h);

/* Squared norms of all orbitals WITHOUT a handle, a workspace or any allocation, for callers that cannot call
 * cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it):
 *     norm2[dom][n] = dv * sum_r |psi[dom][r][n]|^2
 * (the per-orbital norms that the kick of PAPER.md Eq. (2) L138 divides by, reading D27; the diagonal of mlmd_overlap's
 * Gram matrix; sum_n f_n norm2[n] = the electron count of the density).  Same kernel pair as the split step's norm pass,
 * but its per-slab FP64 partial sums live in a file-scope device array of MLMD_STATIC_SCRATCH_BYTES that every GPU
 * loading the library holds until the process exits, instead of in a caller workspace.
 *   psi     DEVICE, complex64 [ndom][ngrid][ld], orbital index fastest (ld = row pitch in complex elements; padded
 *           columns are summed like any other)           norm2   DEVICE, double [ndom][ld]
 *   stream  cudaStream_t the two kernels are enqueued on (NULL = default stream); the call is asynchronous
 * Limit: ndom * 64 * ld * 8 bytes <= MLMD_STATIC_SCRATCH_BYTES (configs[3], 64 x 224, fits), ndom <= 65535; anything
 * larger -> MLMD_ERR_SHAPE with the sizes in mlmd_last_error().  Host pointers -> MLMD_ERR_ARG.  Calls no cudaMalloc,
 * cudaFree or allocating library routine.  All calls share the one array: calls that overlap on the GPU (two streams)
 * race on it - serialise them on one stream.  Nothing needs clearing between calls (every partial sum that is read has
 * been written by the same call). */
#define MLMD_STATIC_SCRATCH_BYTES (8u << 20)
MLMD_API int mlmd_orbital_norms_static(const void *psi_c64, int ndom, long long ngrid, int ld, double dv, double *norm2,
                                       void *stream);

/* Thread-local description of the last failure in this thread; never NULL. */
MLMD_API const char *mlmd_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MLMD_H */
