// Internal declarations of libmlmd (not part of the C ABI; see include/mlmd.h).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <cuda.h>

#include <vector>

#include "../../include/mlmd.h"

namespace mlmd {

// Per-(step, domain) stencil coefficients, computed in FP64 on the host and
// rounded once.  For axis d and offset +-j (j = 1, 2):
//   a_{d,+-j} = p[d][j-1] -+ i q[d][j-1],  p = -1/2 c2_j / h_d^2,  q = A_d c1_{+j} / h_d
// centre (real): c0 + 1/2|A|^2 + V_loc(r).
struct StepCoef {
    float p[3][2];
    float q[3][2];
    float centre;   // c0 + 1/2 |A|^2
    float pad;
};
static_assert(sizeof(StepCoef) == 56, "StepCoef layout");

struct Workspace {              // byte offsets into the caller's workspace
    size_t psi, ua, ub, psi0, vloc, beta, beta_lo, dprime, occ, rho, z, what, what_lo, zpart, coef, coef_cur, flag,
        nrm, nrm_part, scl, occ_eff, avec, gram, rich, total;
};

// Tensor maps are pure functions of (base pointer, shape, box): encoded once per distinct key and kept in the
// handle, instead of 70+ cuTensorMapEncodeTiled calls per time step.
struct TmapKey {
    int kind;                 // which encoder (tag chosen by the caller)
    const void *base;
    unsigned long long a, b, c, d;
    unsigned e, f;
};
struct TmapCache {
    struct Entry { TmapKey key; CUtensorMap map; };
    std::vector<Entry> entries;
    const CUtensorMap *find(const TmapKey &k) const {
        for (const Entry &e : entries)
            if (e.key.kind == k.kind && e.key.base == k.base && e.key.a == k.a && e.key.b == k.b && e.key.c == k.c &&
                e.key.d == k.d && e.key.e == k.e && e.key.f == k.f)
                return &e.map;
        return nullptr;
    }
    void insert(const TmapKey &k, const CUtensorMap &m) {
        if (entries.size() >= 256) entries.clear();     // e.g. a caller cycling through many borrowed buffers
        entries.push_back(Entry{k, m});
    }
    void clear() { entries.clear(); }
};
// *out = the cached map of key k, or build(out) (and remember it).  cache may be NULL (kernel-level test hooks).
template <class Build>
bool cached_tmap(TmapCache *cache, const TmapKey &k, CUtensorMap *out, Build build) {
    if (cache)
        if (const CUtensorMap *m = cache->find(k)) {
            *out = *m;
            return true;
        }
    if (!build(out)) return false;
    if (cache) cache->insert(k, *out);
    return true;
}

constexpr int kCoefCapacity = 256;   // steps per coefficient upload chunk
constexpr int kMaxSplit = 64;        // split-K slices of the projection GEMM
constexpr int kNormSlabs = 64;       // row slabs per domain of the per-orbital norm reduction (split step)

}  // namespace mlmd

struct mlmd_domain {
    int ndom, nx, ny, nz, norb, nproj_max;
    int ld;                     // padded orbital count (row pitch of psi in complex elements)
    long ngrid;
    double hx, hy, hz, dv;
    unsigned flags;
    cudaStream_t stream;
    char *ws;
    size_t ws_bytes;
    mlmd::Workspace off;
    // state
    int nproj;                  // projectors currently set (complex ones count once)
    int beta_complex;           // 1: beta is complex64 -> real GEMM row count P = 2*nproj
    int P;                      // real projector rows
    int ldp;                    // padded P (pitch of beta rows / rows of Z, What)
    int prows;                  // rows allocated for Z/What/zpart = max(ldp(nproj_max), 2*ld)
    int nsplit;                 // split-K factor of the projection (CUDA-core path)
    int nsplit_tc, nsplit_tc_ovl;   // split-K factors of the tcgen05 projection (beta rows / overlap)
    bool tc_ok;                 // shape and device allow the tcgen05 GEMM kernels
    int gemm_mode;
    int opt[MLMD_OPT_COUNT];    // mlmd_set_option values
    bool coef_o2;               // the call in flight takes 2nd-order weights whatever MLMD_OPT_FD_ORDER says (split-operator solver)
    float2 *psi_ptr;            // Psi: inside the workspace, or the caller's buffer (MLMD_BORROW_PSI)
    mutable mlmd::TmapCache tmaps;
    bool have_psi, have_vloc, have_occ, rho_valid;
    bool field_yz;              // any A_y or A_z non-zero in the current propagate call
    double vmax, dmax;
    long long launches;
    // per-kernel-class CUDA-event records (mlmd_profile)
    bool prof_on;
    std::vector<cudaEvent_t> prof_pool;
    struct ProfRec { int kind; int e0, e1; };
    std::vector<ProfRec> prof_recs;
    mlmd::StepCoef *coef_host;  // pinned, kCoefCapacity * ndom
    cudaEvent_t coef_uploaded;  // the pinned staging buffer may be refilled once this has happened
    // CUDA graph of one time step (small, launch-bound problems; see api.cu)
    bool graph_allowed;
    cudaGraphExec_t gexec;
    cudaStream_t gstream;
    cudaEvent_t gfork, gjoin;
    int g_launches;             // kernels per graph launch
    double g_dt;                // the step size the graph was captured with
    bool g_yz;
    bool gram_valid;            // gram() matches the current projectors
    bool split_pending;         // psi in memory is the un-normalised chain of the split step; true psi = scl() * psi
    int ldg;                    // pitch of gram() = ldp_max
    bool g_split;               // the graph holds the Eq. (2) split step, not the Taylor-4 step
    int *flag_host;             // pinned
    // typed views
    float2 *psi() const { return psi_ptr; }
    float2 *ua() const { return (float2 *)(ws + off.ua); }
    float2 *ub() const { return (float2 *)(ws + off.ub); }
    float2 *psi0() const { return (float2 *)(ws + off.psi0); }
    float *vloc() const { return (float *)(ws + off.vloc); }
    float *beta() const { return (float *)(ws + off.beta); }          // the projectors as given (FP32)
    float *beta_lo() const { return (float *)(ws + off.beta_lo); }    // beta - trunc_tf32(beta), exact (back-application)
    float *dprime() const { return (float *)(ws + off.dprime); }
    float *occ() const { return (float *)(ws + off.occ); }
    float *rho() const { return (float *)(ws + off.rho); }
    float *z() const { return (float *)(ws + off.z); }
    float *what() const { return (float *)(ws + off.what); }
    float *what_lo() const { return (float *)(ws + off.what_lo); }
    float *zpart() const { return (float *)(ws + off.zpart); }
    mlmd::StepCoef *coef() const { return (mlmd::StepCoef *)(ws + off.coef); }
    mlmd::StepCoef *coef_cur() const { return (mlmd::StepCoef *)(ws + off.coef_cur); }
    float *rich() const { return (float *)(ws + off.rich); }     // split-operator solver: [ndom][3][8] rotation constants of the step
    int *step_counter() const { return (int *)(ws + off.flag + 64); }
    int *flag() const { return (int *)(ws + off.flag); }
    // split step (Eq. 2): squared orbital norms [4][ndom][ld] (input, after kick 1, after Taylor, after kick 2)
    double *nrm(int which) const { return (double *)(ws + off.nrm) + (size_t)which * ndom * ld; }
    double *nrm_part() const { return (double *)(ws + off.nrm_part); }
    float *scl() const { return (float *)(ws + off.scl); }
    float *occ_eff() const { return (float *)(ws + off.occ_eff); }
    double *avec() const { return (double *)(ws + off.avec); }   // mlmd_current: A[a_ndom][3]
    float *gram() const { return (float *)(ws + off.gram); }      // split step: beta^T beta, [ndom][ldp_max][ldp_max]
};

namespace mlmd {

// One-time-per-device flag (function attributes such as the dynamic shared-memory limit are per device).
struct DeviceOnce {
    unsigned long long mask = 0;
    static int dev() {
        int d = 0;
        cudaGetDevice(&d);
        return d & 63;
    }
    bool done() const { return (mask >> dev()) & 1ull; }
    void mark() { mask |= 1ull << dev(); }
};

// ---- stencil.cu ------------------------------------------------------------------------------
// One Horner stage without the nonlocal term:
//   out(r,n) = psi(r,n) + (-i tau) [ sum_{d,j} a_{d,j} w(r + j e_d, n) + (centre + V(r)) w(r,n) ]
// w, psi, out: [ndom][ngrid][ld] complex64; coef: [ndom] for this step; out may alias psi.
cudaError_t launch_stencil_stage(const mlmd_domain *h, const float2 *w, const float2 *psi, float2 *out,
                                 const StepCoef *coef, const StepCoef *coef_host, float tau, int *nlaunch);
// The same stage that also delivers squared per-orbital norms (split step): norm_mode 1 = of w, 2 = of out,
// into nrm_out[dom][ld]; fused into the TMA pass when that runs, otherwise a separate reduction pass.
cudaError_t launch_stencil_stage_norm(const mlmd_domain *h, const float2 *w, const float2 *psi, float2 *out,
                                      const StepCoef *coef, const StepCoef *coef_host, float tau, int norm_mode,
                                      double *npart, double *nrm_out, int *nlaunch);

// ---- stencil_tma.cu ---------------------------------------------------------------------------
// The same stage with TMA-staged x-planes (needs ny % 16 == 0, nz % 16 == 0).
bool stencil_tma_supported(const mlmd_domain *h);
// coef_host: the one coefficient set of this step when every domain sees the same field (passed by
// value through the constant bank), NULL when coef[dom] differs per domain.
cudaError_t launch_stencil_tma(const mlmd_domain *h, const float2 *w, const float2 *psi, float2 *out, const StepCoef *coef,
                               const StepCoef *coef_host, float tau, int *nlaunch, int norm_mode = 0, double *npart = nullptr);
// (with MLMD_OPT_FD_ORDER = 2 it runs its radius-1 instantiation: same staging, the j = 2 taps neither loaded nor multiplied)
// norm_mode 1 / 2: the pass also writes per-CTA partial sums of |w|^2 / |out|^2 per orbital into
// npart[dom][slot][ld], slot < stencil_tma_norm_slots(h) (split step, reading D27)
int stencil_tma_norm_slots(const mlmd_domain *h);

// ---- richardson.cu ---------------------------------------------------------------------------
// The paper's own local solver (MLMD_OPT_LOCAL_SOLVER = 1; reading D33): psi <- U_loc(dt) psi in place, three passes
// (one per axis); coef: this step's device coefficients [ndom] with the 2nd-order weights.
bool richardson_supported(const mlmd_domain *h);
cudaError_t launch_richardson(const mlmd_domain *h, float2 *psi, const StepCoef *coef, double dt, int *nlaunch);

// ---- gemm_simt.cu ----------------------------------------------------------------------------
// Projection (S2a): zpart[dom][s][p][c] = sum_{r in slice s} B[dom][r][p] * Y[dom][r][c]
//   B: [ndom][ngrid][ldb] float (p fastest), Y: [ndom][ngrid][ldy] float, P rows, N columns used.
//   Blo (may be NULL): B is given as an exact hi + lo pair and summed on load.
cudaError_t launch_proj_simt(cudaStream_t st, int ndom, long ngrid, const float *B, const float *Blo, int ldb, int P,
                             const float *Y, int ldy, int N, float *zpart, int prows, int nsplit,
                             bool fp64, int *nlaunch);
// Back-application (S2d): Y[dom][r][c] += sum_p B[dom][r][p] * What[dom][p][c]  (W stored as hi + lo; Blo may be NULL)
cudaError_t launch_back_simt(cudaStream_t st, int ndom, long ngrid, const float *B, const float *Blo, int ldb, int P,
                             const float *What, const float *Wlo, float *Y, int ldy, int N, int prows, bool fp64,
                             int *nlaunch);

// ---- gemm_tc.cu ------------------------------------------------------------------------------
// The same two contractions on tcgen05 tensor cores, operands staged by TMA.  nprod = 3: 3xTF32
// (FP32-grade), nprod = 2 (back-application only): beta_hi + beta_lo times W_hi, nprod = 1: single TF32 product (psi truncated by the MMA), nprod = 4 (projection only): single product with psi rounded to nearest in shared memory, nprod = 0: single product of operands rounded to BF16
// in shared memory (opt-in low precision).  A_lo == NULL with nprod == 3: the kernel splits A
// itself (overlap, where A is a psi buffer).  Requires ngrid % 128 == 0, N % 32 == 0, lda % 8 == 0.
bool tc_available();
int tc_choose_nsplit(int ndom, long ngrid, int P, int N);
cudaError_t launch_proj_tc(cudaStream_t st, int ndom, long ngrid, const float *A_hi, const float *A_lo, int lda, int P,
                           const float *Y, int ldy, int N, float *zpart, int prows, int nsplit, int nprod,
                           int chain /* 16-row stages per TMEM accumulation chain, 0 = whole slice */, int *nlaunch,
                           TmapCache *cache = nullptr,
                           float *rho = nullptr /* != NULL: also rho[dom][r] = sum_n occ[dom][n] |Y[r][n]|^2 (S3 fused) */,
                           const float *occ = nullptr,
                           const void *A16 = nullptr /* nprod == 0: BF16 copy of A [rows][lda] -> kind::f16 kernel */);
// whether that projection can carry the density (CTA-pair kernel, one row tile of projectors, one column tile)
bool proj_tc_can_fuse_density(int P, int N, int nprod);
cudaError_t launch_back_tc(cudaStream_t st, int ndom, long ngrid, const float *A /* raw FP32 */,
                           const float *A_lo /* A - trunc_tf32(A), or NULL: formed in shared memory */, int lda, int P,
                           const float *W_hi, const float *W_lo, float *Y, int ldy, int N, int prows, int nprod,
                           int *nlaunch, TmapCache *cache = nullptr,
                           const void *A16 = nullptr, const void *W16 = nullptr /* nprod == 0: BF16 copies -> kind::f16 kernel */);

// ---- glue.cu ---------------------------------------------------------------------------------
// S2b: reduce split-K partials in fixed order and build What = (-i tau) D' C in real-GEMM form.
cudaError_t launch_reduce_scale(cudaStream_t st, int ndom, int nproj, int beta_complex, int ld, int prows,
                                int nsplit, const float *zpart, const float *dprime, float tau,
                                float *what, float *what_lo, int lowp /* 1: round W to BF16 in FP32 containers; 2: write W as a
                                BF16 array [prows][2 ld] into `what` */, int *nlaunch);
// S3: rho[dom][r] = sum_n occ[dom][n] |psi[dom][r][n]|^2
cudaError_t launch_density(cudaStream_t st, int ndom, long ngrid, int ld, const float2 *psi, const float *occ,
                           float *rho, int *nlaunch);
// S4 epilogue: S[dom][m][n] = dv * (sum over splits of the complex combination of Z)
cudaError_t launch_overlap_epilogue(cudaStream_t st, int ndom, int norb, int ld, int prows, int nsplit,
                                    const float *zpart, float dv, float2 *S, int *nlaunch);
// y (BF16, round-to-nearest-even) = x
cudaError_t launch_to_bf16(cudaStream_t st, const float *x, void *y, size_t n, int *nlaunch);
// lo = x - (x with the 13 low mantissa bits cleared): the part of x a kind::tf32 operand drops (exact in FP32); x is kept
cudaError_t launch_tf32_remainder(cudaStream_t st, const float *x, float *lo, size_t n, int *nlaunch);
cudaError_t launch_max_abs(cudaStream_t st, const float *x, size_t n, int *flag_bits, int *nlaunch);
cudaError_t launch_check_finite(cudaStream_t st, const float *x, size_t n, int *flag, int *nlaunch);
// graph support: *counter = value;  and  cur[d] = all[*counter * ndom + d], ++*counter
cudaError_t launch_set_counter(cudaStream_t st, int *counter, int value, int *nlaunch);
cudaError_t launch_advance_coef(cudaStream_t st, const StepCoef *all, StepCoef *cur, int *counter, int ndom, int *nlaunch);
// split step (Eq. (2), reading D27): out[dom][c] = sum_r |psi[dom][r][c]|^2 (FP64, fixed order);
// scl = sqrt(n0/na * nc/nd), n0 <- n0 nc/na;  psi *= scl fused with the density pass
cudaError_t launch_colnorm2(cudaStream_t st, int ndom, long ngrid, int ld, const float2 *psi, double *part, double *out,
                            int *nlaunch);
// out[dom][c] = sum_{k < nslabs} part[dom][k][c] in index order
cudaError_t launch_colnorm_final(cudaStream_t st, int ndom, int ld, int nslabs, const double *part, double *out, int *nlaunch);
cudaError_t launch_kick_scale(cudaStream_t st, int n, double *n0, const double *na, const double *nc, const double *nd,
                              float *scl, int *nlaunch);
// NEXT-2 observables (reading D30): E_nl from the projection partials; local current by a forward-neighbour pass
cudaError_t launch_energy_nl(cudaStream_t st, int ndom, int nproj, int beta_complex, int ld, int prows, int nsplit,
                             const float *zpart, const float *dprime, const float *occ, double dv, double *E, int *nlaunch);
cudaError_t launch_current(cudaStream_t st, int ndom, int nx, int ny, int nz, double hx, double hy, double hz, int ld,
                           const float2 *psi, const float *occ, const double *A_dev, int a_ndom, double *part,
                           size_t part_doubles, double *J, int fd_order, int *nlaunch);
// nonlocal part of the current (reading D31): complex projection coefficients from the split-K partials, then
// J[dom][d] = 2 dv sum_n f_n sum_p D'_p Im(conj(G_pn) C_pn)
cudaError_t launch_proj_coeff(cudaStream_t st, int ndom, int nproj, int beta_complex, int ld, int prows, int nsplit,
                              const float *zpart, float2 *cmat, int *nlaunch);
cudaError_t launch_current_nl(cudaStream_t st, int ndom, int nproj, int ld, const float2 *cmat, const float2 *gmat,
                              const float *dprime, const float *occ, double dv, int d, double *J, int *nlaunch);
cudaError_t launch_gram_reduce(cudaStream_t st, int ndom, int P, int ldg, int prows, int N, int nsplit, const float *zpart,
                               float *G, int accumulate, int *nlaunch);
cudaError_t launch_kick_quad(cudaStream_t st, int ndom, int P, int ldg, int ld, int prows, const float *G, const float *what,
                             const float *wlo, const double *nc, double *nd, int *nlaunch);
cudaError_t launch_occ_eff(cudaStream_t st, int n, const float *occ, const float *scl, float *out, int *nlaunch);
cudaError_t launch_occupations(cudaStream_t st, int ndom, int norb, int ld, const float2 *S, const float *occ, double *f,
                               double *nexc, int *nlaunch);
cudaError_t launch_scale_density(cudaStream_t st, int ndom, long ngrid, int ld, float2 *psi, const float *scl,
                                 const float *occ, float *rho, int *nlaunch);

}  // namespace mlmd
