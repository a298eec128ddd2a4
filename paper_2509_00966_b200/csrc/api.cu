// C ABI of libmlmd (include/mlmd.h): argument checking, workspace carving, and the step scheduler
// that strings the kernels into four Horner stages + density per time step.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "mlmd_internal.h"

using namespace mlmd;

// TMEM accumulation chain lengths (16-row stages) of the tcgen05 projection: tensor-core FP32
// accumulation truncates, so long chains drift by ~1 ulp per MMA.
static const int kProjChain = 128, kOverlapChain = 4;
// The drift counts MMAs, not stages: a one-product projection issues a third of the MMAs per stage, so three times
// the stages give the same accumulation error with a third of the chain drains (each drain idles the tensor pipe).
static int proj_chain(int nprod) { return nprod == 3 ? kProjChain : 3 * kProjChain; }
// The three inner Horner stages: whatever error their projections make reaches psi damped by the later stages
// (DESIGN.md 5.6), so their chains are 1024 stages: one or two drains per K slice.
static const int kInnerChain = 8 * kProjChain;
// MLMD_GEMM_FP32GRADE_STAGED: Horner stages 0-2 (tau = dt/4, dt/3, dt/2) run with reduced products; their projection
// is one product with psi rounded to the nearest TF32 in shared memory (nprod code 4)
static const int kStagedMask = 0x7, kStagedProjNprod = 4;

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
// the same for the library's other translation units (noalloc.cu)
namespace mlmd {
int set_error(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
}  // namespace mlmd
#define CU(call)                                                                                    \
    do {                                                                                            \
        cudaError_t e__ = (call);                                                                   \
        if (e__ != cudaSuccess)                                                                     \
            return fail(MLMD_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, __LINE__); \
    } while (0)

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static int round_up_i(int x, int a) { return (x + a - 1) / a * a; }

struct Plan {
    int ld, ldp_max, prows, nsplit, nsplit_tc, nsplit_tc_ovl;
    long ngrid;
    Workspace off;
};

static bool make_plan(int ndom, int nx, int ny, int nz, int norb, int nproj_max, unsigned flags, Plan *pl) {
    if (ndom < 1 || nx < 5 || ny < 5 || nz < 5 || norb < 1 || nproj_max < 0) return false;
    if ((double)ndom * nx * ny * nz > 2.0e9) return false;
    pl->ld = round_up_i(norb, 16);      // 2*ld floats per row = whole 128-byte TMA chunks
    pl->ngrid = (long)nx * ny * nz;
    pl->ldp_max = round_up_i(std::max(nproj_max, 1), 8);
    // rows of Z / W per (domain, slice): whole 128-row accumulator blocks of the tcgen05 projection
    pl->prows = round_up_i(std::max(pl->ldp_max, 2 * pl->ld), 128);
    const long tiles = (long)((2 * pl->ld + 63) / 64) * std::max(1, (nproj_max + 63) / 64) * ndom;
    long ns = (592 + tiles - 1) / tiles;
    ns = std::min<long>(ns, std::min<long>(kMaxSplit, pl->ngrid / 64));
    pl->nsplit = (int)std::max<long>(ns, 1);
    pl->nsplit_tc = tc_choose_nsplit(ndom, pl->ngrid, pl->ldp_max, 2 * pl->ld);
    pl->nsplit_tc_ovl = tc_choose_nsplit(ndom, pl->ngrid, 2 * pl->ld, 2 * pl->ld);
    const size_t npts = (size_t)ndom * pl->ngrid;
    const size_t psi_b = npts * pl->ld * sizeof(float2);
    size_t o = 0;
    auto take = [&](size_t bytes) {
        size_t at = o;
        o = align_up(o + bytes, 256);
        return at;
    };
    Workspace &w = pl->off;
    w.psi = take((flags & MLMD_BORROW_PSI) ? 0 : psi_b);
    w.ua = take(psi_b);
    w.ub = take(psi_b);
    w.psi0 = take((flags & MLMD_KEEP_PSI0) ? psi_b : 0);
    w.vloc = take(npts * sizeof(float));
    // + slack: the last 32-column TMA chunk of a row may read up to 128 B past the row
    w.beta = take(npts * pl->ldp_max * sizeof(float) + 256);      // the projectors as given
    w.beta_lo = take(npts * pl->ldp_max * sizeof(float) + 256);   // what a TF32 operand drops of them (back-application)
    w.dprime = take((size_t)ndom * pl->ldp_max * sizeof(float));
    w.occ = take((size_t)ndom * pl->ld * sizeof(float));
    w.rho = take(npts * sizeof(float));
    const size_t zb = (size_t)ndom * pl->prows * 2 * pl->ld * sizeof(float);
    w.z = take(zb);
    w.what = take(zb);
    w.what_lo = take(zb);
    w.zpart = take(zb * std::max(pl->nsplit, std::max(pl->nsplit_tc, pl->nsplit_tc_ovl)));
    w.coef = take((size_t)kCoefCapacity * ndom * sizeof(StepCoef));
    w.coef_cur = take((size_t)ndom * sizeof(StepCoef));
    w.flag = take(256);
    w.nrm = take((size_t)4 * ndom * pl->ld * sizeof(double));
    w.nrm_part = take((size_t)ndom * kNormSlabs * pl->ld * sizeof(double));
    w.scl = take((size_t)ndom * pl->ld * sizeof(float));
    w.occ_eff = take((size_t)ndom * pl->ld * sizeof(float));
    w.avec = take((size_t)ndom * 3 * sizeof(double));
    w.gram = take((size_t)ndom * pl->ldp_max * pl->ldp_max * sizeof(float));
    w.rich = take((size_t)ndom * 3 * 8 * sizeof(float));
    w.total = o;
    return true;
}

extern "C" {

const char *mlmd_last_error(void) { return g_err; }

size_t mlmd_workspace_bytes(int ndom, int nx, int ny, int nz, int norb, int nproj_max, unsigned flags) {
    Plan pl;
    if (!make_plan(ndom, nx, ny, nz, norb, nproj_max, flags, &pl)) return 0;
    return pl.off.total;
}

int mlmd_domain_create(mlmd_domain_t **out, int ndom, int nx, int ny, int nz, double hx, double hy,
                       double hz, int norb, int nproj_max, void *workspace_dev, size_t workspace_bytes,
                       void *cuda_stream, unsigned flags) {
    if (!out) return fail(MLMD_ERR_ARG, "mlmd_domain_create: out is NULL");
    *out = nullptr;
    if (!workspace_dev) return fail(MLMD_ERR_ARG, "mlmd_domain_create: workspace is NULL");
    if (!(hx > 0) || !(hy > 0) || !(hz > 0)) return fail(MLMD_ERR_ARG, "mlmd_domain_create: grid spacings must be > 0");
    if (flags & ~(MLMD_KEEP_PSI0 | MLMD_CHECK_FINITE | MLMD_BORROW_PSI))
        return fail(MLMD_ERR_ARG, "mlmd_domain_create: unknown flags 0x%x", flags);
    Plan pl;
    if (!make_plan(ndom, nx, ny, nz, norb, nproj_max, flags, &pl))
        return fail(MLMD_ERR_SHAPE, "mlmd_domain_create: bad shape ndom=%d grid=%dx%dx%d norb=%d nproj_max=%d "
                    "(every grid axis must be >= 5)", ndom, nx, ny, nz, norb, nproj_max);
    if ((flags & MLMD_BORROW_PSI) && norb % 16)
        return fail(MLMD_ERR_SHAPE, "mlmd_domain_create: MLMD_BORROW_PSI needs norb %% 16 == 0 (rows of the caller's buffer are "
                    "used unpadded), got norb=%d", norb);
    if (workspace_bytes < pl.off.total)
        return fail(MLMD_ERR_SHAPE, "mlmd_domain_create: workspace has %zu bytes, needs %zu", workspace_bytes, pl.off.total);
    if (((uintptr_t)workspace_dev) % 256) return fail(MLMD_ERR_ARG, "mlmd_domain_create: workspace must be 256-byte aligned");
    int dev = -1;
    CU(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10)
        return fail(MLMD_ERR_CUDA, "mlmd_domain_create: device '%s' is sm_%d%d; this library is built for sm_100a only "
                    "and has no fallback", prop.name, prop.major, prop.minor);
    mlmd_domain *h = new (std::nothrow) mlmd_domain();
    if (!h) return fail(MLMD_ERR_NOMEM, "mlmd_domain_create: out of host memory");
    h->ndom = ndom; h->nx = nx; h->ny = ny; h->nz = nz; h->norb = norb; h->nproj_max = nproj_max;
    h->ld = pl.ld; h->ngrid = pl.ngrid;
    h->hx = hx; h->hy = hy; h->hz = hz; h->dv = hx * hy * hz;
    h->flags = flags;
    h->stream = (cudaStream_t)cuda_stream;
    h->ws = (char *)workspace_dev; h->ws_bytes = workspace_bytes; h->off = pl.off;
    h->nproj = 0; h->beta_complex = 0; h->P = 0; h->ldp = pl.ldp_max; h->prows = pl.prows; h->nsplit = pl.nsplit;
    h->nsplit_tc = pl.nsplit_tc; h->nsplit_tc_ovl = pl.nsplit_tc_ovl;
    h->tc_ok = tc_available() && pl.ngrid % 128 == 0;
    h->gemm_mode = MLMD_GEMM_FP32GRADE;
    for (int k = 0; k < MLMD_OPT_COUNT; ++k) h->opt[k] = 0;
    h->opt[MLMD_OPT_GRAPH] = 1;
    h->opt[MLMD_OPT_FD_ORDER] = 4;
    h->coef_o2 = false;
    h->psi_ptr = (flags & MLMD_BORROW_PSI) ? nullptr : (float2 *)(h->ws + pl.off.psi);
    h->have_psi = h->have_vloc = h->have_occ = false; h->field_yz = false; h->rho_valid = false;
    h->vmax = h->dmax = 0.0; h->launches = 0;
    h->coef_host = nullptr; h->flag_host = nullptr; h->prof_on = false;
    h->coef_uploaded = nullptr; h->gexec = nullptr; h->gstream = nullptr; h->gfork = h->gjoin = nullptr;
    h->g_launches = 0; h->g_dt = 0.0; h->g_yz = false; h->g_split = false;
    h->gram_valid = false; h->ldg = pl.ldp_max; h->split_pending = false;
    h->graph_allowed = true;
    cudaError_t e = cudaMallocHost((void **)&h->coef_host, (size_t)kCoefCapacity * ndom * sizeof(StepCoef));
    if (e == cudaSuccess) e = cudaMallocHost((void **)&h->flag_host, 256);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->coef_uploaded, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->occ(), 0, (size_t)ndom * h->ld * sizeof(float), h->stream);
    // rows >= P of W are read (times zero columns of beta) by the K = 8 slabs of the back-application
    if (e == cudaSuccess) e = cudaMemsetAsync(h->what(), 0, 2 * (pl.off.what_lo - pl.off.what), h->stream);
    if (e != cudaSuccess) {
        if (h->coef_host) cudaFreeHost(h->coef_host);
        if (h->flag_host) cudaFreeHost(h->flag_host);
        delete h;
        return fail(MLMD_ERR_CUDA, "mlmd_domain_create: %s", cudaGetErrorString(e));
    }
    *out = h;
    return MLMD_OK;
}

int mlmd_domain_destroy(mlmd_domain_t *h) {
    if (!h) return MLMD_OK;
    cudaStreamSynchronize(h->stream);
    if (h->coef_host) cudaFreeHost(h->coef_host);
    if (h->flag_host) cudaFreeHost(h->flag_host);
    if (h->coef_uploaded) cudaEventDestroy(h->coef_uploaded);
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    if (h->gstream) {
        cudaStreamSynchronize(h->gstream);
        cudaStreamDestroy(h->gstream);
    }
    if (h->gfork) cudaEventDestroy(h->gfork);
    if (h->gjoin) cudaEventDestroy(h->gjoin);
    for (cudaEvent_t e : h->prof_pool) cudaEventDestroy(e);
    delete h;
    return MLMD_OK;
}

int mlmd_profile(mlmd_domain_t *h, int enable) {
    if (!h) return fail(MLMD_ERR_ARG, "mlmd_profile: NULL handle");
    h->prof_on = enable != 0;
    if (enable) h->prof_recs.clear();
    return MLMD_OK;
}

int mlmd_profile_read(mlmd_domain_t *h, int kind, double *ms_total, long long *launches) {
    if (!h || !ms_total || !launches) return fail(MLMD_ERR_ARG, "mlmd_profile_read: NULL argument");
    if (kind < 0 || kind >= MLMD_K_COUNT) return fail(MLMD_ERR_ARG, "mlmd_profile_read: kind=%d", kind);
    CU(cudaStreamSynchronize(h->stream));
    double ms = 0.0;
    long long n = 0;
    for (const auto &r : h->prof_recs) {
        if (r.kind != kind) continue;
        float t = 0.f;
        CU(cudaEventElapsedTime(&t, h->prof_pool[r.e0], h->prof_pool[r.e1]));
        ms += t;
        ++n;
    }
    *ms_total = ms;
    *launches = n;
    return MLMD_OK;
}

long long mlmd_launch_count(const mlmd_domain_t *h) { return h ? h->launches : 0; }

static bool use_tensor_cores(const mlmd_domain *h) {
    return h->tc_ok && h->opt[MLMD_OPT_GEMM_PATH] == 0 && (h->gemm_mode == MLMD_GEMM_FP32GRADE || h->gemm_mode == MLMD_GEMM_TF32X1 ||
                        h->gemm_mode == MLMD_GEMM_LOWP_BF16 || h->gemm_mode == MLMD_GEMM_FP32GRADE_STAGED);
}
// products per MAC on the tensor-core path: 3 = 3xTF32, 1 = TF32x1, 0 = BF16-rounded operands x1
static int tc_nprod(const mlmd_domain *h) {
    return h->gemm_mode == MLMD_GEMM_TF32X1 ? 1 : (h->gemm_mode == MLMD_GEMM_LOWP_BF16 ? 0 : 3);
}

int mlmd_gemm_path(const mlmd_domain_t *h) { return (h && use_tensor_cores(h)) ? 1 : 0; }

static cudaMemcpyKind kind_in(int where) { return where == MLMD_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice; }
static cudaMemcpyKind kind_out(int where) { return where == MLMD_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice; }
static bool bad_where(int where) { return where != MLMD_HOST && where != MLMD_DEVICE; }

int mlmd_set_orbitals(mlmd_domain_t *h, const void *psi, const double *occ, int where) {
    if (!h || !psi) return fail(MLMD_ERR_ARG, "mlmd_set_orbitals: NULL argument");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_set_orbitals: bad where=%d", where);
    const size_t rows = (size_t)h->ndom * h->ngrid;
    if (occ) {
        std::vector<float> f((size_t)h->ndom * h->ld, 0.f);
        for (int d = 0; d < h->ndom; ++d)
            for (int n = 0; n < h->norb; ++n) {
                const double v = occ[(size_t)d * h->norb + n];
                if (!(v >= 0.0)) return fail(MLMD_ERR_ARG, "mlmd_set_orbitals: occ[%d][%d]=%g is not >= 0", d, n, v);
                f[(size_t)d * h->ld + n] = (float)v;
            }
        CU(cudaMemcpyAsync(h->occ(), f.data(), f.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
        CU(cudaStreamSynchronize(h->stream));   // f is a temporary
        h->have_occ = true;
    } else if (!h->have_occ) {
        std::vector<float> f((size_t)h->ndom * h->ld, 0.f);
        for (int d = 0; d < h->ndom; ++d)
            for (int n = 0; n < h->norb; ++n) f[(size_t)d * h->ld + n] = 2.f;
        CU(cudaMemcpyAsync(h->occ(), f.data(), f.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        h->have_occ = true;
    }
    if (h->flags & MLMD_BORROW_PSI) {
        // adopt the caller's device buffer: every step updates it in place
        if (where != MLMD_DEVICE) return fail(MLMD_ERR_ARG, "mlmd_set_orbitals: MLMD_BORROW_PSI needs a device pointer");
        if (((uintptr_t)psi) % 256) return fail(MLMD_ERR_ARG, "mlmd_set_orbitals: a borrowed Psi buffer must be 256-byte aligned");
        h->psi_ptr = (float2 *)psi;
    } else {
        if (h->ld != h->norb) CU(cudaMemsetAsync(h->psi(), 0, rows * h->ld * sizeof(float2), h->stream));
        CU(cudaMemcpy2DAsync(h->psi(), (size_t)h->ld * sizeof(float2), psi, (size_t)h->norb * sizeof(float2),
                             (size_t)h->norb * sizeof(float2), rows, kind_in(where), h->stream));
    }
    if (h->flags & MLMD_KEEP_PSI0)
        CU(cudaMemcpyAsync(h->psi0(), h->psi(), rows * h->ld * sizeof(float2), cudaMemcpyDeviceToDevice, h->stream));
    if (where == MLMD_HOST) CU(cudaStreamSynchronize(h->stream));
    h->have_psi = true;
    h->rho_valid = false;
    h->split_pending = false;   // a scale left over from a failed split call belongs to the old orbitals
    return MLMD_OK;
}

int mlmd_get_orbitals(mlmd_domain_t *h, void *psi, int where) {
    if (!h || !psi) return fail(MLMD_ERR_ARG, "mlmd_get_orbitals: NULL argument");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_get_orbitals: bad where=%d", where);
    if (!h->have_psi) return fail(MLMD_ERR_STATE, "mlmd_get_orbitals: no orbitals set");
    const size_t rows = (size_t)h->ndom * h->ngrid;
    if (psi != (void *)h->psi())    // a borrowed buffer read back into itself is already there
        CU(cudaMemcpy2DAsync(psi, (size_t)h->norb * sizeof(float2), h->psi(), (size_t)h->ld * sizeof(float2),
                             (size_t)h->norb * sizeof(float2), rows, kind_out(where), h->stream));
    if (where == MLMD_HOST) CU(cudaStreamSynchronize(h->stream));
    return MLMD_OK;
}

int mlmd_set_vloc(mlmd_domain_t *h, const float *vloc, int where) {
    if (!h || !vloc) return fail(MLMD_ERR_ARG, "mlmd_set_vloc: NULL argument");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_set_vloc: bad where=%d", where);
    const size_t n = (size_t)h->ndom * h->ngrid;
    int nl = 0;
    CU(cudaMemcpyAsync(h->vloc(), vloc, n * sizeof(float), kind_in(where), h->stream));
    CU(launch_max_abs(h->stream, h->vloc(), n, h->flag(), &nl));
    CU(cudaMemcpyAsync(h->flag_host, h->flag(), sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    CU(cudaStreamSynchronize(h->stream));
    h->launches += nl;
    float vm;
    memcpy(&vm, h->flag_host, sizeof(float));
    if (!(vm < INFINITY)) return fail(MLMD_ERR_NONFINITE, "mlmd_set_vloc: V_loc contains NaN/Inf");
    h->vmax = vm;
    h->have_vloc = true;
    return MLMD_OK;
}

// the captured step bakes in the projector count, the GEMM mode and dt: reconfiguration discards it
static void drop_graph(mlmd_domain *h) {
    if (h->gexec) {
        cudaStreamSynchronize(h->gstream);
        cudaGraphExecDestroy(h->gexec);
        h->gexec = nullptr;
    }
}

// The second beta-sized buffer holds what the current GEMM mode reads next to the FP32 projectors: the remainder
// beta - trunc_tf32(beta) (lo operand of the 3xTF32 back-application), or, in the opt-in low-precision mode, the BF16
// copy of beta (2 bytes per element) that both kind::f16 GEMMs read INSTEAD of the FP32 array.
static bool lowp_bf16_storage(const mlmd_domain *h) {
    return h->gemm_mode == MLMD_GEMM_LOWP_BF16 && h->tc_ok && h->opt[MLMD_OPT_GEMM_PATH] == 0 && (2 * h->ld) % 64 == 0;
}
static int fill_beta_companion(mlmd_domain *h) {
    if (h->nproj == 0) return MLMD_OK;
    const size_t n = (size_t)h->ndom * h->ngrid * h->ldp;
    int nl = 0;
    if (lowp_bf16_storage(h)) CU(launch_to_bf16(h->stream, h->beta(), h->beta_lo(), n, &nl));
    else CU(launch_tf32_remainder(h->stream, h->beta(), h->beta_lo(), n, &nl));
    // W changes its storage type with the mode too (FP32 hi / lo pair, or one BF16 array): rows beyond the projector
    // count must read as zeros in either view
    CU(cudaMemsetAsync(h->what(), 0, 2 * (h->off.what_lo - h->off.what), h->stream));
    h->launches += nl;
    return MLMD_OK;
}

int mlmd_set_projectors(mlmd_domain_t *h, int nproj, const void *beta, int beta_dtype, const double *D, int where) {
    if (!h) return fail(MLMD_ERR_ARG, "mlmd_set_projectors: NULL handle");
    if (nproj < 0) return fail(MLMD_ERR_ARG, "mlmd_set_projectors: nproj=%d", nproj);
    drop_graph(h);
    h->gram_valid = false;
    if (nproj == 0) {
        h->nproj = h->P = 0;
        h->dmax = 0.0;
        return MLMD_OK;
    }
    if (!beta || !D) return fail(MLMD_ERR_ARG, "mlmd_set_projectors: NULL beta or D");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_set_projectors: bad where=%d", where);
    if (beta_dtype != MLMD_BETA_REAL32 && beta_dtype != MLMD_BETA_COMPLEX64)
        return fail(MLMD_ERR_ARG, "mlmd_set_projectors: bad beta_dtype=%d", beta_dtype);
    const int cplx = beta_dtype == MLMD_BETA_COMPLEX64;
    const int P = cplx ? 2 * nproj : nproj;
    if (P > h->nproj_max)
        return fail(MLMD_ERR_SHAPE, "mlmd_set_projectors: %d %s projectors need %d real rows, handle was created with "
                    "nproj_max=%d", nproj, cplx ? "complex" : "real", P, h->nproj_max);
    const size_t rows = (size_t)h->ndom * h->ngrid;
    const int ldp = round_up_i(P, 8);
    std::vector<float> dp((size_t)h->ndom * nproj);
    double dmax = 0.0;
    for (size_t i = 0; i < dp.size(); ++i) {
        if (!std::isfinite(D[i])) return fail(MLMD_ERR_NONFINITE, "mlmd_set_projectors: D[%zu] is not finite", i);
        dp[i] = (float)(D[i] * h->dv);
        dmax = std::max(dmax, fabs(D[i]));
    }
    CU(cudaMemcpyAsync(h->dprime(), dp.data(), dp.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
    if (ldp != P) CU(cudaMemsetAsync(h->beta(), 0, rows * ldp * sizeof(float), h->stream));
    CU(cudaMemcpy2DAsync(h->beta(), (size_t)ldp * sizeof(float), beta, (size_t)P * sizeof(float), (size_t)P * sizeof(float),
                         rows, kind_in(where), h->stream));
    // rows [P, ldp) of W are read (times zero columns of beta) by the K = 8 slabs of the back-application: a stale NaN
    // left there by an earlier projector set or a diverged run would poison psi
    CU(cudaMemsetAsync(h->what(), 0, 2 * (h->off.what_lo - h->off.what), h->stream));
    h->nproj = nproj; h->beta_complex = cplx; h->P = P; h->ldp = ldp; h->dmax = dmax;
    int rc = fill_beta_companion(h);
    if (rc) return rc;
    CU(cudaStreamSynchronize(h->stream));   // dp is a temporary; host beta may be reused by the caller
    return MLMD_OK;
}

int mlmd_set_gemm_mode(mlmd_domain_t *h, int mode) {
    if (!h) return fail(MLMD_ERR_ARG, "mlmd_set_gemm_mode: NULL handle");
    drop_graph(h);
    if (mode < MLMD_GEMM_FP32GRADE || mode > MLMD_GEMM_FP32GRADE_STAGED) return fail(MLMD_ERR_ARG, "mlmd_set_gemm_mode: bad mode %d", mode);
    const bool was16 = lowp_bf16_storage(h);
    h->gemm_mode = mode;
    if (was16 != lowp_bf16_storage(h)) return fill_beta_companion(h);
    return MLMD_OK;
}

int mlmd_set_option(mlmd_domain_t *h, int key, int value) {
    if (!h) return fail(MLMD_ERR_ARG, "mlmd_set_option: NULL handle");
    static const int nvalues[MLMD_OPT_COUNT] = {2, 3, 2, 2, 0, 2};
    if (key < 0 || key >= MLMD_OPT_COUNT) return fail(MLMD_ERR_ARG, "mlmd_set_option: unknown key %d", key);
    if (key == MLMD_OPT_FD_ORDER) {
        if (value != 2 && value != 4) return fail(MLMD_ERR_ARG, "mlmd_set_option: MLMD_OPT_FD_ORDER takes 2 or 4, got %d", value);
    } else if (value < 0 || value >= nvalues[key]) {
        return fail(MLMD_ERR_ARG, "mlmd_set_option: key %d takes 0..%d, got %d", key, nvalues[key] - 1, value);
    }
    drop_graph(h);      // a captured step bakes the kernel choice in
    const bool was16 = lowp_bf16_storage(h);
    h->opt[key] = value;
    if (was16 != lowp_bf16_storage(h)) return fill_beta_companion(h);
    return MLMD_OK;
}

int mlmd_occupations(mlmd_domain_t *h, double *f, double *n_exc, int where) {
    if (!h || !f || !n_exc) return fail(MLMD_ERR_ARG, "mlmd_occupations: NULL argument");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_occupations: bad where=%d", where);
    // S = dv Psi(0)^H Psi(t) into the Z scratch (argument checks as mlmd_overlap(which = 1))
    int rc = mlmd_overlap(h, 1, h->z(), MLMD_DEVICE);
    if (rc) return rc;
    int nl = 0;
    double *fd = where == MLMD_DEVICE ? f : h->nrm(1);
    double *nd = where == MLMD_DEVICE ? n_exc : h->nrm(2);
    CU(launch_occupations(h->stream, h->ndom, h->norb, h->ld, (const float2 *)h->z(), h->occ(), fd, nd, &nl));
    h->launches += nl;
    if (where == MLMD_HOST) {
        CU(cudaMemcpyAsync(f, fd, (size_t)h->ndom * h->norb * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaMemcpyAsync(n_exc, nd, (size_t)h->ndom * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    return MLMD_OK;
}

int mlmd_energy_nl(mlmd_domain_t *h, double *E, int where) {
    if (!h || !E) return fail(MLMD_ERR_ARG, "mlmd_energy_nl: NULL argument");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_energy_nl: bad where=%d", where);
    if (!h->have_psi) return fail(MLMD_ERR_STATE, "mlmd_energy_nl: no orbitals set");
    double *ed = where == MLMD_DEVICE ? E : h->nrm(3);
    int nl = 0;
    if (h->nproj == 0) {
        CU(cudaMemsetAsync(ed, 0, (size_t)h->ndom * sizeof(double), h->stream));
    } else {
        // the projection GEMM of the hot path (S2a), then a reduction instead of the scaling step
        const bool fp64 = h->gemm_mode == MLMD_GEMM_FP64;
        const bool tc = use_tensor_cores(h);
        const int nsplit = tc ? h->nsplit_tc : h->nsplit;
        if (tc)
            CU(launch_proj_tc(h->stream, h->ndom, h->ngrid, h->beta(), nullptr, h->ldp, h->P, (const float *)h->psi(),
                              2 * h->ld, 2 * h->ld, h->zpart(), h->prows, nsplit, tc_nprod(h), proj_chain(tc_nprod(h)), &nl, &h->tmaps));
        else
            CU(launch_proj_simt(h->stream, h->ndom, h->ngrid, h->beta(), nullptr, h->ldp, h->P, (const float *)h->psi(),
                                2 * h->ld, 2 * h->ld, h->zpart(), h->prows, nsplit, fp64, &nl));
        CU(launch_energy_nl(h->stream, h->ndom, h->nproj, h->beta_complex, h->ld, h->prows, nsplit, h->zpart(), h->dprime(),
                            h->occ(), h->dv, ed, &nl));
    }
    h->launches += nl;
    if (where == MLMD_HOST) {
        CU(cudaMemcpyAsync(E, ed, (size_t)h->ndom * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    return MLMD_OK;
}

int mlmd_current(mlmd_domain_t *h, const double *A, int a_ndom, double *J, int where) {
    if (!h || !A || !J) return fail(MLMD_ERR_ARG, "mlmd_current: NULL argument");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_current: bad where=%d", where);
    if (a_ndom != 1 && a_ndom != h->ndom) return fail(MLMD_ERR_ARG, "mlmd_current: a_ndom=%d must be 1 or ndom=%d", a_ndom, h->ndom);
    if (!h->have_psi) return fail(MLMD_ERR_STATE, "mlmd_current: no orbitals set");
    for (int i = 0; i < 3 * a_ndom; ++i)
        if (!std::isfinite(A[i])) return fail(MLMD_ERR_NONFINITE, "mlmd_current: A[%d] is not finite", i);
    // A goes through the pinned coefficient staging buffer (one StepCoef slot per domain is large enough)
    static_assert(sizeof(StepCoef) >= 3 * sizeof(double), "staging slot holds one field vector");
    CU(cudaEventSynchronize(h->coef_uploaded));
    double *a_host = (double *)h->coef_host;
    memcpy(a_host, A, (size_t)3 * a_ndom * sizeof(double));
    double *a_dev = h->avec();
    CU(cudaMemcpyAsync(a_dev, a_host, (size_t)3 * a_ndom * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CU(cudaEventRecord(h->coef_uploaded, h->stream));
    double *jd = where == MLMD_DEVICE ? J : h->nrm(3);
    int nl = 0;
    CU(launch_current(h->stream, h->ndom, h->nx, h->ny, h->nz, h->hx, h->hy, h->hz, h->ld, h->psi(), h->occ(), a_dev, a_ndom,
                      h->nrm_part(), (size_t)h->ndom * kNormSlabs * h->ld, jd, h->opt[MLMD_OPT_FD_ORDER], &nl));
    h->launches += nl;
    if (where == MLMD_HOST) {
        CU(cudaMemcpyAsync(J, jd, (size_t)h->ndom * 3 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    return MLMD_OK;
}

int mlmd_current_nl(mlmd_domain_t *h, const void *rbeta, int where_rbeta, double *J, int where) {
    if (!h || !J) return fail(MLMD_ERR_ARG, "mlmd_current_nl: NULL argument");
    if (bad_where(where) || bad_where(where_rbeta)) return fail(MLMD_ERR_ARG, "mlmd_current_nl: bad where");
    if (!h->have_psi) return fail(MLMD_ERR_STATE, "mlmd_current_nl: no orbitals set");
    double *jd = where == MLMD_DEVICE ? J : h->nrm(3);
    int nl = 0;
    if (h->nproj == 0) {
        CU(cudaMemsetAsync(jd, 0, (size_t)h->ndom * 3 * sizeof(double), h->stream));
    } else {
        if (!rbeta) return fail(MLMD_ERR_ARG, "mlmd_current_nl: rbeta is NULL");
        // scratch for one direction of rbeta in the layout of beta: the two Horner work buffers (free between steps)
        const size_t rows = (size_t)h->ndom * h->ngrid;
        const size_t need = rows * h->ldp * sizeof(float) + 256, have = h->off.psi0 - h->off.ua;
        // the complex coefficient matrices C, G live in the Z / W scratch ([ndom][nproj][ld] float2 each)
        if (need > have || (size_t)h->nproj * h->ld * sizeof(float2) > (size_t)h->prows * 2 * h->ld * sizeof(float))
            return fail(MLMD_ERR_SHAPE, "mlmd_current_nl: %d projector rows need %zu bytes of staging, the work buffers hold %zu",
                        h->P, need, have);
        float *stage = (float *)h->ua();
        float2 *cmat = (float2 *)h->z(), *gmat = (float2 *)h->what();
        const bool fp64 = h->gemm_mode == MLMD_GEMM_FP64;
        // always FP32-grade (3xTF32 on tensor cores, or the CUDA-core path): it is a measurement
        const bool tc = h->tc_ok && h->opt[MLMD_OPT_GEMM_PATH] == 0 && h->gemm_mode != MLMD_GEMM_FP64 && h->gemm_mode != MLMD_GEMM_FP32_SIMT;
        const int nsplit = tc ? h->nsplit_tc : h->nsplit;
        auto project = [&](const float *B, float2 *out) -> int {
            if (tc)
                CU(launch_proj_tc(h->stream, h->ndom, h->ngrid, B, nullptr, h->ldp, h->P, (const float *)h->psi(), 2 * h->ld, 2 * h->ld,
                                  h->zpart(), h->prows, nsplit, 3, kProjChain, &nl, &h->tmaps));
            else
                CU(launch_proj_simt(h->stream, h->ndom, h->ngrid, B, nullptr, h->ldp, h->P, (const float *)h->psi(), 2 * h->ld, 2 * h->ld,
                                    h->zpart(), h->prows, nsplit, fp64, &nl));
            CU(launch_proj_coeff(h->stream, h->ndom, h->nproj, h->beta_complex, h->ld, h->prows, nsplit, h->zpart(), out, &nl));
            return MLMD_OK;
        };
        int rc = project(h->beta(), cmat);
        if (rc) return rc;
        const size_t elem = h->beta_complex ? sizeof(float2) : sizeof(float);
        for (int d = 0; d < 3; ++d) {
            const char *src = (const char *)rbeta + (size_t)d * rows * h->nproj * elem;
            if (h->ldp != h->P) CU(cudaMemsetAsync(stage, 0, rows * h->ldp * sizeof(float), h->stream));
            CU(cudaMemcpy2DAsync(stage, (size_t)h->ldp * sizeof(float), src, (size_t)h->P * sizeof(float), (size_t)h->P * sizeof(float),
                                 rows, kind_in(where_rbeta), h->stream));
            rc = project(stage, gmat);
            if (rc) return rc;
            CU(launch_current_nl(h->stream, h->ndom, h->nproj, h->ld, cmat, gmat, h->dprime(), h->occ(), h->dv, d, jd, &nl));
        }
        // the W scratch held G: rows of W beyond the projector count must be zero again for the back-application
        CU(cudaMemsetAsync(h->what(), 0, 2 * (h->off.what_lo - h->off.what), h->stream));
    }
    h->launches += nl;
    if (where == MLMD_HOST) {
        CU(cudaMemcpyAsync(J, jd, (size_t)h->ndom * 3 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    } else if (where_rbeta == MLMD_HOST) {
        CU(cudaStreamSynchronize(h->stream));   // the caller may reuse its host rbeta
    }
    return MLMD_OK;
}

// ---- the step --------------------------------------------------------------------------------
// RAII pair of events around one kernel launch when mlmd_profile is on.
struct ProfScope {
    mlmd_domain *h;
    int rec;
    ProfScope(mlmd_domain *hh, int kind) : h(hh), rec(-1) {
        if (!h->prof_on || h->prof_recs.size() >= (1u << 16)) return;
        const size_t need = 2 * (h->prof_recs.size() + 1);
        while (h->prof_pool.size() < need) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return;
            h->prof_pool.push_back(e);
        }
        rec = (int)h->prof_recs.size();
        h->prof_recs.push_back({kind, 2 * rec, 2 * rec + 1});
        cudaEventRecord(h->prof_pool[2 * rec], h->stream);
    }
    ~ProfScope() {
        if (rec >= 0) cudaEventRecord(h->prof_pool[2 * rec + 1], h->stream);
    }
};

static void fill_coef(const mlmd_domain *h, const double *A3, StepCoef *c) {
    // SURVEY.md 8(a) S1; weights of the 4th-order central differences (north_star), or of the paper's own 2nd-order
    // 7-point star (MLMD_OPT_FD_ORDER = 2) written on the same offsets with zero j = 2 weights
    static const double c2_o4[2] = {4.0 / 3.0, -1.0 / 12.0}, c1_o4[2] = {2.0 / 3.0, -1.0 / 12.0};   // j = 1, 2
    static const double c2_o2[2] = {1.0, 0.0}, c1_o2[2] = {0.5, 0.0};
    const bool o2 = h->opt[MLMD_OPT_FD_ORDER] == 2 || h->coef_o2;
    const double *c2 = o2 ? c2_o2 : c2_o4, *c1 = o2 ? c1_o2 : c1_o4;
    const double c2_0 = o2 ? -2.0 : -5.0 / 2.0;
    const double hh[3] = {h->hx, h->hy, h->hz};
    double centre = 0.5 * (A3[0] * A3[0] + A3[1] * A3[1] + A3[2] * A3[2]);
    for (int d = 0; d < 3; ++d) {
        centre += -0.5 * c2_0 / (hh[d] * hh[d]);
        for (int j = 0; j < 2; ++j) {
            c->p[d][j] = (float)(-0.5 * c2[j] / (hh[d] * hh[d]));
            c->q[d][j] = (float)(A3[d] * c1[j] / hh[d]);
        }
    }
    c->centre = (float)centre;
    c->pad = 0.f;
}

// The step's first projection reads every psi row exactly once: on the CTA-pair kernel it can carry the density of
// that state (S3) in its converter warps, so the separate 8 B/element pass over psi runs only once per call.
static bool density_rides_on_projection(const mlmd_domain *h) {
    // (the staged mode's first projection of a step takes one product of rounded operands: it carries the density too)
    // and so does the low-precision mode's BF16 kernel (it sums the FP32 values it packs)
    return h->nproj > 0 && use_tensor_cores(h) &&
           (h->gemm_mode == MLMD_GEMM_FP32GRADE || h->gemm_mode == MLMD_GEMM_FP32GRADE_STAGED || lowp_bf16_storage(h)) &&
           proj_tc_can_fuse_density(h->P, 2 * h->ld, 3);
}

static int nonlocal_project(mlmd_domain *h, const float2 *w, float tau, int *nl, int nprod = -1, int chain = -1,
                            bool with_density = false, const float *density_occ = nullptr) {
    // S2a + S2b: What = (-i tau) D' (beta^H w); nprod >= 0 overrides the mode's products per MAC (staged mode)
    if (nprod < 0) nprod = tc_nprod(h);
    const bool fp64 = h->gemm_mode == MLMD_GEMM_FP64;
    const bool tc = use_tensor_cores(h);
    const int nsplit = tc ? h->nsplit_tc : h->nsplit;
    {
        ProfScope ps(h, MLMD_K_PROJ);
        if (tc)
            CU(launch_proj_tc(h->stream, h->ndom, h->ngrid, h->beta(), nullptr, h->ldp, h->P, (const float *)w,
                              2 * h->ld, 2 * h->ld, h->zpart(), h->prows, nsplit, nprod, chain > 0 ? chain : proj_chain(nprod), nl, &h->tmaps,
                              with_density ? h->rho() : nullptr, density_occ ? density_occ : h->occ(),
                              lowp_bf16_storage(h) ? h->beta_lo() : nullptr));
        else
            CU(launch_proj_simt(h->stream, h->ndom, h->ngrid, h->beta(), nullptr, h->ldp, h->P, (const float *)w,
                                2 * h->ld, 2 * h->ld, h->zpart(), h->prows, nsplit, fp64, nl));
    }
    ProfScope ps(h, MLMD_K_GLUE);
    CU(launch_reduce_scale(h->stream, h->ndom, h->nproj, h->beta_complex, h->ld, h->prows, nsplit, h->zpart(),
                           h->dprime(), tau, h->what(), h->what_lo(),
                           (tc && h->gemm_mode == MLMD_GEMM_LOWP_BF16) ? (lowp_bf16_storage(h) ? 2 : 1) : 0, nl));
    return MLMD_OK;
}

static int nonlocal_back(mlmd_domain *h, float2 *out, int *nl, int nprod = -1) {
    if (nprod < 0) nprod = tc_nprod(h);
    const bool fp64 = h->gemm_mode == MLMD_GEMM_FP64;
    ProfScope ps(h, MLMD_K_BACK);
    if (use_tensor_cores(h))
        CU(launch_back_tc(h->stream, h->ndom, h->ngrid, h->beta(), lowp_bf16_storage(h) ? nullptr : h->beta_lo(), h->ldp, h->P,
                          h->what(), h->what_lo(), (float *)out, 2 * h->ld, 2 * h->ld, h->prows, nprod, nl, &h->tmaps,
                          lowp_bf16_storage(h) ? h->beta_lo() : nullptr, lowp_bf16_storage(h) ? h->what() : nullptr));
    else
        CU(launch_back_simt(h->stream, h->ndom, h->ngrid, h->beta(), nullptr, h->ldp, h->P, h->what(), h->what_lo(),
                            (float *)out, 2 * h->ld, 2 * h->ld, h->prows, fp64, nl));
    return MLMD_OK;
}

// One Taylor-4 time step on h->stream: four Horner stages (projection, glue, fused stencil pass,
// back-application) and the density.  coef: this step's device coefficients [ndom];
// coef_host: the same set on the host when it is identical for all domains (constant-bank path), else NULL.
// last: the final step of a call.  Every step ends with rho of its result (north_star); when the density can ride on a
// projection, the rho of step n is formed by the FIRST projection of step n + 1 (which reads that state anyway) and
// only the last step of a call runs the separate density pass.
static int enqueue_step(mlmd_domain *h, const StepCoef *coef, const StepCoef *coef_host, double dt, bool last, int *nl) {
    const bool fused_rho = density_rides_on_projection(h);
    // Horner form of sum_{m<=4} (-i dt H)^m/m!: w4 = psi, w_{k-1} = psi + (-i dt/k) H w_k
    const float2 *src[4] = {h->psi(), h->ua(), h->ub(), h->ua()};
    float2 *dst[4] = {h->ua(), h->ub(), h->ua(), h->psi()};
    // MLMD_GEMM_FP32GRADE_STAGED: the V_NL term of Horner stage i reaches the result through
    // 3 - i further applications of (dt/k) H, so the three inner stages take a single product of nearest-rounded
    // TF32 operands in the projection and beta_hi + beta_lo times a single-TF32 W in the back-application; the
    // outermost stage (weight dt) stays 3xTF32.
    const bool staged = h->gemm_mode == MLMD_GEMM_FP32GRADE_STAGED && use_tensor_cores(h);
    for (int i = 0; i < 4; ++i) {
        const float tau = (float)(dt / (4 - i));
        const bool reduced = staged && ((kStagedMask >> i) & 1);
        if (h->nproj > 0) {
            // inner stages: their accumulation drift is damped like every other projection error (weights <= dt/2 E
            // ~ 0.05 of the outer stage's), so the chains are 1024 stages: one or two drains per K slice instead of one per 128 stages
            // the three inner stages of every tensor-core mode take the long chains (the products stay as the mode says)
            int rc = nonlocal_project(h, src[i], tau, nl, reduced ? kStagedProjNprod : -1, i < 3 ? kInnerChain : -1,
                                      fused_rho && i == 0);
            if (rc) return rc;
        }
        {
            ProfScope ps(h, MLMD_K_STENCIL);
            CU(launch_stencil_stage(h, src[i], h->psi(), dst[i], coef, coef_host, tau, nl));
        }
        if (h->nproj > 0) {
            int rc = nonlocal_back(h, dst[i], nl, reduced ? 2 : -1);
            if (rc) return rc;
        }
    }
    if (fused_rho && !last) return MLMD_OK;
    ProfScope ps(h, MLMD_K_DENSITY);
    CU(launch_density(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->occ(), h->rho(), nl));
    return MLMD_OK;
}

static int enqueue_split_step(mlmd_domain *h, const StepCoef *coef, const StepCoef *coef_host, double dt, bool last, int *nl);

// Capture one step (coefficients taken from the device slot that advance_coef refills) into h->gexec.
static int capture_step(mlmd_domain *h, double dt, bool yz, bool split) {
    if (!h->gstream) {
        CU(cudaStreamCreateWithFlags(&h->gstream, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&h->gfork, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&h->gjoin, cudaEventDisableTiming));
    }
    cudaStream_t user = h->stream;
    cudaGraph_t graph = nullptr;
    int nl = 0;
    CU(cudaStreamBeginCapture(h->gstream, cudaStreamCaptureModeThreadLocal));
    h->stream = h->gstream;
    cudaError_t e = launch_advance_coef(h->gstream, h->coef(), h->coef_cur(), h->step_counter(), h->ndom, &nl);
    int rc = e != cudaSuccess ? MLMD_ERR_CUDA
             : split ? enqueue_split_step(h, h->coef_cur(), nullptr, dt, false, &nl) : enqueue_step(h, h->coef_cur(), nullptr, dt, false, &nl);
    h->stream = user;
    cudaError_t e2 = cudaStreamEndCapture(h->gstream, &graph);
    if (rc || e != cudaSuccess || e2 != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        h->graph_allowed = false;      // fall back to eager launches for the life of the handle
        return MLMD_OK;
    }
    e = cudaGraphInstantiate(&h->gexec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) {
        h->gexec = nullptr;
        cudaGetLastError();
        h->graph_allowed = false;
        return MLMD_OK;
    }
    h->g_launches = nl;
    h->g_dt = dt;
    h->g_yz = yz;
    h->g_split = split;
    return MLMD_OK;
}

// One step of the paper's literal Eq. (2) (readings D27, D28): normalised first-order
// nonlocal half-kick, Taylor-4 of h_loc alone, half-kick.  The chain runs un-normalised (a per-orbital scale
// commutes with every operator in it); the four squared norms give the two kick scales, which are applied in
// the pass that also computes the density.
static int enqueue_split_step(mlmd_domain *h, const StepCoef *coef, const StepCoef *coef_host, double dt, bool last, int *nl) {
    const bool kicks = h->nproj > 0;
    auto norm2 = [&](int which) -> int {
        ProfScope ps(h, MLMD_K_NORM);
        CU(launch_colnorm2(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->nrm_part(), h->nrm(which), nl));
        return MLMD_OK;
    };
    auto half_kick = [&](int which) -> int {     // psi += (-i dt/2) V_NL psi, then its squared norms -> nrm(which)
        int rc = nonlocal_project(h, h->psi(), (float)(0.5 * dt), nl);
        if (!rc) rc = nonlocal_back(h, h->psi(), nl);
        return rc ? rc : norm2(which);
    };
    // S3 inside a call: the density of the state a step starts from (= the result of the previous step: psi in memory
    // times the pending scale, i.e. occupations occ_eff = f scl^2) rides on the first kick's projection, which reads that
    // state anyway (reading R4, as in the Taylor step); the separate density pass runs for other shapes / modes only
    const bool fused_rho = kicks && density_rides_on_projection(h);
    auto kick_only = [&]() -> int {              // psi += (-i dt/2) V_NL psi
        int rc = nonlocal_project(h, h->psi(), (float)(0.5 * dt), nl, -1, -1, fused_rho, h->occ_eff());
        return rc ? rc : nonlocal_back(h, h->psi(), nl);
    };
    const bool rich = h->opt[MLMD_OPT_LOCAL_SOLVER] == 1;
    // split-operator solver: ||psi_a||^2 after the first kick from the identity the second kick uses (below), with the
    // squared norms of the state in memory at the start of the step, which nrm(3) holds (the previous step's ||psi_d||^2,
    // or the incoming norms at the start of a call)
    const bool quad_a = kicks && rich && h->gram_valid;
    if (quad_a) {
        int rc = nonlocal_project(h, h->psi(), (float)(0.5 * dt), nl, -1, -1, fused_rho, h->occ_eff());
        if (rc) return rc;
        {
            ProfScope ps(h, MLMD_K_GLUE);
            CU(launch_kick_quad(h->stream, h->ndom, h->P, h->ldg, h->ld, h->prows, h->gram(), h->what(), h->what_lo(), h->nrm(3),
                                h->nrm(1), nl));
        }
        rc = nonlocal_back(h, h->psi(), nl);
        if (rc) return rc;
    } else if (kicks) {
        int rc = kick_only();
        if (rc) return rc;
    }
    if (rich) {
        // the paper's own local solver (reading D33): three in-place passes of 2 x 2 nearest-neighbour rotations.  The
        // squared norms the kicks' normalisation needs (reading D27): before the solver by the norm pass; after it they are
        // the same numbers, because U_loc is unitary by construction (exactly so in exact arithmetic; here the passes' FP32 rounding
        // moves a norm by ~1e-7, and handing the second kick the norm BEFORE the solver takes that noise out again).
        // With the projector Gram matrix at hand (quad_a) the norm before the solver needs no pass over psi either
        if (kicks && !quad_a) {
            int rc = norm2(1);
            if (rc) return rc;
        }
        {
            ProfScope ps(h, MLMD_K_STENCIL);
            CU(launch_richardson(h, h->psi(), coef, dt, nl));
        }
        if (kicks)
            CU(cudaMemcpyAsync(h->nrm(2), h->nrm(1), (size_t)h->ndom * h->ld * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    } else {
    // Taylor-4 of h_loc (Horner form).  With kicks, the first stage also sums |psi_a|^2 (its input) and the last
    // |psi_c|^2 (its output) per orbital: the norms ride on passes that read or write those arrays anyway.
    const float2 *src[4] = {h->psi(), h->ua(), h->ub(), h->ua()};
    float2 *dst[4] = {h->ua(), h->ub(), h->ua(), h->psi()};
    for (int i = 0; i < 4; ++i) {
        ProfScope ps(h, MLMD_K_STENCIL);
        const float tau = (float)(dt / (4 - i));
        if (kicks && (i == 0 || i == 3))
            CU(launch_stencil_stage_norm(h, src[i], h->psi(), dst[i], coef, coef_host, tau, i == 0 ? 1 : 2, h->nrm_part(),
                                         h->nrm(i == 0 ? 1 : 2), nl));
        else
            CU(launch_stencil_stage(h, src[i], h->psi(), dst[i], coef, coef_host, tau, nl));
    }
    }
    if (!kicks) {
        ProfScope ps(h, MLMD_K_DENSITY);
        CU(launch_density(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->occ(), h->rho(), nl));
        return MLMD_OK;
    }
    int rc;
    if (h->gram_valid) {
        // ||psi_c + beta W||^2 = ||psi_c||^2 + W^T (beta^T beta) W: no pass over psi for the norm after the second kick
        rc = nonlocal_project(h, h->psi(), (float)(0.5 * dt), nl);
        if (!rc) {
            ProfScope ps(h, MLMD_K_GLUE);
            CU(launch_kick_quad(h->stream, h->ndom, h->P, h->ldg, h->ld, h->prows, h->gram(), h->what(), h->what_lo(), h->nrm(2),
                                h->nrm(3), nl));
        }
        if (!rc) rc = nonlocal_back(h, h->psi(), nl);
    } else {
        rc = half_kick(3);
    }
    if (rc) return rc;
    {
        ProfScope ps(h, MLMD_K_GLUE);
        CU(launch_kick_scale(h->stream, h->ndom * h->ld, h->nrm(0), h->nrm(1), h->nrm(2), h->nrm(3), h->scl(), nl));
    }
    if (last) {
        ProfScope ps(h, MLMD_K_DENSITY);
        CU(launch_scale_density(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->scl(), h->occ(), h->rho(), nl));
        h->split_pending = false;
        return MLMD_OK;
    }
    // Not the last step of the call: psi stays un-normalised in memory (the next step's scale is expressed through the
    // carried true norms nrm(0), so nothing accumulates) and the density takes the scale through the occupations.
    {
        ProfScope ps(h, MLMD_K_GLUE);
        CU(launch_occ_eff(h->stream, h->ndom * h->ld, h->occ(), h->scl(), h->occ_eff(), nl));
    }
    h->split_pending = true;
    if (fused_rho) return MLMD_OK;      // the next step's first projection forms this step's rho; a call ends on a flush
    ProfScope ps(h, MLMD_K_DENSITY);
    CU(launch_density(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->occ_eff(), h->rho(), nl));
    return MLMD_OK;
}

// psi <- scl * psi (and rho from the scaled values) when a call ended on a deferred scale
static int flush_split_scale(mlmd_domain *h, int *nl) {
    if (!h->split_pending) return MLMD_OK;
    ProfScope ps(h, MLMD_K_DENSITY);
    CU(launch_scale_density(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->scl(), h->occ(), h->rho(), nl));
    h->split_pending = false;
    return MLMD_OK;
}

// Shared driver of mlmd_propagate (split = false) and mlmd_propagate_split (split = true).
static int propagate_impl(mlmd_domain_t *h, int nsteps, double dt, const double *A, int a_ndom, bool split) {
    const char *fn = split ? "mlmd_propagate_split" : "mlmd_propagate";
    if (!h) return fail(MLMD_ERR_ARG, "%s: NULL handle", fn);
    if (nsteps < 0 || !(dt == dt) || std::isinf(dt)) return fail(MLMD_ERR_ARG, "%s: nsteps=%d dt=%g", fn, nsteps, dt);
    if (nsteps > 0 && !A) return fail(MLMD_ERR_ARG, "%s: A is NULL", fn);
    if (a_ndom != 1 && a_ndom != h->ndom) return fail(MLMD_ERR_ARG, "%s: a_ndom=%d must be 1 or ndom=%d", fn, a_ndom, h->ndom);
    if (!h->have_psi || !h->have_vloc) return fail(MLMD_ERR_STATE, "%s: call mlmd_set_orbitals and mlmd_set_vloc first", fn);
    // a-priori stability bound of Taylor-4 (reading D14): dt * |lambda|max(H) <= 2 sqrt(2); in the split step the
    // Taylor sum acts on h_loc only and the normalised kick is stable for any dt |D|
    // the paper's own local solver (MLMD_OPT_LOCAL_SOLVER = 1, reading D33) works on the 2nd-order operator whatever
    // MLMD_OPT_FD_ORDER says, pairs neighbouring points on every periodic axis and is unitary for any dt
    const bool rich = split && h->opt[MLMD_OPT_LOCAL_SOLVER] == 1;
    if (rich && !richardson_supported(h))
        return fail(MLMD_ERR_SHAPE, "%s: the split-operator local solver needs even nx, ny, nz (<= 256 each), got %d x %d x %d", fn,
                    h->nx, h->ny, h->nz);
    h->coef_o2 = rich;
    bool yz = false;
    double bound = 0.0;
    for (size_t i = 0; i < (size_t)nsteps * a_ndom; ++i) {
        const double *a = A + 3 * i;
        if (!std::isfinite(a[0]) || !std::isfinite(a[1]) || !std::isfinite(a[2]))
            return fail(MLMD_ERR_NONFINITE, "%s: A[%zu] is not finite", fn, i);
        yz = yz || a[1] != 0.0 || a[2] != 0.0;
        // maxima of the D2 / D1 symbols: 16/3 and 1.3722 (4th order), 4 and 1 (2nd order)
        const bool o2 = h->opt[MLMD_OPT_FD_ORDER] == 2;
        const double b = (o2 ? 2.0 : 8.0 / 3.0) * (1 / (h->hx * h->hx) + 1 / (h->hy * h->hy) + 1 / (h->hz * h->hz)) +
                         (o2 ? 1.0 : 1.3722) * (fabs(a[0]) / h->hx + fabs(a[1]) / h->hy + fabs(a[2]) / h->hz) +
                         0.5 * (a[0] * a[0] + a[1] * a[1] + a[2] * a[2]) + h->vmax + (h->nproj && !split ? h->dmax : 0.0);
        bound = std::max(bound, rich ? 0.0 : b);
    }
    h->field_yz = yz;
    int nl = 0;
    bool rho_flush = false;
    // Small problems are launch-bound (17 launches per step): after one eager step the step is captured
    // into a CUDA graph that reads its stencil coefficients from a device slot.
    const bool want_graph = h->graph_allowed && h->opt[MLMD_OPT_GRAPH] && !h->prof_on && nsteps >= 4 &&
                            (double)h->ndom * (double)h->ngrid * h->ld <= (double)(1 << 23);
    if (h->gexec && (h->g_dt != dt || h->g_yz != yz || h->g_split != split)) drop_graph(h);
    auto one_step = [&](const StepCoef *coef, const StepCoef *coef_host, bool last) {
        return split ? enqueue_split_step(h, coef, coef_host, dt, last, &nl) : enqueue_step(h, coef, coef_host, dt, last, &nl);
    };
    {
        int rc = flush_split_scale(h, &nl);      // only after a split call that failed half-way
        if (rc) return rc;
    }
    if (h->opt[MLMD_OPT_KICK_NORM]) h->gram_valid = false;
    if (split && nsteps > 0 && h->nproj > 0 && !h->gram_valid && h->ldp <= 2 * h->ld && h->P <= 1024 &&
        !h->opt[MLMD_OPT_KICK_NORM]) {
        // one-time per projector set: G = beta^T beta by a CUDA-core projection of beta onto itself (exact FP32 products;
        // the zpart scratch holds [prows][ldp] partials per slice, ldp <= 2 ld)
        ProfScope ps(h, MLMD_K_GLUE);
        CU(launch_proj_simt(h->stream, h->ndom, h->ngrid, h->beta(), nullptr, h->ldp, h->P, h->beta(), h->ldp, h->ldp, h->zpart(),
                            h->prows, h->nsplit, false, &nl));
        CU(launch_gram_reduce(h->stream, h->ndom, h->P, h->ldg, h->prows, h->ldp, h->nsplit, h->zpart(), h->gram(), 0, &nl));
        h->gram_valid = true;
    }
    if (split && nsteps > 0 && h->nproj > 0) {      // squared norms of the incoming orbitals (reading D27)
        ProfScope ps(h, MLMD_K_NORM);
        CU(launch_colnorm2(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->nrm_part(), h->nrm(0), &nl));
        // the incoming state carries no pending scale: its density (riding on the first kick's projection) takes occ itself
        CU(cudaMemcpyAsync(h->occ_eff(), h->occ(), (size_t)h->ndom * h->ld * sizeof(float), cudaMemcpyDeviceToDevice, h->stream));
        // nrm(3) = squared norms of the state in memory at the start of a step (enqueue_split_step, quad_a)
        CU(cudaMemcpyAsync(h->nrm(3), h->nrm(0), (size_t)h->ndom * h->ld * sizeof(double), cudaMemcpyDeviceToDevice, h->stream));
    }
    CU(cudaEventSynchronize(h->coef_uploaded));   // an earlier call's upload has left the pinned staging buffer
    for (int s0 = 0; s0 < nsteps; s0 += kCoefCapacity) {
        const int ns = std::min(kCoefCapacity, nsteps - s0);
        if (s0 > 0) CU(cudaStreamSynchronize(h->stream));   // the pinned staging buffer is reused
        for (int s = 0; s < ns; ++s)
            for (int d = 0; d < h->ndom; ++d)
                fill_coef(h, A + ((size_t)(s0 + s) * a_ndom + (a_ndom == 1 ? 0 : d)) * 3, &h->coef_host[(size_t)s * h->ndom + d]);
        CU(cudaMemcpyAsync(h->coef(), h->coef_host, (size_t)ns * h->ndom * sizeof(StepCoef), cudaMemcpyHostToDevice, h->stream));
        CU(cudaEventRecord(h->coef_uploaded, h->stream));
        int s = 0;
        if (want_graph) {
            if (!h->gexec) {
                // one eager step first: it also sets the per-function attributes, which must not happen in a capture
                int rc = one_step(h->coef(), a_ndom == 1 ? &h->coef_host[0] : nullptr, false);
                if (rc) return rc;
                s = 1;
                rc = capture_step(h, dt, yz, split);
                if (rc) return rc;
            }
            if (h->gexec && s < ns) {
                CU(cudaEventRecord(h->gfork, h->stream));
                CU(cudaStreamWaitEvent(h->gstream, h->gfork, 0));
                CU(launch_set_counter(h->gstream, h->step_counter(), s, &nl));
                for (; s < ns; ++s) {
                    CU(cudaGraphLaunch(h->gexec, h->gstream));
                    nl += h->g_launches;
                }
                CU(cudaEventRecord(h->gjoin, h->gstream));
                CU(cudaStreamWaitEvent(h->stream, h->gjoin, 0));
                if (split && h->nproj > 0) h->split_pending = true;   // every replayed split step defers its scale
                // a replayed Taylor step leaves its rho to the next step's first projection: the call's last step has none
                if (!split && s0 + ns == nsteps && density_rides_on_projection(h)) rho_flush = true;
            }
        }
        for (; s < ns; ++s) {
            int rc = one_step(h->coef() + (size_t)s * h->ndom, a_ndom == 1 ? &h->coef_host[(size_t)s * h->ndom] : nullptr,
                              s0 + s == nsteps - 1);
            if (rc) return rc;
        }
    }
    {
        int rc = flush_split_scale(h, &nl);      // graph replays end on a deferred scale
        if (rc) return rc;
    }
    if (rho_flush) {
        ProfScope ps(h, MLMD_K_DENSITY);
        CU(launch_density(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->occ(), h->rho(), &nl));
    }
    h->launches += nl;
    if (nsteps > 0) h->rho_valid = true;
    if (h->flags & MLMD_CHECK_FINITE) {
        int n2 = 0;
        CU(launch_check_finite(h->stream, (const float *)h->psi(), (size_t)h->ndom * h->ngrid * h->ld * 2, h->flag(), &n2));
        h->launches += n2;
        CU(cudaMemcpyAsync(h->flag_host, h->flag(), sizeof(int), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
        if (*h->flag_host) return fail(MLMD_ERR_NONFINITE, "%s: psi contains NaN/Inf after %d steps", fn, nsteps);
    }
    if (dt * bound > 2.0 * sqrt(2.0)) {
        fail(MLMD_WARN_UNSTABLE, "%s: dt*|%s|max bound = %.3f > 2 sqrt(2): Taylor-4 may be unstable", fn, split ? "h_loc" : "H", dt * bound);
        return MLMD_WARN_UNSTABLE;
    }
    return MLMD_OK;
}

int mlmd_propagate(mlmd_domain_t *h, int nsteps, double dt, const double *A, int a_ndom) {
    return propagate_impl(h, nsteps, dt, A, a_ndom, false);
}

int mlmd_propagate_split(mlmd_domain_t *h, int nsteps, double dt, const double *A, int a_ndom) {
    return propagate_impl(h, nsteps, dt, A, a_ndom, true);
}

int mlmd_density(mlmd_domain_t *h, float *rho, int where) {
    if (!h || !rho) return fail(MLMD_ERR_ARG, "mlmd_density: NULL argument");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_density: bad where=%d", where);
    if (!h->have_psi) return fail(MLMD_ERR_STATE, "mlmd_density: no orbitals set");
    if (!h->rho_valid) {
        int nl = 0;
        CU(launch_density(h->stream, h->ndom, h->ngrid, h->ld, h->psi(), h->occ(), h->rho(), &nl));
        h->launches += nl;
        h->rho_valid = true;
    }
    CU(cudaMemcpyAsync(rho, h->rho(), (size_t)h->ndom * h->ngrid * sizeof(float), kind_out(where), h->stream));
    if (where == MLMD_HOST) CU(cudaStreamSynchronize(h->stream));
    return MLMD_OK;
}

int mlmd_overlap(mlmd_domain_t *h, int which, void *S, int where) {
    if (!h || !S) return fail(MLMD_ERR_ARG, "mlmd_overlap: NULL argument");
    if (bad_where(where)) return fail(MLMD_ERR_ARG, "mlmd_overlap: bad where=%d", where);
    if (which != 0 && which != 1) return fail(MLMD_ERR_ARG, "mlmd_overlap: which=%d", which);
    if (!h->have_psi) return fail(MLMD_ERR_STATE, "mlmd_overlap: no orbitals set");
    if (which == 1 && !(h->flags & MLMD_KEEP_PSI0)) return fail(MLMD_ERR_STATE, "mlmd_overlap: which=1 needs MLMD_KEEP_PSI0 at create");
    const float2 *phi = which == 0 ? h->psi() : h->psi0();
    int nl = 0;
    const bool fp64 = h->gemm_mode == MLMD_GEMM_FP64;
    // projection GEMM with B := float view of Phi (2*ld real rows), S4 of SURVEY.md 8(a); always
    // FP32-grade (3xTF32 on tensor cores, or the CUDA-core path): it is a measurement
    const bool tc = h->tc_ok && h->opt[MLMD_OPT_GEMM_PATH] == 0 && h->gemm_mode != MLMD_GEMM_FP64 &&
                    h->gemm_mode != MLMD_GEMM_FP32_SIMT;
    const int nsplit = tc ? h->nsplit_tc_ovl : h->nsplit;
    if (tc)
        CU(launch_proj_tc(h->stream, h->ndom, h->ngrid, (const float *)phi, nullptr, 2 * h->ld, 2 * h->ld,
                          (const float *)h->psi(), 2 * h->ld, 2 * h->ld, h->zpart(), h->prows, nsplit, 3, kOverlapChain, &nl, &h->tmaps));
    else
        CU(launch_proj_simt(h->stream, h->ndom, h->ngrid, (const float *)phi, nullptr, 2 * h->ld, 2 * h->ld,
                            (const float *)h->psi(), 2 * h->ld, 2 * h->ld, h->zpart(), h->prows, nsplit, fp64, &nl));
    float2 *sdev = where == MLMD_DEVICE ? (float2 *)S : (float2 *)h->z();
    CU(launch_overlap_epilogue(h->stream, h->ndom, h->norb, h->ld, h->prows, nsplit, h->zpart(), (float)h->dv, sdev, &nl));
    h->launches += nl;
    if (where == MLMD_HOST) {
        CU(cudaMemcpyAsync(S, sdev, (size_t)h->ndom * h->norb * h->norb * sizeof(float2), cudaMemcpyDeviceToHost, h->stream));
        CU(cudaStreamSynchronize(h->stream));
    }
    return MLMD_OK;
}

}  // extern "C"
