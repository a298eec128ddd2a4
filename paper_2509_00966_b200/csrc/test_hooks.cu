// Kernel-level test hooks: run one nonlocal GEMM on caller-owned DEVICE buffers so that tests can check the
// tensor-core kernels against a dense reference product.  Not part of include/mlmd.h and NOT linked into
// libmlmd.so: build.py puts this file into libmlmd_test.so only, which tests/ load and the product never does.
#include "mlmd_internal.h"

using namespace mlmd;

#define HOOK __attribute__((visibility("default")))

extern "C" {

// Z partials [ndom][nsplit][prows][N] = per-K-slice sums of A^T Y.  A_lo may be NULL (kernel splits A).
// path: 0 = CUDA cores, 1 = tcgen05.  Returns a cudaError_t value.
HOOK int mlmd_debug_proj(int path, void *stream, int ndom, long ngrid, const float *A_hi, const float *A_lo, int lda, int P,
                    const float *Y, int ldy, int N, float *zpart, int prows, int nsplit, int nprod, int chain) {
    int nl = 0;
    cudaError_t e;
    if (path == 1)
        e = launch_proj_tc((cudaStream_t)stream, ndom, ngrid, A_hi, A_lo, lda, P, Y, ldy, N, zpart, prows, nsplit, nprod, chain, &nl);
    else
        e = launch_proj_simt((cudaStream_t)stream, ndom, ngrid, A_hi, A_lo, lda, P, Y, ldy, N, zpart, prows, nsplit, false, &nl);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
    return (int)e;
}

// Y[dom][r][c] += sum_p A[dom][r][p] * (W_hi + W_lo)[dom][p][c]   (A: plain FP32; A_lo = A - trunc_tf32(A) or NULL)
HOOK int mlmd_debug_back(int path, void *stream, int ndom, long ngrid, const float *A, const float *A_lo, int lda, int P,
                    const float *W_hi, const float *W_lo, float *Y, int ldy, int N, int prows, int nprod) {
    int nl = 0;
    cudaError_t e;
    if (path == 1)
        e = launch_back_tc((cudaStream_t)stream, ndom, ngrid, A, A_lo, lda, P, W_hi, W_lo, Y, ldy, N, prows, nprod, &nl);
    else
        e = launch_back_simt((cudaStream_t)stream, ndom, ngrid, A, nullptr, lda, P, W_hi, W_lo, Y, ldy, N, prows, false, &nl);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
    return (int)e;
}

// The density formed inside the step's first projection (S3 riding on S2a) is overwritten by the separate pass at the
// end of every call, so it cannot be seen through the C ABI: this hook runs that projection on the handle's current
// psi and copies the rho it formed to rho_dev [ndom][ngrid] (device).  Returns a cudaError_t value, -1 if the shape
// cannot carry the density.
// nprod: 3 = the default mode's three-product projection, 4 = the staged mode's one-product projection of rounded operands,
// 0 = the low-precision mode's BF16 projection (the handle must be in that mode: beta's BF16 copy lives in the remainder buffer).
HOOK int mlmd_debug_fused_density_np(mlmd_domain_t *h, float *rho_dev, int nprod);
HOOK int mlmd_debug_fused_density(mlmd_domain_t *h, float *rho_dev) { return mlmd_debug_fused_density_np(h, rho_dev, 3); }
HOOK int mlmd_debug_fused_density_np(mlmd_domain_t *h, float *rho_dev, int nprod) {
    if (!h->tc_ok || !proj_tc_can_fuse_density(h->P, 2 * h->ld, nprod) || h->nproj == 0) return -1;
    int nl = 0;
    cudaError_t e = launch_proj_tc(h->stream, h->ndom, h->ngrid, h->beta(), nullptr, h->ldp, h->P, (const float *)h->psi(), 2 * h->ld,
                                   2 * h->ld, h->zpart(), h->prows, h->nsplit_tc, nprod, 128, &nl, nullptr, h->rho(), h->occ(),
                                   nprod == 0 && h->gemm_mode == MLMD_GEMM_LOWP_BF16 ? h->beta_lo() : nullptr);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(rho_dev, h->rho(), (size_t)h->ndom * h->ngrid * sizeof(float), cudaMemcpyDeviceToDevice, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    h->rho_valid = false;
    return (int)e;
}

// The split step's norm pass as the library runs it, with its partial sums in CALLER scratch part[ndom][64][ld] (device):
// out[dom][c] = sum_r |psi[dom][r][c]|^2 (no dv).  The existing path that mlmd_orbital_norms_static is checked against.
HOOK int mlmd_debug_colnorm2(void *stream, int ndom, long ngrid, int ld, const void *psi, double *part, double *out) {
    int nl = 0;
    cudaError_t e = launch_colnorm2((cudaStream_t)stream, ndom, ngrid, ld, (const float2 *)psi, part, out, &nl);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
    return (int)e;
}

HOOK int mlmd_debug_nsplit(int ndom, long ngrid, int P, int N) { return tc_choose_nsplit(ndom, ngrid, P, N); }

}  // extern "C"
