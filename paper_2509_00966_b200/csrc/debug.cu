// Kernel-level test hooks (not part of include/mlmd.h): run one nonlocal GEMM on caller-owned
// DEVICE buffers so that tests can check the tensor-core kernels against a dense reference product.
#include "mlmd_internal.h"

using namespace mlmd;

extern "C" {

// Z partials [ndom][nsplit][prows][N] = per-K-slice sums of A^T Y.  A_lo may be NULL (kernel splits A).
// path: 0 = CUDA cores, 1 = tcgen05.  Returns a cudaError_t value.
int mlmd_debug_proj(int path, void *stream, int ndom, long ngrid, const float *A_hi, const float *A_lo, int lda, int P,
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

// Y[dom][r][c] += sum_p (A_hi + A_lo)[dom][r][p] * (W_hi + W_lo)[dom][p][c]
int mlmd_debug_back(int path, void *stream, int ndom, long ngrid, const float *A_hi, const float *A_lo, int lda, int P,
                    const float *W_hi, const float *W_lo, float *Y, int ldy, int N, int prows, int nprod) {
    int nl = 0;
    cudaError_t e;
    if (path == 1)
        e = launch_back_tc((cudaStream_t)stream, ndom, ngrid, A_hi, A_lo, lda, P, W_hi, W_lo, Y, ldy, N, prows, nprod, &nl);
    else
        e = launch_back_simt((cudaStream_t)stream, ndom, ngrid, A_hi, A_lo, lda, P, W_hi, W_lo, Y, ldy, N, prows, false, &nl);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
    return (int)e;
}

int mlmd_debug_nsplit(int ndom, long ngrid, int P, int N) { return tc_choose_nsplit(ndom, ngrid, P, N); }

}  // extern "C"
