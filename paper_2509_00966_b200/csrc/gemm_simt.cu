// CUDA-core GEMMs for the nonlocal operator: any shape, FP32 FMA or
// FP64 accumulation of exact FP32 products.  These are the portable path (tiny configs, shapes the
// tcgen05 kernels do not tile, MLMD_GEMM_FP64 / MLMD_GEMM_FP32_SIMT); the tensor-core path lives in
// gemm_tc.cu.
//
// Complex GEMMs are run as REAL GEMMs on the interleaved storage:
//   projection        Z[p][c]  = sum_r B[r][p] * Y[r][c]           (K = grid points)
//   back-application  Y[r][c] += sum_p B[r][p] * What[p][c]        (K = projector rows)
// with Y the float view [ngrid][2*ld] of psi and B the float view of beta ([ngrid][ldb], real
// projectors one column each, complex ones two).
#include "mlmd_internal.h"

namespace mlmd {

constexpr int TM = 64, TN = 64, TK = 16;

template <typename Acc>
__global__ void __launch_bounds__(256)
proj_simt_kernel(long ngrid, const float *__restrict__ B, const float *__restrict__ Blo, int ldb, int P,
                 const float *__restrict__ Y, int ldy, int N, float *__restrict__ zpart, int prows, int nsplit) {
    __shared__ float Bs[TK][TM + 4];
    __shared__ float Ys[TK][TN + 4];
    // grid.x = column tile + ntile_n * (split + nsplit * dom): the batch rides on the x dimension (2^31 - 1 blocks),
    // so neither many domains nor many slices can exceed the 65535 limit of grid.y / grid.z
    const int ntile_n = (N + TN - 1) / TN;
    const int bz = blockIdx.x / ntile_n;
    const int dom = bz / nsplit, split = bz % nsplit;
    const int p0 = blockIdx.y * TM, c0 = (blockIdx.x % ntile_n) * TN;
    const long rlo = ngrid * split / nsplit, rhi = ngrid * (split + 1) / nsplit;
    const float *Bd = B + (size_t)dom * ngrid * ldb;
    const float *Bl = Blo ? Blo + (size_t)dom * ngrid * ldb : nullptr;   // B = hi + lo (exact)
    const float *Yd = Y + (size_t)dom * ngrid * ldy;
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
    Acc acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0;
    for (long r0 = rlo; r0 < rhi; r0 += TK) {
        // 16 rows x 64 columns of each operand: 1024 elements, 4 per thread
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int idx = threadIdx.x + e * 256;
            const int kk = idx / 64, cc = idx % 64;
            const long r = r0 + kk;
            const bool rok = r < rhi;
            Bs[kk][cc] = (rok && p0 + cc < P) ? (Bl ? Bd[r * ldb + p0 + cc] + Bl[r * ldb + p0 + cc] : Bd[r * ldb + p0 + cc]) : 0.f;
            Ys[kk][cc] = (rok && c0 + cc < N) ? Yd[r * ldy + c0 + cc] : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < TK; ++kk) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = Bs[kk][ty * 4 + i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Ys[kk][tx * 4 + j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] += (Acc)a[i] * (Acc)b[j];
        }
        __syncthreads();
    }
    float *zd = zpart + ((size_t)dom * nsplit + split) * prows * N;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int p = p0 + ty * 4 + i;
        if (p >= P) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = c0 + tx * 4 + j;
            if (c < N) zd[(size_t)p * N + c] = (float)acc[i][j];
        }
    }
}

template <typename Acc>
__global__ void __launch_bounds__(256)
back_simt_kernel(long ngrid, const float *__restrict__ B, const float *__restrict__ Blo, int ldb, int P,
                 const float *__restrict__ What, const float *__restrict__ Wlo, float *__restrict__ Y, int ldy, int N,
                 int prows) {
    __shared__ float As[TK][TM + 4];   // As[k][r]
    __shared__ float Ws[TK][TN + 4];
    // grid.x = row tile + nrt * dom (large grids: up to 2^31 - 1 blocks), grid.y = column tile
    const long nrt = (ngrid + TM - 1) / TM;
    const int dom = (int)(blockIdx.x / nrt);
    const long r0 = (long)(blockIdx.x % nrt) * TM;
    const int c0 = blockIdx.y * TN;
    const float *Bd = B + (size_t)dom * ngrid * ldb;
    const float *Bl = Blo ? Blo + (size_t)dom * ngrid * ldb : nullptr;   // optional exact remainder of B
    const float *Wd = What + (size_t)dom * prows * N;
    const float *Wl = Wlo + (size_t)dom * prows * N;
    float *Yd = Y + (size_t)dom * ngrid * ldy;
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
    Acc acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0;
    for (int k0 = 0; k0 < P; k0 += TK) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int idx = threadIdx.x + e * 256;
            {   // A tile: 64 rows x 16 k; consecutive threads walk k (contiguous in memory)
                const int rr = idx / 16, kk = idx % 16;
                const long r = r0 + rr;
                As[kk][rr] = (r < ngrid && k0 + kk < P) ? (Bl ? Bd[r * ldb + k0 + kk] + Bl[r * ldb + k0 + kk] : Bd[r * ldb + k0 + kk]) : 0.f;
            }
            {
                const int kk = idx / 64, cc = idx % 64;
                Ws[kk][cc] = (k0 + kk < P && c0 + cc < N) ? Wd[(size_t)(k0 + kk) * N + c0 + cc] + Wl[(size_t)(k0 + kk) * N + c0 + cc] : 0.f;
            }
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < TK; ++kk) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Ws[kk][tx * 4 + j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] += (Acc)a[i] * (Acc)b[j];
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const long r = r0 + ty * 4 + i;
        if (r >= ngrid) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int c = c0 + tx * 4 + j;
            if (c < N) Yd[r * ldy + c] = (float)((Acc)Yd[r * ldy + c] + acc[i][j]);
        }
    }
}

cudaError_t launch_proj_simt(cudaStream_t st, int ndom, long ngrid, const float *B, const float *Blo, int ldb, int P,
                             const float *Y, int ldy, int N, float *zpart, int prows, int nsplit,
                             bool fp64, int *nlaunch) {
    const long gx = (long)((N + TN - 1) / TN) * ndom * nsplit;
    if (gx > 0x7fffffffL || (P + TM - 1) / TM > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)gx, (P + TM - 1) / TM, 1);
    ++*nlaunch;
    if (fp64)
        proj_simt_kernel<double><<<grid, 256, 0, st>>>(ngrid, B, Blo, ldb, P, Y, ldy, N, zpart, prows, nsplit);
    else
        proj_simt_kernel<float><<<grid, 256, 0, st>>>(ngrid, B, Blo, ldb, P, Y, ldy, N, zpart, prows, nsplit);
    return cudaGetLastError();
}

cudaError_t launch_back_simt(cudaStream_t st, int ndom, long ngrid, const float *B, const float *Blo, int ldb, int P,
                             const float *What, const float *Wlo, float *Y, int ldy, int N, int prows, bool fp64,
                             int *nlaunch) {
    const long gx = ((ngrid + TM - 1) / TM) * ndom;
    if (gx > 0x7fffffffL || (N + TN - 1) / TN > 65535) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)gx, (N + TN - 1) / TN, 1);
    ++*nlaunch;
    if (fp64)
        back_simt_kernel<double><<<grid, 256, 0, st>>>(ngrid, B, Blo, ldb, P, What, Wlo, Y, ldy, N, prows);
    else
        back_simt_kernel<float><<<grid, 256, 0, st>>>(ngrid, B, Blo, ldb, P, What, Wlo, Y, ldy, N, prows);
    return cudaGetLastError();
}

}  // namespace mlmd
