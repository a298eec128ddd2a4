// mlmd_orbital_norms_static: the per-orbital squared norms of the split step (colnorm_part_kernel /
// colnorm_final_kernel of glue.cu, reading D27) for callers that cannot allocate: no handle, no caller workspace,
// no cudaMalloc / cudaFree / allocating library routine anywhere on this path.  The kernel pair needs scratch for its
// per-slab partial sums (part[dom][slab][c], FP64); here that scratch is a file-scope device array of fixed size, so
// every GPU that loads libmlmd.so holds MLMD_STATIC_SCRATCH_BYTES of it until the process exits.
//
// In HOST code the name g_norm_scratch is a host-side stand-in, not a device address: the launcher below takes the
// array's device address once per device with cudaGetSymbolAddress (that device current) and hands THAT to the first
// kernel; the second kernel, being device code of this file, names the array directly.
//
// All calls share the array and it keeps the last call's contents.  Nothing has to start at zero: the first kernel
// writes every partial sum the second one reads (all kNormSlabs slabs of every (domain, orbital column) of THIS call),
// so stale values are never read.  Two calls that overlap on the GPU (different streams, or two host threads on
// different streams) race on the array: serialise them on one stream.
#include <stdio.h>

#include <mutex>

#include "mlmd_internal.h"

namespace mlmd {

int set_error(int code, const char *fmt, ...);   // api.cu: fills the thread-local text of mlmd_last_error

namespace {

constexpr size_t kScratchDoubles = MLMD_STATIC_SCRATCH_BYTES / sizeof(double);
static __device__ __align__(256) double g_norm_scratch[kScratchDoubles];

// part[dom][slab][c] = sum_{r in slab} |psi[dom][r][c]|^2: FP32 squares summed in FP64, one owner per partial sum.
// Same thread mapping and summation order as colnorm_part_kernel (glue.cu), so the two paths agree bit for bit.
__global__ void __launch_bounds__(256)
norms_part_static_kernel(long ngrid, int ld, const float2 *__restrict__ psi, double *__restrict__ part) {
    const int c = blockIdx.z * 64 + threadIdx.x;
    const int dom = blockIdx.y, slab = blockIdx.x;
    const long per = (ngrid + kNormSlabs - 1) / kNormSlabs;
    const long r0 = slab * per, r1 = r0 + per < ngrid ? r0 + per : ngrid;
    double s = 0.0;
    if (c < ld) {
        const float2 *col = psi + (size_t)dom * ngrid * ld + c;
#pragma unroll 4
        for (long r = r0 + threadIdx.y; r < r1; r += 4) {
            const float2 v = __ldcs(col + r * ld);
            s += (double)fmaf(v.x, v.x, v.y * v.y);
        }
    }
    __shared__ double sm[4][64];
    sm[threadIdx.y][threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.y == 0 && c < ld)
        part[((size_t)dom * kNormSlabs + slab) * ld + c] =
            (sm[0][threadIdx.x] + sm[1][threadIdx.x]) + (sm[2][threadIdx.x] + sm[3][threadIdx.x]);
}

// out[dom][c] = dv * sum over slabs (fixed order: reproducible, reading D22); reads the static array by name
__global__ void norms_final_static_kernel(int n, int ld, double dv, double *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;     // i = dom * ld + c
    if (i >= n) return;
    const int dom = i / ld, c = i % ld;
    double s = 0.0;
    for (int k = 0; k < kNormSlabs; ++k) s += g_norm_scratch[((size_t)dom * kNormSlabs + k) * ld + c];
    out[i] = dv * s;
}

// device address of g_norm_scratch on the CURRENT device (taken once per device)
std::mutex g_mu;
double *g_scratch_dev[64] = {nullptr};

cudaError_t scratch_address(double **out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_dev[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_norm_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_dev[dev] = p;
    }
    *out = g_scratch_dev[dev];
    return cudaSuccess;
}

bool on_device(const void *p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace
}  // namespace mlmd

using namespace mlmd;

extern "C" int mlmd_orbital_norms_static(const void *psi, int ndom, long long ngrid, int ld, double dv, double *norm2,
                                         void *stream) {
    const char *fn = "mlmd_orbital_norms_static";
    if (!psi || !norm2) return set_error(MLMD_ERR_ARG, "%s: NULL pointer", fn);
    if (ndom < 1 || ngrid < 1 || ld < 1 || ndom > 65535 || !(dv == dv))
        return set_error(MLMD_ERR_SHAPE, "%s: ndom=%d ngrid=%lld ld=%d dv=%g", fn, ndom, ngrid, ld, dv);
    const unsigned long long need = (unsigned long long)ndom * kNormSlabs * (unsigned long long)ld;
    if (need > kScratchDoubles || (unsigned long long)ndom * (unsigned long long)ld > 0x7fffffffull)
        return set_error(MLMD_ERR_SHAPE,
                         "%s: ndom * ld = %d * %d needs %llu bytes of partial sums, the static scratch array holds %llu "
                         "(MLMD_STATIC_SCRATCH_BYTES); use a handle with a caller workspace for larger batches",
                         fn, ndom, ld, need * 8ull, (unsigned long long)MLMD_STATIC_SCRATCH_BYTES);
    if (!on_device(psi) || !on_device(norm2)) return set_error(MLMD_ERR_ARG, "%s: psi and norm2 must be DEVICE pointers", fn);
    double *part = nullptr;
    cudaError_t e = scratch_address(&part);
    if (e != cudaSuccess)
        return set_error(MLMD_ERR_CUDA, "%s: cudaGetSymbolAddress(static scratch) failed: %s", fn, cudaGetErrorString(e));
    cudaStream_t st = (cudaStream_t)stream;
    norms_part_static_kernel<<<dim3(kNormSlabs, ndom, (ld + 63) / 64), dim3(64, 4), 0, st>>>((long)ngrid, ld, (const float2 *)psi, part);
    e = cudaGetLastError();
    if (e == cudaSuccess) {
        norms_final_static_kernel<<<(ndom * ld + 127) / 128, 128, 0, st>>>(ndom * ld, ld, dv, norm2);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return set_error(MLMD_ERR_CUDA, "%s: kernel launch failed: %s", fn, cudaGetErrorString(e));
    return MLMD_OK;
}
