// Small kernels around the GEMMs and the stencil: split-K reduction + projector scaling (S2b),
// density (S3), overlap epilogue (S4), operand preparation and checks.
#include "mlmd_internal.h"

namespace mlmd {

// x rounded to the nearest TF32 value (ties to even; 13 low mantissa bits cleared afterwards, so a kind::tf32
// tensor-core operand, which drops those bits, keeps it exactly).  Nearest rather than truncated: the hi part
// alone is then an UNBIASED single-product operand (staged mode), and x - hi is still exact in FP32.
__device__ __forceinline__ float tf32_hi(float x) {
    unsigned u = __float_as_uint(x);
    u += 0xfffu + ((u >> 13) & 1u);
    return __uint_as_float(u & 0xffffe000u);
}

__device__ __forceinline__ float bf16_rne(float x) {
    unsigned u = __float_as_uint(x);
    u += 0x7fffu + ((u >> 16) & 1u);
    return __uint_as_float(u & 0xffff0000u);
}

// S2b.  C[p][n] = sum over split slices (fixed order: bit-reproducible, reading D22) of the
// projection, combined to the complex coefficient for complex projectors; then
//   W[p][n] = (-i tau) * D'_p * C[p][n],  D' = D * dv (reading D10)
// written in the real-GEMM form the back-application consumes:
//   real beta:    What[p][2n] = Re W, What[p][2n+1] = Im W
//   complex beta: rows 2p, 2p+1 hold the 2x2 real representation of W.
__global__ void reduce_scale_kernel(int nproj, int beta_complex, int ld, int prows, int nsplit,
                                    const float *__restrict__ zpart, const float *__restrict__ dprime, float tau,
                                    float *__restrict__ what, float *__restrict__ what_lo, int lowp) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const int p = blockIdx.y, dom = blockIdx.z;
    if (n >= ld) return;
    const int N = 2 * ld;
    const float *zp = zpart + (size_t)dom * nsplit * prows * N;
    const size_t slice = (size_t)prows * N;
    float cre = 0.f, cim = 0.f;
    if (!beta_complex) {
        for (int s = 0; s < nsplit; ++s) {
            const float2 v = *(const float2 *)(zp + s * slice + (size_t)p * N + 2 * n);
            cre += v.x;
            cim += v.y;
        }
    } else {
        for (int s = 0; s < nsplit; ++s) {
            const float2 a = *(const float2 *)(zp + s * slice + (size_t)(2 * p) * N + 2 * n);      // Re(beta) row
            const float2 b = *(const float2 *)(zp + s * slice + (size_t)(2 * p + 1) * N + 2 * n);  // Im(beta) row
            cre += a.x + b.y;   // conj(beta) psi
            cim += a.y - b.x;
        }
    }
    const float f = tau * dprime[(size_t)dom * nproj + p];
    const float wre = f * cim, wim = -f * cre;   // (-i f)(cre + i cim)
    // stored as TF32-representable hi part (nearest) + exact FP32 remainder lo (hi + lo == W exactly)
    // low-precision mode: W rounded to BF16 (round-to-nearest-even), no remainder
    const float wre_h = lowp ? bf16_rne(wre) : tf32_hi(wre), wim_h = lowp ? bf16_rne(wim) : tf32_hi(wim);
    const float wre_l = lowp ? 0.f : wre - wre_h, wim_l = lowp ? 0.f : wim - wim_h;
    if (lowp == 2) {
        // low-precision mode proper: W as a BF16 array [dom][prows][N] (the kind::f16 back-application reads it by TMA)
        unsigned short *w16 = (unsigned short *)what + (size_t)dom * prows * N;
        const unsigned short re = (unsigned short)(__float_as_uint(wre_h) >> 16), im = (unsigned short)(__float_as_uint(wim_h) >> 16);
        const unsigned short nim = (unsigned short)(im ^ 0x8000u);
        if (!beta_complex) {
            *(ushort2 *)(w16 + (size_t)p * N + 2 * n) = make_ushort2(re, im);
        } else {
            *(ushort2 *)(w16 + (size_t)(2 * p) * N + 2 * n) = make_ushort2(re, im);
            *(ushort2 *)(w16 + (size_t)(2 * p + 1) * N + 2 * n) = make_ushort2(nim, re);
        }
        return;
    }
    float *wd = what + (size_t)dom * prows * N;
    float *wl = what_lo + (size_t)dom * prows * N;
    if (!beta_complex) {
        *(float2 *)(wd + (size_t)p * N + 2 * n) = make_float2(wre_h, wim_h);
        *(float2 *)(wl + (size_t)p * N + 2 * n) = make_float2(wre_l, wim_l);
    } else {
        *(float2 *)(wd + (size_t)(2 * p) * N + 2 * n) = make_float2(wre_h, wim_h);
        *(float2 *)(wd + (size_t)(2 * p + 1) * N + 2 * n) = make_float2(-wim_h, wre_h);
        *(float2 *)(wl + (size_t)(2 * p) * N + 2 * n) = make_float2(wre_l, wim_l);
        *(float2 *)(wl + (size_t)(2 * p + 1) * N + 2 * n) = make_float2(-wim_l, wre_l);
    }
}

cudaError_t launch_reduce_scale(cudaStream_t st, int ndom, int nproj, int beta_complex, int ld, int prows,
                                int nsplit, const float *zpart, const float *dprime, float tau,
                                float *what, float *what_lo, int lowp, int *nlaunch) {
    dim3 grid((ld + 127) / 128, nproj, ndom);
    ++*nlaunch;
    reduce_scale_kernel<<<grid, 128, 0, st>>>(nproj, beta_complex, ld, prows, nsplit, zpart, dprime, tau, what, what_lo, lowp);
    return cudaGetLastError();
}

// S3: one warp per group of DP consecutive grid points; lanes stride over the orbital rows with 128-bit
// loads (all DP rows are requested before any is reduced, so a warp keeps DP x 512 B per trip in flight)
// and reduce with shuffles (north_star kernel 4).
constexpr int DP = 4;
__global__ void __launch_bounds__(256)
density_kernel(long npoints, long ngrid, int lanes, const float4 *__restrict__ psi, const float *__restrict__ occ,
               float *__restrict__ rho) {
    const long p0 = ((long)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32) * DP;
    if (p0 >= npoints) return;
    const int lane = threadIdx.x % 32;
    float s[DP];
#pragma unroll
    for (int k = 0; k < DP; ++k) s[k] = 0.f;
    // ngrid % DP == 0 is checked by the launcher, so the DP points share a domain
    const float2 *f = (const float2 *)(occ + (size_t)(p0 / ngrid) * lanes * 2);
    for (int l = lane; l < lanes; l += 32) {
        float4 v[DP];
#pragma unroll
        for (int k = 0; k < DP; ++k) v[k] = p0 + k < npoints ? __ldcs(psi + (p0 + k) * lanes + l) : make_float4(0.f, 0.f, 0.f, 0.f);
        const float2 ff = __ldg(f + l);
#pragma unroll
        for (int k = 0; k < DP; ++k) {
            s[k] = fmaf(ff.x, fmaf(v[k].x, v[k].x, v[k].y * v[k].y), s[k]);
            s[k] = fmaf(ff.y, fmaf(v[k].z, v[k].z, v[k].w * v[k].w), s[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < DP; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_xor_sync(0xffffffffu, s[k], o);
    }
    if (lane < DP && p0 + lane < npoints) {
        float out = s[0];
#pragma unroll
        for (int k = 1; k < DP; ++k) out = lane == k ? s[k] : out;
        rho[p0 + lane] = out;
    }
}

// one point per warp: any ngrid
__global__ void __launch_bounds__(256)
density_kernel_1(long npoints, long ngrid, int lanes, const float4 *__restrict__ psi, const float *__restrict__ occ,
                 float *__restrict__ rho) {
    const long pt = (long)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
    if (pt >= npoints) return;
    const int lane = threadIdx.x % 32;
    const float4 *row = psi + pt * lanes;
    const float2 *f = (const float2 *)(occ + (size_t)(pt / ngrid) * lanes * 2);
    float s = 0.f;
    for (int l = lane; l < lanes; l += 32) {
        const float4 v = __ldg(row + l);
        const float2 ff = __ldg(f + l);
        s = fmaf(ff.x, fmaf(v.x, v.x, v.y * v.y), s);
        s = fmaf(ff.y, fmaf(v.z, v.z, v.w * v.w), s);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) rho[pt] = s;
}

cudaError_t launch_density(cudaStream_t st, int ndom, long ngrid, int ld, const float2 *psi, const float *occ,
                           float *rho, int *nlaunch) {
    const long npoints = (long)ndom * ngrid;
    ++*nlaunch;
    if (ngrid % DP == 0) {
        const long nwarps = npoints / DP;
        density_kernel<<<(unsigned)((nwarps + 7) / 8), 256, 0, st>>>(npoints, ngrid, ld / 2, (const float4 *)psi, occ, rho);
    } else {
        density_kernel_1<<<(unsigned)((npoints + 7) / 8), 256, 0, st>>>(npoints, ngrid, ld / 2, (const float4 *)psi, occ, rho);
    }
    return cudaGetLastError();
}

// S4 epilogue: projection run with B := float view of Phi (rows 2m = Re, 2m+1 = Im):
//   S[m][n] = dv * sum_r conj(Phi[r,m]) Psi[r,n]
__global__ void overlap_epilogue_kernel(int norb, int ld, int prows, int nsplit, const float *__restrict__ zpart,
                                        float dv, float2 *__restrict__ S) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const int m = blockIdx.y, dom = blockIdx.z;
    if (n >= norb) return;
    const int N = 2 * ld;
    const float *zp = zpart + (size_t)dom * nsplit * prows * N;
    const size_t slice = (size_t)prows * N;
    float sre = 0.f, sim = 0.f;
    for (int s = 0; s < nsplit; ++s) {
        const float2 a = *(const float2 *)(zp + s * slice + (size_t)(2 * m) * N + 2 * n);
        const float2 b = *(const float2 *)(zp + s * slice + (size_t)(2 * m + 1) * N + 2 * n);
        sre += a.x + b.y;
        sim += a.y - b.x;
    }
    S[((size_t)dom * norb + m) * norb + n] = make_float2(dv * sre, dv * sim);
}

cudaError_t launch_overlap_epilogue(cudaStream_t st, int ndom, int norb, int ld, int prows, int nsplit,
                                    const float *zpart, float dv, float2 *S, int *nlaunch) {
    dim3 grid((norb + 127) / 128, norb, ndom);
    ++*nlaunch;
    overlap_epilogue_kernel<<<grid, 128, 0, st>>>(norb, ld, prows, nsplit, zpart, dv, S);
    return cudaGetLastError();
}

// y = x rounded to BF16 (nearest even): the stored low-precision copy of the projectors (PAPER.md L239 float_to_BF16)
__global__ void to_bf16_kernel(const float *__restrict__ x, unsigned short *__restrict__ y, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        y[i] = (unsigned short)(__float_as_uint(bf16_rne(x[i])) >> 16);
}
cudaError_t launch_to_bf16(cudaStream_t st, const float *x, void *y, size_t n, int *nlaunch) {
    ++*nlaunch;
    to_bf16_kernel<<<2368, 256, 0, st>>>(x, (unsigned short *)y, n);
    return cudaGetLastError();
}

// lo = x - trunc_tf32(x): what a kind::tf32 tensor-core operand drops of x (it ignores the 13 low mantissa bits).
// Exact in FP32.  The back-application reads (x, lo) as the operand pair of 3xTF32; x itself stays as given.
__global__ void tf32_remainder_kernel(const float *__restrict__ x, float *__restrict__ lo, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float v = x[i];
        lo[i] = v - __uint_as_float(__float_as_uint(v) & 0xffffe000u);
    }
}
cudaError_t launch_tf32_remainder(cudaStream_t st, const float *x, float *lo, size_t n, int *nlaunch) {
    ++*nlaunch;
    tf32_remainder_kernel<<<2368, 256, 0, st>>>(x, lo, n);
    return cudaGetLastError();
}

// max |x| as the bit pattern of a non-negative float (atomicMax on ints orders them correctly)
__global__ void max_abs_kernel(const float *__restrict__ x, size_t n, int *out) {
    float m = 0.f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = fabsf(x[i]);
        m = (a > m || a != a) ? a : m;   // NaN propagates as a large bit pattern
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float other = __shfl_xor_sync(0xffffffffu, m, o);
        m = (other > m || other != other) ? other : m;
    }
    if (threadIdx.x % 32 == 0) atomicMax(out, __float_as_int(m));
}
cudaError_t launch_max_abs(cudaStream_t st, const float *x, size_t n, int *flag_bits, int *nlaunch) {
    ++*nlaunch;
    cudaError_t e = cudaMemsetAsync(flag_bits, 0, sizeof(int), st);
    if (e != cudaSuccess) return e;
    max_abs_kernel<<<592, 256, 0, st>>>(x, n, flag_bits);
    return cudaGetLastError();
}

__global__ void check_finite_kernel(const float *__restrict__ x, size_t n, int *flag) {
    bool bad = false;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        bad |= !isfinite(x[i]);
    if (__any_sync(0xffffffffu, bad) && threadIdx.x % 32 == 0) atomicOr(flag, 1);
}
cudaError_t launch_check_finite(cudaStream_t st, const float *x, size_t n, int *flag, int *nlaunch) {
    ++*nlaunch;
    cudaError_t e = cudaMemsetAsync(flag, 0, sizeof(int), st);
    if (e != cudaSuccess) return e;
    check_finite_kernel<<<1184, 256, 0, st>>>(x, n, flag);
    return cudaGetLastError();
}

// ---- CUDA-graph support: the captured step reads its stencil coefficients from a device slot that this
// kernel refills from the uploaded table at the start of every graph launch
__global__ void set_counter_kernel(int *counter, int value) { *counter = value; }
__global__ void advance_coef_kernel(const StepCoef *__restrict__ all, StepCoef *__restrict__ cur, int *counter, int ndom) {
    const int s = *counter;
    for (int d = threadIdx.x; d < ndom; d += blockDim.x) cur[d] = all[(size_t)s * ndom + d];
    __syncthreads();
    if (threadIdx.x == 0) *counter = s + 1;
}
cudaError_t launch_set_counter(cudaStream_t st, int *counter, int value, int *nlaunch) {
    ++*nlaunch;
    set_counter_kernel<<<1, 1, 0, st>>>(counter, value);
    return cudaGetLastError();
}
cudaError_t launch_advance_coef(cudaStream_t st, const StepCoef *all, StepCoef *cur, int *counter, int ndom, int *nlaunch) {
    ++*nlaunch;
    advance_coef_kernel<<<1, 64, 0, st>>>(all, cur, counter, ndom);
    return cudaGetLastError();
}

// ---- the literal Eq. (2) step (mlmd_propagate_split; D27): per-orbital norms and rescaling ----
// part[dom][slab][c] = sum_{r in slab} |psi[dom][r][c]|^2: FP32 squares summed in FP64, one owner per
// partial sum, slabs added in a fixed order by colnorm_final_kernel, so the norms are reproducible.
__global__ void __launch_bounds__(256)
colnorm_part_kernel(long ngrid, int ld, const float2 *__restrict__ psi, double *__restrict__ part) {
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
        part[((size_t)dom * kNormSlabs + slab) * ld + c] = (sm[0][threadIdx.x] + sm[1][threadIdx.x]) + (sm[2][threadIdx.x] + sm[3][threadIdx.x]);
}
__global__ void colnorm_final_kernel(int n, int ld, int nslabs, const double *__restrict__ part, double *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;     // i = dom * ld + c
    if (i >= n) return;
    const int dom = i / ld, c = i % ld;
    double s = 0.0;
    for (int k = 0; k < nslabs; ++k) s += part[((size_t)dom * nslabs + k) * ld + c];
    out[i] = s;
}
cudaError_t launch_colnorm_final(cudaStream_t st, int ndom, int ld, int nslabs, const double *part, double *out, int *nlaunch) {
    ++*nlaunch;
    colnorm_final_kernel<<<(ndom * ld + 127) / 128, 128, 0, st>>>(ndom * ld, ld, nslabs, part, out);
    return cudaGetLastError();
}
cudaError_t launch_colnorm2(cudaStream_t st, int ndom, long ngrid, int ld, const float2 *psi, double *part, double *out,
                            int *nlaunch) {
    ++*nlaunch;
    colnorm_part_kernel<<<dim3(kNormSlabs, ndom, (ld + 63) / 64), dim3(64, 4), 0, st>>>(ngrid, ld, psi, part);
    cudaError_t e = cudaGetLastError();
    return e != cudaSuccess ? e : launch_colnorm_final(st, ndom, ld, kNormSlabs, part, out, nlaunch);
}

// One step's pending scale from the four squared norms (un-normalised chain, D27):
//   kick 1: ||psi|| / ||psi_a||, kick 2: ||psi_c|| / ||psi_d||;  the true squared norm after the step is
//   n0 * nc / na (the kicks keep it, the Taylor step changes it by nc / na).
__global__ void kick_scale_kernel(int n, double *__restrict__ n0, const double *__restrict__ na, const double *__restrict__ nc,
                                  const double *__restrict__ nd, float *__restrict__ scl) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double a = na[i], d = nd[i];
    if (a > 0.0 && d > 0.0) {
        scl[i] = (float)sqrt((n0[i] / a) * (nc[i] / d));
        n0[i] = n0[i] * (nc[i] / a);
    } else {
        scl[i] = 1.f;       // zero (padded) orbitals stay zero
    }
}
cudaError_t launch_kick_scale(cudaStream_t st, int n, double *n0, const double *na, const double *nc, const double *nd,
                              float *scl, int *nlaunch) {
    ++*nlaunch;
    kick_scale_kernel<<<(n + 127) / 128, 128, 0, st>>>(n, n0, na, nc, nd, scl);
    return cudaGetLastError();
}

// psi[r][n] *= scl[n] and rho[r] = sum_n occ[n] |psi[r][n]|^2 of the scaled values, in one pass
// (NP consecutive points of one domain per warp, as density_kernel).
template <int NP>
__global__ void __launch_bounds__(256)
scale_density_kernel(long npoints, long ngrid, int lanes, float4 *__restrict__ psi, const float *__restrict__ scl,
                     const float *__restrict__ occ, float *__restrict__ rho) {
    const long p0 = ((long)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32) * NP;
    if (p0 >= npoints) return;
    const int lane = threadIdx.x % 32;
    float s[NP];
#pragma unroll
    for (int k = 0; k < NP; ++k) s[k] = 0.f;
    const size_t dom = (size_t)(p0 / ngrid);
    const float2 *f = (const float2 *)(occ + dom * lanes * 2);
    const float2 *sc = (const float2 *)(scl + dom * lanes * 2);
    for (int l = lane; l < lanes; l += 32) {
        float4 v[NP];
#pragma unroll
        for (int k = 0; k < NP; ++k) v[k] = psi[(p0 + k) * lanes + l];
        const float2 ff = __ldg(f + l), ss = __ldg(sc + l);
#pragma unroll
        for (int k = 0; k < NP; ++k) {
            v[k].x *= ss.x; v[k].y *= ss.x; v[k].z *= ss.y; v[k].w *= ss.y;
            psi[(p0 + k) * lanes + l] = v[k];
            s[k] = fmaf(ff.x, fmaf(v[k].x, v[k].x, v[k].y * v[k].y), s[k]);
            s[k] = fmaf(ff.y, fmaf(v[k].z, v[k].z, v[k].w * v[k].w), s[k]);
        }
    }
#pragma unroll
    for (int k = 0; k < NP; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_xor_sync(0xffffffffu, s[k], o);
    }
    if (lane < NP) {
        float out = s[0];
#pragma unroll
        for (int k = 1; k < NP; ++k) out = lane == k ? s[k] : out;
        rho[p0 + lane] = out;
    }
}
cudaError_t launch_scale_density(cudaStream_t st, int ndom, long ngrid, int ld, float2 *psi, const float *scl,
                                 const float *occ, float *rho, int *nlaunch) {
    const long npoints = (long)ndom * ngrid;
    ++*nlaunch;
    if (ngrid % 4 == 0)
        scale_density_kernel<4><<<(unsigned)((npoints / 4 + 7) / 8), 256, 0, st>>>(npoints, ngrid, ld / 2, (float4 *)psi, scl, occ, rho);
    else
        scale_density_kernel<1><<<(unsigned)((npoints + 7) / 8), 256, 0, st>>>(npoints, ngrid, ld / 2, (float4 *)psi, scl, occ, rho);
    return cudaGetLastError();
}

// Occupations of the reference orbitals (reading D29): f[dom][s] = sum_n occ[dom][n] |S[dom][s][n]|^2 and
// nexc[dom] = sum_s max(occ[dom][s] - f[dom][s], 0); S from the overlap epilogue.  One block per domain.
__global__ void __launch_bounds__(256)
occupations_kernel(int norb, int ld, const float2 *__restrict__ S, const float *__restrict__ occ, double *__restrict__ f,
                   double *__restrict__ nexc) {
    const int dom = blockIdx.x;
    const float *oc = occ + (size_t)dom * ld;
    double holes = 0.0;
    for (int s = threadIdx.x; s < norb; s += blockDim.x) {
        const float2 *row = S + ((size_t)dom * norb + s) * norb;
        double acc = 0.0;
        for (int n = 0; n < norb; ++n) {
            const float2 v = row[n];
            acc += (double)oc[n] * ((double)v.x * v.x + (double)v.y * v.y);
        }
        f[(size_t)dom * norb + s] = acc;
        const double lost = (double)oc[s] - acc;
        if (lost > 0.0) holes += lost;
    }
    __shared__ double red[256];
    red[threadIdx.x] = holes;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) nexc[dom] = red[0];
}
cudaError_t launch_occupations(cudaStream_t st, int ndom, int norb, int ld, const float2 *S, const float *occ, double *f,
                               double *nexc, int *nlaunch) {
    ++*nlaunch;
    occupations_kernel<<<ndom, 256, 0, st>>>(norb, ld, S, occ, f, nexc);
    return cudaGetLastError();
}

// ---- observables (reading D30) ----
// E_nl[dom] = dv sum_n f_n sum_p D'_p |C[p][n]|^2, C = split-K sum of the projection (as reduce_scale_kernel),
// D' = D dv.  One block per domain, orbitals across threads, fixed summation order.
__global__ void __launch_bounds__(256)
energy_nl_kernel(int nproj, int beta_complex, int ld, int prows, int nsplit, const float *__restrict__ zpart,
                 const float *__restrict__ dprime, const float *__restrict__ occ, double dv, double *__restrict__ E) {
    const int dom = blockIdx.x;
    const int N = 2 * ld;
    const float *zp = zpart + (size_t)dom * nsplit * prows * N;
    const size_t slice = (size_t)prows * N;
    double e = 0.0;
    for (int n = threadIdx.x; n < ld; n += blockDim.x) {
        double en = 0.0;
        for (int p = 0; p < nproj; ++p) {
            float cre = 0.f, cim = 0.f;
            if (!beta_complex) {
                for (int s = 0; s < nsplit; ++s) {
                    const float2 v = *(const float2 *)(zp + s * slice + (size_t)p * N + 2 * n);
                    cre += v.x;
                    cim += v.y;
                }
            } else {
                for (int s = 0; s < nsplit; ++s) {
                    const float2 a = *(const float2 *)(zp + s * slice + (size_t)(2 * p) * N + 2 * n);
                    const float2 b = *(const float2 *)(zp + s * slice + (size_t)(2 * p + 1) * N + 2 * n);
                    cre += a.x + b.y;
                    cim += a.y - b.x;
                }
            }
            en += (double)dprime[(size_t)dom * nproj + p] * ((double)cre * cre + (double)cim * cim);
        }
        e += (double)occ[(size_t)dom * ld + n] * en;
    }
    __shared__ double red[256];
    red[threadIdx.x] = e;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) E[dom] = dv * red[0];
}
cudaError_t launch_energy_nl(cudaStream_t st, int ndom, int nproj, int beta_complex, int ld, int prows, int nsplit,
                             const float *zpart, const float *dprime, const float *occ, double dv, double *E, int *nlaunch) {
    ++*nlaunch;
    energy_nl_kernel<<<ndom, 256, 0, st>>>(nproj, beta_complex, ld, prows, nsplit, zpart, dprime, occ, dv, E);
    return cudaGetLastError();
}

// ---- nonlocal part of the current (mlmd_current_nl, reading D31) ----
// cmat[dom][p][n] = complex projection coefficient C_pn summed over the split-K slices in index order (real beta: row p
// holds (Re, Im) pairs; complex beta: rows 2p, 2p+1 combine as in reduce_scale_kernel).
__global__ void proj_coeff_kernel(int nproj, int beta_complex, int ld, int prows, int nsplit, const float *__restrict__ zpart,
                                  float2 *__restrict__ cmat) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const int p = blockIdx.y, dom = blockIdx.z;
    if (n >= ld) return;
    const int N = 2 * ld;
    const float *zp = zpart + (size_t)dom * nsplit * prows * N;
    const size_t slice = (size_t)prows * N;
    float cre = 0.f, cim = 0.f;
    for (int s = 0; s < nsplit; ++s) {
        if (!beta_complex) {
            const float2 v = *(const float2 *)(zp + s * slice + (size_t)p * N + 2 * n);
            cre += v.x;
            cim += v.y;
        } else {
            const float2 a = *(const float2 *)(zp + s * slice + (size_t)(2 * p) * N + 2 * n);
            const float2 b = *(const float2 *)(zp + s * slice + (size_t)(2 * p + 1) * N + 2 * n);
            cre += a.x + b.y;
            cim += a.y - b.x;
        }
    }
    cmat[((size_t)dom * nproj + p) * ld + n] = make_float2(cre, cim);
}
cudaError_t launch_proj_coeff(cudaStream_t st, int ndom, int nproj, int beta_complex, int ld, int prows, int nsplit,
                              const float *zpart, float2 *cmat, int *nlaunch) {
    dim3 grid((ld + 127) / 128, nproj, ndom);
    ++*nlaunch;
    proj_coeff_kernel<<<grid, 128, 0, st>>>(nproj, beta_complex, ld, prows, nsplit, zpart, cmat);
    return cudaGetLastError();
}
// J[dom][d] = 2 dv sum_n f_n sum_p D'_p Im( conj(G_pn) C_pn ),  D' = D dv;  one block per domain, FP64 sums in a fixed order
__global__ void __launch_bounds__(256)
current_nl_kernel(int nproj, int ld, const float2 *__restrict__ cmat, const float2 *__restrict__ gmat,
                  const float *__restrict__ dprime, const float *__restrict__ occ, double dv, int d, double *__restrict__ J) {
    const int dom = blockIdx.x;
    double acc = 0.0;
    for (int n = threadIdx.x; n < ld; n += blockDim.x) {
        double an = 0.0;
        for (int p = 0; p < nproj; ++p) {
            const float2 c = cmat[((size_t)dom * nproj + p) * ld + n], g = gmat[((size_t)dom * nproj + p) * ld + n];
            an += (double)dprime[(size_t)dom * nproj + p] * ((double)g.x * c.y - (double)g.y * c.x);
        }
        acc += (double)occ[(size_t)dom * ld + n] * an;
    }
    __shared__ double red[256];
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) J[(size_t)dom * 3 + d] = 2.0 * dv * red[0];
}
cudaError_t launch_current_nl(cudaStream_t st, int ndom, int nproj, int ld, const float2 *cmat, const float2 *gmat,
                              const float *dprime, const float *occ, double dv, int d, double *J, int *nlaunch) {
    ++*nlaunch;
    current_nl_kernel<<<ndom, 256, 0, st>>>(nproj, ld, cmat, gmat, dprime, occ, dv, d, J);
    return cudaGetLastError();
}

// Local current: part[dom][blk][0..2] = sum over the block's points and all orbitals of
//   f_n * 2 * sum_{j=1,2} c1_j / h_d * Im( conj(psi(r)) psi(r + j e_d) )      (= f_n Im<psi|D1_d psi> restricted to r;
//   the -j taps are the +j taps of the shifted sum, so only forward neighbours are read)
// and part[..][3] = sum f_n |psi(r)|^2.  One warp per point, lanes stride over the float4 (two orbitals) of the row.
__global__ void __launch_bounds__(256)
current_part_kernel(int nx, int ny, int nz, int lanes, int pts, int nblk, const float4 *__restrict__ psi,
                    const float *__restrict__ occ, float wx1, float wx2, float wy1, float wy2, float wz1, float wz2,
                    double *__restrict__ part) {
    const int dom = blockIdx.x / nblk, blk = blockIdx.x % nblk;
    const long ngrid = (long)nx * ny * nz;
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const float4 *base = psi + (size_t)dom * ngrid * lanes;
    const float2 *f = (const float2 *)(occ + (size_t)dom * lanes * 2);
    double jx = 0.0, jy = 0.0, jz = 0.0, ne = 0.0;
    const long r0 = (long)blk * pts, r1 = r0 + pts < ngrid ? r0 + pts : ngrid;
    for (long r = r0 + warp; r < r1; r += 8) {
        const int iz = (int)(r % nz), iy = (int)((r / nz) % ny), ix = (int)(r / ((long)nz * ny));
        const long rz1 = r + (iz + 1 < nz ? 1 : 1 - nz), rz2 = r + (iz + 2 < nz ? 2 : 2 - nz);
        const long ry1 = r + (long)nz * (iy + 1 < ny ? 1 : 1 - ny), ry2 = r + (long)nz * (iy + 2 < ny ? 2 : 2 - ny);
        const long sx = (long)nz * ny;
        const long rx1 = r + sx * (ix + 1 < nx ? 1 : 1 - nx), rx2 = r + sx * (ix + 2 < nx ? 2 : 2 - nx);
        float ax = 0.f, ay = 0.f, az = 0.f, an = 0.f;
        for (int l = lane; l < lanes; l += 32) {
            const float4 u = __ldg(base + r * lanes + l);
            const float2 ff = __ldg(f + l);
            auto im = [&](const float4 v) {     // f_n Im(conj(u) v) summed over the two orbitals of the float4
                return ff.x * (u.x * v.y - u.y * v.x) + ff.y * (u.z * v.w - u.w * v.z);
            };
            ax += wx1 * im(__ldg(base + rx1 * lanes + l)) + wx2 * im(__ldg(base + rx2 * lanes + l));
            ay += wy1 * im(__ldg(base + ry1 * lanes + l)) + wy2 * im(__ldg(base + ry2 * lanes + l));
            az += wz1 * im(__ldg(base + rz1 * lanes + l)) + wz2 * im(__ldg(base + rz2 * lanes + l));
            an += ff.x * (u.x * u.x + u.y * u.y) + ff.y * (u.z * u.z + u.w * u.w);
        }
        jx += (double)ax;
        jy += (double)ay;
        jz += (double)az;
        ne += (double)an;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        jx += __shfl_xor_sync(0xffffffffu, jx, o);
        jy += __shfl_xor_sync(0xffffffffu, jy, o);
        jz += __shfl_xor_sync(0xffffffffu, jz, o);
        ne += __shfl_xor_sync(0xffffffffu, ne, o);
    }
    __shared__ double red[8][4];
    if (lane == 0) {
        red[warp][0] = jx;
        red[warp][1] = jy;
        red[warp][2] = jz;
        red[warp][3] = ne;
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[w][threadIdx.x];
        part[((size_t)dom * nblk + blk) * 4 + threadIdx.x] = s;
    }
}
// The same sums with each x-plane read once: a block owns an 8(y) x 8(z) patch for one 64-byte orbital chunk
// (thread = point x float4 lane) and marches along x; the x taps come from a three-plane register history,
// the y/z taps are the patch neighbours' own centre loads (L1 hits), only the +2 halo rows add L2 traffic.
__global__ void __launch_bounds__(256)
current_march_kernel(int nx, int ny, int nz, int lanes, int xs, int nxseg, const float4 *__restrict__ psi,
                     const float *__restrict__ occ, float wx1, float wx2, float wy1, float wy2, float wz1, float wz2,
                     double *__restrict__ part) {
    const int l = threadIdx.x % 4, tz = (threadIdx.x / 4) % 8, ty = threadIdx.x / 32;
    int item = blockIdx.x;
    const int seg = item % nxseg;
    item /= nxseg;
    const int nzt = nz / 8, nyt = ny / 8, nchunk = lanes / 4;
    const int zt = item % nzt;
    item /= nzt;
    const int yt = item % nyt;
    item /= nyt;
    const int chunk = item % nchunk;
    const int dom = item / nchunk;
    const int y = yt * 8 + ty, z = zt * 8 + tz;
    const int y1 = y + 1 < ny ? y + 1 : y + 1 - ny, y2 = y + 2 < ny ? y + 2 : y + 2 - ny;
    const int z1 = z + 1 < nz ? z + 1 : z + 1 - nz, z2 = z + 2 < nz ? z + 2 : z + 2 - nz;
    const long sy = (long)nz * lanes, sx = (long)ny * sy;
    const float4 *base = psi + (size_t)dom * nx * sx + chunk * 4 + l;
    const long oc = (long)y * sy + (long)z * lanes;
    const long oy1 = (long)y1 * sy + (long)z * lanes, oy2 = (long)y2 * sy + (long)z * lanes;
    const long oz1 = (long)y * sy + (long)z1 * lanes, oz2 = (long)y * sy + (long)z2 * lanes;
    const float2 ff = __ldg((const float2 *)(occ + (size_t)dom * lanes * 2) + chunk * 4 + l);
    const int x0 = seg * xs, x1 = min(x0 + xs, nx);
    auto xw = [&](int x) { return x < nx ? x : x - nx; };
    float4 u0 = __ldg(base + (long)x0 * sx + oc), u1 = __ldg(base + (long)xw(x0 + 1) * sx + oc);
    float ax = 0.f, ay = 0.f, az = 0.f, an = 0.f;
    // unrolled so that the loads of several planes are in flight per thread (only one load in five is new HBM data)
#pragma unroll 4
    for (int x = x0; x < x1; ++x) {
        const float4 *pl = base + (long)x * sx;
        const float4 u2 = __ldg(base + (long)xw(x + 2) * sx + oc);
        const float4 vy1 = __ldg(pl + oy1), vy2 = __ldg(pl + oy2), vz1 = __ldg(pl + oz1), vz2 = __ldg(pl + oz2);
        auto im = [&](const float4 v) { return ff.x * (u0.x * v.y - u0.y * v.x) + ff.y * (u0.z * v.w - u0.w * v.z); };
        ax += wx1 * im(u1) + wx2 * im(u2);
        ay += wy1 * im(vy1) + wy2 * im(vy2);
        az += wz1 * im(vz1) + wz2 * im(vz2);
        an += ff.x * (u0.x * u0.x + u0.y * u0.y) + ff.y * (u0.z * u0.z + u0.w * u0.w);
        u0 = u1;
        u1 = u2;
    }
    double jx = (double)ax, jy = (double)ay, jz = (double)az, ne = (double)an;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        jx += __shfl_xor_sync(0xffffffffu, jx, o);
        jy += __shfl_xor_sync(0xffffffffu, jy, o);
        jz += __shfl_xor_sync(0xffffffffu, jz, o);
        ne += __shfl_xor_sync(0xffffffffu, ne, o);
    }
    __shared__ double red[8][4];
    if (threadIdx.x % 32 == 0) {
        red[ty][0] = jx;
        red[ty][1] = jy;
        red[ty][2] = jz;
        red[ty][3] = ne;
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double sum = 0.0;
        for (int w = 0; w < 8; ++w) sum += red[w][threadIdx.x];
        part[(size_t)blockIdx.x * 4 + threadIdx.x] = sum;      // blocks of one domain are contiguous
    }
}
// J[dom][d] = dv (sum_blk part[d] + A[dom or 0][d] * sum_blk part[3]); one thread per (dom, d)
__global__ void current_final_kernel(int ndom, int nblk, int a_ndom, double dv, const double *__restrict__ part,
                                     const double *__restrict__ A, double *__restrict__ J) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ndom * 3) return;
    const int dom = i / 3, d = i % 3;
    double s = 0.0, ne = 0.0;
    for (int b = 0; b < nblk; ++b) {
        s += part[((size_t)dom * nblk + b) * 4 + d];
        ne += part[((size_t)dom * nblk + b) * 4 + 3];
    }
    J[i] = dv * (s + A[(size_t)(a_ndom == 1 ? 0 : dom) * 3 + d] * ne);
}
cudaError_t launch_current(cudaStream_t st, int ndom, int nx, int ny, int nz, double hx, double hy, double hz, int ld,
                           const float2 *psi, const float *occ, const double *A_dev, int a_ndom, double *part,
                           size_t part_doubles, double *J, int fd_order, int *nlaunch) {
    const long ngrid = (long)nx * ny * nz;
    const long max_blk = (long)(part_doubles / 4 / ndom);
    if (max_blk < 1) return cudaErrorInvalidValue;
    // 2 c1_j / h_d: c1 = (2/3, -1/12), the 4th-order first difference (north_star), or (1/2, 0), the 2nd-order one
    const float w1 = fd_order == 2 ? 1.0f : (float)(2.0 * 2.0 / 3.0), w2 = fd_order == 2 ? 0.f : (float)(2.0 * -1.0 / 12.0);
    if (ny % 8 == 0 && nz % 8 == 0) {
        const long tiles = (long)(ld / 8) * (ny / 8) * (nz / 8);
        int nxseg = 1;
        while (tiles * ndom * nxseg < 4 * 148 && nx / (nxseg * 2) >= 8) nxseg *= 2;
        const int xs = (nx + nxseg - 1) / nxseg;
        nxseg = (nx + xs - 1) / xs;
        if (tiles * nxseg <= max_blk) {
            const int nblk = (int)(tiles * nxseg);
            *nlaunch += 2;
            current_march_kernel<<<(unsigned)(ndom * nblk), 256, 0, st>>>(nx, ny, nz, ld / 2, xs, nxseg, (const float4 *)psi, occ,
                                                                          (float)(w1 / hx), (float)(w2 / hx), (float)(w1 / hy),
                                                                          (float)(w2 / hy), (float)(w1 / hz), (float)(w2 / hz), part);
            current_final_kernel<<<(ndom * 3 + 127) / 128, 128, 0, st>>>(ndom, nblk, a_ndom, hx * hy * hz, part, A_dev, J);
            return cudaGetLastError();
        }
    }
    // any shape: one warp per point; points per block at least 64, and few enough blocks for the scratch
    long pts = 64;
    if ((ngrid + pts - 1) / pts > max_blk) pts = ((ngrid + max_blk - 1) / max_blk + 7) / 8 * 8;
    const int nblk = (int)((ngrid + pts - 1) / pts);
    *nlaunch += 2;
    current_part_kernel<<<ndom * nblk, 256, 0, st>>>(nx, ny, nz, ld / 2, (int)pts, nblk, (const float4 *)psi, occ,
                                                     (float)(w1 / hx), (float)(w2 / hx), (float)(w1 / hy), (float)(w2 / hy),
                                                     (float)(w1 / hz), (float)(w2 / hz), part);
    current_final_kernel<<<(ndom * 3 + 127) / 128, 128, 0, st>>>(ndom, nblk, a_ndom, hx * hy * hz, part, A_dev, J);
    return cudaGetLastError();
}

// ---- split step: ||psi + beta W||^2 without a pass over psi ----
// Static Gram matrix of the (real-embedded) projector rows, G[dom][p][q] = sum_r beta[r][p] beta[r][q], from the
// split-K partials of a projection of beta onto itself: G (+)= sum_s zpart[dom][s][p][q].
__global__ void gram_reduce_kernel(int P, int ldg, int prows, int N, int nsplit, const float *__restrict__ zpart,
                                   float *__restrict__ G, int accumulate) {
    const int qq = blockIdx.x * blockDim.x + threadIdx.x;
    const int p = blockIdx.y, dom = blockIdx.z;
    if (qq >= P) return;
    const float *zp = zpart + ((size_t)dom * nsplit * prows + p) * N + qq;
    float s = 0.f;
    for (int k = 0; k < nsplit; ++k) s += zp[(size_t)k * prows * N];
    float *g = G + ((size_t)dom * ldg + p) * ldg + qq;
    *g = accumulate ? *g + s : s;
}
cudaError_t launch_gram_reduce(cudaStream_t st, int ndom, int P, int ldg, int prows, int N, int nsplit, const float *zpart,
                               float *G, int accumulate, int *nlaunch) {
    ++*nlaunch;
    gram_reduce_kernel<<<dim3((P + 127) / 128, P, ndom), 128, 0, st>>>(P, ldg, prows, N, nsplit, zpart, G, accumulate);
    return cudaGetLastError();
}
// nd[dom][n] = nc[dom][n] + sum_{c in {2n, 2n+1}} W[:, c]^T G W[:, c], W = what + what_lo ([prows][2 ld], rows < P).
// The cross term 2 Re<psi|beta W> vanishes because W = -i tau D' beta^H psi with a Hermitian V_NL.
// Block = (domain, 32 columns): the W tile [P x 32] sits in shared memory; thread = (column, one of 8 slices of p),
// five rows of G per trip so that one shared-memory read of W feeds five FMAs; FP32 products, FP64 sums.
constexpr int KQ_MAXP = 1024;   // rows of W a block can stage (dynamic shared memory: P * 128 B)
__global__ void __launch_bounds__(256)
kick_quad_kernel(int P, int ldg, int ld, int prows, const float *__restrict__ G, const float *__restrict__ what,
                 const float *__restrict__ wlo, const double *__restrict__ nc, double *__restrict__ nd) {
    extern __shared__ float Ws[];    // [P][32]
    const int dom = blockIdx.y, lane = threadIdx.x % 32, c = blockIdx.x * 32 + lane, slice = threadIdx.x / 32;
    const int N = 2 * ld;
    const float *g = G + (size_t)dom * ldg * ldg;
    const float *wh = what + (size_t)dom * prows * N + c, *wl = wlo + (size_t)dom * prows * N + c;
    for (int p = slice; p < P; p += 8) Ws[p * 32 + lane] = wh[(size_t)p * N] + wl[(size_t)p * N];
    __syncthreads();
    double acc = 0.0;
    for (int p0 = slice * 5; p0 < P; p0 += 40) {
        float t[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
        const float *gr[5];
#pragma unroll
        for (int k = 0; k < 5; ++k) gr[k] = g + (size_t)min(p0 + k, P - 1) * ldg;
        for (int qq = 0; qq < P; ++qq) {
            const float w = Ws[qq * 32 + lane];
#pragma unroll
            for (int k = 0; k < 5; ++k) t[k] = fmaf(__ldg(gr[k] + qq), w, t[k]);
        }
#pragma unroll
        for (int k = 0; k < 5; ++k)
            if (p0 + k < P) acc += (double)Ws[(p0 + k) * 32 + lane] * (double)t[k];
    }
    __shared__ double red[8][32];
    red[slice][lane] = acc;
    __syncthreads();
    if (threadIdx.x < 16) {             // orbital n = columns 2n, 2n+1
        double s = 0.0;
        for (int k = 0; k < 8; ++k) s += red[k][2 * threadIdx.x] + red[k][2 * threadIdx.x + 1];
        const int n = blockIdx.x * 16 + threadIdx.x;
        if (n < ld) nd[(size_t)dom * ld + n] = nc[(size_t)dom * ld + n] + s;
    }
}
cudaError_t launch_kick_quad(cudaStream_t st, int ndom, int P, int ldg, int ld, int prows, const float *G, const float *what,
                             const float *wlo, const double *nc, double *nd, int *nlaunch) {
    ++*nlaunch;
    if (P > KQ_MAXP) return cudaErrorInvalidValue;
    static DeviceOnce attr_set;
    if (!attr_set.done()) {
        cudaError_t e = cudaFuncSetAttribute(kick_quad_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, KQ_MAXP * 128);
        if (e != cudaSuccess) return e;
        attr_set.mark();
    }
    kick_quad_kernel<<<dim3(2 * ld / 32, ndom), 256, (size_t)P * 128, st>>>(P, ldg, ld, prows, G, what, wlo, nc, nd);
    return cudaGetLastError();
}

// occ_eff[i] = occ[i] * scl[i]^2: the density of the true (normalised) orbitals from the un-normalised ones in memory
__global__ void occ_eff_kernel(int n, const float *__restrict__ occ, const float *__restrict__ scl, float *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = occ[i] * scl[i] * scl[i];
}
cudaError_t launch_occ_eff(cudaStream_t st, int n, const float *occ, const float *scl, float *out, int *nlaunch) {
    ++*nlaunch;
    occ_eff_kernel<<<(n + 127) / 128, 128, 0, st>>>(n, occ, scl, out);
    return cudaGetLastError();
}

}  // namespace mlmd
