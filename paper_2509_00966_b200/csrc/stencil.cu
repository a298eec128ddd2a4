// Fused kinetic stencil / local potential / Horner update (north_star kernel 2).
//
//   out(r,n) = psi(r,n) + (-i tau) * [ sum_{d in xyz} sum_{j=1,2} ( p_dj (w(r+j e_d) + w(r-j e_d))
//                                                             - i q_dj (w(r+j e_d) - w(r-j e_d)) )
//                                      + (centre + V_loc(r)) w(r,n) ]
//
// which is -1/2 D2 - i A.D1 + 1/2|A|^2 + V_loc of PAPER.md Eq. (3) (L142) in 4th-order central
// differences, periodic in x, y, z, followed by one Horner stage of the Taylor-4 propagator.  The
// nonlocal term beta (D C) is added by the back-application GEMM.
//
// Layout: [dom][ix][iy][iz][ld] complex64, orbital fastest.  One thread owns one
// float4 = two orbitals of one grid column and marches along x with a five-deep register ring, so
// the x-neighbours cost no memory traffic; the y/z neighbours of the centre plane come through L1.
#include "mlmd_internal.h"

namespace mlmd {

struct StencilParams {
    const float4 *w;
    const float4 *psi;
    float4 *out;
    const float *vloc;
    const StepCoef *coef;   // [ndom]
    float tau;
    int nx, ny, nz;
    int lanes;              // float4 per grid point = ld / 2
    int xseg;               // planes per CTA
    int nxseg;
};

__device__ __forceinline__ float4 ldg4(const float4 *p) { return __ldg(p); }

// acc += p * (a + b)  - i q (a - b)  applied to both complex numbers held in a float4
__device__ __forceinline__ void pair_term(float4 &acc, const float4 a, const float4 b, const float p, const float q) {
    acc.x = fmaf(p, a.x + b.x, acc.x);
    acc.y = fmaf(p, a.y + b.y, acc.y);
    acc.z = fmaf(p, a.z + b.z, acc.z);
    acc.w = fmaf(p, a.w + b.w, acc.w);
    acc.x = fmaf(q, a.y - b.y, acc.x);
    acc.y = fmaf(-q, a.x - b.x, acc.y);
    acc.z = fmaf(q, a.w - b.w, acc.z);
    acc.w = fmaf(-q, a.z - b.z, acc.w);
}
__device__ __forceinline__ void pair_term_real(float4 &acc, const float4 a, const float4 b, const float p) {
    acc.x = fmaf(p, a.x + b.x, acc.x);
    acc.y = fmaf(p, a.y + b.y, acc.y);
    acc.z = fmaf(p, a.z + b.z, acc.z);
    acc.w = fmaf(p, a.w + b.w, acc.w);
}
__device__ __forceinline__ float4 horner_out(const float4 ps, const float4 acc, const float tau) {
    // psi + (-i tau) acc
    return make_float4(fmaf(tau, acc.y, ps.x), fmaf(-tau, acc.x, ps.y), fmaf(tau, acc.w, ps.z),
                       fmaf(-tau, acc.z, ps.w));
}

// ---------------------------------------------------------------------------------------------
// Reference-grade kernel: one thread per output float4, all 13 taps straight from global memory.
// Any grid shape with every axis >= 5.  Kept as the fallback for shapes the marching kernel's
// tiling does not divide, and as the in-library cross-check (MLMD_STENCIL=simple).
__global__ void __launch_bounds__(256) stencil_simple_kernel(StencilParams P, long total) {
    const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= total) return;
    const int lane = (int)(t % P.lanes);
    long r = t / P.lanes;
    const int iz = (int)(r % P.nz);
    r /= P.nz;
    const int iy = (int)(r % P.ny);
    r /= P.ny;
    const int ix = (int)(r % P.nx);
    const int dom = (int)(r / P.nx);
    const StepCoef c = P.coef[dom];
    const long sz = P.lanes, sy = sz * P.nz, sx = sy * P.ny;
    const float4 *wd = P.w + (long)dom * sx * P.nx + lane;
    auto at = [&](int x, int y, int z) { return ldg4(wd + x * sx + y * sy + z * sz); };
    auto wr = [](int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); };
    const long pt = (((long)dom * P.nx + ix) * P.ny + iy) * P.nz + iz;
    const float4 u0 = at(ix, iy, iz);
    const float cen = c.centre + P.vloc[pt];
    float4 acc = make_float4(cen * u0.x, cen * u0.y, cen * u0.z, cen * u0.w);
#pragma unroll
    for (int j = 1; j <= 2; ++j) {
        pair_term(acc, at(wr(ix + j, P.nx), iy, iz), at(wr(ix - j, P.nx), iy, iz), c.p[0][j - 1], c.q[0][j - 1]);
        pair_term(acc, at(ix, wr(iy + j, P.ny), iz), at(ix, wr(iy - j, P.ny), iz), c.p[1][j - 1], c.q[1][j - 1]);
        pair_term(acc, at(ix, iy, wr(iz + j, P.nz)), at(ix, iy, wr(iz - j, P.nz)), c.p[2][j - 1], c.q[2][j - 1]);
    }
    const long e = pt * P.lanes + lane;
    P.out[e] = horner_out(P.psi[e], acc, P.tau);   // plain load: out may alias psi
}

// ---------------------------------------------------------------------------------------------
// Marching kernel.  Block = (CL lanes, TZ, TY) threads covering a TY x TZ patch of the y-z plane for
// CL float4 lanes (CL*16 contiguous bytes per grid point); it walks `xseg` planes along x.
// AYZ: whether A_y or A_z is non-zero for any domain of this step (the configs' pulse is
// x-polarised, so the y/z taps are real and cost half the FMAs).
template <int CL, int TZ, int TY, bool AYZ>
__global__ void __launch_bounds__(CL *TZ *TY) stencil_march_kernel(StencilParams P) {
    const int lane = blockIdx.x * CL + threadIdx.x;
    const int nzt = P.nz / TZ;
    const int iz = (blockIdx.y % nzt) * TZ + threadIdx.y;
    const int iy = (blockIdx.y / nzt) * TY + threadIdx.z;
    const int seg = blockIdx.z % P.nxseg;
    const int dom = blockIdx.z / P.nxseg;
    if (lane >= P.lanes) return;
    const StepCoef c = P.coef[dom];
    const long sz = P.lanes, sy = sz * P.nz, sx = sy * P.ny;
    const long dbase = (long)dom * sx * P.nx;
    const float4 *wd = P.w + dbase + lane;
    auto wr = [](int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); };
    // neighbour offsets inside the plane (periodic)
    const long col = iy * sy + iz * sz;
    const long oyp1 = wr(iy + 1, P.ny) * sy + iz * sz, oym1 = wr(iy - 1, P.ny) * sy + iz * sz;
    const long oyp2 = wr(iy + 2, P.ny) * sy + iz * sz, oym2 = wr(iy - 2, P.ny) * sy + iz * sz;
    const long ozp1 = iy * sy + wr(iz + 1, P.nz) * sz, ozm1 = iy * sy + wr(iz - 1, P.nz) * sz;
    const long ozp2 = iy * sy + wr(iz + 2, P.nz) * sz, ozm2 = iy * sy + wr(iz - 2, P.nz) * sz;

    const int x0 = seg * P.xseg;
    const int x1 = min(x0 + P.xseg, P.nx);
    float4 rm2 = ldg4(wd + wr(x0 - 2, P.nx) * sx + col);
    float4 rm1 = ldg4(wd + wr(x0 - 1, P.nx) * sx + col);
    float4 r0 = ldg4(wd + x0 * sx + col);
    float4 rp1 = ldg4(wd + wr(x0 + 1, P.nx) * sx + col);
    float4 rp2 = ldg4(wd + wr(x0 + 2, P.nx) * sx + col);
    const float4 *psid = P.psi + dbase + lane + col;
    float4 *outd = P.out + dbase + lane + col;
    const float *vd = P.vloc + ((long)dom * P.nx * P.ny + iy) * P.nz + iz;
    float4 ps = psid[x0 * sx];   // plain loads: `out` may alias `psi` (last Horner stage is in place)
    float vv = __ldg(vd + (long)x0 * P.ny * P.nz);

    for (int ix = x0; ix < x1; ++ix) {
        // prefetch the plane three ahead and next psi / V
        const float4 nxt = ldg4(wd + wr(ix + 3, P.nx) * sx + col);
        const int ixn = (ix + 1 < x1) ? ix + 1 : ix;
        const float4 psn = psid[ixn * sx];
        const float vn = __ldg(vd + (long)ixn * P.ny * P.nz);
        const float4 *pl = wd + ix * sx;
        const float4 yp1 = ldg4(pl + oyp1), ym1 = ldg4(pl + oym1), yp2 = ldg4(pl + oyp2), ym2 = ldg4(pl + oym2);
        const float4 zp1 = ldg4(pl + ozp1), zm1 = ldg4(pl + ozm1), zp2 = ldg4(pl + ozp2), zm2 = ldg4(pl + ozm2);
        const float cen = c.centre + vv;
        float4 acc = make_float4(cen * r0.x, cen * r0.y, cen * r0.z, cen * r0.w);
        pair_term(acc, rp1, rm1, c.p[0][0], c.q[0][0]);
        pair_term(acc, rp2, rm2, c.p[0][1], c.q[0][1]);
        if (AYZ) {
            pair_term(acc, yp1, ym1, c.p[1][0], c.q[1][0]);
            pair_term(acc, yp2, ym2, c.p[1][1], c.q[1][1]);
            pair_term(acc, zp1, zm1, c.p[2][0], c.q[2][0]);
            pair_term(acc, zp2, zm2, c.p[2][1], c.q[2][1]);
        } else {
            pair_term_real(acc, yp1, ym1, c.p[1][0]);
            pair_term_real(acc, yp2, ym2, c.p[1][1]);
            pair_term_real(acc, zp1, zm1, c.p[2][0]);
            pair_term_real(acc, zp2, zm2, c.p[2][1]);
        }
        outd[ix * sx] = horner_out(ps, acc, P.tau);
        rm2 = rm1;
        rm1 = r0;
        r0 = rp1;
        rp1 = rp2;
        rp2 = nxt;
        ps = psn;
        vv = vn;
    }
}

template <int CL, int TZ, int TY>
static cudaError_t launch_march(const StencilParams &P, int ndom, bool ayz, cudaStream_t st) {
    dim3 block(CL, TZ, TY);
    dim3 grid((P.lanes + CL - 1) / CL, (P.nz / TZ) * (P.ny / TY), P.nxseg * ndom);
    if (ayz)
        stencil_march_kernel<CL, TZ, TY, true><<<grid, block, 0, st>>>(P);
    else
        stencil_march_kernel<CL, TZ, TY, false><<<grid, block, 0, st>>>(P);
    return cudaGetLastError();
}

cudaError_t launch_stencil_stage(const mlmd_domain *h, const float2 *w, const float2 *psi, float2 *out,
                                 const StepCoef *coef, const StepCoef *coef_host, float tau, int *nlaunch) {
    StencilParams P;
    P.w = (const float4 *)w;
    P.psi = (const float4 *)psi;
    P.out = (float4 *)out;
    P.vloc = h->vloc();
    P.coef = coef;
    P.tau = tau;
    P.nx = h->nx;
    P.ny = h->ny;
    P.nz = h->nz;
    P.lanes = h->ld / 2;
    const int variant = h->opt[MLMD_OPT_STENCIL];   // 0: TMA planes when the shape allows, 1: register marching, 2: simple
    if (variant == 0 && stencil_tma_supported(h)) return launch_stencil_tma(h, w, psi, out, coef, coef_host, tau, nlaunch);
    ++*nlaunch;
    const bool tile_ok = (h->ny % 8 == 0) && (h->nz % 8 == 0);
    if (variant == 2 || !tile_ok) {
        const long total = (long)h->ndom * h->ngrid * P.lanes;
        P.xseg = P.nxseg = 1;
        stencil_simple_kernel<<<(unsigned)((total + 255) / 256), 256, 0, h->stream>>>(P, total);
        return cudaGetLastError();
    }
    const bool ayz = h->field_yz;   // decided on the host per propagate call
    // x segmentation: enough CTAs for >= 4 waves of 148 SMs x 2 CTAs, segments of >= 8 planes
    const long ctas_per_seg = (long)((P.lanes + 7) / 8) * (h->ny / 8) * (h->nz / 8) * h->ndom;
    int nxseg = 1;
    while (ctas_per_seg * nxseg < 4 * 296 && h->nx / (nxseg * 2) >= 8) nxseg *= 2;
    P.xseg = (h->nx + nxseg - 1) / nxseg;
    P.nxseg = (h->nx + P.xseg - 1) / P.xseg;
    if (P.lanes % 8 == 0 || P.lanes > 8)
        return launch_march<8, 8, 8>(P, h->ndom, ayz, h->stream);
    return launch_march<4, 8, 8>(P, h->ndom, ayz, h->stream);
}

cudaError_t launch_stencil_stage_norm(const mlmd_domain *h, const float2 *w, const float2 *psi, float2 *out,
                                      const StepCoef *coef, const StepCoef *coef_host, float tau, int norm_mode,
                                      double *npart, double *nrm_out, int *nlaunch) {
    if (h->opt[MLMD_OPT_STENCIL] == 0 && stencil_tma_supported(h)) {
        const int slots = stencil_tma_norm_slots(h);
        if (slots <= kNormSlabs) {     // npart holds kNormSlabs partial rows per domain
            cudaError_t e = launch_stencil_tma(h, w, psi, out, coef, coef_host, tau, nlaunch, norm_mode, npart);
            return e != cudaSuccess ? e : launch_colnorm_final(h->stream, h->ndom, h->ld, slots, npart, nrm_out, nlaunch);
        }
    }
    // w may alias out only through psi (Horner buffers), never directly, so w is intact after the stage
    cudaError_t e = launch_stencil_stage(h, w, psi, out, coef, coef_host, tau, nlaunch);
    if (e != cudaSuccess) return e;
    return launch_colnorm2(h->stream, h->ndom, h->ngrid, h->ld, norm_mode == 1 ? w : out, npart, nrm_out, nlaunch);
}

}  // namespace mlmd
