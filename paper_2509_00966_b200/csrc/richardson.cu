// The paper's own local solver: block-diagonal split-operator (space splitting) on 2nd-order differences
// ("a block-diagonal split-operator solver for electronic wave functions [41]" performing "uniform
// operations on nearest-neighbor mesh points"; L283 "7-point star stencil"; reading D33).
//
//   U_loc(dt) = P(dt/2)  S_x S_y S_z  P(dt/2),     P(tau) = exp(-i tau (V_loc(r) + 1/2|A|^2 + sum_d 1/h_d^2)),
//   S_d = R_d^even(dt/2) R_d^odd(dt) R_d^even(dt/2),
//   R_d(tau) on a pair (j, j+1):  [[cos(tau|b|), -i u sin(tau|b|)], [-i conj(u) sin(tau|b|), cos(tau|b|)]],
//   b = -1/(2 h_d^2) - i A_d/(2 h_d),  u = b/|b|
// (the scalar phases e^{-i tau a_d/2} of the 2 x 2 block exponentials, a_d = 1/h_d^2, are the same for every point and add
// up to e^{-i dt sum_d a_d} per step: they ride in P, whose argument is then V_loc + the `centre` of the 2nd-order StepCoef).
//
// One pass per axis, in place (16 B per element and pass: 48 B per step against 88 B for the Taylor sum): a thread owns the
// EVEN pair (2p, 2p+1) of its line for one float4 (two orbitals), so the two even sweeps are register-only; for the odd sweep
// the even points go through shared memory once (thread p rotates its point 2p+1 with point 2p+2 of thread p+1; the last
// pair wraps, which is why every axis needs an even number of points).  Eight float4 lanes per line keep every access a full
// 128-byte line whatever the axis.  The rotation constants are computed in FP64 per thread and applied as hi + lo pairs of
// floats: a rounded (cos, sin) pair is off the unit circle by ~6e-8, the SAME factor on every point in every sweep, which
// would be a coherent norm drift of ~5e-7 per step; with the pair the remaining error is the FP32 rounding of the products.
#include "mlmd_internal.h"

namespace mlmd {

namespace {

constexpr int R_LG = 8;       // float4 lanes per line and thread group: 128 bytes

struct RichParams {
    float4 *psi;
    const float *vloc;
    const StepCoef *coef;     // [ndom], 2nd-order weights (fill_coef with the 7-point star)
    double dt;
    int axis;                 // 0 = x, 1 = y, 2 = z
    int n;                    // points along the axis
    long sa;                  // stride along the axis, float4 units
    int n1, n2;               // the two other axes
    long s1, s2;
    long sdom;                // float4 per domain
    int lanes;                // float4 per grid point
    int ngroups;              // lanes / R_LG
    long nlines;              // ndom * n1 * n2 * ngroups
    int nlb;                  // lines per block
};

struct Rot {                  // (c, wr + i wi) = (cos, -i u sin) as hi + lo floats
    float c, cl, wr, wrl, wi, wil;
};
__device__ __forceinline__ Rot make_rot(double theta, double ur, double ui) {
    double s, c;
    sincos(theta, &s, &c);
    const double wr = s * ui, wi = -s * ur;     // -i (ur + i ui) s
    Rot r;
    r.c = (float)c;
    r.cl = (float)(c - (double)r.c);
    r.wr = (float)wr;
    r.wrl = (float)(wr - (double)r.wr);
    r.wi = (float)wi;
    r.wil = (float)(wi - (double)r.wi);
    return r;
}
// one complex number: c * a + (wr + i wi) * b, every constant as hi + lo
__device__ __forceinline__ float2 rot1(const Rot &r, float ax, float ay, float bx, float by, bool conj_w) {
    // upper row: w = (wr, wi); lower row: w' = -i conj(u) s = (-wr, wi)
    const float wr = conj_w ? -r.wr : r.wr, wrl = conj_w ? -r.wrl : r.wrl;
    float lo = fmaf(r.cl, ax, fmaf(wrl, bx, -r.wil * by));
    float x = fmaf(r.c, ax, fmaf(wr, bx, fmaf(-r.wi, by, lo)));
    float lo2 = fmaf(r.cl, ay, fmaf(wrl, by, r.wil * bx));
    float y = fmaf(r.c, ay, fmaf(wr, by, fmaf(r.wi, bx, lo2)));
    return make_float2(x, y);
}
// (a, b) <- R (a, b) for both complex numbers of the float4s; a is the lower-index point of the pair
__device__ __forceinline__ void rotate(const Rot &r, float4 &a, float4 &b) {
    const float2 a0 = rot1(r, a.x, a.y, b.x, b.y, false), a1 = rot1(r, a.z, a.w, b.z, b.w, false);
    const float2 b0 = rot1(r, b.x, b.y, a.x, a.y, true), b1 = rot1(r, b.z, b.w, a.z, a.w, true);
    a = make_float4(a0.x, a0.y, a1.x, a1.y);
    b = make_float4(b0.x, b0.y, b1.x, b1.y);
}
__device__ __forceinline__ float4 phase4(const float4 v, float cs, float sn) {
    return make_float4(v.x * cs - v.y * sn, v.x * sn + v.y * cs, v.z * cs - v.w * sn, v.z * sn + v.w * cs);
}

template <bool PHASE_IN, bool PHASE_OUT>
__global__ void __launch_bounds__(1024) richardson_axis_kernel(const RichParams P) {
    extern __shared__ float4 ev[];      // [nlb][n / 2][R_LG]: the even points of every line of the block
    const int np = P.n / 2;
    const int tid = threadIdx.x;
    const int l = tid % R_LG, p = (tid / R_LG) % np, ql = tid / (R_LG * np);
    long line = (long)blockIdx.x * P.nlb + ql;
    const bool live = line < P.nlines;
    if (!live) line = P.nlines - 1;     // keeps the barriers uniform; nothing is stored
    const int g = (int)(line % P.ngroups);
    long rest = line / P.ngroups;
    const int i2 = (int)(rest % P.n2);
    rest /= P.n2;
    const int i1 = (int)(rest % P.n1);
    const int dom = (int)(rest / P.n1);
    const long base = (long)dom * P.sdom + i1 * P.s1 + i2 * P.s2 + g * R_LG + l;
    const long ad0 = base + (long)(2 * p) * P.sa, ad1 = ad0 + P.sa;

    const StepCoef c = P.coef[dom];
    const double bp = (double)c.p[P.axis][0], bq = (double)c.q[P.axis][0];      // b = bp - i bq
    const double mb = sqrt(bp * bp + bq * bq);
    const double ur = bp / mb, ui = -bq / mb;
    const Rot rh = make_rot(0.5 * P.dt * mb, ur, ui), rf = make_rot(P.dt * mb, ur, ui);

    float4 u0 = P.psi[ad0], u1 = P.psi[ad1];
    float cs0 = 1.f, sn0 = 0.f, cs1 = 1.f, sn1 = 0.f;
    if (PHASE_IN || PHASE_OUT) {
        const float half = (float)(-0.5 * P.dt);
        sincosf(half * (P.vloc[ad0 / P.lanes] + c.centre), &sn0, &cs0);
        sincosf(half * (P.vloc[ad1 / P.lanes] + c.centre), &sn1, &cs1);
    }
    if (PHASE_IN) {
        u0 = phase4(u0, cs0, sn0);
        u1 = phase4(u1, cs1, sn1);
    }
    rotate(rh, u0, u1);                                   // even pairs, dt/2
    float4 *mine = ev + ((size_t)ql * np + p) * R_LG + l;
    float4 *next = ev + ((size_t)ql * np + (p + 1 == np ? 0 : p + 1)) * R_LG + l;
    *mine = u0;
    __syncthreads();
    {
        float4 w = *next;                                 // point 2p + 2 (periodic)
        rotate(rf, u1, w);                                // odd pairs, dt
        *next = w;
    }
    __syncthreads();
    u0 = *mine;
    rotate(rh, u0, u1);                                   // even pairs, dt/2
    if (PHASE_OUT) {
        u0 = phase4(u0, cs0, sn0);
        u1 = phase4(u1, cs1, sn1);
    }
    if (live) {
        P.psi[ad0] = u0;
        P.psi[ad1] = u1;
    }
}

}  // namespace

bool richardson_supported(const mlmd_domain *h) {
    const int n[3] = {h->nx, h->ny, h->nz};
    for (int d = 0; d < 3; ++d)
        if (n[d] % 2 || n[d] / 2 * R_LG > 1024) return false;
    return h->ld % 16 == 0;     // lanes = ld / 2 float4 per point, a multiple of R_LG
}

// psi <- U_loc(dt) psi in place: three launches (z with the leading phase, y, x with the trailing phase).
cudaError_t launch_richardson(const mlmd_domain *h, float2 *psi, const StepCoef *coef, double dt, int *nlaunch) {
    if (!richardson_supported(h)) return cudaErrorInvalidValue;
    const int lanes = h->ld / 2;
    const int n[3] = {h->nx, h->ny, h->nz};
    const long stride[3] = {(long)h->ny * h->nz * lanes, (long)h->nz * lanes, (long)lanes};
    static const int order[3] = {2, 1, 0};
    for (int k = 0; k < 3; ++k) {
        const int d = order[k], o1 = (d + 1) % 3, o2 = (d + 2) % 3;
        RichParams P;
        P.psi = (float4 *)psi;
        P.vloc = h->vloc();
        P.coef = coef;
        P.dt = dt;
        P.axis = d;
        P.n = n[d];
        P.sa = stride[d];
        P.n1 = n[o1];
        P.s1 = stride[o1];
        P.n2 = n[o2];
        P.s2 = stride[o2];
        P.sdom = (long)h->ngrid * lanes;
        P.lanes = lanes;
        P.ngroups = lanes / R_LG;
        P.nlines = (long)h->ndom * P.n1 * P.n2 * P.ngroups;
        const int tpl = (P.n / 2) * R_LG;                 // threads per line
        P.nlb = tpl >= 256 ? 1 : 256 / tpl;
        const long blocks = (P.nlines + P.nlb - 1) / P.nlb;
        if (blocks > 0x7fffffffL) return cudaErrorInvalidConfiguration;
        const size_t smem = (size_t)P.nlb * (P.n / 2) * R_LG * sizeof(float4);
        const dim3 grid((unsigned)blocks), block((unsigned)(tpl * P.nlb));
        ++*nlaunch;
        if (k == 0) richardson_axis_kernel<true, false><<<grid, block, smem, h->stream>>>(P);
        else if (k == 2) richardson_axis_kernel<false, true><<<grid, block, smem, h->stream>>>(P);
        else richardson_axis_kernel<false, false><<<grid, block, smem, h->stream>>>(P);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace mlmd
