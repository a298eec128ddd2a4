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
// EVEN pair (2p, 2p+1) of its line for one or two float4 (two or four orbitals), so the two even sweeps are register-only; for
// the odd sweep the even points go through shared memory once (thread p rotates its point 2p+1 with point 2p+2 of thread p+1;
// the last pair wraps, which is why every axis needs an even number of points).  Eight threads side by side on a point keep
// every access a full 128-byte line (two of them with two float4 per thread) whatever the axis.  The rotation constants of a step are computed in FP64 by a one-block kernel ahead of the
// three passes (from the step's device-resident StepCoef, so a CUDA graph replays them); a rounded (cos, sin) pair is off the
// unit circle by ~6e-8, the SAME factor on every point in every sweep: the last pass takes the product of the nine factors out
// again (see make_rot), so what remains is the FP32 rounding of the products.
#include "mlmd_internal.h"

namespace mlmd {

namespace {

constexpr int R_LG = 8;       // float4 lanes per line and thread group: 128 bytes

struct AxisConst;
struct RichParams {
    float4 *psi;
    const AxisConst *consts;  // [ndom][3], written by richardson_consts_kernel for this step
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
    int nlines;               // ndom * n1 * n2 * ngroups
    int nlb;                  // lines per block
    long pa, p1, p2, pdom;    // the same strides in grid points (index into V_loc)
};

struct Rot {                  // (c, wr + i wi) = (cos, -i u sin), rounded to float
    float c, wr, wi;
};
struct AxisConst {            // one per (domain, axis) and step: 8 floats in the handle's workspace
    Rot half, full;
    float excess;             // axis 0 only: 1 / (product of the nine sweeps' scale factors) - 1
    float pad;
};
static_assert(sizeof(AxisConst) == 32, "AxisConst layout");

// The rounded triple is sqrt(c^2 + wr^2 + wi^2) times an exactly unitary 2 x 2 matrix (its off-diagonal entries are each
// other's negated conjugates bit for bit): that factor, 1 +- 6e-8 and the SAME on every pair in every sweep, would be a
// coherent norm drift.  The constants kernel returns the product of all nine factors (FP64) as `excess` = 1/product - 1
// (a number of size 1e-7 kept to 24 bits), and the last pass multiplies by 1 + excess.
__device__ __forceinline__ Rot make_rot(double theta, double ur, double ui, double *scale) {
    double s, c;
    sincos(theta, &s, &c);
    Rot r;
    r.c = (float)c;
    r.wr = (float)(s * ui);        // -i (ur + i ui) s
    r.wi = (float)(-s * ur);
    *scale *= sqrt((double)r.c * r.c + (double)r.wr * r.wr + (double)r.wi * r.wi);
    return r;
}
// One thread per domain: the constants of the step for the three axes, in FP64, once per step instead of once per thread
// block (B200 has little FP64 throughput: with every thread computing them the three passes took twice as long).
__global__ void richardson_consts_kernel(const StepCoef *__restrict__ coef, double dt, int ndom, AxisConst *__restrict__ out) {
    const int dom = blockIdx.x * blockDim.x + threadIdx.x;
    if (dom >= ndom) return;
    const StepCoef c = coef[dom];
    double sc_all = 1.0;
    AxisConst k[3];
    for (int d = 0; d < 3; ++d) {
        const double bp = (double)c.p[d][0], bq = (double)c.q[d][0];      // b = bp - i bq
        const double mb = sqrt(bp * bp + bq * bq);
        const double ur = bp / mb, ui = -bq / mb;
        double sc = 1.0;
        k[d].half = make_rot(0.5 * dt * mb, ur, ui, &sc);
        sc *= sc;                                                         // two half sweeps
        k[d].full = make_rot(dt * mb, ur, ui, &sc);
        sc_all *= sc;
        k[d].excess = 0.f;
        k[d].pad = 0.f;
    }
    k[0].excess = (float)(1.0 / sc_all - 1.0);
    for (int d = 0; d < 3; ++d) out[dom * 3 + d] = k[d];
}

// (a, b) <- R (a, b) for both complex numbers of the float4s; a is the lower-index point of the pair:
// a' = c a + w b, b' = w' a + c b with w = (wr, wi), w' = -i conj(u) s = (-wr, wi)
__device__ __forceinline__ void rotate(const Rot &r, float4 &a, float4 &b) {
    const float4 x = a, y = b;
    a.x = fmaf(r.c, x.x, fmaf(r.wr, y.x, -r.wi * y.y));
    a.y = fmaf(r.c, x.y, fmaf(r.wr, y.y, r.wi * y.x));
    a.z = fmaf(r.c, x.z, fmaf(r.wr, y.z, -r.wi * y.w));
    a.w = fmaf(r.c, x.w, fmaf(r.wr, y.w, r.wi * y.z));
    b.x = fmaf(r.c, y.x, fmaf(-r.wr, x.x, -r.wi * x.y));
    b.y = fmaf(r.c, y.y, fmaf(-r.wr, x.y, r.wi * x.x));
    b.z = fmaf(r.c, y.z, fmaf(-r.wr, x.z, -r.wi * x.w));
    b.w = fmaf(r.c, y.w, fmaf(-r.wr, x.w, r.wi * x.z));
}
// v (cs + i sn) (1 + ex)
__device__ __forceinline__ float4 phase4(const float4 v, float cs, float sn, float ex) {
    const float4 p = make_float4(v.x * cs - v.y * sn, v.x * sn + v.y * cs, v.z * cs - v.w * sn, v.z * sn + v.w * cs);
    return make_float4(fmaf(ex, p.x, p.x), fmaf(ex, p.y, p.y), fmaf(ex, p.z, p.z), fmaf(ex, p.w, p.w));
}

// LPT: float4 lanes per thread (2 when the lane count allows: the index arithmetic and the phases are shared)
template <bool PHASE_IN, bool PHASE_OUT, int LPT>
__global__ void __launch_bounds__(1024) richardson_axis_kernel(const RichParams P) {
    extern __shared__ float4 ev[];      // [nlb][n / 2][LPT * R_LG]: the even points of every line of the block
    constexpr int LW = LPT * R_LG;      // float4 per line and point
    const int np = P.n / 2;
    const int tid = threadIdx.x;
    const int l = tid % R_LG, p = (tid / R_LG) % np, ql = tid / (R_LG * np);
    int line = (int)blockIdx.x * P.nlb + ql;
    const bool live = line < P.nlines;
    if (!live) line = P.nlines - 1;     // keeps the barriers uniform; nothing is stored
    const int g = line % P.ngroups;
    int rest = line / P.ngroups;
    const int i2 = rest % P.n2;
    rest /= P.n2;
    const int i1 = rest % P.n1;
    const int dom = rest / P.n1;
    const long base = (long)dom * P.sdom + i1 * P.s1 + i2 * P.s2 + g * LW + l;
    const long ad0 = base + (long)(2 * p) * P.sa, ad1 = ad0 + P.sa;
    const long gp0 = (long)dom * P.pdom + i1 * P.p1 + i2 * P.p2 + (long)(2 * p) * P.pa, gp1 = gp0 + P.pa;

    float4 u0[LPT], u1[LPT];
#pragma unroll
    for (int k = 0; k < LPT; ++k) {
        u0[k] = P.psi[ad0 + k * R_LG];
        u1[k] = P.psi[ad1 + k * R_LG];
    }
    const AxisConst ac = P.consts[dom * 3 + P.axis];
    const Rot rh = ac.half, rf = ac.full;
    float cs0 = 1.f, sn0 = 0.f, cs1 = 1.f, sn1 = 0.f, ex = 0.f;
    if (PHASE_IN || PHASE_OUT) {
        const float centre = P.coef[dom].centre;
        const float half = (float)(-0.5 * P.dt);
        sincosf(half * (P.vloc[gp0] + centre), &sn0, &cs0);
        sincosf(half * (P.vloc[gp1] + centre), &sn1, &cs1);
        if (PHASE_OUT) ex = P.consts[dom * 3].excess;
    }
    float4 *mine = ev + ((size_t)ql * np + p) * LW + l;
    float4 *next = ev + ((size_t)ql * np + (p + 1 == np ? 0 : p + 1)) * LW + l;
#pragma unroll
    for (int k = 0; k < LPT; ++k) {
        if (PHASE_IN) {
            u0[k] = phase4(u0[k], cs0, sn0, 0.f);
            u1[k] = phase4(u1[k], cs1, sn1, 0.f);
        }
        rotate(rh, u0[k], u1[k]);                         // even pairs, dt/2
        mine[k * R_LG] = u0[k];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < LPT; ++k) {
        float4 w = next[k * R_LG];                        // point 2p + 2 (periodic)
        rotate(rf, u1[k], w);                             // odd pairs, dt
        next[k * R_LG] = w;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < LPT; ++k) {
        u0[k] = mine[k * R_LG];
        rotate(rh, u0[k], u1[k]);                         // even pairs, dt/2
        if (PHASE_OUT) {
            u0[k] = phase4(u0[k], cs0, sn0, ex);
            u1[k] = phase4(u1[k], cs1, sn1, ex);
        }
        if (live) {
            P.psi[ad0 + k * R_LG] = u0[k];
            P.psi[ad1 + k * R_LG] = u1[k];
        }
    }
}

}  // namespace

bool richardson_supported(const mlmd_domain *h) {
    const int n[3] = {h->nx, h->ny, h->nz};
    for (int d = 0; d < 3; ++d)
        if (n[d] % 2 || n[d] / 2 * R_LG > 1024) return false;
    return h->ld % 16 == 0;     // lanes = ld / 2 float4 per point, a multiple of R_LG
}

// psi <- U_loc(dt) psi in place: the constants kernel and three passes (z with the leading phase, y, x with the trailing phase).
cudaError_t launch_richardson(const mlmd_domain *h, float2 *psi, const StepCoef *coef, double dt, int *nlaunch) {
    if (!richardson_supported(h)) return cudaErrorInvalidValue;
    const int lanes = h->ld / 2;
    const int n[3] = {h->nx, h->ny, h->nz};
    const long stride[3] = {(long)h->ny * h->nz * lanes, (long)h->nz * lanes, (long)lanes};
    static const int order[3] = {2, 1, 0};
    AxisConst *consts = (AxisConst *)h->rich();
    ++*nlaunch;
    richardson_consts_kernel<<<(h->ndom + 63) / 64, 64, 0, h->stream>>>(coef, dt, h->ndom, consts);
    for (int k = 0; k < 3; ++k) {
        const int d = order[k], o1 = (d + 1) % 3, o2 = (d + 2) % 3;
        RichParams P;
        P.psi = (float4 *)psi;
        P.consts = consts;
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
        const int lpt = lanes % (2 * R_LG) == 0 ? 2 : 1;
        P.ngroups = lanes / (lpt * R_LG);
        const long nlines = (long)h->ndom * P.n1 * P.n2 * P.ngroups;
        if (nlines > 0x7fffffffL) return cudaErrorInvalidConfiguration;
        P.nlines = (int)nlines;
        P.pa = stride[d] / lanes;
        P.p1 = stride[o1] / lanes;
        P.p2 = stride[o2] / lanes;
        P.pdom = h->ngrid;
        const int tpl = (P.n / 2) * R_LG;                 // threads per line
        P.nlb = tpl >= 256 ? 1 : 256 / tpl;
        const long blocks = (nlines + P.nlb - 1) / P.nlb;
        const size_t smem = (size_t)P.nlb * (P.n / 2) * lpt * R_LG * sizeof(float4);
        const dim3 grid((unsigned)blocks), block((unsigned)(tpl * P.nlb));
        ++*nlaunch;
        if (lpt == 2) {
            if (k == 0) richardson_axis_kernel<true, false, 2><<<grid, block, smem, h->stream>>>(P);
            else if (k == 2) richardson_axis_kernel<false, true, 2><<<grid, block, smem, h->stream>>>(P);
            else richardson_axis_kernel<false, false, 2><<<grid, block, smem, h->stream>>>(P);
        } else {
            if (k == 0) richardson_axis_kernel<true, false, 1><<<grid, block, smem, h->stream>>>(P);
            else if (k == 2) richardson_axis_kernel<false, true, 1><<<grid, block, smem, h->stream>>>(P);
            else richardson_axis_kernel<false, false, 1><<<grid, block, smem, h->stream>>>(P);
        }
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace mlmd
