// Fused kinetic stencil / local potential / Horner pass with TMA-staged planes (
// north_star kernel 2).  Same arithmetic as stencil.cu:
//
//   out(r,n) = psi(r,n) + (-i tau) [ sum_{d,j} ( p_dj (w(r+j e_d) + w(r-j e_d)) - i q_dj (w(r+j e_d) - w(r-j e_d)) )
//                                   + (centre + V_loc(r)) w(r,n) ]          (Eq. (3), 4th-order FD)
//
// Decomposition (orbital-fastest layout, orbital blocking, y-z planes concurrent):
// one CTA owns a 16(y) x 16(z) patch of the y-z plane for a 64-byte orbital chunk (8 orbitals) and
// marches along x.  Every x-plane of the patch -- centre box plus four 2-deep periodic halo strips --
// is brought into shared memory ONCE by TMA (cp.async.bulk.tensor, 4-D tensor map over
// [x*dom][y][z][orbital]) several planes ahead of the compute; the y/z taps are shared-memory reads, the
// x taps are scattered into a five-deep ring of accumulators held in registers, so no plane is read
// twice and the load latency is hidden by the asynchronous pipeline instead of by occupancy.
#include "mlmd_internal.h"
#include "tc_ptx.cuh"

namespace mlmd {

using namespace ptx;

namespace {

constexpr int SY = 16, SZ = 16, SL = 4;            // patch: 16 y x 16 z x 4 float4 lanes
constexpr int S_CENTER = SY * SZ * 64;             // bytes
constexpr int S_STRIP = 2 * 16 * 64;
constexpr int S_PLANE_W = S_CENTER + 4 * S_STRIP;  // w: centre, z-lo, z-hi, y-lo, y-hi
constexpr int S_PLANE = S_PLANE_W + S_CENTER;      // + the Horner base psi of the plane completed by this step
constexpr int S_NBUF = 5, S_PF = 3;                // NBUF = unroll factor of the march: buffer index is static
constexpr int S_THREADS = (SY / 2) * SZ * SL;      // 512: every thread owns the points (y, z) and (y + 1, z), y even
constexpr int S_SMEM = S_NBUF * S_PLANE + 256;

struct TmaStencilParams {
    float4 *out;
    const float *vloc;
    const StepCoef *coef;    // per-domain coefficients (PERDOM variant)
    StepCoef cval;           // the single coefficient set when the field is the same for every domain
    float tau;
    int nx, ny, nz, lanes;   // lanes = float4 per grid point
    int xs, nxseg;           // planes per CTA, segments per domain
    int nchunk;              // 64-byte chunks per grid point
    int chunk_fast;          // CTA order: orbital chunk fastest (else patch fastest)
    double *npart;           // NORM variants: [dom][slot][ld] partial squared norms, slot = (yt, zt, seg)
    int ld;
};

__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *m, uint64_t *bar, int c0, int c1, int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(smem_u32(dst)), "l"(m), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ float4 lds4(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
// acc += (p + s*i*q) * u for both complex numbers of the float4 (s = +1 or -1 folded into q)
__device__ __forceinline__ void cmul_acc(float4 &acc, const float4 u, const float p, const float q) {
    acc.x = fmaf(p, u.x, acc.x);
    acc.x = fmaf(-q, u.y, acc.x);
    acc.y = fmaf(p, u.y, acc.y);
    acc.y = fmaf(q, u.x, acc.y);
    acc.z = fmaf(p, u.z, acc.z);
    acc.z = fmaf(-q, u.w, acc.z);
    acc.w = fmaf(p, u.w, acc.w);
    acc.w = fmaf(q, u.z, acc.w);
}
__device__ __forceinline__ void pair_acc(float4 &acc, const float4 a, const float4 b, const float p, const float q) {
    acc.x = fmaf(p, a.x + b.x, acc.x);
    acc.y = fmaf(p, a.y + b.y, acc.y);
    acc.z = fmaf(p, a.z + b.z, acc.z);
    acc.w = fmaf(p, a.w + b.w, acc.w);
    acc.x = fmaf(q, a.y - b.y, acc.x);
    acc.y = fmaf(-q, a.x - b.x, acc.y);
    acc.z = fmaf(q, a.w - b.w, acc.z);
    acc.w = fmaf(-q, a.z - b.z, acc.w);
}
__device__ __forceinline__ void pair_acc_real(float4 &acc, const float4 a, const float4 b, const float p) {
    acc.x = fmaf(p, a.x + b.x, acc.x);
    acc.y = fmaf(p, a.y + b.y, acc.y);
    acc.z = fmaf(p, a.z + b.z, acc.z);
    acc.w = fmaf(p, a.w + b.w, acc.w);
}

// NORM (split step, reading D27): 1 = also sum |w|^2 of the CTA's own points per orbital, 2 = |out|^2;
// one partial sum per (CTA, orbital), reduced in a fixed order, so the norms are reproducible.
// R1: radius-1 instantiation for the paper's own 2nd-order / 7-point stencil (MLMD_OPT_FD_ORDER = 2;
// SURVEY.md 8(f) NEXT-3): same staging and march, but the j = 2 taps are neither read from shared memory nor
// multiplied (their coefficients are zero): 8 instead of 16 shared-memory loads per plane and thread.
// SAMEBASE: the Horner base IS the stencil input (the k = 4 stage, w == psi): the base of the plane completed at step n
// is read from the shared-memory copy of plane n - 2 that the march already holds, instead of being loaded a second
// time.  That buffer is released two steps later than usual, so the prefetch distance is two planes instead of three.
template <bool AYZ, bool PERDOM, int NORM, bool R1, bool SAMEBASE>
__global__ void __launch_bounds__(S_THREADS, 1)
stencil_tma_kernel(const __grid_constant__ CUtensorMap map_c, const __grid_constant__ CUtensorMap map_z,
                   const __grid_constant__ CUtensorMap map_y, const __grid_constant__ CUtensorMap map_p,
                   const TmaStencilParams P) {
    extern __shared__ __align__(1024) uint8_t smem[];
    uint64_t *full = (uint64_t *)(smem + S_NBUF * S_PLANE), *empty = full + S_NBUF;
    const int tid = threadIdx.x;
    const int l = tid % SL, tz = (tid / SL) % SZ, ty = 2 * (tid / (SL * SZ));   // a warp = 8 z x 4 lanes: 512 contiguous bytes

    // work item
    int item = blockIdx.x;
    const int seg = item % P.nxseg;
    item /= P.nxseg;
    // orbital chunk fastest: CTAs that run together read adjacent 64-byte pieces of the same rows (DRAM pages)
    const int nzt = P.nz / SZ, nyt = P.ny / SY;
    int chunk, zt, yt, dom;
    if (P.chunk_fast) {
        chunk = item % P.nchunk;
        item /= P.nchunk;
        zt = item % nzt;
        item /= nzt;
        yt = item % nyt;
        dom = item / nyt;
    } else {
        zt = item % nzt;
        item /= nzt;
        yt = item % nyt;
        item /= nyt;
        chunk = item % P.nchunk;
        dom = item / P.nchunk;
    }
    const int x0 = seg * P.xs;
    const int x1 = min(x0 + P.xs, P.nx);
    const int nplanes = (x1 - x0) + 4;
    const int nout = x1 - x0;
    const int y0 = yt * SY, z0 = zt * SZ;

    if (tid == 0) {
        for (int b = 0; b < S_NBUF; ++b) {
            mbar_init(&full[b], 1);
            mbar_init(&empty[b], S_THREADS / 32);
        }
        fence_barrier_init();
        prefetch_tmap(&map_c);
        prefetch_tmap(&map_z);
        prefetch_tmap(&map_y);
        prefetch_tmap(&map_p);
    }
    __syncthreads();

    const int zlo = (z0 - 2 + P.nz) % P.nz, zhi = (z0 + SZ) % P.nz;
    const int ylo = (y0 - 2 + P.ny) % P.ny, yhi = (y0 + SY) % P.ny;
    auto issue = [&](int n) {   // plane n of this march: x = x0 - 2 + n (periodic)
        const int b = n % S_NBUF;
        int x = x0 - 2 + n;
        x = x < 0 ? x + P.nx : (x >= P.nx ? x - P.nx : x);
        const int xr = dom * P.nx + x;
        uint8_t *buf = smem + b * S_PLANE;
        const int po = n - 4;   // output plane completed by step n: its Horner base travels with plane n
        const bool with_psi = !SAMEBASE && po >= 0 && po < nout;
        mbar_expect_tx(&full[b], with_psi ? S_PLANE : S_PLANE_W);
        if (with_psi) tma_load_4d(buf + S_PLANE_W, &map_p, &full[b], chunk * 16, z0, y0, dom * P.nx + x0 + po);
        tma_load_4d(buf, &map_c, &full[b], chunk * 16, z0, y0, xr);
        tma_load_4d(buf + S_CENTER, &map_z, &full[b], chunk * 16, zlo, y0, xr);
        tma_load_4d(buf + S_CENTER + S_STRIP, &map_z, &full[b], chunk * 16, zhi, y0, xr);
        tma_load_4d(buf + S_CENTER + 2 * S_STRIP, &map_y, &full[b], chunk * 16, z0, ylo, xr);
        tma_load_4d(buf + S_CENTER + 3 * S_STRIP, &map_y, &full[b], chunk * 16, z0, yhi, xr);
    };
    constexpr int PF = SAMEBASE ? 2 : S_PF;
    if (tid == 0)
        for (int n = 0; n < PF && n < nplanes; ++n) issue(n);

    // Byte offsets inside a plane buffer.  Point A = (ty, tz), point B = (ty + 1, tz), ty even: the six rows
    // ty-2 .. ty+3 at the own z serve as centre and y-neighbours of BOTH points (6 loads instead of 10); the
    // z-neighbours of B are those of A one row up (+1024 in the centre box, +128 in a z halo strip).
    const uint32_t own = (uint32_t)((ty * SZ + tz) * 64 + l * 16);
    auto zoff = [&](int t) -> uint32_t {
        if (t < 0) return (uint32_t)(S_CENTER + (ty * 2 + (t + 2)) * 64 + l * 16);
        if (t >= SZ) return (uint32_t)(S_CENTER + S_STRIP + (ty * 2 + (t - SZ)) * 64 + l * 16);
        return (uint32_t)((ty * SZ + t) * 64 + l * 16);
    };
    auto yoff = [&](int t) -> uint32_t {
        if (t < 0) return (uint32_t)(S_CENTER + 2 * S_STRIP + ((t + 2) * SZ + tz) * 64 + l * 16);
        if (t >= SY) return (uint32_t)(S_CENTER + 3 * S_STRIP + ((t - SY) * SZ + tz) * 64 + l * 16);
        return (uint32_t)((t * SZ + tz) * 64 + l * 16);
    };
    const uint32_t ozm1 = zoff(tz - 1), ozm2 = zoff(tz - 2), ozp1 = zoff(tz + 1), ozp2 = zoff(tz + 2);
    const uint32_t dzm = tz < 2 ? 128u : 1024u, dzp = tz >= SZ - 2 ? 128u : 1024u;   // B's z offsets = A's + these
    const uint32_t dzm1 = tz < 1 ? 128u : 1024u, dzp1 = tz >= SZ - 1 ? 128u : 1024u;
    const uint32_t oym2 = yoff(ty - 2), oym1 = yoff(ty - 1), oyp2 = yoff(ty + 2), oyp3 = yoff(ty + 3);

    const StepCoef c = PERDOM ? P.coef[dom] : P.cval;   // by-value copy lives in the constant bank: no registers
    const long sz = P.lanes, sy = sz * P.nz, sx = sy * P.ny;
    const long pbase = (long)dom * sx * P.nx + (long)(y0 + ty) * sy + (long)(z0 + tz) * sz + chunk * SL + l;
    const float *vd = P.vloc + ((long)dom * P.nx * P.ny + (y0 + ty)) * P.nz + (z0 + tz);   // B: + nz
    const long vsx = (long)P.ny * P.nz;
    const uint32_t sbase = smem_u32(smem);

    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 a0 = zero4, a1 = zero4, a2 = zero4, a3 = zero4, a4 = zero4;   // point A, planes q-2 .. q+2
    float4 b0 = zero4, b1 = zero4, b2 = zero4, b3 = zero4, b4 = zero4;   // point B
    // running element offsets (no per-step 64-bit index arithmetic): Horner base / output of the plane
    // being completed, V_loc of the plane being consumed.  B = A + one grid row along y.
    const long dB = sy;
    float4 *out_p = P.out + pbase + (long)x0 * sx;
    int xq = x0 - 2;
    xq = xq < 0 ? xq + P.nx : xq;
    const float *vp = vd + (long)xq * vsx;
    const long vwrap = (long)P.nx * vsx;
    // V_loc of the plane consumed by the NEXT step, loaded one step ahead so that its latency is off the
    // critical path of the first FMA
    float vAn = __ldg(vp), vBn = __ldg(vp + P.nz);

    float nrm0 = 0.f, nrm1 = 0.f;   // NORM: this thread's two orbitals, summed over its points
    // centre, y and z taps of one point: u = centre value, (yp1, ym1), (yp2, ym2) its y-neighbours (already loaded)
    auto point = [&](const uint32_t buf, const float4 u, const float4 yp1, const float4 ym1, const float4 yp2, const float4 ym2,
                     const uint32_t zm1, const uint32_t zm2, const uint32_t zp1, const uint32_t zp2, const float cen,
                     const bool own_plane, float4 &A0, float4 &A1, float4 &A2, float4 &A3, float4 &A4) {
        if (NORM == 1 && own_plane) {
            nrm0 = fmaf(u.x, u.x, fmaf(u.y, u.y, nrm0));
            nrm1 = fmaf(u.z, u.z, fmaf(u.w, u.w, nrm1));
        }
        A2.x = fmaf(cen, u.x, A2.x);
        A2.y = fmaf(cen, u.y, A2.y);
        A2.z = fmaf(cen, u.z, A2.z);
        A2.w = fmaf(cen, u.w, A2.w);
        if (AYZ) pair_acc(A2, yp1, ym1, c.p[1][0], c.q[1][0]); else pair_acc_real(A2, yp1, ym1, c.p[1][0]);
        if (!R1) {
            if (AYZ) pair_acc(A2, yp2, ym2, c.p[1][1], c.q[1][1]); else pair_acc_real(A2, yp2, ym2, c.p[1][1]);
        }
        {
            const float4 p1 = lds4(buf + zp1), m1 = lds4(buf + zm1);
            if (AYZ) pair_acc(A2, p1, m1, c.p[2][0], c.q[2][0]); else pair_acc_real(A2, p1, m1, c.p[2][0]);
            if (!R1) {
                const float4 p2 = lds4(buf + zp2), m2 = lds4(buf + zm2);
                if (AYZ) pair_acc(A2, p2, m2, c.p[2][1], c.q[2][1]); else pair_acc_real(A2, p2, m2, c.p[2][1]);
            }
        }
        // x taps: u = w(plane q) is the +j neighbour of plane q-j (coefficient p_j - i q_j) and the -j
        // neighbour of plane q+j (coefficient p_j + i q_j)
        cmul_acc(A1, u, c.p[0][0], -c.q[0][0]);
        cmul_acc(A3, u, c.p[0][0], c.q[0][0]);
        if (!R1) {
            cmul_acc(A0, u, c.p[0][1], -c.q[0][1]);
            cmul_acc(A4, u, c.p[0][1], c.q[0][1]);
        }
    };
    // One plane step.  A0..A4 / B0..B4 are the accumulators of planes q-2..q+2; the caller rotates the
    // names, so the ring costs no register moves.
    auto step = [&](const int n, const int k, const int it, float4 &A0, float4 &A1, float4 &A2, float4 &A3, float4 &A4,
                    float4 &B0, float4 &B1, float4 &B2, float4 &B3, float4 &B4) {
        // n = 5 it + k: plane n lives in buffer k; its barrier phase is it & 1
        if (tid == 0 && n + PF < nplanes) {
            const int m = n + PF, bm = (k + PF) % S_NBUF, um = it + (k + PF) / S_NBUF;   // um-th use of buffer bm
            if (um >= 1) mbar_wait(&empty[bm], (um - 1) & 1);
            issue(m);
        }
        const float vA = vAn, vB = vBn;
        vp += vsx;
        if (++xq == P.nx) {
            xq = 0;
            vp -= vwrap;
        }
        vAn = __ldg(vp);
        vBn = __ldg(vp + P.nz);
        mbar_wait(&full[k], it & 1);
        const uint32_t buf = sbase + k * S_PLANE;
        const bool own_plane = n >= 2 && n < nplanes - 2;
        {
            const float4 rm1 = lds4(buf + oym1), r0 = lds4(buf + own), r1 = lds4(buf + own + 1024), r2 = lds4(buf + oyp2);
            const float4 rm2 = R1 ? zero4 : lds4(buf + oym2), r3 = R1 ? zero4 : lds4(buf + oyp3);
            point(buf, r0, r1, rm1, r2, rm2, ozm1, ozm2, ozp1, ozp2, c.centre + vA, own_plane, A0, A1, A2, A3, A4);
            point(buf, r1, r2, r0, r3, rm1, ozm1 + dzm1, ozm2 + dzm, ozp1 + dzp1, ozp2 + dzp, c.centre + vB, own_plane, B0, B1, B2,
                  B3, B4);
        }
        // plane q-2 (output n - 4) is complete: out = psi + (-i tau) acc
        if (n >= 4) {
            // SAMEBASE: plane n - 2 lives in buffer (k + 3) % 5
            const uint32_t pb = SAMEBASE ? sbase + ((k + 3) % S_NBUF) * S_PLANE : buf + S_PLANE_W;
            const float4 psA = lds4(pb + own), psB = lds4(pb + own + 1024);
            const float4 oA = make_float4(fmaf(P.tau, A0.y, psA.x), fmaf(-P.tau, A0.x, psA.y), fmaf(P.tau, A0.w, psA.z),
                                          fmaf(-P.tau, A0.z, psA.w));
            const float4 oB = make_float4(fmaf(P.tau, B0.y, psB.x), fmaf(-P.tau, B0.x, psB.y), fmaf(P.tau, B0.w, psB.z),
                                          fmaf(-P.tau, B0.z, psB.w));
            out_p[0] = oA;
            out_p[dB] = oB;
            out_p += sx;
            if (NORM == 2) {
                nrm0 = fmaf(oA.x, oA.x, fmaf(oA.y, oA.y, nrm0));
                nrm1 = fmaf(oA.z, oA.z, fmaf(oA.w, oA.w, nrm1));
                nrm0 = fmaf(oB.x, oB.x, fmaf(oB.y, oB.y, nrm0));
                nrm1 = fmaf(oB.z, oB.z, fmaf(oB.w, oB.w, nrm1));
            }
        }
        __syncwarp();
        if (SAMEBASE) {
            if (n >= 2 && tid % 32 == 0) mbar_arrive(&empty[(k + 3) % S_NBUF]);   // plane n - 2 has served as base
        } else if (tid % 32 == 0) {
            mbar_arrive(&empty[k]);
        }
        A0 = zero4;
        B0 = zero4;
    };
    for (int n = 0, it = 0; n < nplanes; n += 5, ++it) {
        step(n, 0, it, a0, a1, a2, a3, a4, b0, b1, b2, b3, b4);
        if (n + 1 < nplanes) step(n + 1, 1, it, a1, a2, a3, a4, a0, b1, b2, b3, b4, b0);
        if (n + 2 < nplanes) step(n + 2, 2, it, a2, a3, a4, a0, a1, b2, b3, b4, b0, b1);
        if (n + 3 < nplanes) step(n + 3, 3, it, a3, a4, a0, a1, a2, b3, b4, b0, b1, b2);
        if (n + 4 < nplanes) step(n + 4, 4, it, a4, a0, a1, a2, a3, b4, b0, b1, b2, b3);
    }
    if (NORM != 0) {
        // threads with the same l hold the same two orbitals: lanes l, l+4, .. of a warp, then the 16 warps
        __shared__ float red[S_THREADS / 32][SL][2];
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            nrm0 += __shfl_xor_sync(0xffffffffu, nrm0, o);
            nrm1 += __shfl_xor_sync(0xffffffffu, nrm1, o);
        }
        if (tid % 32 < SL) {
            red[tid / 32][l][0] = nrm0;
            red[tid / 32][l][1] = nrm1;
        }
        __syncthreads();
        if (tid < 2 * SL) {
            double sum = 0.0;
            for (int wq = 0; wq < S_THREADS / 32; ++wq) sum += (double)red[wq][tid / 2][tid % 2];
            const int nslots = nyt * nzt * P.nxseg;
            const int slot = (yt * nzt + zt) * P.nxseg + seg;
            P.npart[((size_t)dom * nslots + slot) * P.ld + chunk * 2 * SL + tid] = sum;
        }
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_fn2() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}
bool make_plane_map_raw(CUtensorMap *m, const float *base, int F, int nz, int ny, long nxd, int bz, int by) {
    EncodeTiledFn f = encode_fn2();
    if (!f) return false;
    cuuint64_t dims[4] = {(cuuint64_t)F, (cuuint64_t)nz, (cuuint64_t)ny, (cuuint64_t)nxd};
    cuuint64_t strides[3] = {(cuuint64_t)F * 4, (cuuint64_t)F * 4 * nz, (cuuint64_t)F * 4 * nz * ny};
    cuuint32_t box[4] = {16, (cuuint32_t)bz, (cuuint32_t)by, 1};
    cuuint32_t es[4] = {1, 1, 1, 1};
    return f(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool make_plane_map(TmapCache *cache, CUtensorMap *m, const float *base, int F, int nz, int ny, long nxd, int bz, int by) {
    const TmapKey k{4, base, (unsigned long long)F, (unsigned long long)nz, (unsigned long long)ny, (unsigned long long)nxd,
                    (unsigned)bz, (unsigned)by};
    return cached_tmap(cache, k, m, [&](CUtensorMap *o) { return make_plane_map_raw(o, base, F, nz, ny, nxd, bz, by); });
}

}  // namespace

bool stencil_tma_supported(const mlmd_domain *h) {
    return encode_fn2() != nullptr && h->ny % SY == 0 && h->nz % SZ == 0 && h->nx >= 5 && h->ld % 8 == 0;
}

namespace {
template <int NORM, bool R1, bool SB>
cudaError_t set_attrs() {
    cudaError_t e = cudaFuncSetAttribute(stencil_tma_kernel<false, false, NORM, R1, SB>, cudaFuncAttributeMaxDynamicSharedMemorySize, S_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stencil_tma_kernel<true, false, NORM, R1, SB>, cudaFuncAttributeMaxDynamicSharedMemorySize, S_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stencil_tma_kernel<false, true, NORM, R1, SB>, cudaFuncAttributeMaxDynamicSharedMemorySize, S_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(stencil_tma_kernel<true, true, NORM, R1, SB>, cudaFuncAttributeMaxDynamicSharedMemorySize, S_SMEM);
    return e;
}
template <int NORM, bool R1, bool SB>
void launch_variant(bool yz, bool perdom, unsigned g, cudaStream_t st, const CUtensorMap &mc, const CUtensorMap &mz,
                    const CUtensorMap &my, const CUtensorMap &mp, const TmaStencilParams &P) {
    if (!perdom) {
        if (yz) stencil_tma_kernel<true, false, NORM, R1, SB><<<g, S_THREADS, S_SMEM, st>>>(mc, mz, my, mp, P);
        else stencil_tma_kernel<false, false, NORM, R1, SB><<<g, S_THREADS, S_SMEM, st>>>(mc, mz, my, mp, P);
    } else {
        if (yz) stencil_tma_kernel<true, true, NORM, R1, SB><<<g, S_THREADS, S_SMEM, st>>>(mc, mz, my, mp, P);
        else stencil_tma_kernel<false, true, NORM, R1, SB><<<g, S_THREADS, S_SMEM, st>>>(mc, mz, my, mp, P);
    }
}
template <int NORM, bool R1>
void launch_variant2(bool same, bool yz, bool perdom, unsigned g, cudaStream_t st, const CUtensorMap &mc, const CUtensorMap &mz,
                     const CUtensorMap &my, const CUtensorMap &mp, const TmaStencilParams &P) {
    if (same) launch_variant<NORM, R1, true>(yz, perdom, g, st, mc, mz, my, mp, P);
    else launch_variant<NORM, R1, false>(yz, perdom, g, st, mc, mz, my, mp, P);
}
}  // namespace

// x-march segments per (domain, chunk, patch): enough CTAs to fill the GPU twice on small batches
static void x_segments(const mlmd_domain *h, int *xs, int *nxseg) {
    const long base = (long)h->ndom * (h->ld / 8) * (h->ny / SY) * (h->nz / SZ);
    int n = 1;
    while (base * n < 2 * 148 && h->nx / (n * 2) >= 8) n *= 2;
    *xs = (h->nx + n - 1) / n;
    *nxseg = (h->nx + *xs - 1) / *xs;
}
int stencil_tma_norm_slots(const mlmd_domain *h) {
    int xs, nxseg;
    x_segments(h, &xs, &nxseg);
    return (h->ny / SY) * (h->nz / SZ) * nxseg;
}

cudaError_t launch_stencil_tma(const mlmd_domain *h, const float2 *w, const float2 *psi, float2 *out, const StepCoef *coef,
                               const StepCoef *coef_host, float tau, int *nlaunch, int norm_mode, double *npart) {
    static DeviceOnce attr_set;      // the opt-in shared-memory size is a per-device function attribute
    if (!attr_set.done()) {
        cudaError_t e = set_attrs<0, false, false>();
        if (e == cudaSuccess) e = set_attrs<1, false, false>();
        if (e == cudaSuccess) e = set_attrs<2, false, false>();
        if (e == cudaSuccess) e = set_attrs<0, true, false>();
        if (e == cudaSuccess) e = set_attrs<1, true, false>();
        if (e == cudaSuccess) e = set_attrs<2, true, false>();
        if (e == cudaSuccess) e = set_attrs<0, false, true>();
        if (e == cudaSuccess) e = set_attrs<1, false, true>();
        if (e == cudaSuccess) e = set_attrs<2, false, true>();
        if (e == cudaSuccess) e = set_attrs<0, true, true>();
        if (e == cudaSuccess) e = set_attrs<1, true, true>();
        if (e == cudaSuccess) e = set_attrs<2, true, true>();
        if (e != cudaSuccess) return e;
        attr_set.mark();
    }
    const int F = 2 * h->ld;
    CUtensorMap mc, mz, my, mp;
    const long nxd = (long)h->nx * h->ndom;
    if (!make_plane_map(&h->tmaps, &mc, (const float *)w, F, h->nz, h->ny, nxd, SZ, SY)) return cudaErrorInvalidValue;
    if (!make_plane_map(&h->tmaps, &mz, (const float *)w, F, h->nz, h->ny, nxd, 2, SY)) return cudaErrorInvalidValue;
    if (!make_plane_map(&h->tmaps, &my, (const float *)w, F, h->nz, h->ny, nxd, SZ, 2)) return cudaErrorInvalidValue;
    if (!make_plane_map(&h->tmaps, &mp, (const float *)psi, F, h->nz, h->ny, nxd, SZ, SY)) return cudaErrorInvalidValue;
    TmaStencilParams P;
    P.out = (float4 *)out;
    P.vloc = h->vloc();
    P.coef = coef;
    P.tau = tau;
    P.nx = h->nx;
    P.ny = h->ny;
    P.nz = h->nz;
    P.lanes = h->ld / 2;
    P.nchunk = h->ld / 8;
    P.npart = npart;
    {
        // CTA order.  Patch-fastest keeps neighbouring patches (shared halos) together in time, but the CTAs resident
        // at once then cover only 148 / npatch adjacent 64-byte chunks of a row; when that is under 1 KB (many patches,
        // e.g. 64^2 planes) DRAM page locality wins: chunk-fastest (configs[4]: 4.31 -> 3.58 ms; configs[3] stays, 1 % the other way).
        const int npatch = (h->ny / SY) * (h->nz / SZ);
        P.chunk_fast = 64 * 148 / npatch < 1024 ? 1 : 0;
    }
    P.ld = h->ld;
    const long base = (long)h->ndom * P.nchunk * (h->ny / SY) * (h->nz / SZ);
    x_segments(h, &P.xs, &P.nxseg);
    const long grid = base * P.nxseg;
    ++*nlaunch;
    const unsigned g = (unsigned)grid;
    P.cval = coef_host ? *coef_host : StepCoef();
    const bool r1 = h->opt[MLMD_OPT_FD_ORDER] == 2;
    const bool same = (const void *)w == (const void *)psi;      // the k = 4 stage: the Horner base is the stencil input
    if (norm_mode == 1) r1 ? launch_variant2<1, true>(same, h->field_yz, !coef_host, g, h->stream, mc, mz, my, mp, P)
                           : launch_variant2<1, false>(same, h->field_yz, !coef_host, g, h->stream, mc, mz, my, mp, P);
    else if (norm_mode == 2) r1 ? launch_variant2<2, true>(same, h->field_yz, !coef_host, g, h->stream, mc, mz, my, mp, P)
                                : launch_variant2<2, false>(same, h->field_yz, !coef_host, g, h->stream, mc, mz, my, mp, P);
    else r1 ? launch_variant2<0, true>(same, h->field_yz, !coef_host, g, h->stream, mc, mz, my, mp, P)
            : launch_variant2<0, false>(same, h->field_yz, !coef_host, g, h->stream, mc, mz, my, mp, P);
    return cudaGetLastError();
}

}  // namespace mlmd
