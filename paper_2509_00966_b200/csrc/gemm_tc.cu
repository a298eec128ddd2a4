// tcgen05 tensor-core GEMMs of the nonlocal operator (north_star kernel 3).
//
// Complex GEMMs run as REAL GEMMs on the interleaved storage:
//   projection        Z[p][c]  = sum_r B[r][p] * Y[r][c]        K = grid points   (PAPER.md L283 CGEMM(1))
//   back-application  Y[r][c] += sum_p B[r][p] * W[p][c]        K = projector rows (PAPER.md L283 CGEMM(2))
// with Y the float view [ngrid][2*ld] of a psi-like buffer and B the float view of beta.
//
// Operands are staged by TMA (cp.async.bulk.tensor, SWIZZLE_128B_ATOM_32B) straight from their natural
// row-major HBM layouts: a [rows x 32 floats] box IS one column-chunk of the canonical UMMA
// MN-major SWIZZLE_128B_BASE32B layout (K = rows), so neither GEMM needs a transposed copy of psi or beta.
// Accumulators live in TMEM; one thread issues tcgen05.mma; warp roles: 0 = TMA producer,
// 1 = MMA issuer (+ TMEM allocation), the rest convert (hi/lo split) and run the epilogue.
//
// FP32-grade accuracy = 3xTF32 (PAPER.md L239 describes the same idea as BF16x3):
//   a*b ~= a_hi*b_hi + a_lo*b_hi + a_hi*b_lo,  x_hi = a TF32-representable value within one TF32 ulp of x
// (beta, W: nearest, rounded when they are written; psi: the 13 low mantissa bits cleared, which is what a
// kind::tf32 operand keeps of the tile as loaded), x_lo = x - x_hi (exact in FP32); FP32 accumulation in TMEM.
// beta_hi / beta_lo are split once at mlmd_set_projectors; psi-side lo tiles are produced in shared
// memory by the converter warps; W hi/lo are written by the glue kernel.
#include <stdio.h>
#include <stdlib.h>

#include "mlmd_internal.h"
#include "tc_ptx.cuh"

namespace mlmd {

using namespace ptx;

namespace {

// ---- tensor maps --------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
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

// Column-chunked view of a row-major float matrix [rows][pitch]: dims (32 floats, rows, chunks of 32
// columns); a box (32, box_rows, box_chunks) lands in shared memory as box_chunks consecutive
// [box_rows x 128 B] regions in the 128B-span / 32B-atom swizzle = UMMA MN-major SWIZZLE_128B_BASE32B
// atoms (4 K-rows x 32 MN-elements each; the only MN-major layout tcgen05 takes for TF32 operands).
bool make_chunk_map(TmapCache *cache, CUtensorMap *m, const float *base, uint64_t rows, uint64_t pitch, uint64_t nchunk,
                    uint32_t box_rows, uint32_t box_chunks);
bool make_chunk_map_raw(CUtensorMap *m, const float *base, uint64_t rows, uint64_t pitch, uint64_t nchunk, uint32_t box_rows,
                        uint32_t box_chunks) {
    EncodeTiledFn f = encode_fn();
    if (!f) return false;
    cuuint64_t dims[3] = {32, rows, nchunk};
    cuuint64_t strides[2] = {pitch * sizeof(float), 32 * sizeof(float)};
    cuuint32_t box[3] = {32, box_rows, box_chunks};
    cuuint32_t es[3] = {1, 1, 1};
    return f(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Plain 2-D view (cols, rows) with a (8 floats = 32 B, box_rows) box and the 32-byte swizzle = UMMA
// K-major SWIZZLE_32B layout of one K = 8 slab.
bool make_k8_map_raw(CUtensorMap *m, const float *base, uint64_t rows, uint64_t cols, uint64_t pitch, uint32_t box_rows) {
    EncodeTiledFn f = encode_fn();
    if (!f) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {pitch * sizeof(float)};
    cuuint32_t box[2] = {8, box_rows};
    cuuint32_t es[2] = {1, 1};
    return f(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// (cols, rows) view with a [128 rows x 32 floats] box in the plain 128-byte swizzle: epilogue staging tiles
bool make_out_map_raw(CUtensorMap *m, const float *base, uint64_t rows, uint64_t cols, uint64_t pitch) {
    EncodeTiledFn f = encode_fn();
    if (!f) return false;
    cuuint64_t dims[2] = {cols, rows};
    cuuint64_t strides[1] = {pitch * sizeof(float)};
    cuuint32_t box[2] = {32, 128};
    cuuint32_t es[2] = {1, 1};
    return f(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// the same three encoders through the handle's cache
bool make_chunk_map(TmapCache *cache, CUtensorMap *m, const float *base, uint64_t rows, uint64_t pitch, uint64_t nchunk,
                    uint32_t box_rows, uint32_t box_chunks) {
    const TmapKey k{1, base, rows, pitch, nchunk, 0, box_rows, box_chunks};
    return cached_tmap(cache, k, m, [&](CUtensorMap *o) { return make_chunk_map_raw(o, base, rows, pitch, nchunk, box_rows, box_chunks); });
}
bool make_k8_map(TmapCache *cache, CUtensorMap *m, const float *base, uint64_t rows, uint64_t cols, uint64_t pitch, uint32_t box_rows) {
    const TmapKey k{2, base, rows, cols, pitch, 0, box_rows, 0};
    return cached_tmap(cache, k, m, [&](CUtensorMap *o) { return make_k8_map_raw(o, base, rows, cols, pitch, box_rows); });
}
bool make_out_map(TmapCache *cache, CUtensorMap *m, const float *base, uint64_t rows, uint64_t cols, uint64_t pitch) {
    const TmapKey k{3, base, rows, cols, pitch, 0, 0, 0};
    return cached_tmap(cache, k, m, [&](CUtensorMap *o) { return make_out_map_raw(o, base, rows, cols, pitch); });
}

// BF16 operands (opt-in low-precision mode).  MN-major tiles keep the 32-column chunk granularity of the FP32 path:
// dims (32 bf16 = 64 B, rows, chunks of 32 columns), 64-byte swizzle = UMMA MN-major SWIZZLE_64B atoms (8 K-rows x 32
// MN-elements), so a CTA of a pair can hold any number of chunks of a column tile.
bool make_chunk16_map(TmapCache *cache, CUtensorMap *m, const void *base, uint64_t rows, uint64_t pitch, uint64_t nchunk,
                      uint32_t box_rows, uint32_t box_chunks) {
    const TmapKey k{5, base, rows, pitch, nchunk, 0, box_rows, box_chunks};
    return cached_tmap(cache, k, m, [&](CUtensorMap *o) {
        EncodeTiledFn f = encode_fn();
        if (!f) return false;
        cuuint64_t dims[3] = {32, rows, nchunk};
        cuuint64_t strides[2] = {pitch * 2, 64};
        cuuint32_t box[3] = {32, box_rows, box_chunks};
        cuuint32_t es[3] = {1, 1, 1};
        return f(o, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                 CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
    });
}
// K-major BF16 slab: (cols, rows) view with a (64 bf16 = 128 B, box_rows) box in the 128-byte swizzle = UMMA K-major
// SWIZZLE_128B (four K = 16 steps per row)
bool make_k64_map(TmapCache *cache, CUtensorMap *m, const void *base, uint64_t rows, uint64_t cols, uint64_t pitch, uint32_t box_rows) {
    const TmapKey k{6, base, rows, cols, pitch, 0, box_rows, 0};
    return cached_tmap(cache, k, m, [&](CUtensorMap *o) {
        EncodeTiledFn f = encode_fn();
        if (!f) return false;
        cuuint64_t dims[2] = {cols, rows};
        cuuint64_t strides[1] = {pitch * 2};
        cuuint32_t box[2] = {64, box_rows};
        cuuint32_t es[2] = {1, 1};
        return f(o, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                 CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
    });
}

constexpr int EPI_TILE_BYTES = 128 * 128;   // one staging tile: 128 rows x 32 floats
constexpr int EPI_BAR = 1;                  // named barrier of the 128 epilogue threads

// The 128 epilogue threads hand one [128 x 32] FP32 tile (thread r holds row r in v) to the TMA engine,
// which stores it or adds it (L2 reduction, round-to-nearest) into global memory at (c0, row0).
// NB staging tiles rotate; `slot` counts tiles issued so far by this group.
template <int NB>
__device__ __forceinline__ void epi_tile_out(uint8_t *stage, int &slot, const CUtensorMap *map, int c0, int row0,
                                             const uint32_t (&v)[32], int r, bool add) {
    uint8_t *buf = stage + (slot % NB) * EPI_TILE_BYTES;
    if (r == 0) bulk_wait_read<NB - 1>();     // the tile issued NB slots ago has left this buffer
    named_bar_sync(EPI_BAR, 128);
    const uint32_t rowaddr = smem_u32(buf) + r * 128;
#pragma unroll
    for (int j = 0; j < 8; ++j)
        sts4(rowaddr + (((uint32_t)j ^ ((uint32_t)r & 7u)) << 4), v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
    fence_proxy_async_smem();
    named_bar_sync(EPI_BAR, 128);
    if (r == 0) {
        if (add) tma_reduce_add_2d(map, buf, c0, row0);
        else tma_store_2d(map, buf, c0, row0);
        bulk_commit();
    }
    ++slot;
}

__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }
// in place: v -> hi (TF32-representable), returns lo = v - hi (exact)
__device__ __forceinline__ float4 split4(float4 &v) {
    const float4 h = make_float4(tf32_hi(v.x), tf32_hi(v.y), tf32_hi(v.z), tf32_hi(v.w));
    const float4 l = make_float4(v.x - h.x, v.y - h.y, v.z - h.z, v.w - h.w);
    v = h;
    return l;
}

// round-to-nearest-even to TF32 precision (13 low mantissa bits cleared afterwards)
__device__ __forceinline__ float tf32_rn(float x) {
    uint32_t u = __float_as_uint(x);
    u += 0xfffu + ((u >> 13) & 1u);
    return __uint_as_float(u & 0xffffe000u);
}
__device__ __forceinline__ float4 tf32_rn4(const float4 v) { return make_float4(tf32_rn(v.x), tf32_rn(v.y), tf32_rn(v.z), tf32_rn(v.w)); }

// in place: v -> nearest TF32 value hi, returns lo = v - hi (exact in FP32; |lo| <= half a TF32 ulp of v)
__device__ __forceinline__ float4 split4_rn(float4 &v) {
    const float4 h = tf32_rn4(v);
    const float4 l = make_float4(v.x - h.x, v.y - h.y, v.z - h.z, v.w - h.w);
    v = h;
    return l;
}

// round-to-nearest-even to BF16 precision, kept in an FP32 container (every BF16 value is a TF32 value)
__device__ __forceinline__ float bf16_round(float x) {
    uint32_t u = __float_as_uint(x);
    u += 0x7fffu + ((u >> 16) & 1u);
    return __uint_as_float(u & 0xffff0000u);
}
__device__ __forceinline__ float4 bf16_round4(const float4 v) {
    return make_float4(bf16_round(v.x), bf16_round(v.y), bf16_round(v.z), bf16_round(v.w));
}

// two floats -> packed BF16 pair (round-to-nearest-even), low half = first
__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    uint32_t ua = __float_as_uint(a), ub = __float_as_uint(b);
    ua += 0x7fffu + ((ua >> 16) & 1u);
    ub += 0x7fffu + ((ub >> 16) & 1u);
    return (ua >> 16) | (ub & 0xffff0000u);
}

// =================================================================================================
// Projection: Z[p][c] = sum_r A[r][p] * Y[r][c] over one K slice; FP32 partials per slice.
// CTA tile: up to 256 rows p (two M = 128 UMMA blocks) x BN <= 224 columns; K pipeline of 16 rows.
// CTAs run as clusters of two on neighbouring column tiles of the same (domain, row tile, K slice): the
// beta tile of a stage is the same for both, so each fetches half of its chunks and TMA-multicasts them.
// =================================================================================================
constexpr int PJ_BK = 16;               // grid points per pipeline stage (two K = 8 UMMA steps)
constexpr int PJ_STAGES = 3;
constexpr int PJ_MAXBN = 224;
constexpr int PJ_A_BYTES = 8 * PJ_BK * 128;            // 8 chunks of 32 p  = 256 rows p
constexpr int PJ_Y_BYTES = (PJ_MAXBN / 32) * PJ_BK * 128;
constexpr int PJ_STAGE_BYTES = 2 * PJ_A_BYTES + 2 * PJ_Y_BYTES;
constexpr int PJ_SMEM = PJ_STAGES * PJ_STAGE_BYTES + 2 * EPI_TILE_BYTES + 1024 /*align*/ + 256 /*barriers*/;
constexpr int PJ_THREADS = 192;          // warp 0 TMA, warp 1 MMA, warps 2-5 convert + epilogue

// Column tiles of the CTA-pair kernels: N / 64 units of 64 columns over ntile = ceil(N / 448) tiles: `wt` wide tiles of
// `wu` units followed by narrow tiles of `nu` units.  A tile is issued as UMMA pieces of n0 = min(width, 256) and
// n1 = width - n0 columns (each CTA of the pair stages h0 = n0 / 64 and h1 = n1 / 64 chunks); a 64-column piece costs
// as much as a 128-column one (its MMAs are bound by the A-operand reads), so the split avoids them where it can:
// configs[4], 1408 columns = 448 + 448 + 256 + 256, nothing padded.
struct ColSplit {
    int ntile, wt, wu, nu;
};
struct ColTile {
    int start, width, n0, n1, h0, h1;
};
__host__ __device__ inline ColTile col_tile(const ColSplit cs, int nt) {
    ColTile t;
    t.width = (nt < cs.wt ? cs.wu : cs.nu) * 64;
    t.start = (nt < cs.wt ? nt * cs.wu : cs.wt * cs.wu + (nt - cs.wt) * cs.nu) * 64;
    t.n0 = t.width < 256 ? t.width : 256;
    t.n1 = t.width - t.n0;
    t.h0 = t.n0 / 64;
    t.h1 = t.n1 / 64;
    return t;
}
inline ColSplit choose_col_split(int N) {
    const int units = N / 64, ntile = (N + 447) / 448;
    auto piece = [](int n) { return n == 0 ? 0 : (n < 128 ? 128 : n); };
    auto cost = [&](int u) { const int w = u * 64, n0 = w < 256 ? w : 256; return piece(n0) + piece(w - n0); };
    ColSplit best{ntile, ntile, (units + ntile - 1) / ntile, (units + ntile - 1) / ntile};
    long best_cost = -1;
    for (int wt = 1; wt <= ntile; ++wt)
        for (int wu = 1; wu <= 7; ++wu) {
            const int left = units - wt * wu, nn = ntile - wt;
            if (left < 0 || (nn == 0 ? left != 0 : (left % nn != 0 || left / nn > wu || left / nn < 1))) continue;
            const int nu = nn ? left / nn : wu;
            const long c = (long)wt * cost(wu) + (long)nn * cost(nu);
            if (best_cost < 0 || c < best_cost) {
                best_cost = c;
                best = ColSplit{ntile, wt, wu, nu};
            }
        }
    return best;
}

struct ProjParams {
    int ndom, ngrid, P, N, BN, ntile_m, ntile_n, nsplit, prows, nprod, conv_a, chain, lowp, rn;
    float *zpart;
    // fused density (S3 riding on the step's first projection): rho[dom][r] += sum_n occ[dom][n] |Y[r][n]|^2 over this
    // CTA's columns of the psi tile it holds anyway; NULL = off
    float *rho;
    const float *occ;
    ColSplit cs;                 // column tiles of the CTA-pair kernel
};

// LO = true: stages hold hi and lo tiles of both operands (3xTF32), 3 stages; LO = false (one product per MAC):
// one tile per operand, so the same shared memory gives a 6-stage pipeline for the then HBM-latency-bound kernel.
template <bool LO>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PJ_THREADS, 1)
proj_tc_kernel(const __grid_constant__ CUtensorMap map_ahi, const __grid_constant__ CUtensorMap map_alo,
               const __grid_constant__ CUtensorMap map_y, const __grid_constant__ CUtensorMap map_z, const ProjParams q) {
    constexpr int NST = LO ? PJ_STAGES : 2 * PJ_STAGES;
    constexpr int YOFF = (LO ? 2 : 1) * PJ_A_BYTES;            // Y tile(s) follow the beta tile(s)
    constexpr int SB = LO ? PJ_STAGE_BYTES : PJ_STAGE_BYTES / 2;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *stage = smem + NST * SB;
    uint64_t *bars = (uint64_t *)(stage + 2 * EPI_TILE_BYTES);
    uint64_t *full = bars, *empty = bars + NST, *conv = bars + 2 * NST;
    uint64_t *acc_full = bars + 3 * NST, *acc_empty = acc_full + 1;
    uint32_t *tmem_slot = (uint32_t *)(acc_empty + 1);
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 2);    // this CTA's MMAs and the peer's (its multicast half lands here too)
            mbar_init(&conv[s], 128);
        }
        mbar_init(acc_full, 1);
        mbar_init(acc_empty, 128);
        fence_barrier_init();
        prefetch_tmap(&map_ahi);
        prefetch_tmap(&map_alo);
        prefetch_tmap(&map_y);
        prefetch_tmap(&map_z);
    }
    if (warp == 1) tmem_alloc(tmem_slot, 512);
    tc_fence_before();
    cluster_sync_all();          // barrier inits visible to the peer before any remote arrive / multicast
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int crank = (int)cluster_ctarank();
    const int ncl = gridDim.x / 2, cl = blockIdx.x / 2;

    const int nkb = q.ngrid / PJ_BK;
    const int nntp = (q.ntile_n + 1) / 2;          // pairs of column tiles: one per cluster unit
    const int total = q.ndom * q.ntile_m * nntp * q.nsplit;   // cluster units
    const bool need_lo = q.nprod == 3;
    const bool need_conv = true;        // beta arrives as one raw FP32 copy: the converter warps touch every stage
    const bool load_alo = need_lo && !q.conv_a;
    const uint32_t y_bytes = (uint32_t)(q.BN / 32) * PJ_BK * 128;
    const uint32_t tx_bytes = PJ_A_BYTES * (load_alo ? 2u : 1u) + y_bytes;

    auto decode = [&](int u, int &dom, int &mt, int &nt, int &kb0, int &kb1) {
        nt = 2 * (u % nntp) + crank;   // may be == ntile_n (odd tile count): that CTA only keeps the protocol going
        u /= nntp;
        const int sp = u % q.nsplit;
        u /= q.nsplit;
        mt = u % q.ntile_m;
        dom = u / q.ntile_m;
        kb0 = (int)((long)nkb * sp / q.nsplit);
        kb1 = (int)((long)nkb * (sp + 1) / q.nsplit);
    };

    if (warp == 0) {
        if (lane == 0) {
            int it = 0;
            for (int u = cl; u < total; u += ncl) {
                int dom, mt, nt, kb0, kb1;
                decode(u, dom, mt, nt, kb0, kb1);
                for (int kb = kb0; kb < kb1; ++kb, ++it) {
                    const int s = it % NST;
                    mbar_wait(&empty[s], ((it / NST) & 1) ^ 1);
                    uint8_t *st = smem + s * SB;
                    mbar_expect_tx(&full[s], tx_bytes);
                    const int row = dom * q.ngrid + kb * PJ_BK;
                    const int ahalf = crank * 4 * (PJ_BK * 128);   // this CTA fetches 4 of the 8 beta chunks for both
                    tma_load_3d_mc(st + ahalf, &map_ahi, &full[s], 0, row, mt * 8 + crank * 4, (uint16_t)3);
                    if (load_alo)
                        tma_load_3d_mc(st + PJ_A_BYTES + ahalf, &map_alo, &full[s], 0, row, mt * 8 + crank * 4, (uint16_t)3);
                    tma_load_3d(st + YOFF, &map_y, &full[s], 0, row, nt * (q.BN / 32));
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            const uint32_t idesc = instr_desc(FMT_TF32, 1, 1, 128, (uint32_t)q.BN);
            int it = 0, nd = 0;   // nd: accumulator hand-overs (drains) so far
            for (int u = cl; u < total; u += ncl) {
                int dom, mt, nt, kb0, kb1;
                decode(u, dom, mt, nt, kb0, kb1);
                const int nblk = (q.P - mt * 256 > 128) ? 2 : 1;
                for (int kb = kb0; kb < kb1; ++kb, ++it) {
                    // a chain = at most q.chain stages accumulated in TMEM before the epilogue warps add
                    // it to the FP32 partial sums (tensor-core accumulation truncates)
                    const bool first = (kb - kb0) % q.chain == 0;
                    if (first) {
                        mbar_wait(acc_empty, (nd & 1) ^ 1);
                        tc_fence_after();
                    }
                    const int s = it % NST;
                    const uint32_t ph = (it / NST) & 1;
                    mbar_wait(&full[s], ph);
                    if (need_conv) mbar_wait(&conv[s], ph);
                    tc_fence_after();
                    const uint32_t st = smem_u32(smem + s * SB);
                    const uint32_t a_hi = st, a_lo = st + PJ_A_BYTES, y_hi = st + YOFF,
                                   y_lo = st + YOFF + PJ_Y_BYTES;
#pragma unroll
                    for (int k8 = 0; k8 < PJ_BK / 8; ++k8) {
                        const uint64_t dy = smem_desc(y_hi + k8 * 1024, PJ_BK * 128, 512, LAYOUT_SW128_32B);
                        const uint64_t dyl = smem_desc(y_lo + k8 * 1024, PJ_BK * 128, 512, LAYOUT_SW128_32B);
                        for (int mb = 0; mb < nblk; ++mb) {
                            const uint32_t aoff = mb * 4 * (PJ_BK * 128) + k8 * 1024;
                            const uint64_t da = smem_desc(a_hi + aoff, PJ_BK * 128, 512, LAYOUT_SW128_32B);
                            const uint32_t d = tmem + mb * q.BN;
                            umma_tf32(d, da, dy, idesc, (!first || k8 > 0) ? 1u : 0u);
                            if (need_lo) {
                                const uint64_t dal = smem_desc(a_lo + aoff, PJ_BK * 128, 512, LAYOUT_SW128_32B);
                                umma_tf32(d, dal, dy, idesc, 1u);
                                umma_tf32(d, da, dyl, idesc, 1u);
                            }
                        }
                    }
                    umma_commit_mc(&empty[s], (uint16_t)3);   // frees the stage in both CTAs of the cluster
                    if ((kb - kb0 + 1) % q.chain == 0 || kb + 1 == kb1) {
                        umma_commit(acc_full);
                        ++nd;
                    }
                }
            }
        }
    } else {
        const int t = threadIdx.x - 64;   // 0..127
        const int quarter = warp % 4;
        const int er = quarter * 32 + lane;   // TMEM lane = accumulator row of this thread; er == 0 leads the TMA stores
        int it = 0, nd = 0, slot = 0;
        const int ny4 = q.BN / 32 * PJ_BK * 8;    // float4 count of the Y tile
        for (int u = cl; u < total; u += ncl) {
            int dom, mt, nt, kb0, kb1;
            decode(u, dom, mt, nt, kb0, kb1);
            const int sp = (u / nntp) % q.nsplit;
            const int nblk = (q.P - mt * 256 > 128) ? 2 : 1;
            for (int c0k = kb0; c0k < kb1; c0k += q.chain) {
                const int c1k = min(c0k + q.chain, kb1);
                if (q.lowp) {
                    // opt-in low precision (PAPER.md L207, L239 float_to_BF16): both operands rounded to BF16
                    for (int kb = c0k; kb < c1k; ++kb, ++it) {
                        const int s = it % NST;
                        mbar_wait(&full[s], (it / NST) & 1);
                        uint8_t *st = smem + s * SB;
                        float4 *y4 = (float4 *)(st + YOFF);
                        for (int i = t; i < ny4; i += 128) y4[i] = bf16_round4(y4[i]);
                        float4 *a4 = (float4 *)st;
                        for (int i = t; i < PJ_A_BYTES / 16; i += 128) a4[i] = bf16_round4(a4[i]);
                        fence_proxy_async_smem();
                        mbar_arrive(&conv[s]);
                    }
                } else if (!need_lo) {
                    // one product: beta rounded to the nearest TF32 in place (an unbiased operand; the MMA alone would
                    // truncate), and psi too when q.rn (staged inner stages); plain TF32x1 leaves psi to the MMA
                    for (int kb = c0k; kb < c1k; ++kb, ++it) {
                        const int s = it % NST;
                        mbar_wait(&full[s], (it / NST) & 1);
                        uint8_t *st = smem + s * SB;
                        float4 *a4 = (float4 *)st;
                        for (int i = t; i < PJ_A_BYTES / 16; i += 128) a4[i] = tf32_rn4(a4[i]);
                        if (q.rn) {
                            float4 *y4 = (float4 *)(st + YOFF);
                            for (int i = t; i < ny4; i += 128) y4[i] = tf32_rn4(y4[i]);
                        }
                        fence_proxy_async_smem();
                        mbar_arrive(&conv[s]);
                    }
                } else {
                    for (int kb = c0k; kb < c1k; ++kb, ++it) {
                        const int s = it % NST;
                        mbar_wait(&full[s], (it / NST) & 1);
                        uint8_t *st = smem + s * SB;
                        // elementwise on the swizzled image: the lo tile has the same layout as the hi tile
                        float4 *ysrc = (float4 *)(st + YOFF);
                        float4 *ydst = (float4 *)(st + YOFF + PJ_Y_BYTES);
                        for (int i = t; i < ny4; i += 128) {
                            float4 v = ysrc[i];
                            ydst[i] = split4(v);   // the hi tile stays as loaded: kind::tf32 ignores the 13 low bits
                        }
                        if (q.conv_a) {
                            // beta / Phi: nearest TF32 in place + exact remainder (as round 1's stored hi / lo pair)
                            float4 *asrc = (float4 *)st;
                            float4 *adst = (float4 *)(st + PJ_A_BYTES);
                            for (int i = t; i < PJ_A_BYTES / 16; i += 128) {
                                float4 v = asrc[i];
                                adst[i] = split4_rn(v);
                                asrc[i] = v;
                            }
                        }
                        fence_proxy_async_smem();
                        mbar_arrive(&conv[s]);
                    }
                }
                // drain this chain: TMEM -> (+)= FP32 partial sums of this K slice (round-to-nearest adds)
                mbar_wait(acc_full, nd & 1);
                ++nd;
                tc_fence_after();
                const bool add = c0k > kb0;
                // the store of the slice's first chain must have landed before later chains add to it
                if (add && c0k == kb0 + q.chain && er == 0) bulk_wait<0>();
                const int zrow = (dom * q.nsplit + sp) * q.prows + mt * 256;
                for (int mb = 0; mb < nblk; ++mb) {
                    for (int cb = 0; cb < q.BN / 32; ++cb) {
                        uint32_t v[32];
                        tmem_ld32(tmem + ((uint32_t)(quarter * 32) << 16) + mb * q.BN + cb * 32, v);
                        tmem_ld_wait();
                        const int c0 = nt * q.BN + cb * 32;
                        if (c0 < q.N && nt < q.ntile_n) epi_tile_out<2>(stage, slot, &map_z, c0, zrow + mb * 128, v, er, add);
                    }
                }
                tc_fence_before();
                mbar_arrive(acc_empty);
            }
        }
        if (er == 0) bulk_wait<0>();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();          // the peer may still multicast into / arrive on this CTA's shared memory
    if (warp == 1) {
        __syncwarp();
        tmem_dealloc(tmem, 512);
    }
}

// =================================================================================================
// Projection on CTA PAIRS (tcgen05 cta_group::2): Z[p][c] = sum_r A[r][p] * Y[r][c] over one K slice.
// One UMMA spans two SMs: M = 256 projector rows (128 per CTA: each CTA stages only its own 4 chunks of the beta
// tile) x BN <= 448 columns, the psi tile split by columns between the two shared memories.  With single-CTA UMMAs
// (proj_tc_kernel) every CTA re-reads the psi tile once per 128-row block and the operand reads alone take ~98 of the
// 128 B/cycle of shared-memory bandwidth (tensor pipe 67 % active, round 1); the pair reads every operand byte once:
// ~49 B/cycle.  beta and psi both arrive as plain FP32; the four converter / epilogue warps of EACH CTA form the
// operand pairs of their own tiles in shared memory (beta: nearest TF32 in place + exact remainder; psi: remainder
// only, the hi product reads the raw tile, whose 13 low bits kind::tf32 ignores), so the leader's single MMA thread
// needs to know that BOTH CTAs have converted a stage: the leader's converters arrive on its `conv` barrier directly,
// the peer's arrive on a local barrier that four otherwise idle lanes of the peer's MMA warp (round-robin over the
// stages, so a slow cluster-scope arrive is off everybody's critical path) forward to the leader.
// =================================================================================================
constexpr int P2_A_BYTES = 4 * PJ_BK * 128;             // this CTA's 128 projector rows: 4 chunks of [16 r x 32 p]
constexpr int P2_Y_BYTES = 7 * PJ_BK * 128;             // this CTA's half of the psi tile: <= 224 columns
constexpr int P2_STAGE_BYTES = 2 * P2_A_BYTES + 2 * P2_Y_BYTES;   // 44 KB (3xTF32); one-product modes use half
constexpr int P2_STAGES = 4;
constexpr int P2_SMEM = P2_STAGES * P2_STAGE_BYTES + 2 * EPI_TILE_BYTES + 1024 + 512;
constexpr int P2_FWD = 4;                               // forwarding lanes of the peer's MMA warp; must divide the stage count, so
                                                        // that one lane sees all uses of a barrier in order (parity waits)

static_assert(P2_STAGES % P2_FWD == 0, "one forwarding lane must see every use of a stage barrier in order");

template <bool LO>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PJ_THREADS, 1)
proj2_tc_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_y0,
                const __grid_constant__ CUtensorMap map_y1, const __grid_constant__ CUtensorMap map_y0n,
                const __grid_constant__ CUtensorMap map_y1n, const __grid_constant__ CUtensorMap map_z, const ProjParams q) {
    // map_y0 / map_y1: boxes of the WIDE column tiles' two pieces, map_y0n / map_y1n: of the tiles one unit narrower
    constexpr int NST = LO ? P2_STAGES : 2 * P2_STAGES;
    constexpr int SB = LO ? P2_STAGE_BYTES : P2_STAGE_BYTES / 2;
    constexpr int YOFF = (LO ? 2 : 1) * P2_A_BYTES;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *stage = smem + NST * SB;
    uint64_t *bars = (uint64_t *)(stage + 2 * EPI_TILE_BYTES);
    uint64_t *full = bars, *empty = bars + NST, *conv = bars + 2 * NST, *cdone = bars + 3 * NST;
    uint64_t *acc_full = bars + 4 * NST, *acc_empty = acc_full + 1;
    uint32_t *tmem_slot = (uint32_t *)(acc_empty + 1);
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int crank = (int)cluster_ctarank();
    const bool leader = crank == 0;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; ++s) {
            mbar_init(&full[s], 1);          // LOCAL: this CTA's tiles have landed
            mbar_init(&empty[s], 1);         // the leader's tcgen05.commit, multicast to both CTAs
            mbar_init(&conv[s], 128 + 1);    // used in the leader: its 128 converter threads + the peer's forwarder
            mbar_init(&cdone[s], 128);       // used in the peer: its 128 converter threads
        }
        mbar_init(acc_full, 1);              // commit multicast
        mbar_init(acc_empty, 2);             // one elected epilogue thread per CTA (remote arrive on the leader)
        fence_barrier_init();
        prefetch_tmap(&map_a);
        prefetch_tmap(&map_y0);
        prefetch_tmap(&map_y1);
        prefetch_tmap(&map_y0n);
        prefetch_tmap(&map_y1n);
        prefetch_tmap(&map_z);
    }
    if (warp == 1) tmem_alloc_2cta(tmem_slot, 512);
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int ncl = gridDim.x / 2, cl = blockIdx.x / 2;

    const int nkb = q.ngrid / PJ_BK;
    const int total = q.ndom * q.ntile_m * q.ntile_n * q.nsplit;   // pair units
    const bool need_lo = q.nprod == 3;

    auto decode = [&](int u, int &dom, int &mt, int &nt, int &sp, int &kb0, int &kb1) {
        nt = u % q.ntile_n;
        u /= q.ntile_n;
        sp = u % q.nsplit;
        u /= q.nsplit;
        mt = u % q.ntile_m;
        dom = u / q.ntile_m;
        kb0 = (int)((long)nkb * sp / q.nsplit);
        kb1 = (int)((long)nkb * (sp + 1) / q.nsplit);
    };

    if (warp == 0) {
        if (lane == 0) {
            int it = 0;
            for (int u = cl; u < total; u += ncl) {
                int dom, mt, nt, sp, kb0, kb1;
                decode(u, dom, mt, nt, sp, kb0, kb1);
                const ColTile ct = col_tile(q.cs, nt);
                const int h0 = ct.h0, h1 = ct.h1;
                const int ch0 = ct.start / 32 + crank * h0, ch1 = ct.start / 32 + ct.n0 / 32 + crank * h1;
                const bool narrow = nt >= q.cs.wt;
                const CUtensorMap *my0 = narrow ? &map_y0n : &map_y0, *my1 = narrow ? &map_y1n : &map_y1;
                const uint32_t tx_bytes = P2_A_BYTES + (uint32_t)(h0 + h1) * PJ_BK * 128;
                for (int kb = kb0; kb < kb1; ++kb, ++it) {
                    const int s = it % NST;
                    mbar_wait(&empty[s], ((it / NST) & 1) ^ 1);
                    uint8_t *st = smem + s * SB;
                    mbar_expect_tx(&full[s], tx_bytes);
                    const int row = dom * q.ngrid + kb * PJ_BK;
                    tma_load_3d(st, &map_a, &full[s], 0, row, mt * 8 + crank * 4);
                    tma_load_3d(st + YOFF, my0, &full[s], 0, row, ch0);
                    if (h1) tma_load_3d(st + YOFF + h0 * (PJ_BK * 128), my1, &full[s], 0, row, ch1);
                }
            }
        }
    } else if (warp == 1) {
        if (leader) {
            if (lane == 0) {
                int it = 0, nd = 0;   // nd: accumulator hand-overs (drains) so far
                for (int u = cl; u < total; u += ncl) {
                    int dom, mt, nt, sp, kb0, kb1;
                    decode(u, dom, mt, nt, sp, kb0, kb1);
                    const ColTile ct = col_tile(q.cs, nt);
                    const int n0 = ct.n0, h0 = ct.h0, h1 = ct.h1;
                    const uint32_t id0 = instr_desc(FMT_TF32, 1, 1, 256, (uint32_t)n0);
                    const uint32_t id1 = instr_desc(FMT_TF32, 1, 1, 256, (uint32_t)(ct.n1 ? ct.n1 : 64));
                    for (int kb = kb0; kb < kb1; ++kb, ++it) {
                        const bool first = (kb - kb0) % q.chain == 0;
                        if (first) {
                            mbar_wait(acc_empty, (nd & 1) ^ 1);
                            tc_fence_after();
                        }
                        const int s = it % NST;
                        mbar_wait(&conv[s], (it / NST) & 1);   // both CTAs' tiles landed and converted
                        tc_fence_after();
                        const uint32_t st = smem_u32(smem + s * SB);
                        const uint32_t a_hi = st, a_lo = st + P2_A_BYTES, y_hi = st + YOFF, y_lo = st + YOFF + P2_Y_BYTES;
#pragma unroll
                        for (int k8 = 0; k8 < PJ_BK / 8; ++k8) {
                            const uint32_t acc = (!first || k8 > 0) ? 1u : 0u;
                            const uint64_t da = smem_desc(a_hi + k8 * 1024, PJ_BK * 128, 512, LAYOUT_SW128_32B);
                            const uint64_t dal = smem_desc(a_lo + k8 * 1024, PJ_BK * 128, 512, LAYOUT_SW128_32B);
                            {
                                const uint64_t dy = smem_desc(y_hi + k8 * 1024, PJ_BK * 128, 512, LAYOUT_SW128_32B);
                                umma_tf32_2cta(tmem, da, dy, id0, acc);
                                if (need_lo) {
                                    umma_tf32_2cta(tmem, dal, dy, id0, 1u);
                                    umma_tf32_2cta(tmem, da, smem_desc(y_lo + k8 * 1024, PJ_BK * 128, 512, LAYOUT_SW128_32B), id0, 1u);
                                }
                            }
                            if (h1) {
                                const uint32_t yo = (uint32_t)h0 * (PJ_BK * 128) + k8 * 1024;
                                const uint64_t dy = smem_desc(y_hi + yo, PJ_BK * 128, 512, LAYOUT_SW128_32B);
                                umma_tf32_2cta(tmem + n0, da, dy, id1, acc);
                                if (need_lo) {
                                    umma_tf32_2cta(tmem + n0, dal, dy, id1, 1u);
                                    umma_tf32_2cta(tmem + n0, da, smem_desc(y_lo + yo, PJ_BK * 128, 512, LAYOUT_SW128_32B), id1, 1u);
                                }
                            }
                        }
                        umma_commit_2cta_mc(&empty[s], (uint16_t)3);
                        if ((kb - kb0 + 1) % q.chain == 0 || kb + 1 == kb1) {
                            umma_commit_2cta_mc(acc_full, (uint16_t)3);
                            ++nd;
                        }
                    }
                }
            }
        } else if (lane < P2_FWD) {
            // the peer's MMA warp has nothing to issue: its first lanes forward "stage converted" to the leader
            int it = 0;
            for (int u = cl; u < total; u += ncl) {
                int dom, mt, nt, sp, kb0, kb1;
                decode(u, dom, mt, nt, sp, kb0, kb1);
                for (int kb = kb0; kb < kb1; ++kb, ++it) {
                    if (it % P2_FWD != lane) continue;
                    const int s = it % NST;
                    mbar_wait(&cdone[s], (it / NST) & 1);
                    mbar_arrive_remote(&conv[s], 0);
                }
            }
        }
    } else {
        const int t = threadIdx.x - 64;   // 0..127
        const int quarter = warp % 4;
        const int er = quarter * 32 + lane;   // TMEM lane = accumulator row of this thread; er == 0 leads the TMA stores
        uint64_t *done = leader ? conv : cdone;
        int it = 0, nd = 0, slot = 0;
        for (int u = cl; u < total; u += ncl) {
            int dom, mt, nt, sp, kb0, kb1;
            decode(u, dom, mt, nt, sp, kb0, kb1);
            const ColTile ct = col_tile(q.cs, nt);
            const int n0 = ct.n0, h0 = ct.h0, h1 = ct.h1;
            const int ny4 = (h0 + h1) * PJ_BK * 8;    // float4 count of this CTA's psi tile
            const bool rows_live = q.P - mt * 256 - crank * 128 > 0;
            for (int c0k = kb0; c0k < kb1; c0k += q.chain) {
                const int c1k = min(c0k + q.chain, kb1);
                for (int kb = c0k; kb < c1k; ++kb, ++it) {
                    const int s = it % NST;
                    mbar_wait(&full[s], (it / NST) & 1);
                    uint8_t *st = smem + s * SB;
                    float4 *a4 = (float4 *)st;
                    float4 *y4 = (float4 *)(st + YOFF);
                    if (q.lowp) {
                        // opt-in low precision (PAPER.md L207, L239 float_to_BF16): both operands rounded to BF16
                        for (int i = t; i < ny4; i += 128) y4[i] = bf16_round4(y4[i]);
                        for (int i = t; i < P2_A_BYTES / 16; i += 128) a4[i] = bf16_round4(a4[i]);
                    } else if (!LO) {
                        for (int i = t; i < P2_A_BYTES / 16; i += 128) a4[i] = tf32_rn4(a4[i]);
                        if (q.rn && q.rho) {
                            // S3 fused, as in the three-product branch below (same tile layout, same thread -> row / orbital map):
                            // the density is summed from the values as loaded, then psi is rounded in place
                            const int r = (t >> 3) & 15, w = t & 7;
                            const int pair_in_chunk = (((w >> 1) ^ (r & 3)) << 1) | (w & 1);
                            const float2 *f2 = (const float2 *)(q.occ + (size_t)dom * (q.N / 2));
                            float acc = 0.f;
                            int j = 0;
                            for (int i = t; i < ny4; i += 128, ++j) {
                                const float4 v = y4[i];
                                const int gch = j < h0 ? ct.start / 32 + crank * h0 + j : ct.start / 32 + n0 / 32 + crank * h1 + (j - h0);
                                const float2 ff = __ldg(f2 + gch * 8 + pair_in_chunk);
                                acc = fmaf(ff.x, fmaf(v.x, v.x, v.y * v.y), acc);
                                acc = fmaf(ff.y, fmaf(v.z, v.z, v.w * v.w), acc);
                                y4[i] = tf32_rn4(v);
                            }
                            acc += __shfl_xor_sync(0xffffffffu, acc, 1);
                            acc += __shfl_xor_sync(0xffffffffu, acc, 2);
                            acc += __shfl_xor_sync(0xffffffffu, acc, 4);
                            if (w == 0) atomicAdd(q.rho + (size_t)dom * q.ngrid + (size_t)kb * PJ_BK + r, acc);
                        } else if (q.rn)
                            for (int i = t; i < ny4; i += 128) y4[i] = tf32_rn4(y4[i]);
                    } else {
                        // elementwise on the swizzled image: the lo tile has the same layout as the hi tile
                        float4 *yl = (float4 *)(st + YOFF + P2_Y_BYTES);
                        if (q.rho) {
                            // S3 fused: thread t always holds row (t >> 3) & 15 of every chunk (a chunk = 16 rows x 8 units of
                            // 16 B) and, undoing the 32-byte-atom swizzle (atom index ^ row & 3), the same pair of orbitals
                            // inside each chunk; the 8 threads of a row are neighbouring lanes.  One FP32 sum per (CTA, row),
                            // added to rho by ONE atomic: two addends per row (the pair's two column halves), so the result
                            // does not depend on their order (reading D22).
                            const int r = (t >> 3) & 15, w = t & 7;
                            const int pair_in_chunk = (((w >> 1) ^ (r & 3)) << 1) | (w & 1);
                            const float2 *f2 = (const float2 *)(q.occ + (size_t)dom * (q.N / 2));
                            float acc = 0.f;
                            int j = 0;
                            for (int i = t; i < ny4; i += 128, ++j) {
                                float4 v = y4[i];
                                const int gch = j < h0 ? ct.start / 32 + crank * h0 + j : ct.start / 32 + n0 / 32 + crank * h1 + (j - h0);
                                const float2 ff = __ldg(f2 + gch * 8 + pair_in_chunk);
                                acc = fmaf(ff.x, fmaf(v.x, v.x, v.y * v.y), acc);
                                acc = fmaf(ff.y, fmaf(v.z, v.z, v.w * v.w), acc);
                                yl[i] = split4(v);
                            }
                            acc += __shfl_xor_sync(0xffffffffu, acc, 1);
                            acc += __shfl_xor_sync(0xffffffffu, acc, 2);
                            acc += __shfl_xor_sync(0xffffffffu, acc, 4);
                            if (w == 0) atomicAdd(q.rho + (size_t)dom * q.ngrid + (size_t)kb * PJ_BK + r, acc);
                        } else
                        for (int i = t; i < ny4; i += 128) {
                            float4 v = y4[i];
                            yl[i] = split4(v);   // the hi tile stays as loaded: kind::tf32 ignores the 13 low bits
                        }
                        float4 *al = (float4 *)(st + P2_A_BYTES);
                        for (int i = t; i < P2_A_BYTES / 16; i += 128) {
                            float4 v = a4[i];
                            al[i] = split4_rn(v);
                            a4[i] = v;
                        }
                    }
                    fence_proxy_async_smem();
                    mbar_arrive(&done[s]);
                }
                // drain this chain: TMEM -> (+)= FP32 partial sums of this K slice (round-to-nearest adds)
                mbar_wait(acc_full, nd & 1);
                ++nd;
                tc_fence_after();
                const bool add = c0k > kb0;
                // the store of the slice's first chain must have landed before later chains add to it
                if (add && c0k == kb0 + q.chain && er == 0) bulk_wait<0>();
                const int zrow = (dom * q.nsplit + sp) * q.prows + mt * 256 + crank * 128;
                for (int cb = 0; cb < ct.width / 32; ++cb) {
                    uint32_t v[32];
                    tmem_ld32(tmem + ((uint32_t)(quarter * 32) << 16) + cb * 32, v);
                    tmem_ld_wait();
                    const int c0 = ct.start + cb * 32;
                    if (rows_live) epi_tile_out<2>(stage, slot, &map_z, c0, zrow, v, er, add);
                }
                tc_fence_before();
                named_bar_sync(EPI_BAR, 128);
                if (er == 0) mbar_arrive_remote(acc_empty, 0);   // this CTA's half of the accumulator is drained
            }
        }
        if (er == 0) bulk_wait<0>();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 1) {
        __syncwarp();
        tmem_dealloc_2cta(tmem, 512);
    }
}

// =================================================================================================
// Opt-in low-precision projection (PAPER.md L207, L239 float_to_BF16; L296): BF16 x BF16 -> FP32 on CTA pairs with
// tcgen05.mma.kind::f16 (K = 16 per instruction: one instruction per 16-row stage and column piece).  beta is read as
// its stored BF16 copy (2 bytes per element instead of round 1's 8); psi arrives as FP32 (its only copy) and the
// converter warps of each CTA write its BF16 image, re-laid-out from the FP32 tile's 32-byte-atom swizzle to the
// 64-byte swizzle of a BF16 MN-major operand, next to it.  Same unit / chain / handshake structure as proj2_tc_kernel.
// =================================================================================================
constexpr int PH_A_BYTES = 4 * PJ_BK * 64;              // this CTA's 128 projector rows: 4 chunks of [16 r x 32 p] BF16
constexpr int PH_Y16_BYTES = 7 * PJ_BK * 64;            // BF16 image of this CTA's half of the psi tile
constexpr int PH_STAGE_BYTES = 4096 + P2_Y_BYTES + 7168;     // beta16 (4 KB) + psi FP32 staging (14 KB) + psi16 (7 KB)
constexpr int PH_STAGES = 7;
constexpr int PH_FWD = PH_STAGES;                       // one forwarding lane per stage
constexpr int PH_SMEM = PH_STAGES * PH_STAGE_BYTES + 2 * EPI_TILE_BYTES + 1024 + 512;
static_assert(PH_A_BYTES == 4096 && PH_Y16_BYTES == 7168, "stage carving");
static_assert(PH_SMEM <= 232448, "shared memory of proj2h_tc_kernel");

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PJ_THREADS, 1)
proj2h_tc_kernel(const __grid_constant__ CUtensorMap map_a16, const __grid_constant__ CUtensorMap map_y0,
                 const __grid_constant__ CUtensorMap map_y1, const __grid_constant__ CUtensorMap map_y0n,
                 const __grid_constant__ CUtensorMap map_y1n, const __grid_constant__ CUtensorMap map_z, const ProjParams q) {
    constexpr int NST = PH_STAGES, SB = PH_STAGE_BYTES, YOFF = PH_A_BYTES, Y16OFF = PH_A_BYTES + P2_Y_BYTES;
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *stage = smem + NST * SB;
    uint64_t *bars = (uint64_t *)(stage + 2 * EPI_TILE_BYTES);
    uint64_t *full = bars, *empty = bars + NST, *conv = bars + 2 * NST, *cdone = bars + 3 * NST;
    uint64_t *acc_full = bars + 4 * NST, *acc_empty = acc_full + 1;
    uint32_t *tmem_slot = (uint32_t *)(acc_empty + 1);
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int crank = (int)cluster_ctarank();
    const bool leader = crank == 0;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NST; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 1);
            mbar_init(&conv[s], 128 + 1);
            mbar_init(&cdone[s], 128);
        }
        mbar_init(acc_full, 1);
        mbar_init(acc_empty, 2);
        fence_barrier_init();
        prefetch_tmap(&map_a16);
        prefetch_tmap(&map_y0);
        prefetch_tmap(&map_y1);
        prefetch_tmap(&map_z);
    }
    if (warp == 1) tmem_alloc_2cta(tmem_slot, 512);
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int ncl = gridDim.x / 2, cl = blockIdx.x / 2;
    const int nkb = q.ngrid / PJ_BK;
    const int total = q.ndom * q.ntile_m * q.ntile_n * q.nsplit;

    auto decode = [&](int u, int &dom, int &mt, int &nt, int &sp, int &kb0, int &kb1) {
        nt = u % q.ntile_n;
        u /= q.ntile_n;
        sp = u % q.nsplit;
        u /= q.nsplit;
        mt = u % q.ntile_m;
        dom = u / q.ntile_m;
        kb0 = (int)((long)nkb * sp / q.nsplit);
        kb1 = (int)((long)nkb * (sp + 1) / q.nsplit);
    };

    if (warp == 0) {
        if (lane == 0) {
            int it = 0;
            for (int u = cl; u < total; u += ncl) {
                int dom, mt, nt, sp, kb0, kb1;
                decode(u, dom, mt, nt, sp, kb0, kb1);
                const ColTile ct = col_tile(q.cs, nt);
                const int h0 = ct.h0, h1 = ct.h1;
                const int ch0 = ct.start / 32 + crank * h0, ch1 = ct.start / 32 + ct.n0 / 32 + crank * h1;
                const bool narrow = nt >= q.cs.wt;
                const CUtensorMap *my0 = narrow ? &map_y0n : &map_y0, *my1 = narrow ? &map_y1n : &map_y1;
                const uint32_t tx_bytes = PH_A_BYTES + (uint32_t)(h0 + h1) * PJ_BK * 128;
                for (int kb = kb0; kb < kb1; ++kb, ++it) {
                    const int s = it % NST;
                    mbar_wait(&empty[s], ((it / NST) & 1) ^ 1);
                    uint8_t *st = smem + s * SB;
                    mbar_expect_tx(&full[s], tx_bytes);
                    const int row = dom * q.ngrid + kb * PJ_BK;
                    tma_load_3d(st, &map_a16, &full[s], 0, row, mt * 8 + crank * 4);
                    tma_load_3d(st + YOFF, my0, &full[s], 0, row, ch0);
                    if (h1) tma_load_3d(st + YOFF + h0 * (PJ_BK * 128), my1, &full[s], 0, row, ch1);
                }
            }
        }
    } else if (warp == 1) {
        if (leader) {
            if (lane == 0) {
                int it = 0, nd = 0;
                for (int u = cl; u < total; u += ncl) {
                    int dom, mt, nt, sp, kb0, kb1;
                    decode(u, dom, mt, nt, sp, kb0, kb1);
                    const ColTile ct = col_tile(q.cs, nt);
                    const uint32_t id0 = instr_desc(FMT_BF16, 1, 1, 256, (uint32_t)ct.n0);
                    const uint32_t id1 = instr_desc(FMT_BF16, 1, 1, 256, (uint32_t)(ct.n1 ? ct.n1 : 64));
                    for (int kb = kb0; kb < kb1; ++kb, ++it) {
                        const bool first = (kb - kb0) % q.chain == 0;
                        if (first) {
                            mbar_wait(acc_empty, (nd & 1) ^ 1);
                            tc_fence_after();
                        }
                        const int s = it % NST;
                        mbar_wait(&conv[s], (it / NST) & 1);
                        tc_fence_after();
                        const uint32_t st = smem_u32(smem + s * SB);
                        // MN-major BF16 chunks of [16 rows x 64 B]: chunk stride 1024, 8-row group stride 512
                        const uint64_t da = smem_desc(st, PJ_BK * 64, 512, LAYOUT_SW64);
                        const uint64_t dy0 = smem_desc(st + Y16OFF, PJ_BK * 64, 512, LAYOUT_SW64);
                        umma_f16_2cta(tmem, da, dy0, id0, first ? 0u : 1u);
                        if (ct.h1) {
                            const uint64_t dy1 = smem_desc(st + Y16OFF + ct.h0 * (PJ_BK * 64), PJ_BK * 64, 512, LAYOUT_SW64);
                            umma_f16_2cta(tmem + ct.n0, da, dy1, id1, first ? 0u : 1u);
                        }
                        umma_commit_2cta_mc(&empty[s], (uint16_t)3);
                        if ((kb - kb0 + 1) % q.chain == 0 || kb + 1 == kb1) {
                            umma_commit_2cta_mc(acc_full, (uint16_t)3);
                            ++nd;
                        }
                    }
                }
            }
        } else if (lane < PH_FWD) {
            int it = 0;
            for (int u = cl; u < total; u += ncl) {
                int dom, mt, nt, sp, kb0, kb1;
                decode(u, dom, mt, nt, sp, kb0, kb1);
                for (int kb = kb0; kb < kb1; ++kb, ++it) {
                    if (it % PH_FWD != lane) continue;
                    const int s = it % NST;
                    mbar_wait(&cdone[s], (it / NST) & 1);
                    mbar_arrive_remote(&conv[s], 0);
                }
            }
        }
    } else {
        const int t = threadIdx.x - 64;
        const int quarter = warp % 4;
        const int er = quarter * 32 + lane;
        uint64_t *done = leader ? conv : cdone;
        // thread t holds row r, 16-byte unit w of every FP32 chunk; logical float column c of that unit (32-byte-atom
        // swizzle undone); its four BF16 go to row r of the BF16 chunk at bytes 2c .. 2c + 7, 16-byte units swizzled by
        // (r >> 1) & 3 (64-byte swizzle)
        const int r = (t >> 3) & 15, w = t & 7;
        const int c = (((w >> 1) ^ (r & 3)) << 3) | ((w & 1) << 2);
        const uint32_t dst_off = (uint32_t)(r * 64 + ((((c >> 3) ^ ((r >> 1) & 3))) << 4) + ((c >> 2) & 1) * 8);
        int it = 0, nd = 0, slot = 0;
        for (int u = cl; u < total; u += ncl) {
            int dom, mt, nt, sp, kb0, kb1;
            decode(u, dom, mt, nt, sp, kb0, kb1);
            const ColTile ct = col_tile(q.cs, nt);
            const int nch = ct.h0 + ct.h1;
            const bool rows_live = q.P - mt * 256 - crank * 128 > 0;
            for (int c0k = kb0; c0k < kb1; c0k += q.chain) {
                const int c1k = min(c0k + q.chain, kb1);
                for (int kb = c0k; kb < c1k; ++kb, ++it) {
                    const int s = it % NST;
                    mbar_wait(&full[s], (it / NST) & 1);
                    uint8_t *st = smem + s * SB;
                    const float4 *y4 = (const float4 *)(st + YOFF);
                    const uint32_t y16 = smem_u32(st + Y16OFF) + dst_off;
                    if (q.rho) {
                        // S3 fused, as in proj2_tc_kernel (same FP32 tile layout, same thread -> row / orbital map): the density
                        // is summed from the FP32 values as loaded, before they are packed to BF16
                        const int pair_in_chunk = (((w >> 1) ^ (r & 3)) << 1) | (w & 1);
                        const float2 *f2 = (const float2 *)(q.occ + (size_t)dom * (q.N / 2));
                        float acc = 0.f;
                        for (int j = 0; j < nch; ++j) {
                            const float4 v = y4[j * 128 + t];
                            const int gch = j < ct.h0 ? ct.start / 32 + crank * ct.h0 + j
                                                      : ct.start / 32 + ct.n0 / 32 + crank * ct.h1 + (j - ct.h0);
                            const float2 ff = __ldg(f2 + gch * 8 + pair_in_chunk);
                            acc = fmaf(ff.x, fmaf(v.x, v.x, v.y * v.y), acc);
                            acc = fmaf(ff.y, fmaf(v.z, v.z, v.w * v.w), acc);
                            sts2(y16 + j * (PJ_BK * 64), pack_bf16(v.x, v.y), pack_bf16(v.z, v.w));
                        }
                        acc += __shfl_xor_sync(0xffffffffu, acc, 1);
                        acc += __shfl_xor_sync(0xffffffffu, acc, 2);
                        acc += __shfl_xor_sync(0xffffffffu, acc, 4);
                        if (w == 0) atomicAdd(q.rho + (size_t)dom * q.ngrid + (size_t)kb * PJ_BK + r, acc);
                    } else
                    for (int j = 0; j < nch; ++j) {
                        const float4 v = y4[j * 128 + t];
                        sts2(y16 + j * (PJ_BK * 64), pack_bf16(v.x, v.y), pack_bf16(v.z, v.w));
                    }
                    fence_proxy_async_smem();
                    mbar_arrive(&done[s]);
                }
                mbar_wait(acc_full, nd & 1);
                ++nd;
                tc_fence_after();
                const bool add = c0k > kb0;
                if (add && c0k == kb0 + q.chain && er == 0) bulk_wait<0>();
                const int zrow = (dom * q.nsplit + sp) * q.prows + mt * 256 + crank * 128;
                for (int cb = 0; cb < ct.width / 32; ++cb) {
                    uint32_t v[32];
                    tmem_ld32(tmem + ((uint32_t)(quarter * 32) << 16) + cb * 32, v);
                    tmem_ld_wait();
                    if (rows_live) epi_tile_out<2>(stage, slot, &map_z, ct.start + cb * 32, zrow, v, er, add);
                }
                tc_fence_before();
                named_bar_sync(EPI_BAR, 128);
                if (er == 0) mbar_arrive_remote(acc_empty, 0);
            }
        }
        if (er == 0) bulk_wait<0>();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 1) {
        __syncwarp();
        tmem_dealloc_2cta(tmem, 512);
    }
}

// =================================================================================================
// Back-application: Y[r][c] += sum_p A[r][p] * W[p][c].
// CTA tile: 128 grid points x BN <= 448 columns (TMEM accumulator), K pipeline of 8 projector rows.
// CTAs run as clusters of two on neighbouring row tiles: the W slab of a stage is the same for both, so
// each CTA fetches half of it and TMA-multicasts it into both shared memories (the GEMM is otherwise
// bound by L2->SM bandwidth, ~43 B/cycle/SM measured, not by the tensor pipe).
// =================================================================================================
constexpr int BK_STAGES = 5;
constexpr int BK_EPI_NB = 2;                            // staging tiles of the epilogue in flight
constexpr int BK_MAXBN = 448;
constexpr int BK_A_BYTES = 128 * 32;                    // [128 rows x 8 floats], SWIZZLE_32B
constexpr int BK_W_BYTES = (BK_MAXBN / 32) * 1024;      // chunks of [8 rows x 128 B], SWIZZLE_128B
constexpr int BK_STAGE_BYTES = 2 * BK_A_BYTES + 2 * BK_W_BYTES;
constexpr int BK_SMEM = BK_STAGES * BK_STAGE_BYTES + BK_EPI_NB * EPI_TILE_BYTES + 1024 + 512;
constexpr int BK_EPI_WARPS = 4;
constexpr int BK_THREADS = 64 + 32 * BK_EPI_WARPS;

struct BackParams {
    int ndom, ngrid, P, N, BN, ntile_n, prows, nprod, ldy, lowp;
    float *Y;
    ColSplit cs;                 // column tiles of the CTA-pair kernel
};

// beta arrives as ONE FP32 copy (raw); the operand pair of 3xTF32 is formed in shared memory:
//   hi = beta rounded to the nearest TF32 (in place), lo = beta - hi (exact) into the second slot.
// mode: 0 = hi/lo pair, 1 = hi only (one-product modes), 2 = BF16 rounding in place (low precision)
__device__ __forceinline__ void convert_a_slab(uint8_t *st, int t, int nthreads, int mode) {
    float4 *a4 = (float4 *)st;
    float4 *l4 = (float4 *)(st + BK_A_BYTES);
    if (mode == 0) {
        for (int i = t; i < BK_A_BYTES / 16; i += nthreads) {
            float4 v = a4[i];
            l4[i] = split4_rn(v);
            a4[i] = v;
        }
    } else if (mode == 1) {
        for (int i = t; i < BK_A_BYTES / 16; i += nthreads) a4[i] = tf32_rn4(a4[i]);
    } else {
        for (int i = t; i < BK_A_BYTES / 16; i += nthreads) a4[i] = bf16_round4(a4[i]);
    }
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(BK_THREADS, 1)
back_tc_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_whi,
               const __grid_constant__ CUtensorMap map_wlo, const __grid_constant__ CUtensorMap map_out, const BackParams q) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *stage = smem + BK_STAGES * BK_STAGE_BYTES;
    uint64_t *bars = (uint64_t *)(stage + BK_EPI_NB * EPI_TILE_BYTES);
    uint64_t *full = bars, *empty = bars + BK_STAGES, *conv = bars + 2 * BK_STAGES;
    uint64_t *acc_full = bars + 3 * BK_STAGES, *acc_empty = acc_full + 1;
    uint32_t *tmem_slot = (uint32_t *)(acc_empty + 1);
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;

    if (threadIdx.x == 0) {
        for (int s = 0; s < BK_STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 2);    // this CTA's MMAs and the peer's (its multicast half lands here too)
            mbar_init(&conv[s], 32 * BK_EPI_WARPS);
        }
        mbar_init(acc_full, 1);
        mbar_init(acc_empty, 32 * BK_EPI_WARPS);
        fence_barrier_init();
        prefetch_tmap(&map_a);
        prefetch_tmap(&map_whi);
        prefetch_tmap(&map_wlo);
        prefetch_tmap(&map_out);
    }
    if (warp == 1) tmem_alloc(tmem_slot, 512);
    tc_fence_before();
    cluster_sync_all();          // barrier inits visible to the peer before any remote arrive / multicast
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const int crank = (int)cluster_ctarank();

    const int nrt = q.ngrid / 128;                 // row tiles per domain
    const int nrp = (nrt + 1) / 2;                 // pairs of row tiles: one per cluster unit
    const int total = q.ndom * nrp * q.ntile_n;    // cluster units
    const int ncl = gridDim.x / 2, cl = blockIdx.x / 2;
    const int nk = (q.P + 7) / 8;
    // nprod 3: beta_hi W_hi + beta_lo W_hi + beta_hi W_lo; nprod 2 (staged mode): the first two (W taken as one TF32)
    const bool need_lo = q.nprod >= 2, need_wlo = q.nprod == 3;
    const int cmode = q.lowp ? 2 : (need_lo ? 0 : 1);
    const int nchunk = q.BN / 32, chalf = (nchunk + 1) / 2;   // W chunks: this CTA fetches `chalf` of them
    const uint32_t w_bytes = (uint32_t)(2 * chalf) * 1024;
    const uint32_t tx_bytes = BK_A_BYTES + (need_wlo ? 2u : 1u) * w_bytes;
    const int ninstr = q.BN > 256 ? 2 : 1;
    const int NI = q.BN / ninstr;                   // columns per UMMA instruction (multiple of 32)

    if (warp == 0) {
        if (lane == 0) {
            int it = 0;
            for (int u = cl; u < total; u += ncl) {
                const int nt = u % q.ntile_n, rt = 2 * ((u / q.ntile_n) % nrp) + crank, dom = u / (q.ntile_n * nrp);
                const int row = dom * q.ngrid + rt * 128;
                for (int k = 0; k < nk; ++k, ++it) {
                    const int s = it % BK_STAGES;
                    mbar_wait(&empty[s], ((it / BK_STAGES) & 1) ^ 1);
                    uint8_t *st = smem + s * BK_STAGE_BYTES;
                    mbar_expect_tx(&full[s], tx_bytes);
                    tma_load_2d(st, &map_a, &full[s], k * 8, row);
                    tma_load_3d_mc(st + 2 * BK_A_BYTES + crank * chalf * 1024, &map_whi, &full[s], 0, dom * q.prows + k * 8,
                                   nt * nchunk + crank * chalf, (uint16_t)3);
                    if (need_wlo)
                        tma_load_3d_mc(st + 2 * BK_A_BYTES + BK_W_BYTES + crank * chalf * 1024, &map_wlo, &full[s], 0,
                                       dom * q.prows + k * 8, nt * nchunk + crank * chalf, (uint16_t)3);
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            const uint32_t idesc = instr_desc(FMT_TF32, 0, 1, 128, (uint32_t)NI);
            int it = 0, nu = 0;
            for (int u = cl; u < total; u += ncl, ++nu) {
                mbar_wait(acc_empty, (nu & 1) ^ 1);
                tc_fence_after();
                for (int k = 0; k < nk; ++k, ++it) {
                    const int s = it % BK_STAGES;
                    mbar_wait(&full[s], (it / BK_STAGES) & 1);
                    mbar_wait(&conv[s], (it / BK_STAGES) & 1);
                    tc_fence_after();
                    const uint32_t st = smem_u32(smem + s * BK_STAGE_BYTES);
                    const uint64_t da = smem_desc(st, 16, 256, LAYOUT_SW32);
                    const uint64_t dal = smem_desc(st + BK_A_BYTES, 16, 256, LAYOUT_SW32);
                    for (int h = 0; h < ninstr; ++h) {
                        const uint32_t woff = (uint32_t)h * (NI / 32) * 1024;
                        const uint64_t dw = smem_desc(st + 2 * BK_A_BYTES + woff, 1024, 512, LAYOUT_SW128_32B);
                        const uint32_t d = tmem + h * NI;
                        umma_tf32(d, da, dw, idesc, k > 0 ? 1u : 0u);
                        if (need_lo) umma_tf32(d, dal, dw, idesc, 1u);
                        if (need_wlo) {
                            const uint64_t dwl = smem_desc(st + 2 * BK_A_BYTES + BK_W_BYTES + woff, 1024, 512, LAYOUT_SW128_32B);
                            umma_tf32(d, da, dwl, idesc, 1u);
                        }
                    }
                    umma_commit_mc(&empty[s], (uint16_t)3);   // frees the stage in both CTAs of the cluster
                }
                umma_commit(acc_full);
            }
        }
    } else {
        const int quarter = warp % 4;
        const int er = quarter * 32 + lane;         // accumulator row of this thread
        int nu = 0, slot = 0, it = 0;
        for (int u = cl; u < total; u += ncl, ++nu) {
            const int nt = u % q.ntile_n, rt = 2 * ((u / q.ntile_n) % nrp) + crank, dom = u / (q.ntile_n * nrp);
            const int row0 = dom * q.ngrid + rt * 128;
            const bool live = rt < nrt;           // odd tile count: the last pair's second CTA only keeps the protocol going
            // the epilogue warps (idle during the main loop) form the operand pair of every beta slab in place
            for (int k = 0; k < nk; ++k, ++it) {
                const int s = it % BK_STAGES;
                mbar_wait(&full[s], (it / BK_STAGES) & 1);
                convert_a_slab(smem + s * BK_STAGE_BYTES, er, 32 * BK_EPI_WARPS, cmode);
                fence_proxy_async_smem();
                mbar_arrive(&conv[s]);
            }
            mbar_wait(acc_full, nu & 1);
            tc_fence_after();
            for (int cb = 0; cb < q.BN / 32; ++cb) {
                uint32_t v[32];
                tmem_ld32(tmem + ((uint32_t)(quarter * 32) << 16) + cb * 32, v);
                tmem_ld_wait();
                const int c0 = nt * q.BN + cb * 32;
                // Y += tile through the TMA engine: the add happens in L2, nothing is read back into the SM
                if (c0 < q.N && live) epi_tile_out<BK_EPI_NB>(stage, slot, &map_out, c0, row0, v, er, true);
            }
            tc_fence_before();
            mbar_arrive(acc_empty);
        }
        if (er == 0) bulk_wait<0>();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();          // the peer may still multicast into / arrive on this CTA's shared memory
    if (warp == 1) {
        __syncwarp();
        tmem_dealloc(tmem, 512);
    }
}

// =================================================================================================
// Back-application on CTA PAIRS (tcgen05 cta_group::2): Y[r][c] += sum_p A[r][p] * W[p][c].
// One UMMA spans two SMs: M = 256 grid points (128 per CTA, each CTA stages only its own beta slab)
// and the W slab is split by columns between the two shared memories, so every operand byte is read
// from shared memory once per pair instead of once per CTA.  With single-CTA UMMAs (M = 128) the
// operand reads alone take ~98 of the 128 B/cycle of shared-memory bandwidth and, together with the
// TMA fills, cap the tensor pipe near 75 % (measured); this is what cta_group::2 exists for.
// Per CTA: 128 x BN accumulator in TMEM (BN <= 448, BN % 64 == 0), UMMA pieces of N = 256 and BN - 256.
//
// Operands of 3xTF32: the hi product reads the RAW FP32 beta slab (kind::tf32 ignores the 13 low mantissa bits, i.e.
// uses beta truncated to TF32), the lo product the stored remainder beta - trunc(beta) (exact; written once by
// mlmd_set_projectors).  Forming that remainder in shared memory instead (as the projection does) was built and
// measured here in round 2: the leader's MMA thread then has to wait for a "slab converted" signal from BOTH CTAs
// per K = 8 stage, and the kernel went from 9.3 to 11.3 ms at configs[3] although it read 6.8 GB less
// (profiles/r2_negative_results.md), so this kernel keeps the second HBM stream.
// =================================================================================================
constexpr int B2_STAGES = 7;
constexpr int B2_WH_BYTES = 7 * 1024;                  // this CTA's half of the W slab: <= 224 columns
constexpr int B2_STAGE_BYTES = 2 * BK_A_BYTES + 2 * B2_WH_BYTES;
constexpr int B2_SMEM = B2_STAGES * B2_STAGE_BYTES + 2 * EPI_TILE_BYTES + 1024 + 512;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(BK_THREADS, 1)
back2_tc_kernel(const __grid_constant__ CUtensorMap map_ahi, const __grid_constant__ CUtensorMap map_alo,
                const __grid_constant__ CUtensorMap map_w0h, const __grid_constant__ CUtensorMap map_w0l,
                const __grid_constant__ CUtensorMap map_w1h, const __grid_constant__ CUtensorMap map_w1l,
                const __grid_constant__ CUtensorMap map_n0h, const __grid_constant__ CUtensorMap map_n0l,
                const __grid_constant__ CUtensorMap map_n1h, const __grid_constant__ CUtensorMap map_n1l,
                const __grid_constant__ CUtensorMap map_out, const BackParams q) {
    // column tiles as in the projection (col_tile): map_w* are the boxes of the wide tiles' two pieces (hi, lo),
    // map_n* those of the tiles one 64-column unit narrower
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *stage = smem + B2_STAGES * B2_STAGE_BYTES;
    uint64_t *bars = (uint64_t *)(stage + 2 * EPI_TILE_BYTES);
    uint64_t *full = bars, *empty = bars + B2_STAGES;
    uint64_t *acc_full = bars + 2 * B2_STAGES, *acc_empty = acc_full + 1;
    uint32_t *tmem_slot = (uint32_t *)(acc_empty + 1);
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int crank = (int)cluster_ctarank();
    const bool leader = crank == 0;

    if (threadIdx.x == 0) {
        for (int s = 0; s < B2_STAGES; ++s) {
            mbar_init(&full[s], 1);     // used in the leader: its own expect_tx arrive; both CTAs' TMA bytes land on it
            mbar_init(&empty[s], 1);    // the leader's tcgen05.commit, multicast to both CTAs
        }
        mbar_init(acc_full, 1);         // commit multicast
        mbar_init(acc_empty, 2);        // one elected epilogue thread per CTA (remote arrive on the leader)
        fence_barrier_init();
        prefetch_tmap(&map_ahi);
        prefetch_tmap(&map_alo);
        prefetch_tmap(&map_w0h);
        prefetch_tmap(&map_w0l);
        prefetch_tmap(&map_out);
    }
    if (warp == 1) tmem_alloc_2cta(tmem_slot, 512);
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    const int nrt = q.ngrid / 128, nrp = (nrt + 1) / 2;
    const int total = q.ndom * nrp * q.ntile_n;    // cluster units: a pair of row tiles x one column tile
    const int ncl = gridDim.x / 2, cl = blockIdx.x / 2;
    const int nk = (q.P + 7) / 8;
    const bool need_lo = q.nprod >= 2, need_wlo = q.nprod == 3;   // as in back_tc_kernel

    if (warp == 0) {
        if (lane == 0) {
            int it = 0;
            for (int u = cl; u < total; u += ncl) {
                const int nt = u % q.ntile_n, rt = 2 * ((u / q.ntile_n) % nrp) + crank, dom = u / (q.ntile_n * nrp);
                const int row = dom * q.ngrid + rt * 128;
                const ColTile ct = col_tile(q.cs, nt);
                const int h0 = ct.h0, h1 = ct.h1;
                const int ch0 = ct.start / 32 + crank * h0, ch1 = ct.start / 32 + ct.n0 / 32 + crank * h1;
                const bool narrow = nt >= q.cs.wt;
                const CUtensorMap *m0h = narrow ? &map_n0h : &map_w0h, *m0l = narrow ? &map_n0l : &map_w0l;
                const CUtensorMap *m1h = narrow ? &map_n1h : &map_w1h, *m1l = narrow ? &map_n1l : &map_w1l;
                const uint32_t cta_bytes = (need_lo ? 2u : 1u) * BK_A_BYTES + (need_wlo ? 2u : 1u) * (uint32_t)(h0 + h1) * 1024;
                for (int k = 0; k < nk; ++k, ++it) {
                    const int s = it % B2_STAGES;
                    mbar_wait(&empty[s], ((it / B2_STAGES) & 1) ^ 1);
                    uint8_t *st = smem + s * B2_STAGE_BYTES;
                    if (leader) mbar_expect_tx(&full[s], 2 * cta_bytes);
                    const int wrow = dom * q.prows + k * 8;
                    tma_load_2d_2cta(st, &map_ahi, &full[s], k * 8, row);
                    tma_load_3d_2cta(st + 2 * BK_A_BYTES, m0h, &full[s], 0, wrow, ch0);
                    if (h1) tma_load_3d_2cta(st + 2 * BK_A_BYTES + h0 * 1024, m1h, &full[s], 0, wrow, ch1);
                    if (need_lo) tma_load_2d_2cta(st + BK_A_BYTES, &map_alo, &full[s], k * 8, row);
                    if (need_wlo) {
                        tma_load_3d_2cta(st + 2 * BK_A_BYTES + B2_WH_BYTES, m0l, &full[s], 0, wrow, ch0);
                        if (h1)
                            tma_load_3d_2cta(st + 2 * BK_A_BYTES + B2_WH_BYTES + h0 * 1024, m1l, &full[s], 0, wrow, ch1);
                    }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0 && leader) {
            int it = 0, nu = 0;
            for (int u = cl; u < total; u += ncl, ++nu) {
                const ColTile ct = col_tile(q.cs, u % q.ntile_n);
                const int n0 = ct.n0, h0 = ct.h0, h1 = ct.h1;
                const uint32_t id0 = instr_desc(FMT_TF32, 0, 1, 256, (uint32_t)n0);
                const uint32_t id1 = instr_desc(FMT_TF32, 0, 1, 256, (uint32_t)(ct.n1 ? ct.n1 : 64));
                mbar_wait(acc_empty, (nu & 1) ^ 1);
                tc_fence_after();
                for (int k = 0; k < nk; ++k, ++it) {
                    const int s = it % B2_STAGES;
                    mbar_wait(&full[s], (it / B2_STAGES) & 1);
                    tc_fence_after();
                    const uint32_t st = smem_u32(smem + s * B2_STAGE_BYTES);
                    const uint64_t da = smem_desc(st, 16, 256, LAYOUT_SW32);
                    const uint64_t dal = smem_desc(st + BK_A_BYTES, 16, 256, LAYOUT_SW32);
                    const uint32_t wh = st + 2 * BK_A_BYTES, wl = wh + B2_WH_BYTES;
                    const uint32_t acc = k > 0 ? 1u : 0u;
                    {
                        const uint64_t dw = smem_desc(wh, 1024, 512, LAYOUT_SW128_32B);
                        umma_tf32_2cta(tmem, da, dw, id0, acc);
                        if (need_lo) umma_tf32_2cta(tmem, dal, dw, id0, 1u);
                        if (need_wlo) umma_tf32_2cta(tmem, da, smem_desc(wl, 1024, 512, LAYOUT_SW128_32B), id0, 1u);
                    }
                    if (h1) {
                        const uint64_t dw = smem_desc(wh + h0 * 1024, 1024, 512, LAYOUT_SW128_32B);
                        umma_tf32_2cta(tmem + n0, da, dw, id1, acc);
                        if (need_lo) umma_tf32_2cta(tmem + n0, dal, dw, id1, 1u);
                        if (need_wlo)
                            umma_tf32_2cta(tmem + n0, da, smem_desc(wl + h0 * 1024, 1024, 512, LAYOUT_SW128_32B), id1, 1u);
                    }
                    umma_commit_2cta_mc(&empty[s], (uint16_t)3);
                }
                umma_commit_2cta_mc(acc_full, (uint16_t)3);
            }
        }
    } else {
        const int quarter = warp % 4;
        const int er = quarter * 32 + lane;         // accumulator row of this thread
        int nu = 0, slot = 0;
        for (int u = cl; u < total; u += ncl, ++nu) {
            const int nt = u % q.ntile_n, rt = 2 * ((u / q.ntile_n) % nrp) + crank, dom = u / (q.ntile_n * nrp);
            const int row0 = dom * q.ngrid + rt * 128;
            const bool live = rt < nrt;
            mbar_wait(acc_full, nu & 1);
            tc_fence_after();
            const ColTile ct = col_tile(q.cs, nt);
            for (int cb = 0; cb < ct.width / 32; ++cb) {
                uint32_t v[32];
                tmem_ld32(tmem + ((uint32_t)(quarter * 32) << 16) + cb * 32, v);
                tmem_ld_wait();
                const int c0 = ct.start + cb * 32;
                if (live) epi_tile_out<2>(stage, slot, &map_out, c0, row0, v, er, true);
            }
            tc_fence_before();
            named_bar_sync(EPI_BAR, 128);
            if (er == 0) mbar_arrive_remote(acc_empty, 0);   // this CTA's half of the accumulator is drained
        }
        if (er == 0) bulk_wait<0>();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 1) {
        __syncwarp();
        tmem_dealloc_2cta(tmem, 512);
    }
}

// =================================================================================================
// Opt-in low-precision back-application on CTA pairs: Y[r][c] += sum_p A16[r][p] * W16[p][c], BF16 x BF16 -> FP32
// (tcgen05.mma.kind::f16).  beta is read as its stored BF16 copy (K-major [128 rows x 64 p] slabs, 128-byte swizzle,
// four K = 16 steps per slab), W as the BF16 array the glue kernel wrote (MN-major 32-column chunks, 64-byte
// swizzle).  With a sixth of the MMA work of 3xTF32 the kernel is bound by its HBM traffic (beta 2 bytes per element,
// Y read-modify-write) and by the epilogue, which is the one of back2_tc_kernel.
// =================================================================================================
constexpr int BH_KB = 64;                               // projector rows per stage
constexpr int BH_A_BYTES = 128 * 128;                   // [128 rows x 64 BF16]
constexpr int BH_W_BYTES = 7 * BH_KB * 64;              // this CTA's half of the W slab: <= 224 columns
constexpr int BH_STAGE_BYTES = BH_A_BYTES + BH_W_BYTES; // 44 KB
constexpr int BH_STAGES = 4;
constexpr int BH_SMEM = BH_STAGES * BH_STAGE_BYTES + 2 * EPI_TILE_BYTES + 1024 + 512;

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(BK_THREADS, 1)
back2h_tc_kernel(const __grid_constant__ CUtensorMap map_a16, const __grid_constant__ CUtensorMap map_w0,
                 const __grid_constant__ CUtensorMap map_w1, const __grid_constant__ CUtensorMap map_n0,
                 const __grid_constant__ CUtensorMap map_n1, const __grid_constant__ CUtensorMap map_out, const BackParams q) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t *stage = smem + BH_STAGES * BH_STAGE_BYTES;
    uint64_t *bars = (uint64_t *)(stage + 2 * EPI_TILE_BYTES);
    uint64_t *full = bars, *empty = bars + BH_STAGES;
    uint64_t *acc_full = bars + 2 * BH_STAGES, *acc_empty = acc_full + 1;
    uint32_t *tmem_slot = (uint32_t *)(acc_empty + 1);
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int crank = (int)cluster_ctarank();
    const bool leader = crank == 0;

    if (threadIdx.x == 0) {
        for (int s = 0; s < BH_STAGES; ++s) {
            mbar_init(&full[s], 1);     // used in the leader: its own expect_tx arrive; both CTAs' TMA bytes land on it
            mbar_init(&empty[s], 1);    // the leader's tcgen05.commit, multicast to both CTAs
        }
        mbar_init(acc_full, 1);
        mbar_init(acc_empty, 2);
        fence_barrier_init();
        prefetch_tmap(&map_a16);
        prefetch_tmap(&map_w0);
        prefetch_tmap(&map_w1);
        prefetch_tmap(&map_out);
    }
    if (warp == 1) tmem_alloc_2cta(tmem_slot, 512);
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    const int nrt = q.ngrid / 128, nrp = (nrt + 1) / 2;
    const int total = q.ndom * nrp * q.ntile_n;
    const int ncl = gridDim.x / 2, cl = blockIdx.x / 2;
    const int nk = (q.P + BH_KB - 1) / BH_KB;      // columns of beta16 / rows of W16 past P are zero (out-of-bounds fill / memset)

    if (warp == 0) {
        if (lane == 0) {
            int it = 0;
            for (int u = cl; u < total; u += ncl) {
                const int nt = u % q.ntile_n, rt = 2 * ((u / q.ntile_n) % nrp) + crank, dom = u / (q.ntile_n * nrp);
                const int row = dom * q.ngrid + rt * 128;
                const ColTile ct = col_tile(q.cs, nt);
                const int h0 = ct.h0, h1 = ct.h1;
                const int ch0 = ct.start / 32 + crank * h0, ch1 = ct.start / 32 + ct.n0 / 32 + crank * h1;
                const bool narrow = nt >= q.cs.wt;
                const CUtensorMap *m0 = narrow ? &map_n0 : &map_w0, *m1 = narrow ? &map_n1 : &map_w1;
                const uint32_t cta_bytes = BH_A_BYTES + (uint32_t)(h0 + h1) * BH_KB * 64;
                for (int k = 0; k < nk; ++k, ++it) {
                    const int s = it % BH_STAGES;
                    mbar_wait(&empty[s], ((it / BH_STAGES) & 1) ^ 1);
                    uint8_t *st = smem + s * BH_STAGE_BYTES;
                    if (leader) mbar_expect_tx(&full[s], 2 * cta_bytes);
                    const int wrow = dom * q.prows + k * BH_KB;
                    tma_load_2d_2cta(st, &map_a16, &full[s], k * BH_KB, row);
                    tma_load_3d_2cta(st + BH_A_BYTES, m0, &full[s], 0, wrow, ch0);
                    if (h1) tma_load_3d_2cta(st + BH_A_BYTES + h0 * (BH_KB * 64), m1, &full[s], 0, wrow, ch1);
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0 && leader) {
            int it = 0, nu = 0;
            for (int u = cl; u < total; u += ncl, ++nu) {
                const ColTile ct = col_tile(q.cs, u % q.ntile_n);
                const uint32_t id0 = instr_desc(FMT_BF16, 0, 1, 256, (uint32_t)ct.n0);
                const uint32_t id1 = instr_desc(FMT_BF16, 0, 1, 256, (uint32_t)(ct.n1 ? ct.n1 : 64));
                mbar_wait(acc_empty, (nu & 1) ^ 1);
                tc_fence_after();
                for (int k = 0; k < nk; ++k, ++it) {
                    const int s = it % BH_STAGES;
                    mbar_wait(&full[s], (it / BH_STAGES) & 1);
                    tc_fence_after();
                    const uint32_t st = smem_u32(smem + s * BH_STAGE_BYTES);
                    const uint32_t wb = st + BH_A_BYTES;
#pragma unroll
                    for (int k16 = 0; k16 < BH_KB / 16; ++k16) {
                        const uint32_t acc = (k > 0 || k16 > 0) ? 1u : 0u;
                        // A: K-major, 128-byte rows, 8-row atoms of 1024 B; a K = 16 step is 32 B further along the row
                        const uint64_t da = smem_desc(st + k16 * 32, 16, 1024, LAYOUT_SW128);
                        // W: MN-major chunks of [64 rows x 64 B] (chunk stride 4096), 8-row groups of 512 B; 16 rows per step
                        const uint64_t dw0 = smem_desc(wb + k16 * 1024, BH_KB * 64, 512, LAYOUT_SW64);
                        umma_f16_2cta(tmem, da, dw0, id0, acc);
                        if (ct.h1) {
                            const uint64_t dw1 = smem_desc(wb + ct.h0 * (BH_KB * 64) + k16 * 1024, BH_KB * 64, 512, LAYOUT_SW64);
                            umma_f16_2cta(tmem + ct.n0, da, dw1, id1, acc);
                        }
                    }
                    umma_commit_2cta_mc(&empty[s], (uint16_t)3);
                }
                umma_commit_2cta_mc(acc_full, (uint16_t)3);
            }
        }
    } else {
        const int quarter = warp % 4;
        const int er = quarter * 32 + lane;
        int nu = 0, slot = 0;
        for (int u = cl; u < total; u += ncl, ++nu) {
            const int nt = u % q.ntile_n, rt = 2 * ((u / q.ntile_n) % nrp) + crank, dom = u / (q.ntile_n * nrp);
            const int row0 = dom * q.ngrid + rt * 128;
            const bool live = rt < nrt;
            const ColTile ct = col_tile(q.cs, nt);
            mbar_wait(acc_full, nu & 1);
            tc_fence_after();
            for (int cb = 0; cb < ct.width / 32; ++cb) {
                uint32_t v[32];
                tmem_ld32(tmem + ((uint32_t)(quarter * 32) << 16) + cb * 32, v);
                tmem_ld_wait();
                if (live) epi_tile_out<2>(stage, slot, &map_out, ct.start + cb * 32, row0, v, er, true);
            }
            tc_fence_before();
            named_bar_sync(EPI_BAR, 128);
            if (er == 0) mbar_arrive_remote(acc_empty, 0);
        }
        if (er == 0) bulk_wait<0>();
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    if (warp == 1) {
        __syncwarp();
        tmem_dealloc_2cta(tmem, 512);
    }
}

// column tiles of the projection: <= 224 columns each.  (An odd count leaves one CTA of the last cluster
// without a tile; rounding up to an even count of narrower tiles measured slower on configs[4].)
int proj_ntile_n(int N) { return (N + PJ_MAXBN - 1) / PJ_MAXBN; }

int g_num_sms = 0;
int num_sms() {
    if (!g_num_sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev);
        if (g_num_sms <= 0) g_num_sms = 148;
    }
    return g_num_sms;
}

}  // namespace

bool tc_available() { return encode_fn() != nullptr; }

int tc_choose_nsplit(int ndom, long ngrid, int P, int N) {
    const int ntile_m = (P + 255) / 256;
    const int ntile_n = proj_ntile_n(N);
    const long base = (long)ndom * ntile_m * ((ntile_n + 1) / 2);   // cluster units per K slice
    const int sms = 74;                                               // clusters of two CTAs
    const long nkb = ngrid / PJ_BK;
    int best = 1;
    double best_eff = 0.0;
    for (int ns = 1; ns <= kMaxSplit && ns <= nkb / 8; ++ns) {
        const long units = base * ns;
        const double eff = (double)units / (double)(((units + sms - 1) / sms) * sms);
        if (eff > best_eff + 1e-9) {
            best_eff = eff;
            best = ns;
        }
        if (eff >= 0.97) return ns;
    }
    return best;
}

bool proj_tc_can_fuse_density(int P, int N, int nprod) {
    // one pair of CTAs sees every psi row exactly once, each CTA half of its columns: two addends per rho element
    // (nprod 0: the BF16 kind::f16 kernel, i.e. only with a BF16 copy of A)
    return (nprod == 3 || nprod == 4 || nprod == 0) && N % 64 == 0 && N <= BK_MAXBN && P <= 256;
}

cudaError_t launch_proj_tc(cudaStream_t st, int ndom, long ngrid, const float *A_hi, const float *A_lo, int lda, int P,
                           const float *Y, int ldy, int N, float *zpart, int prows, int nsplit, int nprod,
                           int chain, int *nlaunch, TmapCache *cache, float *rho, const float *occ, const void *A16) {
    static DeviceOnce attr_set;      // the opt-in shared-memory size is a per-device function attribute
    if (!attr_set.done()) {
        cudaError_t e = cudaFuncSetAttribute(proj_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, PJ_SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(proj_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, PJ_SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(proj2_tc_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, P2_SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(proj2_tc_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, P2_SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(proj2h_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, PH_SMEM);
        if (e != cudaSuccess) return e;
        attr_set.mark();
    }
    ProjParams q;
    q.ndom = ndom;
    q.ngrid = (int)ngrid;
    q.P = P;
    q.N = N;
    q.ntile_m = (P + 255) / 256;
    q.nsplit = nsplit;
    q.prows = prows;
    q.nprod = nprod;
    q.conv_a = (nprod == 3 && A_lo == nullptr) ? 1 : 0;
    q.zpart = zpart;
    q.chain = chain > 0 ? chain : (1 << 30);
    q.lowp = nprod == 0 ? 1 : 0;     // nprod 0 = one product of BF16-rounded operands
    q.rn = nprod == 4 ? 1 : 0;       // nprod 4 = one product, psi rounded to the nearest TF32 in shared memory
    if (q.lowp || q.rn) q.nprod = 1;
    q.rho = nullptr;
    q.occ = occ;
    if (rho) {
        if (!(A_lo == nullptr && proj_tc_can_fuse_density(P, N, nprod)) || ldy != N || (nprod == 0 && !A16)) return cudaErrorInvalidValue;
        cudaError_t e = cudaMemsetAsync(rho, 0, (size_t)ndom * ngrid * sizeof(float), st);
        if (e != cudaSuccess) return e;
        q.rho = rho;
    }
    const uint64_t rows = (uint64_t)ndom * ngrid;
    CUtensorMap mz;
    if (!make_out_map(cache, &mz, zpart, (uint64_t)ndom * nsplit * prows, N, N)) return cudaErrorInvalidValue;
    if (N % 64 == 0 && A_lo == nullptr) {
        // CTA pairs (cta_group::2): one pair per (domain, 256-row tile, column tile of <= 448, K slice)
        q.cs = choose_col_split(N);
        q.ntile_n = q.cs.ntile;
        const ColTile wide = col_tile(q.cs, 0), narrow = col_tile(q.cs, q.ntile_n - 1);
        q.BN = wide.width;
        CUtensorMap ma, my0, my1, my0n, my1n;
        if (!make_chunk_map(cache, &ma, A_hi, rows, lda, (lda + 31) / 32, PJ_BK, 4)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &my0, Y, rows, ldy, N / 32, PJ_BK, wide.h0)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &my1, Y, rows, ldy, N / 32, PJ_BK, wide.h1 ? wide.h1 : 1)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &my0n, Y, rows, ldy, N / 32, PJ_BK, narrow.h0)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &my1n, Y, rows, ldy, N / 32, PJ_BK, narrow.h1 ? narrow.h1 : 1)) return cudaErrorInvalidValue;
        const int total = ndom * q.ntile_m * q.ntile_n * nsplit;
        const int grid = 2 * (total < num_sms() / 2 ? total : num_sms() / 2);
        ++*nlaunch;
        if (q.lowp && A16) {
            // low-precision mode proper: beta from its BF16 copy, kind::f16 MMAs
            CUtensorMap ma16;
            if (!make_chunk16_map(cache, &ma16, A16, rows, lda, (lda + 31) / 32, PJ_BK, 4)) return cudaErrorInvalidValue;
            proj2h_tc_kernel<<<grid, PJ_THREADS, PH_SMEM, st>>>(ma16, my0, my1, my0n, my1n, mz, q);
            return cudaGetLastError();
        }
        if (q.nprod == 3) proj2_tc_kernel<true><<<grid, PJ_THREADS, P2_SMEM, st>>>(ma, my0, my1, my0n, my1n, mz, q);
        else proj2_tc_kernel<false><<<grid, PJ_THREADS, P2_SMEM, st>>>(ma, my0, my1, my0n, my1n, mz, q);
        return cudaGetLastError();
    }
    q.ntile_n = proj_ntile_n(N);
    q.BN = ((N + q.ntile_n - 1) / q.ntile_n + 31) / 32 * 32;
    CUtensorMap ma, mal, my;
    // 4-chunk boxes: each CTA of a cluster fetches (and multicasts) half of the 8 beta chunks of a stage
    if (!make_chunk_map(cache, &ma, A_hi, rows, lda, (lda + 31) / 32, PJ_BK, 4)) return cudaErrorInvalidValue;
    if (!make_chunk_map(cache, &mal, A_lo ? A_lo : A_hi, rows, lda, (lda + 31) / 32, PJ_BK, 4)) return cudaErrorInvalidValue;
    if (!make_chunk_map(cache, &my, Y, rows, ldy, N / 32, PJ_BK, q.BN / 32)) return cudaErrorInvalidValue;
    const int total = ndom * q.ntile_m * ((q.ntile_n + 1) / 2) * nsplit;   // cluster units
    const int grid = 2 * (total < num_sms() / 2 ? total : num_sms() / 2);
    ++*nlaunch;
    if (q.nprod == 3) proj_tc_kernel<true><<<grid, PJ_THREADS, PJ_SMEM, st>>>(ma, mal, my, mz, q);
    else proj_tc_kernel<false><<<grid, PJ_THREADS, PJ_SMEM, st>>>(ma, mal, my, mz, q);
    return cudaGetLastError();
}

cudaError_t launch_back_tc(cudaStream_t st, int ndom, long ngrid, const float *A, const float *A_lo, int lda, int P,
                           const float *W_hi, const float *W_lo, float *Y, int ldy, int N, int prows, int nprod,
                           int *nlaunch, TmapCache *cache, const void *A16, const void *W16) {
    static DeviceOnce attr_set;
    if (!attr_set.done()) {
        cudaError_t e = cudaFuncSetAttribute(back_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, BK_SMEM);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(back2h_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, BH_SMEM);
        if (e != cudaSuccess) return e;
        attr_set.mark();
    }
    BackParams q;
    q.ndom = ndom;
    q.ngrid = (int)ngrid;
    q.P = P;
    q.N = N;
    q.ntile_n = (N + BK_MAXBN - 1) / BK_MAXBN;
    const int per = (N + q.ntile_n - 1) / q.ntile_n;
    q.BN = per <= 256 ? (per + 31) / 32 * 32 : (per + 63) / 64 * 64;
    q.prows = prows;
    q.lowp = nprod == 0 ? 1 : 0;
    q.nprod = nprod == 0 ? 1 : nprod;
    q.ldy = ldy;
    q.Y = Y;
    const uint64_t rows = (uint64_t)ndom * ngrid;
    CUtensorMap ma, mw, mwl;
    if (!make_k8_map(cache, &ma, A, rows, lda, lda, 128)) return cudaErrorInvalidValue;
    CUtensorMap mo;
    if (!make_out_map(cache, &mo, Y, rows, N, ldy)) return cudaErrorInvalidValue;
    const int total = ndom * (int)((ngrid / 128 + 1) / 2) * q.ntile_n;   // cluster units (pairs of row tiles)
    const int grid = 2 * (total < num_sms() / 2 ? total : num_sms() / 2);
    ++*nlaunch;
    if (q.lowp && A16 && W16 && N % 64 == 0) {
        // low-precision mode proper: BF16 copies of beta and W, kind::f16 MMAs on CTA pairs
        q.cs = choose_col_split(N);
        const ColTile wide = col_tile(q.cs, 0), narrow = col_tile(q.cs, q.ntile_n - 1);
        const uint64_t wrows = (uint64_t)ndom * prows;
        CUtensorMap ma16, w0, w1, n0m, n1m;
        if (!make_k64_map(cache, &ma16, A16, rows, lda, lda, 128)) return cudaErrorInvalidValue;
        if (!make_chunk16_map(cache, &w0, W16, wrows, N, N / 32, BH_KB, wide.h0)) return cudaErrorInvalidValue;
        if (!make_chunk16_map(cache, &w1, W16, wrows, N, N / 32, BH_KB, wide.h1 ? wide.h1 : 1)) return cudaErrorInvalidValue;
        if (!make_chunk16_map(cache, &n0m, W16, wrows, N, N / 32, BH_KB, narrow.h0)) return cudaErrorInvalidValue;
        if (!make_chunk16_map(cache, &n1m, W16, wrows, N, N / 32, BH_KB, narrow.h1 ? narrow.h1 : 1)) return cudaErrorInvalidValue;
        back2h_tc_kernel<<<grid, BK_THREADS, BH_SMEM, st>>>(ma16, w0, w1, n0m, n1m, mo, q);
        return cudaGetLastError();
    }
    // CTA pairs for the modes that take beta as (raw, stored remainder): 3xTF32 and the staged mode's two products;
    // one-product modes want beta ROUNDED (an unbiased operand), which the single-CTA kernel forms in shared memory
    if (N % 64 == 0 && !q.lowp && q.nprod >= 2 && A_lo) {
        static DeviceOnce attr2;
        if (!attr2.done()) {
            cudaError_t e = cudaFuncSetAttribute(back2_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, B2_SMEM);
            if (e != cudaSuccess) return e;
            attr2.mark();
        }
        q.cs = choose_col_split(N);
        const ColTile wide = col_tile(q.cs, 0), narrow = col_tile(q.cs, q.ntile_n - 1);
        q.BN = wide.width;
        const uint64_t wrows = (uint64_t)ndom * prows;
        CUtensorMap mal, w0h, w0l, w1h, w1l, n0h, n0l, n1h, n1l;
        if (!make_k8_map(cache, &mal, A_lo, rows, lda, lda, 128)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &w0h, W_hi, wrows, N, N / 32, 8, wide.h0)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &w0l, W_lo, wrows, N, N / 32, 8, wide.h0)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &w1h, W_hi, wrows, N, N / 32, 8, wide.h1 ? wide.h1 : 1)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &w1l, W_lo, wrows, N, N / 32, 8, wide.h1 ? wide.h1 : 1)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &n0h, W_hi, wrows, N, N / 32, 8, narrow.h0)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &n0l, W_lo, wrows, N, N / 32, 8, narrow.h0)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &n1h, W_hi, wrows, N, N / 32, 8, narrow.h1 ? narrow.h1 : 1)) return cudaErrorInvalidValue;
        if (!make_chunk_map(cache, &n1l, W_lo, wrows, N, N / 32, 8, narrow.h1 ? narrow.h1 : 1)) return cudaErrorInvalidValue;
        back2_tc_kernel<<<grid, BK_THREADS, B2_SMEM, st>>>(ma, mal, w0h, w0l, w1h, w1l, n0h, n0l, n1h, n1l, mo, q);
        return cudaGetLastError();
    }
    const int chalf = (q.BN / 32 + 1) / 2;   // each CTA of a cluster fetches (and multicasts) half of the W chunks
    if (!make_chunk_map(cache, &mw, W_hi, (uint64_t)ndom * prows, N, N / 32, 8, chalf)) return cudaErrorInvalidValue;
    if (!make_chunk_map(cache, &mwl, W_lo, (uint64_t)ndom * prows, N, N / 32, 8, chalf)) return cudaErrorInvalidValue;
    back_tc_kernel<<<grid, BK_THREADS, BK_SMEM, st>>>(ma, mw, mwl, mo, q);
    return cudaGetLastError();
}

}  // namespace mlmd
