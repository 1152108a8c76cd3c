// gridff_eval_tma.cu — gridff_eval variant 3: the 4 x 4 x 4-node stencil of PAPER.md:L136 fetched as ONE 3-D TMA box per point.
//
// The ZFAST store (gridff_internal.cuh) is a dense tensor of 16-byte nodes with extents (nx+3) x (ny+3) x nzp; with its 3-node periodic halo
// every stencil is an axis-aligned box {4 x, 4 y, 4 z} = 16 rows of 64 contiguous bytes = 1 KB.  That is exactly what the tensor memory
// accelerator moves: one `cp.async.bulk.tensor.3d` (SASS UTMALDG) per point lands the box in shared memory and signals an mbarrier, without
// occupying the LSU / L1 data pipe that bounds the warp-cooperative LDG gather (k_eval_coop: one L1 cycle per distinct 128-byte line, 22 per
// stencil).  The tensor is described to the TMA unit as fp32 elements {nzp * 4, ny + 3, nx + 3} (z and channel merged: TMA has no
// 16-byte element type), box {16, 4, 4}, no swizzle, 64-byte L2 promotion.  The 8-copy micro-brick store (gridff_derive.cu) is a 5-D tensor
// {32 floats = a brick, nbz, nby, nbx, 8 copies}; a stencil is the box {32, 2, 2, 2, 1} in the copy of its corner's parity: 8 whole 128-byte lines
// (UTMALDG.5D) — the template parameter BRICKS.
//
// A warp owns 32 consecutive points and walks over its tiles persistently.  Per tile the boxes arrive in 4 groups of 8 points that alternate
// between two raw buffers of 8 KB with their own mbarriers; the warp folds each group with the points' channel factors into the same XOR-swizzled
// 8 KB tile that k_eval_coop builds (lanes read consecutive 16-byte chunks of the raw box: conflict-free), re-arms the buffer with the group
// after next (of this tile or of the warp's next one), and finally every lane contracts its own point (interp_tile).  The folded tile and the
// contraction are bit-identical to k_eval_coop's, so variant 3 returns exactly variant 2's numbers (test).  24.6 KB per warp: 8 warps and 128 KB
// in flight per SM behind the arithmetic (16-point groups, 41 KB and 5 warps: 10 % slower on the HBM-bound brick store, profiles/r2_hbm.md).
#include "gridff_interp.cuh"
#include <cuda.h>
#include <stdio.h>
#include <string.h>

using namespace gridff;

namespace {

constexpr int kTmaWarps = 1;                       // warps per block: a warp is self-contained (own buffers, own barriers)
constexpr int kGroupPts = 8;                       // points whose boxes share a raw buffer and an mbarrier: a tile of 32 points arrives in 32 / kGroupPts groups,
constexpr int kGroups = 32 / kGroupPts;            // alternating between two buffers (kGroups even).  8 points: 24.6 KB per warp, 8 warps per SM (16: 41 KB, 5 warps)
constexpr int kRawHalf = kGroupPts * 1024;         // one raw buffer
constexpr size_t kWarpSmem = 2 * kRawHalf + 32 * 64 * 4 + 32 * 16 + 32 * 4 + 2 * 8;      // raw A, raw B, folded tile, cf, base, 2 mbarriers

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one {16 floats, 4, 4} box: fastest coordinate first (z * 4 + channel, y, x), in elements
__device__ __forceinline__ void tma_box(void* dst, const CUtensorMap* map, int c0, int c1, int c2, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
// 8-copy micro-brick store: one {32 floats = a brick, 2, 2, 2, 1} box: (0, brick z, brick y, brick x, copy) — 8 whole 128-byte lines
__device__ __forceinline__ void tma_box5(void* dst, const CUtensorMap* map, int bz, int by, int bx, int copy, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(0), "r"(bz), "r"(by), "r"(bx), "r"(copy) : "memory");
}

// base: the stencil's corner in the z-fastest store (BRICKS: the packed corner for gather_bricks); kNoStencil = above the domain
struct Pt { unsigned base; float tx, ty, tz; int c0, c1, c2, c3; float4 cf; };

template <bool BRICKS>
__device__ __forceinline__ Pt load_point(const GridGeom& g, long long p, long long n, const float* __restrict__ pos, const float4* __restrict__ coef) {
    Pt q; q.base = kNoStencil; q.tx = q.ty = q.tz = 0.f; q.c0 = q.c1 = q.c2 = q.c3 = 0; q.cf = make_float4(0.f, 0.f, 0.f, 0.f);
    if (p < n) {
        int ix, iy, iz;
        cell_periodic(pos[3 * p], g.inv_hx_hi, g.inv_hx_lo, g.fnx, g.inv_nx, ix, q.tx);
        cell_periodic(pos[3 * p + 1], g.inv_hy_hi, g.inv_hy_lo, g.fny, g.inv_ny, iy, q.ty);
        if (cell_z(pos[3 * p + 2], g, iz, q.tz)) {
            if (BRICKS) {
                // corner (ix, iy, iz - 1) in stored indices; the copy with the corner's parity holds it brick-aligned: brick (X + (X & 1)) >> 1
                const int Z0 = iz - 1;
                q.base = pack_corner(ix, iy, Z0);
                q.c0 = (Z0 + (Z0 & 1)) >> 1; q.c1 = (iy + (iy & 1)) >> 1; q.c2 = (ix + (ix & 1)) >> 1;
                q.c3 = ((ix & 1) << 2) | ((iy & 1) << 1) | (Z0 & 1);
            } else {
                q.base = (unsigned)corner_zfast(g, ix, iy, iz);        // same validity flag and offsets as the LDG kernels
                q.c0 = 4 * (iz - 1); q.c1 = iy; q.c2 = ix;             // stored index s holds node s - 1: the stencil corner (ix-1, iy-1) is stored at (ix, iy)
            }
        } else q.tz = 0.f;
        q.cf = coef[p];
    }
    return q;
}

template <bool BRICKS>
__global__ void __launch_bounds__(kTmaWarps * 32) k_eval_tma(const __grid_constant__ CUtensorMap tmap, GridGeom g, long long n, const float* __restrict__ pos,
                                                             const float4* __restrict__ coef, float* __restrict__ E, float* __restrict__ F,
                                                             const unsigned* __restrict__ choice) {
    if (choice && *choice != kChoiceTma) return;          // gridff_eval's device-side choice (k_eval_classify) went to the LDG kernel
    extern __shared__ __align__(16) unsigned char smem[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned char* base = smem + ((128u - (smem_u32(smem) & 127u)) & 127u) + (size_t)w * ((kWarpSmem + 1023) & ~(size_t)1023);    // TMA destinations: 128-byte aligned
    float4* raw[2] = {reinterpret_cast<float4*>(base), reinterpret_cast<float4*>(base + kRawHalf)};
    float* tile = reinterpret_cast<float*>(base + 2 * kRawHalf);
    float4* s_cf = reinterpret_cast<float4*>(tile + 32 * 64);
    unsigned* s_base = reinterpret_cast<unsigned*>(s_cf + 32);
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(s_base + 32);
    if (lane == 0) { mbar_init(bar, 1); mbar_init(bar + 1, 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    warp_sync();

    const long long n_tiles = (n + 31) / 32, stride = (long long)gridDim.x * kTmaWarps;
    long long t = (long long)blockIdx.x * kTmaWarps + w;
    const int my_group = lane / kGroupPts;
    // arm buffer (grp & 1) with the boxes of group `grp` of the points `q` (the lanes of that group own them)
    auto issue = [&](const Pt& q, int grp) {
        const int hb = grp & 1;
        const unsigned valid = __ballot_sync(0xFFFFFFFFu, q.base != kNoStencil);
        const unsigned mine = (valid >> (kGroupPts * grp)) & ((1u << kGroupPts) - 1u);
        if (lane == 0) mbar_expect_tx(bar + hb, 1024u * (unsigned)__popc(mine));
        warp_sync();
        if (my_group == grp && q.base != kNoStencil) {
            if (BRICKS) tma_box5(reinterpret_cast<unsigned char*>(raw[hb]) + (lane & (kGroupPts - 1)) * 1024, &tmap, q.c0, q.c1, q.c2, q.c3, bar + hb);
            else tma_box(reinterpret_cast<unsigned char*>(raw[hb]) + (lane & (kGroupPts - 1)) * 1024, &tmap, q.c0, q.c1, q.c2, bar + hb);
        }
    };
    // raw box -> tile element: z-fastest rows land in tile order (node lane = 4 row + k); a brick box lands as [bx][by][bz][dx dy dz]: float4 lane of
    // the first half is node a = dx, b = 2 by + dy, k = 2 bz + dz (the second half: a + 2)
    const int e0 = BRICKS ? (((lane >> 2) & 1) << 4) | (((((lane >> 4) & 1) << 1) | ((lane >> 1) & 1)) << 2) | ((((lane >> 3) & 1) << 1) | (lane & 1)) : lane;
    // A tile whose points share stencil lines (spatially sorted input: warp_points_are_local) is gathered through the L1 instead, as k_eval_coop
    // does: L1 / L2 hits are worth more than the TMA's independence from the LSU.  Its buffers are simply not armed.
    auto is_clustered = [&](const Pt& q) {
        if (BRICKS) return warp_points_are_local((int)(q.base & 2047u), (int)((q.base >> kCornerBits) & 2047u), (int)(q.base >> (2 * kCornerBits)), q.base != kNoStencil, lane);
        return warp_points_are_local(q.c2, q.c1, q.c0 >> 2, q.base != kNoStencil, lane);
    };
    Pt cur = load_point<BRICKS>(g, t * 32 + lane, n, pos, coef);
    bool cur_cl = is_clustered(cur);
    if (t < n_tiles && !cur_cl) { issue(cur, 0); issue(cur, 1); }
    unsigned parity[2] = {0u, 0u};
    for (; t < n_tiles; t += stride) {
        const long long tn = t + stride;
        Pt nxt = load_point<BRICKS>(g, tn < n_tiles ? tn * 32 + lane : n, n, pos, coef);       // p = n: an empty point
        const bool nxt_cl = is_clustered(nxt);
        s_cf[lane] = cur.cf; s_base[lane] = cur.base;
        warp_sync();
        if (cur_cl) {
#pragma unroll 8
            for (int q = 0; q < 32; ++q) {
                const unsigned b = s_base[q];
                if (b != kNoStencil) { if (BRICKS) gather_bricks<false>(g, b, s_cf[q], lane, q, tile); else gather_rows<false>(g, b, s_cf[q], lane, q, tile); }
            }
            if (tn < n_tiles && !nxt_cl) { issue(nxt, 0); issue(nxt, 1); }
        } else {
#pragma unroll
            for (int grp = 0; grp < kGroups; ++grp) {
                const int hb = grp & 1;
                mbar_wait(bar + hb, parity[hb]);
                parity[hb] ^= 1u;
                stress_delay();
                const float4* r4 = raw[hb];
#pragma unroll 4
                for (int q = 0; q < kGroupPts; ++q) {
                    if (s_base[kGroupPts * grp + q] != kNoStencil)
                        store_rows(s_cf[kGroupPts * grp + q], r4[q * 64 + lane], r4[q * 64 + 32 + lane], e0, kGroupPts * grp + q, tile);
                }
                warp_sync();                              // every lane has read this buffer: it can take the boxes of the group after next
                if (grp + 2 < kGroups) issue(cur, grp + 2);
                else if (tn < n_tiles && !nxt_cl) issue(nxt, grp + 2 - kGroups);
            }
        }
        warp_sync();
        const long long p = t * 32 + lane;
        if (p < n) {
            Stencil s; s.base = cur.base; s.tx = cur.tx; s.ty = cur.ty; s.tz = cur.tz;
            float e, fx, fy, fz;
            interp_tile(g, s, lane, tile, e, fx, fy, fz);
            if (E) E[p] = e;
            if (F) { F[3 * p] = fx; F[3 * p + 1] = fy; F[3 * p + 2] = fz; }
        }
        warp_sync();                                      // the folded tile and s_cf / s_base are rewritten in the next trip
        cur = nxt; cur_cl = nxt_cl;
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

namespace gridff {

// Encode the ZFAST store as a 3-D tensor of fp32 {nzp * 4, sy, sx} with a {16, 4, 4} box (driver entry point looked up at run time: the
// library does not link libcuda).  Returns 0 and fills grid->tmap on success.
int make_tensor_map(gridff_grid* grid) {
    grid->tmap_ok = 0;
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr; cudaDriverEntryPointQueryResult qr;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
        if (e != cudaSuccess || !fn || qr != cudaDriverEntryPointSuccess) { cudaGetLastError(); set_error("cuTensorMapEncodeTiled is not available in this driver"); return GRIDFF_EUNSUPPORTED; }
        encode = (EncodeTiledFn)fn;
    }
    const GridGeom& G = grid->geom;
    static_assert(sizeof(CUtensorMap) <= sizeof(grid->tmap), "tensor map storage");
    if (G.n_copies == 8) {
        // 8-copy micro-brick store: fp32 {32 (a brick), nbz, nby, nbx, 8 copies}, box {32, 2, 2, 2, 1} = the 8 bricks of a stencil in its aligned copy
        const cuuint64_t dims[5] = {32, (cuuint64_t)G.nbz, (cuuint64_t)G.nby, (cuuint64_t)G.nbx, 8};
        const cuuint64_t strides[4] = {128, (cuuint64_t)G.nbz * 128, (cuuint64_t)G.nby * G.nbz * 128, (cuuint64_t)G.copy_stride * 16};
        const cuuint32_t box[5] = {32, 2, 2, 2, 1}, estr[5] = {1, 1, 1, 1, 1};
        CUtensorMap m;
        CUresult r = encode(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, (void*)G.store, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled (bricks) failed (%d)", (int)r); return GRIDFF_ECUDA; }
        memcpy(grid->tmap, &m, sizeof(m));
        grid->tmap_ok = 1;
        return GRIDFF_OK;
    }
    const cuuint64_t dims[3] = {(cuuint64_t)G.nzp * 4, (cuuint64_t)G.sy, (cuuint64_t)G.sx};
    const cuuint64_t strides[2] = {(cuuint64_t)G.nzp * 16, (cuuint64_t)G.sy * G.nzp * 16};         // bytes, dims 1 and 2
    const cuuint32_t box[3] = {16, 4, 4}, estr[3] = {1, 1, 1};
    CUtensorMap m;
    // L2 promotion: measured on the 1.09 GB store, random points: NONE 2.20e9, 64 B 2.30e9, 128 B 2.20e9, 256 B 1.96e9 evals/s (every setting
    // moves whole 128-byte lines from DRAM: 2.6 KB per point, profiles/r2_hbm.md)
    const CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
    CUresult r = encode(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)G.store, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed (%d)", (int)r); return GRIDFF_ECUDA; }
    memcpy(grid->tmap, &m, sizeof(m));
    grid->tmap_ok = 1;
    return GRIDFF_OK;
}

int eval_tma(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F, const unsigned* d_choice, cudaStream_t st) {
    if (!grid->tmap_ok) { set_error("this grid has no tensor map (TMA needs the z-fastest fp32 store)"); return GRIDFF_EUNSUPPORTED; }
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const size_t smem = kTmaWarps * ((kWarpSmem + 1023) & ~(size_t)1023) + 128;
    const bool bricks = grid->geom.n_copies == 8;
    auto kern = bricks ? k_eval_tma<true> : k_eval_tma<false>;
    static bool attr_set[64][2] = {};                     // per device: function attributes belong to the device that is current when they are set
    if (dev < 0 || dev >= 64 || !attr_set[dev][bricks]) {
        GRIDFF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        GRIDFF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        if (dev >= 0 && dev < 64) attr_set[dev][bricks] = true;
    }
    int per_sm = 1;
    GRIDFF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kTmaWarps * 32, smem));
    if (per_sm < 1) per_sm = 1;
    const long long n_tiles = (n + 31) / 32;
    long long blocks = (long long)sms * per_sm;
    if (blocks * kTmaWarps > n_tiles) blocks = (n_tiles + kTmaWarps - 1) / kTmaWarps;
    CUtensorMap m;
    memcpy(&m, grid->tmap, sizeof(m));
    cudaError_t e = launch_with_window(grid, kern, dim3((unsigned)blocks), dim3(kTmaWarps * 32), smem, st, m, grid->geom, n, d_pos, (const float4*)d_coef, d_E, d_F, d_choice);
    count_launch();
    if (e != cudaSuccess) return cuda_fail(e, "gridff_eval (TMA) launch");
    return GRIDFF_OK;
}

}  // namespace gridff
