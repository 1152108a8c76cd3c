// gridff_eval.cu — gridff_eval (step a5) and the bandwidth probe.  PAPER.md:L128-138; DESIGN.md §5.
#include "gridff_interp.cuh"
#include <stdio.h>
#include <atomic>

using namespace gridff;

namespace {

// variant 1: one thread per point, 64 independent 16-byte loads (the paper's per-atom loop moved to a thread)
__global__ void __launch_bounds__(128) k_eval_direct(GridGeom g, long long n, const float* __restrict__ pos, const float4* __restrict__ coef,
                                                     float* __restrict__ E, float* __restrict__ F) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const Stencil s = locate(g, pos[3 * p], pos[3 * p + 1], pos[3 * p + 2]);
    float e, fx, fy, fz;
    interp_direct(g, s, coef[p], e, fx, fy, fz);
    if (E) E[p] = e;
    if (F) { F[3 * p] = fx; F[3 * p + 1] = fy; F[3 * p + 2] = fz; }
}

// variant 2: warp-cooperative row gather.  A warp owns 32 consecutive points; for each of them 4 lanes fetch each 64-byte
// stencil row (8 rows per LDG.128), fold the channels and park the 64 scalars in shared memory; then every lane contracts
// its own point from the (swizzled) tile.
constexpr int kEvalWarps = 4;

// `choice` (may be NULL): device word written by k_eval_classify; the kernel runs only when it holds kChoiceCoop
// `rec` (may be NULL; gridff_eval_binned): the points as 32-byte records {x, y, z, index}, {coef} in bin order; the results then go, as
// float4 {E, Fx, Fy, Fz} per slot, to `out4` (k_bin_gather_out hands them to the points' own indices)
__global__ void __launch_bounds__(kEvalWarps * 32) k_eval_coop(GridGeom g, long long n, const float* __restrict__ pos, const float4* __restrict__ coef,
                                                               float* __restrict__ E, float* __restrict__ F, const unsigned* __restrict__ choice,
                                                               const float4* __restrict__ rec, float4* __restrict__ out4) {
    if (choice && *choice != kChoiceCoop) return;
    __shared__ __align__(16) float s_tile[kEvalWarps][32 * 64];
    __shared__ __align__(16) float4 s_cf[kEvalWarps][32];
    __shared__ unsigned s_base[kEvalWarps][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const long long p = ((long long)blockIdx.x * kEvalWarps + w) * 32 + lane;
    Stencil s; s.base = kNoStencil; s.tx = s.ty = s.tz = 0.f;
    float4 cf = make_float4(0.f, 0.f, 0.f, 0.f);
    int ix = 0, iy = 0, iz = 0;
    if (p < n) {
        if (rec) { const float4 a = rec[2 * p]; s = locate(g, a.x, a.y, a.z, ix, iy, iz); cf = rec[2 * p + 1]; }
        else { s = locate(g, pos[3 * p], pos[3 * p + 1], pos[3 * p + 2], ix, iy, iz); cf = coef[p]; }
    }
    s_base[w][lane] = s.base; s_cf[w][lane] = cf;
    warp_sync();
    float* tile = s_tile[w];
    // do this warp's points share stencil lines?  (spatially sorted input)  Then the L1 pays; otherwise gather past it
    const bool clustered = warp_points_are_local(ix, iy, iz, s.base != kNoStencil, lane);
    if (clustered) {
#pragma unroll 8
        for (int q = 0; q < 32; ++q) {
            const unsigned b = s_base[w][q];
            if (b != kNoStencil) gather_rows<false>(g, b, s_cf[w][q], lane, q, tile);
        }
    } else {
#pragma unroll 8
        for (int q = 0; q < 32; ++q) {
            const unsigned b = s_base[w][q];
            if (b != kNoStencil) gather_rows<true>(g, b, s_cf[w][q], lane, q, tile);
        }
    }
    warp_sync();
    if (p >= n) return;
    float e, fx, fy, fz;
    interp_tile(g, s, lane, tile, e, fx, fy, fz);
    if (out4) { out4[p] = make_float4(e, fx, fy, fz); return; }
    if (E) E[p] = e;
    if (F) { F[3 * p] = fx; F[3 * p + 1] = fy; F[3 * p + 2] = fz; }
}

// ---- gridff_eval_binned: a counting sort of the points by coarse cell block, so that scattered points are gathered with the locality of sorted ones ----
// Bins are blocks of 4 x 4 x 8 cells in [x][y][z] order (z fastest, like the store); points above the domain go to one extra bin at the end.
constexpr int kBinX = 2, kBinY = 2, kBinZ = 3;            // log2 of the block's cells per axis
__device__ __forceinline__ unsigned bin_of(const GridGeom& g, const float* __restrict__ pos, long long p, int nby, int nbz, unsigned n_bins) {
    int ix, iy, iz;
    const Stencil s = locate(g, pos[3 * p], pos[3 * p + 1], pos[3 * p + 2], ix, iy, iz);
    if (s.base == kNoStencil) return n_bins - 1;
    return (unsigned)(((ix >> kBinX) * nby + (iy >> kBinY)) * nbz + (iz >> kBinZ));
}
// pass 1: count[bin]++, the value before the increment is the point's rank within its bin
__global__ void __launch_bounds__(256) k_bin_count(GridGeom g, long long n, const float* __restrict__ pos, int nby, int nbz, unsigned n_bins,
                                                   unsigned* __restrict__ count, unsigned* __restrict__ rank) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    rank[p] = atomicAdd(count + bin_of(g, pos, p, nby, nbz, n_bins), 1u);
}
// pass 2: exclusive scan of the counts in place: one block walks over tiles of 1024 counts (coalesced), scanning each with warp shuffles
__global__ void __launch_bounds__(1024) k_bin_scan(unsigned n_bins, unsigned* __restrict__ count) {
    __shared__ unsigned s_warp[32];
    __shared__ unsigned s_run;
    const unsigned lane = threadIdx.x & 31u, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_run = 0u;
    __syncthreads();
    unsigned next = threadIdx.x < n_bins ? count[threadIdx.x] : 0u;
    for (unsigned t0 = 0; t0 < n_bins; t0 += 1024u) {
        const unsigned b = t0 + threadIdx.x;
        const unsigned c = next;
        next = b + 1024u < n_bins ? count[b + 1024u] : 0u;     // the next tile's counts are on their way while this one is scanned
        unsigned inc = c;
#pragma unroll
        for (unsigned o = 1; o < 32u; o <<= 1) { const unsigned v = __shfl_up_sync(0xFFFFFFFFu, inc, o); if (lane >= o) inc += v; }
        if (lane == 31u) s_warp[w] = inc;
        __syncthreads();
        unsigned wsum = s_warp[lane];                          // every warp scans the 32 warp totals
#pragma unroll
        for (unsigned o = 1; o < 32u; o <<= 1) { const unsigned v = __shfl_up_sync(0xFFFFFFFFu, wsum, o); if (lane >= o) wsum += v; }
        const unsigned before = __shfl_sync(0xFFFFFFFFu, wsum, w) - s_warp[w], total = __shfl_sync(0xFFFFFFFFu, wsum, 31);
        const unsigned run = s_run;
        if (b < n_bins) count[b] = run + before + inc - c;
        __syncthreads();                                       // s_warp and s_run have been read
        if (threadIdx.x == 0) s_run = run + total;
        __syncthreads();
    }
}
// pass 3: slot = offset[bin] + rank; the point's 32-byte record {x, y, z, index}, {coef} goes to rec[slot] (one whole sector), slot to rank[p]
__global__ void __launch_bounds__(256) k_bin_scatter(GridGeom g, long long n, const float* __restrict__ pos, const float4* __restrict__ coef, int nby, int nbz,
                                                     unsigned n_bins, const unsigned* __restrict__ offset, unsigned* __restrict__ rank, float4* __restrict__ rec) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const unsigned slot = offset[bin_of(g, pos, p, nby, nbz, n_bins)] + rank[p];
    rank[p] = slot;
    rec[2 * (size_t)slot] = make_float4(pos[3 * p], pos[3 * p + 1], pos[3 * p + 2], __uint_as_float((unsigned)p));
    rec[2 * (size_t)slot + 1] = coef[p];
}
// pass 5: the results back to the points' own indices (random 16-byte reads, coalesced writes)
__global__ void __launch_bounds__(256) k_bin_gather_out(long long n, const unsigned* __restrict__ slot, const float4* __restrict__ out4,
                                                        float* __restrict__ E, float* __restrict__ F) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const float4 o = __ldcg(out4 + slot[p]);
    if (E) E[p] = o.x;
    if (F) { F[3 * p] = o.y; F[3 * p + 1] = o.z; F[3 * p + 2] = o.w; }
}

// Which kernel for a store that does not fit the L2?  Scattered points: the TMA box kernel (DRAM-bound, it keeps more bytes in flight: +26 %);
// spatially sorted points: the LDG gather at full occupancy (L2 hits: 2.3x).  The order of the caller's points is not known at launch, so a
// one-block kernel samples 64 warp tiles spread over the array, applies warp_points_are_local and leaves the choice in a device word that both
// kernels read first; the one not chosen exits at once.  No host round-trip.
__global__ void __launch_bounds__(256) k_eval_classify(GridGeom g, long long n, const float* __restrict__ pos, unsigned* __restrict__ choice) {
    __shared__ int s_local[8];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const long long n_tiles = (n + 31) / 32;
    int local = 0;
    for (int k = 0; k < 8; ++k) {
        const long long t = (long long)((double)(8 * w + k) * (double)n_tiles / 64.0);
        const long long p = t * 32 + lane;
        int ix = 0, iy = 0, iz = 0; bool valid = false;
        if (p < n) valid = locate(g, pos[3 * p], pos[3 * p + 1], pos[3 * p + 2], ix, iy, iz).base != kNoStencil;
        local += warp_points_are_local(ix, iy, iz, valid, lane) ? 1 : 0;
    }
    if (lane == 0) s_local[w] = local;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
        for (int k = 0; k < 8; ++k) tot += s_local[k];
        *choice = tot >= 32 ? kChoiceCoop : kChoiceTma;
    }
}

__device__ unsigned g_eval_choice[64];        // one word per launch in flight (round robin): concurrent streams do not share a word

// brick layout, thread per point (layout study)
__device__ __forceinline__ size_t brick_index(const GridGeom& g, int s_x, int s_y, int iz) {
    const int by_n = (g.sy + 3) >> 2, bz_n = g.nzp >> 2;
    const size_t brick = ((size_t)(s_x >> 2) * by_n + (s_y >> 2)) * bz_n + (iz >> 2);
    return brick * 64 + (size_t)(((s_x & 3) << 4) | ((s_y & 3) << 2) | (iz & 3));
}

__global__ void __launch_bounds__(128) k_eval_brick(GridGeom g, long long n, const float* __restrict__ pos, const float4* __restrict__ coef,
                                                    float* __restrict__ E, float* __restrict__ F) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    int ix, iy, iz; float tx, ty, tz;
    cell_periodic(pos[3 * p], g.inv_hx_hi, g.inv_hx_lo, g.fnx, g.inv_nx, ix, tx);
    cell_periodic(pos[3 * p + 1], g.inv_hy_hi, g.inv_hy_lo, g.fny, g.inv_ny, iy, ty);
    float e = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
    if (cell_z(pos[3 * p + 2], g, iz, tz)) {
        const float4 cf = coef[p];
        Contract C; C.init(tx, ty, tz);
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                float c[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) c[k] = fold4(cf, __ldg(g.store + brick_index(g, ix + a, iy + b, iz - 1 + k)));
                C.row(a, b, c[0], c[1], c[2], c[3]);
            }
        e = C.e; fx = -C.gx * g.inv_hx; fy = -C.gy * g.inv_hy; fz = -C.gz * g.inv_hz;
    }
    if (E) E[p] = e;
    if (F) { F[3 * p] = fx; F[3 * p + 1] = fy; F[3 * p + 2] = fz; }
}

// ---- bandwidth probe ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned hash32(unsigned x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

__global__ void __launch_bounds__(256) k_probe_stream(const float4* __restrict__ buf, size_t n16, int iters, float* sink) {
    float acc = 0.f;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int it = 0; it < iters; ++it) {
        // rotate the block -> data assignment every pass so that no SM finds its previous pass in its own L1
        size_t i = (size_t)((blockIdx.x + (unsigned)it) % gridDim.x) * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < n16; i += 4 * stride) {
            const float4 a = __ldcg(buf + i), b = __ldcg(buf + i + stride), c = __ldcg(buf + i + 2 * stride), d = __ldcg(buf + i + 3 * stride);   // L2 only, no L1
            acc += (a.x + b.y) + (c.z + d.w);
        }
        for (; i < n16; i += stride) acc += __ldcg(buf + i).x;
    }
    if (acc == 1.2345678e-30f) *sink = acc;
}

// LANES = 4: 4 lanes read one 64-byte row at a random 16-byte-aligned offset (the z-fastest stencil's access granule);
// LANES = 8: 8 lanes read one whole, aligned 128-byte line at a random position (the micro-brick stencil's granule)
template <int LANES>
__global__ void __launch_bounds__(256) k_probe_rows(const float4* __restrict__ buf, size_t n16, int iters, float* sink) {
    float acc = 0.f;
    const unsigned quad = (blockIdx.x * blockDim.x + threadIdx.x) / LANES, k = threadIdx.x % LANES;
    const unsigned nquads = (gridDim.x * blockDim.x) / LANES;
    const size_t rows = n16 / LANES;               // rows to read per pass
    const unsigned span = (unsigned)(n16 - LANES);
    for (int it = 0; it < iters; ++it) {
        for (size_t r = quad; r < rows; r += (size_t)nquads * 4) {
            unsigned h = hash32((unsigned)r * 2654435761u + (unsigned)it);
            float4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const size_t rr = r + (size_t)u * nquads;
                if (rr < rows) { const size_t o = (size_t)(h % span); v[u] = __ldcg(buf + (LANES == 8 ? (o & ~(size_t)7) : o) + k); } else v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                h = hash32(h + 0x9e3779b9u);
            }
            acc += (v[0].x + v[1].y) + (v[2].z + v[3].w);
        }
    }
    if (acc == 1.2345678e-30f) *sink = acc;
}

bool store_exceeds_l2(const gridff_grid* grid) {
    static int l2_bytes = -1;
    if (l2_bytes < 0) {
        int dev = 0, v = 0;
        cudaGetDevice(&dev);
        l2_bytes = cudaDeviceGetAttribute(&v, cudaDevAttrL2CacheSize, dev) == cudaSuccess ? v : 0;
    }
    return l2_bytes > 0 && grid->store_bytes > (size_t)l2_bytes;
}

}  // namespace


namespace gridff {

// enqueue k_eval_classify; *choice = the device word it writes (kChoiceCoop: spatially sorted points, kChoiceTma: scattered)
int classify_points(const gridff_grid* grid, long long n, const float* d_pos, cudaStream_t st, const unsigned** choice) {
    static std::atomic<unsigned> next{0};
    unsigned* words = nullptr;
    GRIDFF_CUDA(cudaGetSymbolAddress((void**)&words, g_eval_choice));
    unsigned* w = words + (next.fetch_add(1, std::memory_order_relaxed) & 63u);
    k_eval_classify<<<1, 256, 0, st>>>(grid->geom, n, d_pos, w);
    GRIDFF_LAUNCH_CHECK("k_eval_classify");
    *choice = w;
    return GRIDFF_OK;
}

}  // namespace gridff

extern "C" {

int gridff_eval_variant(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F,
                        int variant, void* cuda_stream) {
    if (!grid) { set_error("grid is NULL"); return GRIDFF_EINVAL; }
    if (n < 0) { set_error("n < 0"); return GRIDFF_EINVAL; }
    if (n == 0) return GRIDFF_OK;
    if (!d_pos || !d_coef) { set_error("d_pos / d_coef is NULL"); return GRIDFF_EINVAL; }
    if ((uintptr_t)d_coef & 15) { set_error("d_coef must be 16-byte aligned"); return GRIDFF_EINVAL; }
    const GridGeom& G = grid->geom;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (G.layout == GRIDFF_LAYOUT_HALF || G.layout == GRIDFF_LAYOUT_TRILINEAR) return eval_derived(grid, n, d_pos, d_coef, d_E, d_F, st);
    if (G.n_copies > 0) return eval_bricks(grid, n, d_pos, d_coef, d_E, d_F, variant, st);
    if (G.layout == GRIDFF_LAYOUT_BRICK) {
        e = launch_with_window(grid, k_eval_brick, dim3((unsigned)((n + 127) / 128)), dim3(128), 0, st, G, n, d_pos, (const float4*)d_coef, d_E, d_F);
    } else if (variant == 1) {
        e = launch_with_window(grid, k_eval_direct, dim3((unsigned)((n + 127) / 128)), dim3(128), 0, st, G, n, d_pos, (const float4*)d_coef, d_E, d_F);
    } else if (variant == 3) {
        return eval_tma(grid, n, d_pos, d_coef, d_E, d_F, nullptr, st);
    } else if (variant == 0 || variant == 2) {
        // default for a store that does not fit the L2: classify the point order on the device, then launch both kernels (see k_eval_classify).
        // L2-resident stores: the LDG gather alone (1.4x the TMA kernel there).
        const unsigned* choice = nullptr;
        if (variant == 0 && grid->tmap_ok && n >= 4096 && store_exceeds_l2(grid)) {
            int rc = classify_points(grid, n, d_pos, st, &choice);
            if (rc) return rc;
            rc = eval_tma(grid, n, d_pos, d_coef, d_E, d_F, choice, st);
            if (rc) return rc;
        }
        const long long per_block = kEvalWarps * 32;
        e = launch_with_window(grid, k_eval_coop, dim3((unsigned)((n + per_block - 1) / per_block)), dim3(kEvalWarps * 32), 0, st, G, n, d_pos, (const float4*)d_coef, d_E, d_F,
                               choice, (const float4*)nullptr, (float4*)nullptr);
    } else { set_error("unknown eval variant %d", variant); return GRIDFF_EINVAL; }
    count_launch();
    if (e != cudaSuccess) return cuda_fail(e, "gridff_eval launch");
    return GRIDFF_OK;
}

int gridff_eval(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F, void* cuda_stream) {
    return gridff_eval_variant(grid, n, d_pos, d_coef, d_E, d_F, 0, cuda_stream);
}

static unsigned binned_bins(const GridGeom& G, int& nby, int& nbz) {
    const int nbx = (G.nx + (1 << kBinX) - 1) >> kBinX;
    nby = (G.ny + (1 << kBinY) - 1) >> kBinY; nbz = (G.nz + (1 << kBinZ) - 1) >> kBinZ;
    return (unsigned)(nbx * nby * nbz) + 1u;                    // + the bin of the points above the domain
}

size_t gridff_eval_binned_work_bytes(const gridff_grid* grid, long long n) {
    if (!grid || n < 0) return 0;
    int nby, nbz;
    const size_t bins = binned_bins(grid->geom, nby, nbz);
    return (((size_t)n * 4 + 255) & ~(size_t)255) + (size_t)n * 32 + (((size_t)n * 16 + 255) & ~(size_t)255) + ((bins * 4 + 255) & ~(size_t)255) + 256;
}

int gridff_eval_binned(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F,
                       void* d_work, size_t work_bytes, void* cuda_stream) {
    if (!grid) { set_error("grid is NULL"); return GRIDFF_EINVAL; }
    if (n < 0) { set_error("n < 0"); return GRIDFF_EINVAL; }
    if (n == 0) return GRIDFF_OK;
    if (n > 0xFFFFFFF0ll) { set_error("gridff_eval_binned takes at most 2^32 - 16 points per call"); return GRIDFF_EUNSUPPORTED; }
    if (!d_pos || !d_coef) { set_error("d_pos / d_coef is NULL"); return GRIDFF_EINVAL; }
    if ((uintptr_t)d_coef & 15) { set_error("d_coef must be 16-byte aligned"); return GRIDFF_EINVAL; }
    if (grid->geom.layout != GRIDFF_LAYOUT_ZFAST) { set_error("gridff_eval_binned reads the z-fastest store"); return GRIDFF_EUNSUPPORTED; }
    if (!d_work || work_bytes < gridff_eval_binned_work_bytes(grid, n)) { set_error("d_work too small"); return GRIDFF_ESIZE; }
    if ((uintptr_t)d_work & 255) { set_error("d_work must be 256-byte aligned"); return GRIDFF_EINVAL; }
    const GridGeom& G = grid->geom;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int nby, nbz;
    const unsigned n_bins = binned_bins(G, nby, nbz);
    const size_t np4 = ((size_t)n * 4 + 255) & ~(size_t)255;
    unsigned* rank = (unsigned*)d_work;                                   // rank within the bin, then the slot
    float4* rec = (float4*)((char*)d_work + np4);                          // [n] x 32 B
    float4* out4 = (float4*)((char*)d_work + np4 + (size_t)n * 32);        // [n] x 16 B
    unsigned* count = (unsigned*)((char*)d_work + np4 + (size_t)n * 32 + (((size_t)n * 16 + 255) & ~(size_t)255));
    GRIDFF_CUDA(cudaMemsetAsync(count, 0, (size_t)n_bins * 4, st));
    const unsigned blocks = (unsigned)((n + 255) / 256);
    k_bin_count<<<blocks, 256, 0, st>>>(G, n, d_pos, nby, nbz, n_bins, count, rank);
    GRIDFF_LAUNCH_CHECK("k_bin_count");
    k_bin_scan<<<1, 1024, 0, st>>>(n_bins, count);
    GRIDFF_LAUNCH_CHECK("k_bin_scan");
    k_bin_scatter<<<blocks, 256, 0, st>>>(G, n, d_pos, (const float4*)d_coef, nby, nbz, n_bins, count, rank, rec);
    GRIDFF_LAUNCH_CHECK("k_bin_scatter");
    const long long per_block = kEvalWarps * 32;
    cudaError_t e = launch_with_window(grid, k_eval_coop, dim3((unsigned)((n + per_block - 1) / per_block)), dim3(kEvalWarps * 32), 0, st, G, n, d_pos, (const float4*)d_coef,
                                       d_E, d_F, (const unsigned*)nullptr, (const float4*)rec, out4);
    count_launch();
    if (e != cudaSuccess) return cuda_fail(e, "gridff_eval_binned launch");
    k_bin_gather_out<<<blocks, 256, 0, st>>>(n, rank, out4, d_E, d_F);
    GRIDFF_LAUNCH_CHECK("k_bin_gather_out");
    return GRIDFF_OK;
}

}  // extern "C"

// ---- gridff_eval_binned_noalloc: the same passes with their work space in a file-scope device array (callers that cannot allocate) ----
// In host code `g_binned_scratch` is only a host-side stand-in for the symbol, never a device address: binned_scratch_ptr() asks the runtime for
// the device address once per device (with that device current) and the entry point hands that pointer to the kernels.
constexpr size_t kNoAllocScratchBytes = (size_t)GRIDFF_NOALLOC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_binned_scratch[kNoAllocScratchBytes];
constexpr int kNoAllocMaxDevices = 64;
static std::atomic<void*> g_binned_scratch_ptr[kNoAllocMaxDevices];

static int binned_scratch_ptr(void** out) {
    int dev = -1;
    GRIDFF_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) { set_error("device ordinal %d outside the %d the no-alloc path keeps addresses for", dev, kNoAllocMaxDevices); return GRIDFF_EUNSUPPORTED; }
    void* p = g_binned_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        cudaError_t e = cudaGetSymbolAddress(&p, g_binned_scratch);      // the address on the CURRENT device; two racing threads store the same value
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_binned_scratch)");
        if (!p || ((uintptr_t)p & 255)) { set_error("the scratch symbol resolved to an unusable address"); return GRIDFF_ECUDA; }
        g_binned_scratch_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return GRIDFF_OK;
}

extern "C" {

size_t gridff_eval_binned_noalloc_max_bytes(void) { return kNoAllocScratchBytes; }

int gridff_eval_binned_noalloc(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F, void* cuda_stream) {
    if (!grid) { set_error("grid is NULL"); return GRIDFF_EINVAL; }
    if (n < 0) { set_error("n < 0"); return GRIDFF_EINVAL; }
    if (n > (long long)GRIDFF_NOALLOC_MAX_POINTS) {
        set_error("gridff_eval_binned_noalloc takes at most %lld points per call (got %lld): split the batch or use gridff_eval_binned with your own work space",
                  (long long)GRIDFF_NOALLOC_MAX_POINTS, n);
        return GRIDFF_ESIZE;
    }
    const size_t need = gridff_eval_binned_work_bytes(grid, n);
    if (need > kNoAllocScratchBytes) {
        set_error("gridff_eval_binned_noalloc: %lld points on this grid need %zu bytes of work space, the built-in scratch holds %zu (4 bytes per block of 4x4x8 cells + 52 per point)",
                  n, need, kNoAllocScratchBytes);
        return GRIDFF_ESIZE;
    }
    void* scratch = nullptr;
    int rc = binned_scratch_ptr(&scratch);
    if (rc) return rc;
    // the same passes as gridff_eval_binned over the built-in scratch; its bin counters are cleared there (cudaMemsetAsync on the stream) on every call
    return gridff_eval_binned(grid, n, d_pos, d_coef, d_E, d_F, scratch, kNoAllocScratchBytes, cuda_stream);
}

size_t gridff_eval_work_bytes(long long n) {
    if (n < 0) n = 0;
    return (size_t)n * (12 + 16 + 4 + 12) + 256;
}

int gridff_eval_host(const gridff_grid* grid, long long n, const float* h_pos, const float* h_coef, float* h_E, float* h_F,
                     void* d_work, size_t work_bytes, void* cuda_stream) {
    if (!grid) { set_error("grid is NULL"); return GRIDFF_EINVAL; }
    if (n < 0 || !h_pos || !h_coef) { set_error("bad n / host pointers"); return GRIDFF_EINVAL; }
    if (n == 0) return GRIDFF_OK;
    if (!d_work || work_bytes < gridff_eval_work_bytes(n)) { set_error("d_work too small"); return GRIDFF_ESIZE; }
    if ((uintptr_t)d_work & 255) { set_error("d_work must be 256-byte aligned"); return GRIDFF_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* w = (char*)d_work;
    float* d_coef = (float*)w;                       // [n][4]  (16-byte aligned)
    float* d_pos = (float*)(w + (size_t)n * 16);     // [n][3]
    float* d_F = (float*)(w + (size_t)n * 28);       // [n][3]
    float* d_E = (float*)(w + (size_t)n * 40);       // [n]
    // Pipelined in chunks over three streams so that, with pinned host buffers, the upload of chunk c+1, the kernel of chunk c and the
    // download of chunk c-1 overlap (PCIe is full duplex): the call is then bound by max(upload, download), not by their sum.
    static thread_local cudaStream_t s_in = nullptr, s_out = nullptr;
    static thread_local cudaEvent_t ev_start = nullptr, ev_in[2] = {nullptr, nullptr}, ev_k[2] = {nullptr, nullptr}, ev_out = nullptr;
    if (!s_in) {
        GRIDFF_CUDA(cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking));
        GRIDFF_CUDA(cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking));
        GRIDFF_CUDA(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
        GRIDFF_CUDA(cudaEventCreateWithFlags(&ev_out, cudaEventDisableTiming));
        for (int k = 0; k < 2; ++k) {
            GRIDFF_CUDA(cudaEventCreateWithFlags(&ev_in[k], cudaEventDisableTiming));
            GRIDFF_CUDA(cudaEventCreateWithFlags(&ev_k[k], cudaEventDisableTiming));
        }
    }
    const long long chunk = 1ll << 22;                  // 4 Mi points: 117 MB up, 67 MB down per chunk
    GRIDFF_CUDA(cudaEventRecord(ev_start, st));         // work already enqueued on the caller's stream (e.g. the grid build) comes first
    GRIDFF_CUDA(cudaStreamWaitEvent(s_in, ev_start, 0));
    GRIDFF_CUDA(cudaStreamWaitEvent(s_out, ev_start, 0));
    int c = 0;
    for (long long p0 = 0; p0 < n; p0 += chunk, ++c) {
        const long long m = n - p0 < chunk ? n - p0 : chunk;
        const int k = c & 1;
        GRIDFF_CUDA(cudaMemcpyAsync(d_coef + 4 * p0, h_coef + 4 * p0, (size_t)m * 16, cudaMemcpyHostToDevice, s_in));
        GRIDFF_CUDA(cudaMemcpyAsync(d_pos + 3 * p0, h_pos + 3 * p0, (size_t)m * 12, cudaMemcpyHostToDevice, s_in));
        GRIDFF_CUDA(cudaEventRecord(ev_in[k], s_in));
        GRIDFF_CUDA(cudaStreamWaitEvent(st, ev_in[k], 0));
        int rc = gridff_eval(grid, m, d_pos + 3 * p0, d_coef + 4 * p0, h_E ? d_E + p0 : nullptr, h_F ? d_F + 3 * p0 : nullptr, cuda_stream);
        if (rc) return rc;
        GRIDFF_CUDA(cudaEventRecord(ev_k[k], st));
        GRIDFF_CUDA(cudaStreamWaitEvent(s_out, ev_k[k], 0));
        if (h_E) GRIDFF_CUDA(cudaMemcpyAsync(h_E + p0, d_E + p0, (size_t)m * 4, cudaMemcpyDeviceToHost, s_out));
        if (h_F) GRIDFF_CUDA(cudaMemcpyAsync(h_F + 3 * p0, d_F + 3 * p0, (size_t)m * 12, cudaMemcpyDeviceToHost, s_out));
    }
    GRIDFF_CUDA(cudaEventRecord(ev_out, s_out));
    GRIDFF_CUDA(cudaStreamWaitEvent(st, ev_out, 0));
    GRIDFF_CUDA(cudaStreamSynchronize(st));
    return GRIDFF_OK;
}

int gridff_probe_read(const void* d_buf, size_t bytes, int iters, int mode, void* d_sink, void* cuda_stream) {
    if (!d_buf || !d_sink || bytes < 4096 || iters < 1) { set_error("bad probe arguments"); return GRIDFF_EINVAL; }
    if ((uintptr_t)d_buf & 15) { set_error("d_buf must be 16-byte aligned"); return GRIDFF_EINVAL; }
    if (bytes / 16 > 0xFFFFFFF0ull && mode >= 1) { set_error("row probe supports < 64 GB"); return GRIDFF_EINVAL; }
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (mode == 0) k_probe_stream<<<sms * 8, 256, 0, st>>>((const float4*)d_buf, bytes / 16, iters, (float*)d_sink);
    else if (mode == 1) k_probe_rows<4><<<sms * 8, 256, 0, st>>>((const float4*)d_buf, bytes / 16, iters, (float*)d_sink);
    else if (mode == 2) k_probe_rows<8><<<sms * 8, 256, 0, st>>>((const float4*)d_buf, bytes / 16, iters, (float*)d_sink);
    else { set_error("unknown probe mode %d", mode); return GRIDFF_EINVAL; }
    GRIDFF_LAUNCH_CHECK("gridff_probe_read");
    return GRIDFF_OK;
}

}  // extern "C"
