// gridff_derive.cu — derived coefficient stores for the interpolation trade study.
//   GRIDFF_LAYOUT_HALF       fp16 coefficients (8 B per node), tricubic B-spline with fp32 accumulation
//   GRIDFF_LAYOUT_TRILINEAR  the trilinear foil the paper compares against ("the force components (Fx, Fy, Fz) and
//                            energy E were stored and interpolated independently"; L140: tricubic "only about two times slower")
//   GRIDFF_LAYOUT_MBRICK*    the fp32 coefficients in 2 x 2 x 2-node bricks of one 128-byte line, 1 / 2 / 8 shifted copies: the layout for
//                            stores that exceed the L2, where DRAM moves whole lines and the z-fastest rows waste 1.7 of every 2.7 bytes
// All are built from a ZFAST fp32 grid and are read by gridff_eval only.
#include "gridff_interp.cuh"
#include <cuda_fp16.h>
#include <string.h>
#include <new>

using namespace gridff;

namespace {

inline unsigned blocks_for(long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

// ---- fp16 store: same extents and indexing as the parent, uint2 = 4 halves per node ---------------------------------------------------
__global__ void k_to_half(const float4* __restrict__ src, long n, uint2* __restrict__ dst) {
    const long k = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const float4 v = src[k];
    const __half2 a = __floats2half2_rn(v.x, v.y), b = __floats2half2_rn(v.z, v.w);
    uint2 o; o.x = *reinterpret_cast<const unsigned*>(&a); o.y = *reinterpret_cast<const unsigned*>(&b);
    dst[k] = o;
}

__device__ __forceinline__ float fold_half(const float4 c, const uint2 n) {
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&n.x)), b = __half22float2(*reinterpret_cast<const __half2*>(&n.y));
    return fmaf(c.x, a.x, fmaf(c.y, a.y, fmaf(c.z, b.x, c.w * b.y)));
}

// warp-cooperative gather as k_eval_coop: a stencil row is 4 nodes x 8 B = 32 B; 4 lanes read one row, 8 rows per LDG.64
constexpr int kWarps = 4;
__global__ void __launch_bounds__(kWarps * 32) k_eval_half(GridGeom g, long long n, const float* __restrict__ pos, const float4* __restrict__ coef,
                                                           float* __restrict__ E, float* __restrict__ F) {
    __shared__ __align__(16) float s_tile[kWarps][32 * 64];
    __shared__ __align__(16) float4 s_cf[kWarps][32];
    __shared__ unsigned s_base[kWarps][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const long long p = ((long long)blockIdx.x * kWarps + w) * 32 + lane;
    Stencil s; s.base = kNoStencil; s.tx = s.ty = s.tz = 0.f;
    float4 cf = make_float4(0.f, 0.f, 0.f, 0.f);
    if (p < n) { s = locate(g, pos[3 * p], pos[3 * p + 1], pos[3 * p + 2]); cf = coef[p]; }
    s_base[w][lane] = s.base; s_cf[w][lane] = cf;
    warp_sync();
    float* tile = s_tile[w];
    const uint2* store = reinterpret_cast<const uint2*>(g.store);
    const int k = lane & 3, r0 = lane >> 2;
    const int rs = g.nzp, ps = g.sy * g.nzp;
    const int off = (r0 >> 2) * ps + (r0 & 3) * rs + k;
    // per-warp load path as in k_eval_coop: through the L1 when the warp's points share cells, past it otherwise
    const unsigned prev = __shfl_up_sync(0xFFFFFFFFu, s.base, 1);
    const bool clustered = __popc(__ballot_sync(0xFFFFFFFFu, lane > 0 && prev == s.base)) >= 8;
#pragma unroll 8
    for (int q = 0; q < 32; ++q) {
        const unsigned b = s_base[w][q];
        if (b != kNoStencil) {
            const uint2* a = store + b + off;
            const uint2 n0 = clustered ? __ldg(a) : __ldcg(a), n1 = clustered ? __ldg(a + 2 * ps) : __ldcg(a + 2 * ps);
            const float4 c = s_cf[w][q];
            tile[tile_word(q, lane)] = fold_half(c, n0);
            tile[tile_word(q, lane + 32)] = fold_half(c, n1);
        }
    }
    warp_sync();
    if (p >= n) return;
    float e, fx, fy, fz;
    interp_tile(g, s, lane, tile, e, fx, fy, fz);
    if (E) E[p] = e;
    if (F) { F[3 * p] = fx; F[3 * p + 1] = fy; F[3 * p + 2] = fz; }
}

// ---- trilinear foil ------------------------------------------------------------------------------------------------------------------
// store: [nx + 1][ny + 1][nzt] nodes of 4 float4 {V, dV/dx, dV/dy, dV/dz} (each float4 = the 4 channels), stored x / y index s holds
// node s mod n; nzt = nz rounded up to 2 so that the two z corners of a cell share a 128-byte line when iz is even.
// Node values: the parent spline and its analytic gradient at the node (t = 0: weights (1/6, 4/6, 1/6), derivative weights (-1/2, 0, 1/2)),
// for iz in [1, nz-2]; zero elsewhere (never read: cells are clamped to [1, nz-3] like the spline's).
__global__ void k_to_trilinear(GridGeom g, int nzt, float4* __restrict__ dst) {
    const long k = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long total = (long)(g.nx + 1) * (g.ny + 1) * nzt;
    if (k >= total) return;
    const int iz = (int)(k % nzt); const long r = k / nzt;
    const int sy_ = (int)(r % (g.ny + 1)), sx_ = (int)(r / (g.ny + 1));
    float4 V = make_float4(0.f, 0.f, 0.f, 0.f), Gx = V, Gy = V, Gz = V;
    if (iz >= 1 && iz <= g.nz - 2) {
        const int ix = sx_ % g.nx, iy = sy_ % g.ny;
        const float w[3] = {1.0f / 6.0f, 4.0f / 6.0f, 1.0f / 6.0f}, d[3] = {-0.5f, 0.0f, 0.5f};
        // parent stored index of node (ix - 1 + a) is ix + a (halo: stored s holds node s - 1)
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b)
                for (int c = 0; c < 3; ++c) {
                    const float4 nd = g.store[((size_t)(ix + a) * g.sy + (iy + b)) * g.nzp + (iz - 1 + c)];
                    const float wv = w[a] * w[b] * w[c], wx = d[a] * w[b] * w[c] * g.inv_hx, wy = w[a] * d[b] * w[c] * g.inv_hy, wz = w[a] * w[b] * d[c] * g.inv_hz;
                    V.x = fmaf(wv, nd.x, V.x); V.y = fmaf(wv, nd.y, V.y); V.z = fmaf(wv, nd.z, V.z); V.w = fmaf(wv, nd.w, V.w);
                    Gx.x = fmaf(wx, nd.x, Gx.x); Gx.y = fmaf(wx, nd.y, Gx.y); Gx.z = fmaf(wx, nd.z, Gx.z); Gx.w = fmaf(wx, nd.w, Gx.w);
                    Gy.x = fmaf(wy, nd.x, Gy.x); Gy.y = fmaf(wy, nd.y, Gy.y); Gy.z = fmaf(wy, nd.z, Gy.z); Gy.w = fmaf(wy, nd.w, Gy.w);
                    Gz.x = fmaf(wz, nd.x, Gz.x); Gz.y = fmaf(wz, nd.y, Gz.y); Gz.z = fmaf(wz, nd.z, Gz.z); Gz.w = fmaf(wz, nd.w, Gz.w);
                }
    }
    float4* o = dst + k * 4;
    o[0] = V; o[1] = Gx; o[2] = Gy; o[3] = Gz;
}

// 4 lanes per point: lane j of the quad reads float4 j (V, Gx, Gy or Gz) of each of the 8 corners (one 64-byte node per quad per load),
// folds it with the point's channel factors and accumulates its own output component
__global__ void __launch_bounds__(256) k_eval_trilinear(GridGeom g, int nzt, long long n, const float* __restrict__ pos, const float4* __restrict__ coef,
                                                        float* __restrict__ E, float* __restrict__ F) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long p = t >> 2; const int j = (int)(t & 3);
    if (p >= n) return;
    int ix, iy, iz; float tx, ty, tz;
    cell_periodic(pos[3 * p], g.inv_hx_hi, g.inv_hx_lo, g.fnx, g.inv_nx, ix, tx);
    cell_periodic(pos[3 * p + 1], g.inv_hy_hi, g.inv_hy_lo, g.fny, g.inv_ny, iy, ty);
    float out = 0.f;
    if (cell_z(pos[3 * p + 2], g, iz, tz)) {
        const float4 cf = coef[p];
        const float4* base = g.store + ((((size_t)ix * (g.ny + 1) + iy) * nzt + iz) << 2) + j;
        const size_t sz = 4, sy_ = (size_t)nzt * 4, sx_ = (size_t)(g.ny + 1) * nzt * 4;
        float4 v[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) v[c] = __ldg(base + (c >> 2) * sx_ + ((c >> 1) & 1) * sy_ + (c & 1) * sz);
        const float wx[2] = {1.0f - tx, tx}, wy[2] = {1.0f - ty, ty}, wz[2] = {1.0f - tz, tz};
#pragma unroll
        for (int c = 0; c < 8; ++c) out = fmaf(wx[c >> 2] * wy[(c >> 1) & 1] * wz[c & 1], fold4(cf, v[c]), out);
    }
    if (j == 0) { if (E) E[p] = out; }
    else if (F) F[3 * p + (j - 1)] = -out;
}

// ---- micro-brick stores (addressing: gridff_interp.cuh) ----------------------------------------------------------------------------------
__global__ void k_to_bricks(GridGeom parent, GridGeom g, float4* __restrict__ dst) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.copy_stride * g.n_copies) return;
    const int copy = (int)(k / g.copy_stride);
    const long long r = k - (long long)copy * g.copy_stride;
    const int in = (int)(r & 7); long long b = r >> 3;
    const int bz = (int)(b % g.nbz); b /= g.nbz;
    const int by = (int)(b % g.nby), bx = (int)(b / g.nby);
    const int sh = brick_shift_bits(g.n_copies, copy);
    const int X = 2 * bx - ((sh >> 2) & 1) + ((in >> 2) & 1), Y = 2 * by - ((sh >> 1) & 1) + ((in >> 1) & 1), Z = 2 * bz - (sh & 1) + (in & 1);
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (X >= 0 && X < parent.sx && Y >= 0 && Y < parent.sy && Z >= 0 && Z < parent.nzp) v = parent.store[((size_t)X * parent.sy + Y) * parent.nzp + Z];
    dst[k] = v;
}

// k_eval_coop over bricks: a warp owns 32 points, gathers each stencil cooperatively (lane <-> node as over the z-fastest store, so the folded
// tile, the contraction and the results are the same bit for bit), every lane then contracts its own point
__global__ void __launch_bounds__(kWarps * 32) k_eval_bricks(GridGeom g, long long n, const float* __restrict__ pos, const float4* __restrict__ coef,
                                                             float* __restrict__ E, float* __restrict__ F, const unsigned* __restrict__ choice) {
    if (choice && *choice != kChoiceCoop) return;         // the device-side choice (k_eval_classify) went to the TMA kernel
    __shared__ __align__(16) float s_tile[kWarps][32 * 64];
    __shared__ __align__(16) float4 s_cf[kWarps][32];
    __shared__ unsigned s_corner[kWarps][32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const long long p = ((long long)blockIdx.x * kWarps + w) * 32 + lane;
    Stencil s; s.base = kNoStencil; s.tx = s.ty = s.tz = 0.f;
    float4 cf = make_float4(0.f, 0.f, 0.f, 0.f);
    int ix = 0, iy = 0, iz = 0;
    if (p < n) { s = locate(g, pos[3 * p], pos[3 * p + 1], pos[3 * p + 2], ix, iy, iz); cf = coef[p]; }
    s_corner[w][lane] = s.base == kNoStencil ? kNoStencil : pack_corner(ix, iy, iz - 1);
    s_cf[w][lane] = cf;
    warp_sync();
    float* tile = s_tile[w];
    if (warp_points_are_local(ix, iy, iz, s.base != kNoStencil, lane)) {
#pragma unroll 8
        for (int q = 0; q < 32; ++q) {
            const unsigned c = s_corner[w][q];
            if (c != kNoStencil) gather_bricks<false>(g, c, s_cf[w][q], lane, q, tile);
        }
    } else {
#pragma unroll 8
        for (int q = 0; q < 32; ++q) {
            const unsigned c = s_corner[w][q];
            if (c != kNoStencil) gather_bricks<true>(g, c, s_cf[w][q], lane, q, tile);
        }
    }
    warp_sync();
    if (p >= n) return;
    float e, fx, fy, fz;
    interp_tile(g, s, lane, tile, e, fx, fy, fz);
    if (E) E[p] = e;
    if (F) { F[3 * p] = fx; F[3 * p + 1] = fy; F[3 * p + 2] = fz; }
}

inline int brick_copies(int layout) { return layout == GRIDFF_LAYOUT_MBRICK8 ? 8 : layout == GRIDFF_LAYOUT_MBRICK2 ? 2 : layout == GRIDFF_LAYOUT_MBRICK ? 1 : 0; }
inline void brick_extents(const GridGeom& P, int& nbx, int& nby, int& nbz) { nbx = (P.sx >> 1) + 1; nby = (P.sy >> 1) + 1; nbz = (P.nzp >> 1) + 1; }

}  // namespace

namespace gridff {

int eval_bricks(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F, int variant, cudaStream_t st) {
    const GridGeom& G = grid->geom;
    if (variant != 0 && variant != 2 && variant != 3) { set_error("micro-brick stores have variants 0, 2 (LDG gather) and 3 (TMA, 8 copies)"); return GRIDFF_EINVAL; }
    if (variant == 3 && !(G.n_copies == 8 && grid->tmap_ok)) { set_error("the TMA variant needs the 8-copy micro-brick store and a tensor map"); return GRIDFF_EUNSUPPORTED; }
    if (variant == 3) return eval_tma(grid, n, d_pos, d_coef, d_E, d_F, nullptr, st);
    // 8-copy store, default: scattered points go to the TMA box kernel, spatially sorted ones to the LDG gather (L1 / L2 hits at full occupancy);
    // the order of the caller's points is classified on the device and both kernels are enqueued (gridff_eval.cu: k_eval_classify)
    const unsigned* choice = nullptr;
    if (variant == 0 && G.n_copies == 8 && grid->tmap_ok && n >= 4096) {
        int rc = classify_points(grid, n, d_pos, st, &choice);
        if (rc) return rc;
        rc = eval_tma(grid, n, d_pos, d_coef, d_E, d_F, choice, st);
        if (rc) return rc;
    }
    const long long per_block = kWarps * 32;
    cudaError_t e = launch_with_window(grid, k_eval_bricks, dim3((unsigned)((n + per_block - 1) / per_block)), dim3(kWarps * 32), 0, st, G, n, d_pos, (const float4*)d_coef, d_E, d_F, choice);
    count_launch();
    if (e != cudaSuccess) return cuda_fail(e, "gridff_eval (micro-brick store) launch");
    return GRIDFF_OK;
}

int eval_derived(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F, cudaStream_t st) {
    const GridGeom& G = grid->geom;
    cudaError_t e;
    if (G.layout == GRIDFF_LAYOUT_HALF) {
        const long long per_block = kWarps * 32;
        e = launch_with_window(grid, k_eval_half, dim3((unsigned)((n + per_block - 1) / per_block)), dim3(kWarps * 32), 0, st, G, n, d_pos, (const float4*)d_coef, d_E, d_F);
    } else if (G.layout == GRIDFF_LAYOUT_TRILINEAR) {
        const int nzt = (G.nz + 1) & ~1;
        e = launch_with_window(grid, k_eval_trilinear, dim3((unsigned)((4 * n + 255) / 256)), dim3(256), 0, st, G, nzt, n, d_pos, (const float4*)d_coef, d_E, d_F);
    } else { set_error("not a derived layout"); return GRIDFF_EINVAL; }
    count_launch();
    if (e != cudaSuccess) return cuda_fail(e, "gridff_eval (derived store) launch");
    return GRIDFF_OK;
}

}  // namespace gridff

extern "C" {

size_t gridff_derive_bytes(const gridff_grid* parent, int layout) {
    if (!parent) return 0;
    const GridGeom& G = parent->geom;
    if (layout == GRIDFF_LAYOUT_HALF) return (size_t)G.sx * G.sy * G.nzp * 8;
    if (layout == GRIDFF_LAYOUT_TRILINEAR) return (size_t)(G.nx + 1) * (G.ny + 1) * ((G.nz + 1) & ~1) * 64;
    if (brick_copies(layout)) { int bx, by, bz; brick_extents(G, bx, by, bz); return (size_t)brick_copies(layout) * bx * by * bz * 128; }
    return 0;
}

int gridff_grid_derive(const gridff_grid* parent, int layout, void* d_store, size_t store_bytes, void* cuda_stream, gridff_grid** out) {
    if (!parent || !out) { set_error("parent / out is NULL"); return GRIDFF_EINVAL; }
    *out = nullptr;
    if (parent->geom.layout != GRIDFF_LAYOUT_ZFAST) { set_error("derived stores are built from a z-fastest fp32 grid"); return GRIDFF_EUNSUPPORTED; }
    if (layout != GRIDFF_LAYOUT_HALF && layout != GRIDFF_LAYOUT_TRILINEAR && !brick_copies(layout)) { set_error("unknown derived layout %d", layout); return GRIDFF_EINVAL; }
    if (brick_copies(layout) && (parent->geom.sx > 2047 || parent->geom.sy > 2047 || parent->geom.nzp > 1023)) {
        set_error("micro-brick stores need nx + 3, ny + 3 <= 2047 and nz <= 1023"); return GRIDFF_EUNSUPPORTED;
    }
    const size_t need = gridff_derive_bytes(parent, layout);
    if (!d_store || store_bytes < need) { set_error("derived store buffer too small: %zu < %zu", store_bytes, need); return GRIDFF_ESIZE; }
    if ((uintptr_t)d_store & 255) { set_error("d_store must be 256-byte aligned"); return GRIDFF_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const GridGeom& G = parent->geom;
    if (layout == GRIDFF_LAYOUT_HALF) {
        const long nn = (long)G.sx * G.sy * G.nzp;
        k_to_half<<<blocks_for(nn, 256), 256, 0, st>>>(G.store, nn, (uint2*)d_store);
        GRIDFF_LAUNCH_CHECK("k_to_half");
    } else if (layout == GRIDFF_LAYOUT_TRILINEAR) {
        const int nzt = (G.nz + 1) & ~1;
        const long nn = (long)(G.nx + 1) * (G.ny + 1) * nzt;
        k_to_trilinear<<<blocks_for(nn, 128), 128, 0, st>>>(G, nzt, (float4*)d_store);
        GRIDFF_LAUNCH_CHECK("k_to_trilinear");
    }
    gridff_grid* g = new (std::nothrow) gridff_grid();
    if (!g) { set_error("out of host memory"); return GRIDFF_EINVAL; }
    *g = *parent;
    g->geom.layout = layout;
    g->geom.store = (const float4*)d_store;
    g->store_bytes = need;
    g->tmap_ok = 0;
    if (brick_copies(layout)) {
        GridGeom& B = g->geom;
        brick_extents(G, B.nbx, B.nby, B.nbz);
        B.n_copies = brick_copies(layout);
        B.copy_stride = (long long)B.nbx * B.nby * B.nbz * 8;
        const long long nn = B.copy_stride * B.n_copies;
        k_to_bricks<<<(unsigned)((nn + 255) / 256), 256, 0, st>>>(G, B, (float4*)d_store);
        count_launch();
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) { delete g; return cuda_fail(e, "k_to_bricks"); }
        if (B.n_copies == 8 && make_tensor_map(g) != GRIDFF_OK) g->tmap_ok = 0;      // variant 3 then reports it; the LDG gather serves
    }
    *out = g;
    return GRIDFF_OK;
}

}  // extern "C"
