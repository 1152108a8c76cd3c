// gridff_internal.cuh — shared declarations of the CUDA GridFF library (sm_100a).  Product code: shares nothing
// with oracle/.  Public surface is include/gridff.h; everything here is internal.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/gridff.h"

struct gridff_grid;

namespace gridff {

constexpr double kKe = 14.3996454784;      // eV·Å/e²
constexpr double kAcc = 9.648533212e-3;    // 1 eV/(Å·amu) in Å/fs²
constexpr int kMaxAtoms = 64;
constexpr int kHalo = 3;                   // stored x/y extent = n + 3: stored index s holds node (s - 1) mod n

// Geometry of the fp32 coefficient store, passed by value to every kernel that interpolates.
// Node (jx, jy, jz), jx in [-1, nx+1], is the float4 at  store[((jx+1) * sy + (jy+1)) * nzp + jz]   (ZFAST)
struct GridGeom {
    int nx, ny, nz;              // nodes per axis
    int sx, sy, nzp;             // stored extents: nx+3, ny+3, nz rounded up to 8 nodes (128 B lines)
    int layout;
    int n_channels;
    // 1/h split into hi + lo floats so that t = fma(x, hi, -i) + x*lo keeps ~1e-7 of a cell at any |x|
    float inv_hx_hi, inv_hx_lo, inv_hy_hi, inv_hy_lo, inv_hz_hi, inv_hz_lo;
    float z0_hi, z0_lo;          // z of node 0 (z_ref + z_lo), split
    float inv_hx, inv_hy, inv_hz;
    float fnx, inv_nx, fny, inv_ny;   // (float)nx, 1/nx, ...: cell wrap without an integer division
    const float4* store;
    // micro-brick stores (GRIDFF_LAYOUT_MBRICK*, gridff_derive.cu): bricks per axis and nodes per copy; 0 otherwise
    int nbx, nby, nbz, n_copies;
    long long copy_stride;
};

struct MolDev;   // packed molecule in device memory (gridff_replica.cu)
int molecule_n_atoms(const gridff_molecule* mol);     // gridff_replica.cu (the handle's layout is private to that file)

void set_error(const char* fmt, ...);
int eval_derived(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F, cudaStream_t st);   // gridff_derive.cu
constexpr unsigned kChoiceCoop = 1u, kChoiceTma = 2u;     // device-side kernel choice of gridff_eval (gridff_eval.cu: k_eval_classify)
int eval_tma(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F, const unsigned* d_choice, cudaStream_t st);       // gridff_eval_tma.cu
int classify_points(const gridff_grid* grid, long long n, const float* d_pos, cudaStream_t st, const unsigned** choice);       // gridff_eval.cu: device-side choice word
int make_tensor_map(gridff_grid* grid);               // gridff_eval_tma.cu: CUtensorMap of a z-fastest fp32 store or of an 8-copy micro-brick store (0 on success)
int eval_bricks(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef, float* d_E, float* d_F, int variant, cudaStream_t st);   // gridff_derive.cu
int cuda_fail(cudaError_t e, const char* what);
void count_launch(int n = 1);

#define GRIDFF_CUDA(call)                                        \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return gridff::cuda_fail(e__, #call); \
    } while (0)

#define GRIDFF_LAUNCH_CHECK(name)                                \
    do {                                                         \
        gridff::count_launch();                                  \
        cudaError_t e__ = cudaGetLastError();                    \
        if (e__ != cudaSuccess) return gridff::cuda_fail(e__, name); \
    } while (0)

// ---- race stress build (-DGRIDFF_STRESS; csrc/build.py build_stress, tests/test_gpu_stress.py) ------------------
// compute-sanitizer's racecheck is not available on the GPU pool, so the hand-overs through shared memory are tested by perturbing the
// schedule instead: in the stress build every synchronisation point is surrounded by a pseudo-random per-LANE delay (one lane in four sleeps
// up to ~1 us, keyed on the clock, the lane and the warp), so that lanes and warps that normally run in lock-step reach the hand-overs at
// very different times.  A missing or misplaced barrier then changes results; the test compares the stress build with the plain build bit
// for bit.  In the product build stress_delay() is empty.
#ifdef GRIDFF_STRESS
__device__ __forceinline__ void stress_delay() {
    unsigned c, l, w;
    asm volatile("mov.u32 %0, %%clock;" : "=r"(c));
    asm volatile("mov.u32 %0, %%laneid;" : "=r"(l));
    asm volatile("mov.u32 %0, %%warpid;" : "=r"(w));
    unsigned h = c ^ (l * 0x9E3779B9u) ^ (w * 0x85EBCA6Bu);
    h ^= h >> 15; h *= 0x2C1B3C6Du; h ^= h >> 12; h *= 0x297A2D39u; h ^= h >> 15;
    if ((h & 3u) == 0u) __nanosleep(h >> 22);
}
#else
__device__ __forceinline__ void stress_delay() {}
#endif
// __syncwarp() with the stress delays around it
__device__ __forceinline__ void warp_sync() { stress_delay(); __syncwarp(); stress_delay(); }
// before an ALIGNED barrier (bar.sync, __syncthreads: every lane of a warp must arrive together): delay, then re-converge the warp
__device__ __forceinline__ void stress_before_barrier() {
#ifdef GRIDFF_STRESS
    stress_delay(); __syncwarp();
#endif
}

// ---- B-spline weights (Eqs. 5-6; polynomial pieces of B(t+1-j), j = 0..3) -------------------
__device__ __forceinline__ void bspline_w(float t, float w[4], float d[4]) {
    const float s = 1.0f - t, t2 = t * t, s2 = s * s;
    const float k6 = 1.0f / 6.0f;
    w[0] = s2 * s * k6;
    w[3] = t2 * t * k6;
    w[1] = fmaf(t2, fmaf(0.5f, t, -1.0f), 2.0f / 3.0f);      // t^3/2 - t^2 + 2/3
    w[2] = fmaf(s2, fmaf(0.5f, s, -1.0f), 2.0f / 3.0f);      // mirror image: (1-t)
    d[0] = -0.5f * s2;
    d[3] = 0.5f * t2;
    d[1] = t * fmaf(1.5f, t, -2.0f);                          // 3/2 t^2 - 2 t
    d[2] = -s * fmaf(1.5f, s, -2.0f);
}

// cell index (wrapped into [0,n)) and fraction along a periodic axis
__device__ __forceinline__ void cell_periodic(float x, float inv_hi, float inv_lo, float fn, float inv_n, int& i, float& t) {
    float fi = floorf(x * inv_hi);
    float tt = fmaf(x, inv_hi, -fi) + x * inv_lo;
    if (tt < 0.0f) { tt += 1.0f; fi -= 1.0f; }
    if (tt >= 1.0f) { tt -= 1.0f; fi += 1.0f; }
    // fi mod n in floats: fi is an integer with |fi| < 2^24 for any sane coordinate, so fi - q n is exact; the rounded
    // quotient can be off by one either way
    float r = fmaf(-floorf(fi * inv_n), fn, fi);
    if (r < 0.0f) r += fn;
    if (r >= fn) r -= fn;
    int ii = (int)r;                      // NaN -> 0
    ii = min(max(ii, 0), (int)fn - 1);    // and never outside the store, whatever x was
    i = ii; t = tt;
}

// z axis: returns false when the point is above the stored domain (E = F = 0, gridff.h); below node 1 the lowest
// cell's polynomial is continued (t < 0).
__device__ __forceinline__ bool cell_z(float z, const GridGeom& g, int& i, float& t) {
    const float dz = (z - g.z0_hi) - g.z0_lo;
    const float q = dz * g.inv_hz_hi;
    if (!(q < (float)(g.nz - 2))) {
        // q rounds to nz-2 from below only within 1 ulp: treat as above as well (E there is ~0 by construction)
        return false;
    }
    float fi = floorf(q);
    fi = fminf(fmaxf(fi, 1.0f), (float)(g.nz - 3));
    t = fmaf(dz, g.inv_hz_hi, -fi) + dz * g.inv_hz_lo;
    i = (int)fi;
    return true;
}

// stored-array offset (in float4 nodes) of the stencil corner (ix-1, iy-1, iz-1) in the ZFAST layout
__device__ __forceinline__ size_t corner_zfast(const GridGeom& g, int ix, int iy, int iz) {
    return ((size_t)ix * g.sy + iy) * g.nzp + (iz - 1);
}

}  // namespace gridff

// opaque handles ------------------------------------------------------------------------------------------------
struct gridff_grid {
    gridff::GridGeom geom;
    gridff_grid_desc desc;
    double h[3], origin[3];
    size_t store_bytes;
    int l2_window_ok;     // 1 when an access-policy window could be applied
    int tmap_ok;          // 1 when tmap describes the store (z-fastest fp32 stores; gridff_eval variant 3)
    alignas(64) unsigned char tmap[128];      // CUtensorMap (opaque here: <cuda.h> is needed only where it is encoded and used)
};
