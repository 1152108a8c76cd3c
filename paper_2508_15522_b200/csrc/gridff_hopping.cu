// gridff_hopping.cu — minima hopping with an on-device unique-structure filter.
//   PAPER.md:L222  "perturbing the molecular structure (i.e., by performing 1000 steps of Langevin molecular dynamics at ... 300 K,
//                   followed by dynamical relaxation to the nearest local minimum"
//   PAPER.md:L241  "each optimized geometry is compared with all previously minimized structures using a root-mean-square deviation
//                   criterion (with a threshold of 0.1 Å) ... geometries are downloaded from the GPU and the comparison is performed on
//                   the CPU" — here the comparison stays on the device, so a whole run of cycles is enqueued without a host round-trip.
// Same-structure criterion: DESIGN.md R16.  Filter semantics: sequential greedy in replica order (what a CPU loop would do), obtained
// in two launches: (A) every converged replica against the records that existed before this cycle, one warp per replica;
// (B) one block walks the survivors in replica order against the records appended in this cycle and appends the new ones.
#include "gridff_internal.cuh"
#include <string.h>

using namespace gridff;

namespace {

struct FilterParams {
    int n, n_rep, cap, tag;
    float Lx, Ly, inv_Lx, inv_Ly, e_tol, rmsd_tol2;
    const float* pos; const float* E; const int* steps; const int* ok;
    float* lib; int* n_lib; int* stats; int* flags;
};

// candidate (E_c, x_c) vs record rec = {.,.,.,E, x[3n]}: |dE| < e_tol and mean |dx|^2 < rmsd_tol^2 after removing the cell translation
// nearest to the mean displacement (two passes over the atoms)
__device__ __forceinline__ bool same_structure(const FilterParams& P, float Ec, const float* __restrict__ xc, const float* __restrict__ rec) {
    if (!(fabsf(Ec - rec[3]) < P.e_tol)) return false;
    const float* xr = rec + 4;
    float mx = 0.f, my = 0.f;
    for (int i = 0; i < P.n; ++i) { mx += xc[3 * i] - xr[3 * i]; my += xc[3 * i + 1] - xr[3 * i + 1]; }
    const float inv_n = 1.0f / (float)P.n;
    const float sx = rintf(mx * inv_n * P.inv_Lx) * P.Lx, sy = rintf(my * inv_n * P.inv_Ly) * P.Ly;
    float s2 = 0.f;
    for (int i = 0; i < P.n; ++i) {
        const float dx = xc[3 * i] - xr[3 * i] - sx, dy = xc[3 * i + 1] - xr[3 * i + 1] - sy, dz = xc[3 * i + 2] - xr[3 * i + 2];
        s2 += fmaf(dx, dx, fmaf(dy, dy, dz * dz));
    }
    return s2 * inv_n < P.rmsd_tol2;
}

// (A) flags[r] = -1 not a candidate, 1 matches an existing record, 0 survivor
__global__ void __launch_bounds__(256) k_filter_library(const FilterParams P) {
    const int r = (int)((blockIdx.x * (unsigned)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (r >= P.n_rep) return;
    if (!P.ok[r]) { if (lane == 0) P.flags[r] = -1; return; }
    const int n_lib = min(*P.n_lib, P.cap);
    const float Ec = P.E[r];
    const float* xc = P.pos + (size_t)r * 3 * P.n;
    const size_t stride = 4 + 3 * (size_t)P.n;
    bool hit = false;
    for (int j0 = 0; j0 < n_lib && !hit; j0 += 32) {
        const int j = j0 + lane;
        const bool m = j < n_lib && same_structure(P, Ec, xc, P.lib + (size_t)j * stride);
        hit = __any_sync(0xFFFFFFFFu, m);
    }
    if (lane == 0) P.flags[r] = hit ? 1 : 0;
}

// (B) one block: survivors in replica order against the records appended during this launch; appends the new ones
__global__ void __launch_bounds__(1024) k_filter_append(const FilterParams P) {
    __shared__ int s_hit;
    const size_t stride = 4 + 3 * (size_t)P.n;
    const int n0 = min(*P.n_lib, P.cap);
    int n_cur = n0, n_cand = 0, n_new = 0, n_drop = 0;
    for (int r = 0; r < P.n_rep; ++r) {
        const int f = P.flags[r];                     // uniform over the block
        if (f < 0) continue;
        ++n_cand;
        if (f > 0) continue;
        if (threadIdx.x == 0) s_hit = 0;
        stress_before_barrier(); __syncthreads(); stress_delay();
        const float Ec = P.E[r];
        const float* xc = P.pos + (size_t)r * 3 * P.n;
        bool m = false;
        for (int j = n0 + threadIdx.x; j < n_cur; j += blockDim.x) m = m || same_structure(P, Ec, xc, P.lib + (size_t)j * stride);
        if (m) s_hit = 1;
        stress_before_barrier(); __syncthreads(); stress_delay();
        const bool hit = s_hit != 0;
        stress_before_barrier(); __syncthreads(); stress_delay();
        if (hit) continue;
        if (n_cur >= P.cap) { ++n_drop; continue; }
        float* rec = P.lib + (size_t)n_cur * stride;
        if (threadIdx.x == 0) { rec[0] = (float)r; rec[1] = (float)P.tag; rec[2] = P.steps ? (float)P.steps[r] : 0.f; rec[3] = Ec; }
        for (int i = threadIdx.x; i < 3 * P.n; i += blockDim.x) rec[4 + i] = xc[i];
        ++n_cur; ++n_new;
        stress_before_barrier(); __syncthreads(); stress_delay();                              // the record is visible to the block before the next survivor is compared
    }
    if (threadIdx.x == 0) {
        *P.n_lib = n_cur;
        if (P.stats) { P.stats[0] = n_cand; P.stats[1] = n_new; P.stats[2] = n_drop; P.stats[3] = n_cur; }
    }
}

// E_total = sum of the 7 potential terms; ok = converged flag of the FIRE launch
__global__ void k_hop_collect(int n_rep, const float* __restrict__ energy, const int* __restrict__ status, float* __restrict__ E,
                              int* __restrict__ ok, int* __restrict__ steps) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_rep) return;
    float e = 0.f;
    for (int c = 0; c < 7; ++c) e += energy[8 * r + c];
    E[r] = e; steps[r] = status[2 * r]; ok[r] = status[2 * r + 1] == 1;
}

inline size_t up256(size_t v) { return (v + 255) & ~(size_t)255; }

int enqueue_filter(const gridff_grid* grid, int n, int n_rep, const float* d_pos, const float* d_E, const int* d_steps, const int* d_ok,
                   float e_tol, float rmsd_tol, int tag, float* d_library, int cap, int* d_n_library, int* d_stats4, int* d_flags, cudaStream_t st) {
    FilterParams P;
    memset(&P, 0, sizeof(P));
    P.n = n; P.n_rep = n_rep; P.cap = cap; P.tag = tag;
    P.Lx = (float)grid->desc.Lx; P.Ly = (float)grid->desc.Ly; P.inv_Lx = (float)(1.0 / grid->desc.Lx); P.inv_Ly = (float)(1.0 / grid->desc.Ly);
    P.e_tol = e_tol; P.rmsd_tol2 = rmsd_tol * rmsd_tol;
    P.pos = d_pos; P.E = d_E; P.steps = d_steps; P.ok = d_ok; P.lib = d_library; P.n_lib = d_n_library; P.stats = d_stats4; P.flags = d_flags;
    k_filter_library<<<(unsigned)((n_rep + 7) / 8), 256, 0, st>>>(P);
    GRIDFF_LAUNCH_CHECK("k_filter_library");
    k_filter_append<<<1, 1024, 0, st>>>(P);
    GRIDFF_LAUNCH_CHECK("k_filter_append");
    return GRIDFF_OK;
}

}  // namespace

extern "C" {

int gridff_unique_filter(const gridff_grid* grid, const gridff_molecule* mol, int n_rep, const float* d_pos, const float* d_E,
                         const int* d_steps, const int* d_ok, float e_tol, float rmsd_tol, int tag,
                         float* d_library, int cap, int* d_n_library, int* d_stats4, int* d_flags, void* cuda_stream) {
    if (!grid || !mol) { set_error("grid / mol is NULL (the cell defines the lattice translations)"); return GRIDFF_EINVAL; }
    if (n_rep < 0 || cap < 0) { set_error("n_rep / cap < 0"); return GRIDFF_EINVAL; }
    if (n_rep == 0) return GRIDFF_OK;
    if (!d_pos || !d_E || !d_ok || !d_library || !d_n_library || !d_flags) { set_error("a required device pointer is NULL"); return GRIDFF_EINVAL; }
    if (!(e_tol > 0) || !(rmsd_tol > 0)) { set_error("e_tol and rmsd_tol must be > 0"); return GRIDFF_EINVAL; }
    return enqueue_filter(grid, molecule_n_atoms(mol), n_rep, d_pos, d_E, d_steps, d_ok, e_tol, rmsd_tol, tag, d_library, cap, d_n_library,
                          d_stats4, d_flags, (cudaStream_t)cuda_stream);
}

size_t gridff_hopping_work_bytes(const gridff_molecule* mol, int n_rep) {
    if (!mol || n_rep < 0) return 0;
    const size_t nr = (size_t)n_rep, n = (size_t)molecule_n_atoms(mol);
    // vel, fire, energy, status, E, ok, steps, flags
    return up256(nr * n * 12) + up256(nr * 16) + up256(nr * 32) + up256(nr * 8) + 4 * up256(nr * 4) + 256;
}

int gridff_minima_hopping(const gridff_grid* grid, const gridff_molecule* mol, const gridff_hopping* H, int n_rep,
                          float* d_pos, float* d_library, int cap, int* d_n_library, int* d_stats,
                          void* d_work, size_t work_bytes, void* cuda_stream) {
    if (!grid || !mol || !H) { set_error("grid / mol / hop is NULL"); return GRIDFF_EINVAL; }
    if (n_rep < 0 || cap < 0 || H->n_cycles < 0) { set_error("n_rep / cap / n_cycles < 0"); return GRIDFF_EINVAL; }
    if (n_rep == 0 || H->n_cycles == 0) return GRIDFF_OK;
    if (!d_pos || !d_library || !d_n_library) { set_error("a required device pointer is NULL"); return GRIDFF_EINVAL; }
    if (H->md_steps < 0 || H->relax_steps < 0 || !(H->md_dt > 0) || !(H->relax_dt > 0)) { set_error("bad step counts / time steps"); return GRIDFF_EINVAL; }
    if (!(H->e_tol > 0) || !(H->rmsd_tol > 0) || !(H->f_tol > 0)) { set_error("e_tol, rmsd_tol, f_tol must be > 0"); return GRIDFF_EINVAL; }
    if (!d_work || work_bytes < gridff_hopping_work_bytes(mol, n_rep)) { set_error("d_work too small"); return GRIDFF_ESIZE; }
    if ((uintptr_t)d_work & 255) { set_error("d_work must be 256-byte aligned"); return GRIDFF_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t nr = (size_t)n_rep, n = (size_t)molecule_n_atoms(mol);
    char* w = (char*)d_work;
    float* d_vel = (float*)w; w += up256(nr * n * 12);
    float* d_fire = (float*)w; w += up256(nr * 16);
    float* d_energy = (float*)w; w += up256(nr * 32);
    int* d_status = (int*)w; w += up256(nr * 8);
    float* d_E = (float*)w; w += up256(nr * 4);
    int* d_ok = (int*)w; w += up256(nr * 4);
    int* d_steps = (int*)w; w += up256(nr * 4);
    int* d_flags = (int*)w;

    gridff_integrator md;
    memset(&md, 0, sizeof(md));
    md.kind = 2; md.n_steps = H->md_steps; md.dt = H->md_dt; md.temperature = H->temperature; md.gamma = H->gamma;
    md.seed = H->seed; md.fixed_mask = H->fixed_mask;
    gridff_integrator fi;
    memset(&fi, 0, sizeof(fi));
    fi.kind = 1; fi.n_steps = H->relax_steps; fi.dt = H->relax_dt; fi.f_tol = H->f_tol; fi.dt_max = H->dt_max; fi.max_step = H->max_step;
    fi.fixed_mask = H->fixed_mask;

    for (int c = 0; c < H->n_cycles; ++c) {
        md.step0 = (unsigned)(H->cycle0 + c) * (unsigned)H->md_steps;
        GRIDFF_CUDA(cudaMemsetAsync(d_vel, 0, nr * n * 12, st));                     // Langevin from rest
        int rc = gridff_run_replicas(grid, mol, &md, n_rep, d_pos, d_vel, nullptr, nullptr, nullptr, nullptr, 0, nullptr, cuda_stream);
        if (rc) return rc;
        GRIDFF_CUDA(cudaMemsetAsync(d_vel, 0, nr * n * 12, st));                     // FIRE from rest, fresh scalars
        GRIDFF_CUDA(cudaMemsetAsync(d_fire, 0, nr * 16, st));
        rc = gridff_run_replicas(grid, mol, &fi, n_rep, d_pos, d_vel, d_fire, d_energy, d_status, nullptr, 0, nullptr, cuda_stream);
        if (rc) return rc;
        k_hop_collect<<<(unsigned)((n_rep + 255) / 256), 256, 0, st>>>(n_rep, d_energy, d_status, d_E, d_ok, d_steps);
        GRIDFF_LAUNCH_CHECK("k_hop_collect");
        rc = enqueue_filter(grid, (int)n, n_rep, d_pos, d_E, d_steps, d_ok, H->e_tol, H->rmsd_tol, H->cycle0 + c, d_library, cap, d_n_library,
                            d_stats ? d_stats + 4 * c : nullptr, d_flags, st);
        if (rc) return rc;
    }
    return GRIDFF_OK;
}

}  // extern "C"
