/*
 * gridff.h — C-ABI of the B200-native GridFF hot path (arxiv 2508.15522).
 *
 * The library implements, as hand-written CUDA for sm_100a, the data-parallel path of the paper:
 *   substrate atoms + periodic cell + voxel size  ->  B-spline coefficient grids
 *   positions + per-atom channel factors          ->  E_i, F_i by tricubic B-splines    (Eq.1, L128-138 Eqs.5-6)
 *   N replicas + topology + integrator            ->  final states and energies
 *
 * Conventions
 *   - Units: Å, eV, e, amu, fs.  k_e = 14.3996454784 eV·Å/e²;  1 eV/(Å·amu) = 9.648533212e-3 Å/fs².
 *   - Every function returns 0 (GRIDFF_OK) or a negative error code; gridff_last_error() gives a thread-local
 *     message.  No exception crosses the ABI.
 *   - Pointers named d_* are DEVICE pointers, h_* / unprefixed array pointers are HOST pointers.
 *   - The library never allocates, frees or keeps caller memory beyond what is stated: device buffers
 *     (store, scratch, topology buffer, work buffers) are owned by the caller (e.g. torch tensors) and must stay
 *     alive while the handle that refers to them is in use.  Opaque handles are small host objects owned by the
 *     library and released by gridff_free_grid / gridff_free_molecule.
 *   - All device work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = default stream) and is
 *     asynchronous unless stated.  Host input arrays are consumed before the call returns.
 *   - Arrays are row-major, atom-major xyz.  Out-of-domain atoms are not an error (rules at gridff_eval);
 *     a replica that produces NaN sets bit 30 of its status flag, the call still returns 0.
 *   - There is no CPU fallback anywhere: without a CUDA device every compute entry point returns GRIDFF_ECUDA.
 */
#ifndef GRIDFF_H
#define GRIDFF_H
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GRIDFF_OK 0
#define GRIDFF_EINVAL (-1)        /* bad argument */
#define GRIDFF_EUNSUPPORTED (-2)  /* e.g. non-neutral substrate with a Coulomb channel, > 64 atoms per molecule */
#define GRIDFF_ESIZE (-3)         /* a caller buffer is too small */
#define GRIDFF_ECUDA (-4)         /* CUDA runtime error (message in gridff_last_error) */

const char* gridff_last_error(void);
int gridff_version(void);

/* ---------------------------------------------------------------------------------------------------------
 * Grid build  (steps a1-a4; Eqs. 2-4)
 * --------------------------------------------------------------------------------------------------------- */

typedef struct gridff_grid gridff_grid;

typedef enum { GRIDFF_CH_PAULI = 0, GRIDFF_CH_LONDON = 1, GRIDFF_CH_COULOMB = 2, GRIDFF_CH_ZERO = 3 } gridff_channel;

typedef enum {
    GRIDFF_LAYOUT_ZFAST = 0,  /* [x][y][z] nodes, z contiguous (the paper's order), x/y halo of 3 nodes */
    GRIDFF_LAYOUT_BRICK = 1,  /* 4x4x4-node bricks of 1 KB, bricks in [x][y][z] order, x/y halo                     */
    /* derived stores (gridff_grid_derive; gridff_eval only — SURVEY.md §8(f) row 3): */
    GRIDFF_LAYOUT_HALF = 2,   /* ZFAST with the 4 coefficients of a node rounded to fp16 (8 B per node), fp32 arithmetic */
    GRIDFF_LAYOUT_TRILINEAR = 3, /* the trilinear foil of PAPER.md:L118-120, L140: per node V and the three gradient components for
                                   each channel (4 x float4 = 64 B), each interpolated independently over the 8 cell corners   */
    /* derived fp32 stores for grids that do not fit the L2 (the HBM-bound gather): the same coefficients in
       2x2x2-node bricks of 128 B (one memory line), bricks in [x][y][z] order.  The 4x4x4 stencil of PAPER.md:L136 then touches
       whole lines only; the results are bit-identical to the z-fastest store's (variant 2). */
    GRIDFF_LAYOUT_MBRICK = 4,    /* one copy: a stencil touches 8 / 12 / 18 / 27 lines by the parity of its corner (15.6 on average; the
                                   z-fastest store: 22 partly used lines)                                                         */
    GRIDFF_LAYOUT_MBRICK2 = 5,   /* two copies, the second anchored one node further in x, y and z: the better aligned copy is read
                                   (8 or 12 lines, 11 on average), 2 x the memory                                                  */
    GRIDFF_LAYOUT_MBRICK8 = 6    /* eight copies, one per parity of the corner: EVERY stencil is exactly 8 whole lines = the 1024
                                   algorithmic bytes, 8 x the memory (sized for 180 GB of HBM: a 1 GB grid becomes 8.7 GB)        */
} gridff_layout;

typedef struct {
    double Lx, Ly;        /* periodic orthorhombic surface cell, Å                               */
    double z_ref;         /* z of the top substrate layer                                                               */
    double z_lo, z_hi;    /* grid z range above z_ref; node k sits at z_ref + z_lo + k*spacing                          */
    double spacing;       /* target voxel size: nx = round(Lx/spacing), hx = Lx/nx (same for y); nz = round((z_hi-z_lo)/spacing), hz = spacing */
    double alpha;         /* Morse alpha, 1/Å                                                         */
    double r_cut;         /* lateral images with |a| <= ceil(r_cut/Lx), |b| <= ceil(r_cut/Ly) are summed  */
    int n_channels;       /* 1..4; every node is stored as 4 floats (16 B), missing channels are zero                    */
    int channel[4];       /* gridff_channel per stored component                                                        */
    int layout;           /* gridff_layout                                                                              */
    int l2_persist;       /* 1: ask for an L2 access-policy window over the store on the streams that use the grid; honoured
                             only when the store fits the device's largest persisting carve-out (a window that cannot hold the
                             store costs the HBM-bound gathers 10-19 %: DESIGN.md §5) */
    int morse_window;     /* Morse sampling (a1): 0 = library's choice, 1 = always skip the terms below fp64 rounding of the node's
                             sum (the magnitude window), 2 = never (every image term is evaluated); same coefficients  */
} gridff_grid_desc;

/* nodes per axis, spacings and origin {0, 0, z_ref+z_lo} implied by a descriptor. */
int gridff_grid_dims(const gridff_grid_desc* desc, int dims[3], double h[3], double origin[3]);

/* Bytes the caller must provide for the coefficient store (kept for the life of the grid) and for the build
 * scratch (may be released once the stream has finished the build). */
int gridff_grid_bytes(const gridff_grid_desc* desc, int n_sub, size_t* store_bytes, size_t* scratch_bytes);

/* Sample the channels on the grid, prefilter them to interpolating cubic B-spline coefficients (cyclic in x,y;
 * not-a-knot in z) and write the interleaved fp32 store.
 *   sub_pos [n_sub][3], sub_e (sqrt(eps_j), eV^1/2), sub_R (Å), sub_q (e): HOST doubles; sub_q may be NULL without a
 *   Coulomb channel.  A Coulomb channel needs |sum q| < 1e-9 e (GRIDFF_EUNSUPPORTED otherwise) and z_ref at or above the
 *   topmost substrate atom (an adatom or a step included: z_ref is THEIR z; GRIDFF_EINVAL otherwise), so that the lowest
 *   grid plane lies at least z_lo > 0 above every atom — the Fourier sum is cut where exp(-|G| z_lo) < 1e-16.
 *   Sampling and prefilter run in fp64 on the device; the store is fp32.
 *   Synchronises the stream once (host -> device copy of the substrate from pageable memory).                    */
int gridff_build_grid(const gridff_grid_desc* desc, int n_sub,
                      const double* sub_pos, const double* sub_e, const double* sub_R, const double* sub_q,
                      void* d_store, size_t store_bytes, void* d_scratch, size_t scratch_bytes,
                      void* cuda_stream, gridff_grid** out);

/* Same, but the node samples are supplied by the caller (density-derived or imported potentials):
 * d_samples [nx][ny][nz][n_channels] fp32 on the device. */
int gridff_grid_from_samples(const gridff_grid_desc* desc, const float* d_samples,
                             void* d_store, size_t store_bytes, void* d_scratch, size_t scratch_bytes,
                             void* cuda_stream, gridff_grid** out);

/* Parity hook: write the stored coefficients in canonical order, d_coef [nx][ny][nz][n_channels] fp32. */
int gridff_grid_export(const gridff_grid* grid, float* d_coef, void* cuda_stream);

int gridff_grid_info(const gridff_grid* grid, int dims[3], double h[3], double origin[3], int* n_channels, int* layout);

/* Frees the handle only; d_store stays the caller's. */
int gridff_free_grid(gridff_grid* grid);

/* Derived stores for the interpolation trade study.  `parent` must be a ZFAST grid.
 *   GRIDFF_LAYOUT_HALF       every stored fp32 coefficient rounded to nearest-even fp16; same tricubic evaluation, fp32 accumulate.
 *   GRIDFF_LAYOUT_TRILINEAR  node values V_c = the parent spline at the node and G_c = its analytic gradient there (R20);
 *                            gridff_eval then returns E = sum_c coef_c lerp(V_c), F = -sum_c coef_c lerp(G_c) ("the force components
 *                            and energy were stored and interpolated independently", L120), cell and domain rules as for the spline.
 *   GRIDFF_LAYOUT_MBRICK / MBRICK2 / MBRICK8   the parent's fp32 coefficients re-laid in 2x2x2-node bricks, 1 / 2 / 8 copies (see
 *                            gridff_layout); needs nx + 3, ny + 3 <= 2047 and nz <= 1023; gridff_eval returns the parent's numbers bit for bit.
 * d_store (>= gridff_derive_bytes) stays the caller's; the handle is freed with gridff_free_grid.                          */
size_t gridff_derive_bytes(const gridff_grid* parent, int layout);
int gridff_grid_derive(const gridff_grid* parent, int layout, void* d_store, size_t store_bytes, void* cuda_stream, gridff_grid** out);

/* Per-atom channel factors of PAPER.md:L83-85 Eq. 4 with e_i = sqrt(eps_i):
 *   coef[i] = { e_i exp(2 alpha R_i), -2 e_i exp(alpha R_i), q_i, 0 }.   HOST arrays, computed on the host in fp64. */
int gridff_atom_coefs(double alpha, int n, const float* e, const float* R, const float* q, float* coef);

/* ---------------------------------------------------------------------------------------------------------
 * Interpolation  (step a5)
 * --------------------------------------------------------------------------------------------------------- */

/* E_i = sum_c coef[i][c] V_c(r_i),  F_i = -sum_c coef[i][c] grad V_c(r_i) for n points.
 *   d_pos [n][3] Å, d_coef [n][4], d_E [n] eV (may be NULL), d_F [n][3] eV/Å (may be NULL): device, fp32.
 *   x,y are wrapped into the cell.  z above the stored domain (node index >= nz-2): E = F = 0;
 *   z below node 1: the lowest cell's polynomial is continued.                                                 */
int gridff_eval(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef,
                float* d_E, float* d_F, void* cuda_stream);

/* Same with an explicit kernel variant (layout / gather study): 0 = library default, 1 = one thread per point
 * (64 independent 16-byte loads), 2 = warp-cooperative row gather, 3 = one 3-D TMA box (cp.async.bulk.tensor, 1 KB) per point into shared
 * memory (z-fastest fp32 stores only; GRIDFF_EUNSUPPORTED when the driver has no tensor-map entry point).  Variants 2 and 3 return
 * bit-identical results.  A brick-layout grid always uses its own kernel.  Micro-brick stores (GRIDFF_LAYOUT_MBRICK*): 0 / 2 = the
 * warp-cooperative gather over bricks, 3 = one 5-D TMA box {brick, 2, 2, 2, copy} per point (MBRICK8 only; the default there). */
int gridff_eval_variant(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef,
                        float* d_E, float* d_F, int variant, void* cuda_stream);

/* Same results as gridff_eval (bit for bit) for SCATTERED points on a z-fastest store that does not fit the L2 ("limited by global
 * memory access"): the points are first counting-sorted on the device by blocks of 4 x 4 x 8 cells (one atomic pass for count and rank, a scan,
 * a scatter of 32-byte point records), evaluated block by block, and the results gathered back to the points' own indices — neighbouring points
 * then share stencil lines in L1 / L2 as spatially sorted input does, without any extra copy of the grid.  d_work needs gridff_eval_binned_work_bytes(grid, n)
 * bytes (52 n + 4 per bin), 256-byte aligned; n < 2^32 - 16.  The order inside a bin depends on the atomics' order; the results do not. */
size_t gridff_eval_binned_work_bytes(const gridff_grid* grid, long long n);
int gridff_eval_binned(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef,
                       float* d_E, float* d_F, void* d_work, size_t work_bytes, void* cuda_stream);

/* gridff_eval_binned for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the
 * same passes and the same numbers, bit for bit, with the work space in a device array built into the library — GRIDFF_NOALLOC_SCRATCH_BYTES
 * (16 MiB) of every GPU that loads the library, held until the process exits.  The call allocates nothing: no cudaMalloc / cudaFree, no allocating
 * library routine; d_pos, d_coef, d_E, d_F are the caller's as in gridff_eval.  Limits: n <= GRIDFF_NOALLOC_MAX_POINTS (262,144) and
 * gridff_eval_binned_work_bytes(grid, n) <= gridff_eval_binned_noalloc_max_bytes() (52 bytes per point + 4 per block of 4 x 4 x 8 cells: at the full
 * point count that leaves 3.1 MB for the counters: grids up to 7.8e5 blocks = 1e8 cells, e.g. 512 x 512 x 256; larger grids take fewer points per call);
 * beyond either, GRIDFF_ESIZE with the numbers in gridff_last_error() and nothing launched.  ALL calls on one device share the one array, which keeps
 * the previous call's contents: the bin counters are cleared on the stream at the start of every call, everything else is written before it is read;
 * two calls that overlap on the GPU (different streams, no dependency between them) race on it — order them on one stream or with events. */
#define GRIDFF_NOALLOC_SCRATCH_BYTES (16u << 20)
#define GRIDFF_NOALLOC_MAX_POINTS (1 << 18)
size_t gridff_eval_binned_noalloc_max_bytes(void);
int gridff_eval_binned_noalloc(const gridff_grid* grid, long long n, const float* d_pos, const float* d_coef,
                               float* d_E, float* d_F, void* cuda_stream);

/* Same through HOST buffers: copies pos/coef to d_work, evaluates, copies E/F back, synchronises the stream.
 * d_work needs gridff_eval_work_bytes(n) bytes.  The work is pipelined in chunks of 2^22 points over two library-owned copy streams
 * and the caller's stream (upload of chunk c+1, kernel of chunk c and download of chunk c-1 overlap); the overlap needs pinned
 * host buffers, pageable ones are correct but serialise. */
size_t gridff_eval_work_bytes(long long n);
int gridff_eval_host(const gridff_grid* grid, long long n, const float* h_pos, const float* h_coef,
                     float* h_E, float* h_F, void* d_work, size_t work_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------------------
 * Fused replica step  (steps a5-a9)
 * --------------------------------------------------------------------------------------------------------- */

typedef struct {
    int n_atoms;                                   /* 1..64 */
    const float* mass;                             /* [n] amu */
    const float* coef;                             /* [n][4] channel factors (gridff_atom_coefs) */
    const float* q; const float* lj_e; const float* lj_R;   /* [n] e, sqrt(eps) eV^1/2, Å (R_ij = R_i + R_j) */
    int n_bonds;  const int* bond;  const float* bond_k_r0;      /* [.][2] i,j;       [.][2] k (eV/Å²), r0 (Å)      E = k/2 (r-r0)²        */
    int n_angles; const int* angle; const float* angle_k_t0;     /* [.][3] i,j,k (j centre); k (eV/rad²), theta0    E = k/2 (th-th0)²      */
    int n_tors;   const int* tors;  const float* tors_k_n_p0;    /* [.][4] i,j,k,l;   k (eV), n, phi0               E = k [1+cos(n phi-phi0)] */
    const unsigned char* excl;                     /* [n][n], 1 = pair excluded from LJ + Coulomb; NULL = all excluded */
    /* restart generator (used with integrator.restart = 1) */
    int n_rot; const int* rot_bond;                /* [.][2] rotatable bonds j0 -> j1 */
    const unsigned char* rot_mask;                 /* [.][n] 1 = atom turns with j1 */
    const float* ref_pos;                          /* [n][3] template conformation; required by integrator.restart = 1 (GRIDFF_EINVAL without it) */
} gridff_topology;                                 /* HOST arrays; copied by gridff_create_molecule */

typedef struct gridff_molecule gridff_molecule;

size_t gridff_molecule_bytes(const gridff_topology* topo);
/* Pack the topology into the caller's device buffer d_buf (>= gridff_molecule_bytes).  Synchronises the stream. */
int gridff_create_molecule(const gridff_topology* topo, void* d_buf, size_t buf_bytes, void* cuda_stream,
                           gridff_molecule** out);
int gridff_free_molecule(gridff_molecule* mol);

typedef struct {
    int kind;                 /* 0 velocity Verlet, 1 FIRE (ref 72), 2 Langevin dynamics (BAOAB, R18) */
    int n_steps;              /* steps per launch (FIRE: upper bound) */
    float dt;                 /* fs (FIRE: initial dt) */
    float f_tol;              /* FIRE stops when max_i |F_i| < f_tol, eV/Å */
    float dt_max, f_inc, f_dec, a_start, f_a; int n_min;    /* FIRE parameters; defaults 10 dt, 1.1, 0.5, 0.1, 0.99, 5 */
    float max_step;           /* FIRE: cap on the largest atomic displacement per step, Å; 0 = none */
    int restart;              /* FIRE: 0 stop when converged; 1 record the minimum and re-seed from Philox4x32-10(seed, replica, restart#) */
    unsigned long long seed;
    float z_ref, place_z_lo, place_z_hi, place_z_min, clash;   /* restart placement (3, 6, 2 Å above z_ref; clash factor 0.4) */
    int variant;              /* kernel variant: 0 = default (library's choice), 1 = one thread per atom gathers its 64 nodes, 2 = warp-cooperative row gather every step,
                                 3 = 2 + the folded stencils cached in shared memory and re-gathered only when an atom changes cell.
                                 Molecules of 33-64 atoms: variants 1, 2 put two atoms on a lane; variant 3 puts the replica on a pair of warps
                                 (one atom per lane); variant 4 = variant 3's stencil cache on ONE warp with two atoms per lane (the older kernel, kept
                                 for the design comparison; for <= 32 atoms it is variant 3); variant 5 = variant 3 with the pair loop of molecules of
                                 <= 32 atoms as a full shell with a warp-uniform partner instead of the half shell on a ring (design comparison: slower;
                                 for 33-64 atoms it is variant 3).  All variants compute the same forces; they differ in rounding order only. */
    /* SURVEY.md §8(f) rows 1-2 (0 / unset = off) */
    float temperature;        /* K, kind 2 */
    float gamma;              /* friction 1/fs, kind 2: per step  B: v += dt/2 a;  A: x += dt/2 v;  O: v = c1 v + c2 sqrt(kT/m) xi;  A;  F(x);  B,
                                 c1 = exp(-gamma dt), c2 = sqrt(1 - c1^2); xi = Box-Muller normals from Philox4x32-10 with counter
                                 (step0 + step, atom, 'Lang', replica), key = seed, u = ((x >> 9) + 1/2) 2^-23 */
    unsigned step0;           /* kind 2: index of this launch's first step in the noise stream (1 x N == k x N/k launches) */
    int n_scan;               /* gridff_run_scan only: number of scan points */
    unsigned long long fixed_mask;   /* bit i: atom i is held (the restrained atom of PAPER.md:L178, L184): it feels no force, has no velocity and takes
                                        no part in the convergence test; only a scan moves it */
    float scan_dx[3];         /* gridff_run_scan: displacement of the held atoms per scan point, Å */
} gridff_integrator;

/* Advance n_rep independent replicas of one molecule for integ->n_steps steps in ONE launch sequence without host
 * round-trips: per step, grid forces by interpolation + intramolecular terms + integrator.
 *   d_pos, d_vel   [n_rep][n][3]  in/out, fp32
 *   d_fire         [n_rep][4]     in/out FIRE scalars {dt, a, steps since P<=0, restarts done}; dt <= 0 = fresh.  May be NULL (VV, or fresh FIRE)
 *   d_energy       [n_rep][8]     out: grid ch0, ch1, ch2 (+ ch3 when the grid has a 4th channel), bond, angle, torsion, non-bonded, kinetic (eV)
 *                                 at the final state: the first 7 sum to the potential whose gradient the forces are.  May be NULL
 *   d_status       [n_rep][2]     out: {steps taken, converged flag (restart=0) or minima recorded (restart=1)}.  May be NULL
 *   d_minima       [cap][4+3n]    out, restart=1: {replica, restart#, steps, E_total, positions}; d_n_minima (1 int, device, caller zeroes it)
 *                                 counts records (may exceed cap; excess dropped).  May be NULL
 * `grid` may be NULL (gas-phase molecule).                                                                          */
int gridff_run_replicas(const gridff_grid* grid, const gridff_molecule* mol, const gridff_integrator* integ, int n_rep,
                        float* d_pos, float* d_vel, float* d_fire, float* d_energy, int* d_status,
                        float* d_minima, int minima_cap, int* d_n_minima, void* cuda_stream);

/* Driven scan ("restrained the position of one atom ... displaced the z-component ... by 0.1 Å ... let the position of
 * the other atoms relax"; L184 dragging): for each of integ->n_scan points, every replica moves its held atoms (fixed_mask) by
 * scan_dx, then relaxes the others with FIRE (fresh scalars, v = 0) until max_i |F_i| < f_tol or n_steps iterations, all inside
 * one launch.  integ->kind must be 1, restart 0.
 *   d_scan  [n_rep][n_scan][4]  out: {E_total (eV), FIRE iterations, converged 0/1, max_i |F_i| over the free atoms} per point
 *   d_pos / d_vel in/out as in gridff_run_replicas; d_energy / d_status (may be NULL) describe the last point
 *   (status = {total iterations, points converged}).                                                                 */
int gridff_run_scan(const gridff_grid* grid, const gridff_molecule* mol, const gridff_integrator* integ, int n_rep,
                    float* d_pos, float* d_vel, float* d_energy, int* d_status, float* d_scan, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------------------
 * Minima hopping with an on-device unique-structure filter
 * --------------------------------------------------------------------------------------------------------- */
typedef struct {
    int n_cycles;                       /* hops per call */
    int cycle0;                         /* index of this call's first cycle (noise stream position = (cycle0 + c) * md_steps; record tag) */
    int md_steps; float md_dt;          /* perturbation: Langevin dynamics from rest (1000 steps ...) */
    float temperature, gamma;           /* ... at 300 K; friction 1/fs */
    int relax_steps; float relax_dt;    /* FIRE relaxation from rest: at most relax_steps iterations */
    float f_tol, dt_max, max_step;      /* FIRE: converged when max_i |F_i| < f_tol; dt_max 0 = 10 relax_dt; max_step 0 = none */
    float e_tol, rmsd_tol;              /* same structure: |dE| < e_tol (1e-3 eV) and RMSD < rmsd_tol (0.1 Å) after removing the
                                           whole cell translation nearest to the mean displacement (R16) */
    unsigned long long seed;
    unsigned long long fixed_mask;
} gridff_hopping;

/* n_cycles times, without host round-trips: Langevin -> FIRE -> filter.  Every replica continues from its relaxed state.
 * The filter is the sequential greedy one in replica order: a converged replica whose structure matches no library record
 * (older, or appended earlier in the same cycle) is appended.
 *   d_pos      [n_rep][n][3]      in/out
 *   d_library  [cap][4+3n]        in/out records {replica, cycle, FIRE iterations, E_total, positions}
 *   d_n_library 1 int (device)    in/out number of records stored (<= cap)
 *   d_stats    [n_cycles][4] int  out (may be NULL): converged candidates, new records, dropped because the library was full, library size after
 *   d_work     gridff_hopping_work_bytes(mol, n_rep) bytes, 256-byte aligned                                           */
size_t gridff_hopping_work_bytes(const gridff_molecule* mol, int n_rep);
int gridff_minima_hopping(const gridff_grid* grid, const gridff_molecule* mol, const gridff_hopping* hop, int n_rep,
                          float* d_pos, float* d_library, int cap, int* d_n_library, int* d_stats,
                          void* d_work, size_t work_bytes, void* cuda_stream);
/* The filter alone (parity hook and building block): candidates = replicas with d_ok[r] != 0, energies d_E [n_rep], positions d_pos. */
int gridff_unique_filter(const gridff_grid* grid, const gridff_molecule* mol, int n_rep, const float* d_pos, const float* d_E,
                         const int* d_steps /*may be NULL*/, const int* d_ok, float e_tol, float rmsd_tol, int tag,
                         float* d_library, int cap, int* d_n_library, int* d_stats4 /*may be NULL*/,
                         int* d_flags /*[n_rep] scratch*/, void* cuda_stream);

/* Same through HOST buffers (pinned or pageable): copies pos/vel(/fire) to d_work, runs, copies pos/vel/fire/energy/
 * status back, synchronises the stream.  d_work needs gridff_run_work_bytes(mol, n_rep) bytes. */
size_t gridff_run_work_bytes(const gridff_molecule* mol, int n_rep);
int gridff_run_replicas_host(const gridff_grid* grid, const gridff_molecule* mol, const gridff_integrator* integ, int n_rep,
                             float* h_pos, float* h_vel, float* h_fire, float* h_energy, int* h_status,
                             void* d_work, size_t work_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------------------
 * Measurement helpers (roofline denominators; not part of the method)
 * --------------------------------------------------------------------------------------------------------- */

/* Read `bytes` of d_buf `iters` times with coalesced 16-byte loads (mode 0), with the 64-byte-row gather pattern of
 * the z-fastest stencil at random 16-byte offsets (mode 1), or as whole aligned 128-byte lines at random positions, the
 * micro-brick stencil's granule (mode 2); one launch.  d_sink: >= 4 bytes.  Used to measure L2 / HBM read bandwidth. */
int gridff_probe_read(const void* d_buf, size_t bytes, int iters, int mode, void* d_sink, void* cuda_stream);

/* Number of kernel launches the library has enqueued since it was loaded (for bench.py's gpu_launches). */
long long gridff_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif
