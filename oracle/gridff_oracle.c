/*
 * gridff_oracle.c — fp64 CPU oracle for the GridFF hot path (arxiv 2508.15522).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2508_15522_b200/csrc and is
 * never tuned: plain loops in the paper's order, fp64 throughout, `omp parallel for`
 * over independent units (grid nodes, points, replicas) only.
 *
 * Citations are "PAPER.md:Lnn" (+ equation) and "DESIGN.md Rn" for the readings taken
 * where the paper is silent or garbled.
 *
 * Pins (tests/test_oracle_*.py, `-m "not gpu"`):
 *   weights          partition of unity, Eq. 6 at the four offsets            pinned
 *   prefilter        scipy CubicSpline (periodic / not-a-knot), cubics        pinned
 *   interpolation    FD gradient, periodicity, polynomial reproduction        pinned
 *   Morse sums       single-atom closed form, sub-cell periodicity            pinned
 *   Coulomb          scipy-erfc 2D Ewald, direct image sum, antisymmetry,
 *                    decay constant, Laplace                                  pinned
 *   force field      textbook 2/3/4-atom cases, FD, zero net force/torque     pinned
 *   velocity Verlet  harmonic-diatomic closed forms, reversibility            pinned
 *   FIRE             quadratic-bowl minimum, launch-split invariance;         pinned
 *                    time-step schedule and mixing order: closed forms on a constant force
 *   Philox4x32-10    brute-force big-integer restatement in Python            pinned
 *   restart geometry bond lengths/angles invariant under torsion moves        pinned
 *   Langevin (BAOAB) gamma = 0 -> velocity Verlet, exact OU decay and equilibrium
 *                    variance of free particles, equipartition, normal moments  pinned
 *   held atoms/scan  one-atom scan = the interpolated potential itself;
 *                    held atoms never move; relaxed E <= unrelaxed E            pinned
 *   basin assignment parity unpinned: WHICH minimum a given start relaxes to has no external reference (only
 *                    oracle-vs-GPU agreement); that the end state IS a minimum (max |F_i| < f_tol, E <= E_start) and the
 *                    same-structure criterion itself (gridff_oracle.py same_structure) are pinned
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_KE 14.3996454784        /* eV·Å/e²   (DESIGN.md units) */
#define ORC_ACC 9.648533212e-3      /* 1 eV/(Å·amu) in Å/fs² */
#define ORC_PI 3.14159265358979323846

/* ------------------------------------------------------------------ */
/* 1. Cubic B-spline basis and per-cell weights                        */
/* ------------------------------------------------------------------ */

/* B(t), Eq. 6 */
double orc_bspline_basis(double t) {
    double a = fabs(t);
    if (a < 1.0) return 2.0 / 3.0 - a * a + 0.5 * a * a * a;
    if (a < 2.0) { double c = 2.0 - a; return c * c * c / 6.0; }
    return 0.0;
}

/* Weights of the four coefficients b_{i-1..i+2} for a point at fraction t in cell i
 * (Eq. 5 with the index reading DESIGN.md R1): w_j = B(t + 1 - j), j=0..3,
 * written out as polynomials, and their derivatives with respect to t. */
void orc_bspline_weights(double t, double w[4], double dw[4]) {
    double t2 = t * t, t3 = t2 * t, m = 1.0 - t;
    w[0] = m * m * m / 6.0;
    w[1] = (3.0 * t3 - 6.0 * t2 + 4.0) / 6.0;
    w[2] = (-3.0 * t3 + 3.0 * t2 + 3.0 * t + 1.0) / 6.0;
    w[3] = t3 / 6.0;
    dw[0] = -m * m / 2.0;
    dw[1] = (3.0 * t2 - 4.0 * t) / 2.0;
    dw[2] = (-3.0 * t2 + 2.0 * t + 1.0) / 2.0;
    dw[3] = t2 / 2.0;
}

/* ------------------------------------------------------------------ */
/* 2. Un-approximated substrate potentials at arbitrary points         */
/* ------------------------------------------------------------------ */

static double fold(double x, double L) { return x - floor(x / L) * L; }

/* Morse channels, Eq. 4:
 *   V^P(r) = sum_j e_j exp(-2 alpha (|r - r_j - T| - R_j)),  V^L same with alpha,
 * over substrate atoms j and lateral images T = (a Lx, b Ly, 0), |a|<=Nx, |b|<=Ny, with the
 * point and the atoms folded into [0,L) first (R10).  e_j = sqrt(eps_j) (R9).
 * grad* may be NULL; otherwise [n][3] = dV/dr. */
void orc_morse_points(int n_sub, const double* sub_pos, const double* sub_e, const double* sub_R,
                      double alpha, double Lx, double Ly, int Nx, int Ny,
                      long n, const double* pts, double* VP, double* VL, double* gradP, double* gradL) {
#pragma omp parallel for schedule(static)
    for (long p = 0; p < n; ++p) {
        double x = fold(pts[3 * p], Lx), y = fold(pts[3 * p + 1], Ly), z = pts[3 * p + 2];
        double vp = 0, vl = 0, gp[3] = {0, 0, 0}, gl[3] = {0, 0, 0};
        for (int j = 0; j < n_sub; ++j) {
            double xj = fold(sub_pos[3 * j], Lx), yj = fold(sub_pos[3 * j + 1], Ly), zj = sub_pos[3 * j + 2];
            for (int a = -Nx; a <= Nx; ++a)
                for (int b = -Ny; b <= Ny; ++b) {
                    double dx = x - xj - a * Lx, dy = y - yj - b * Ly, dz = z - zj;
                    double d = sqrt(dx * dx + dy * dy + dz * dz);
                    double tp = sub_e[j] * exp(-2.0 * alpha * (d - sub_R[j]));
                    double tl = sub_e[j] * exp(-alpha * (d - sub_R[j]));
                    vp += tp; vl += tl;
                    double cp = -2.0 * alpha * tp / d, cl = -alpha * tl / d;
                    gp[0] += cp * dx; gp[1] += cp * dy; gp[2] += cp * dz;
                    gl[0] += cl * dx; gl[1] += cl * dy; gl[2] += cl * dz;
                }
        }
        VP[p] = vp; VL[p] = vl;
        if (gradP) { gradP[3 * p] = gp[0]; gradP[3 * p + 1] = gp[1]; gradP[3 * p + 2] = gp[2]; }
        if (gradL) { gradL[3 * p] = gl[0]; gradL[3 * p + 1] = gl[1]; gradL[3 * p + 2] = gl[2]; }
    }
}

/* Coulomb channel: exact potential of a neutral, laterally periodic slab above its top layer
 * (Eq. 2 summed over the 2D lattice; R11):
 *   V^C(rho,z) = k_e (2 pi/A) [ sum_{G!=0} S(G)/|G| e^{iG.rho} e^{-|G| z} + sum_j Q_j z_j ],
 *   S(G) = sum_j Q_j e^{-iG.rho_j} e^{|G| z_j},   G = 2 pi (m/Lx, n/Ly),  A = Lx Ly.
 * z and z_j are taken relative to z_top = max_j z_j so every exponent is <= 0; terms with
 * |G| (z - z_top) > g_cut (37: < 1e-16) are dropped.  The +G/-G pair is added as 2 Re[...].
 * Valid for z > z_top only.  Structure factors with |S| < 1e-14 sum|Q| are exact zeros of
 * a crystalline slab and are skipped.  Returns V in eV/e; grad may be NULL.             */
typedef struct { double gx, gy, g, sre, sim; } orc_gvec;

static int build_gvecs(int n_sub, const double* sub_pos, const double* sub_q, double Lx, double Ly,
                       double gmax, double* z_top_out, double* qz_out, orc_gvec** out) {
    double z_top = -1e300, qabs = 0, qz = 0;
    for (int j = 0; j < n_sub; ++j) { if (sub_pos[3 * j + 2] > z_top) z_top = sub_pos[3 * j + 2]; qabs += fabs(sub_q[j]); }
    for (int j = 0; j < n_sub; ++j) qz += sub_q[j] * (sub_pos[3 * j + 2] - z_top);
    int M = (int)floor(gmax * Lx / (2 * ORC_PI)), N = (int)floor(gmax * Ly / (2 * ORC_PI));
    long cap = (long)(2 * M + 1) * (N + 1);
    orc_gvec* g = (orc_gvec*)malloc(sizeof(orc_gvec) * (size_t)(cap > 0 ? cap : 1));
    int cnt = 0;
    /* half plane: n > 0, or n == 0 and m > 0 */
    for (int nn = 0; nn <= N; ++nn)
        for (int m = -M; m <= M; ++m) {
            if (nn == 0 && m <= 0) continue;
            double gx = 2 * ORC_PI * m / Lx, gy = 2 * ORC_PI * nn / Ly, gg = sqrt(gx * gx + gy * gy);
            if (gg > gmax) continue;
            double sre = 0, sim = 0;
            for (int j = 0; j < n_sub; ++j) {
                double ph = gx * sub_pos[3 * j] + gy * sub_pos[3 * j + 1];
                double w = sub_q[j] * exp(gg * (sub_pos[3 * j + 2] - z_top));
                sre += w * cos(ph); sim -= w * sin(ph);
            }
            if (sqrt(sre * sre + sim * sim) < 1e-14 * qabs) continue;
            g[cnt].gx = gx; g[cnt].gy = gy; g[cnt].g = gg; g[cnt].sre = sre; g[cnt].sim = sim; ++cnt;
        }
    *z_top_out = z_top; *qz_out = qz; *out = g;
    return cnt;
}

void orc_coulomb_points(int n_sub, const double* sub_pos, const double* sub_q, double Lx, double Ly,
                        double g_cut, double z_min_above_top,
                        long n, const double* pts, double* VC, double* gradC) {
    double z_top, qz; orc_gvec* g;
    int ng = build_gvecs(n_sub, sub_pos, sub_q, Lx, Ly, g_cut / z_min_above_top, &z_top, &qz, &g);
    double pref = ORC_KE * 2 * ORC_PI / (Lx * Ly);
#pragma omp parallel for schedule(dynamic, 64)
    for (long p = 0; p < n; ++p) {
        double x = pts[3 * p], y = pts[3 * p + 1], z = pts[3 * p + 2] - z_top;
        double v = qz, gx = 0, gy = 0, gz = 0;
        for (int k = 0; k < ng; ++k) {
            double a = g[k].g * z;
            if (a > g_cut) continue;
            double ph = g[k].gx * x + g[k].gy * y, c = cos(ph), s = sin(ph);
            double damp = exp(-a) / g[k].g;
            double re = 2.0 * (g[k].sre * c - g[k].sim * s) * damp;   /* 2 Re[S e^{i ph}] e^{-gz}/g */
            double im = 2.0 * (g[k].sre * s + g[k].sim * c) * damp;   /* 2 Im[...] */
            v += re;
            gx -= g[k].gx * im; gy -= g[k].gy * im; gz -= g[k].g * re;
        }
        VC[p] = pref * v;
        if (gradC) { gradC[3 * p] = pref * gx; gradC[3 * p + 1] = pref * gy; gradC[3 * p + 2] = pref * gz; }
    }
    free(g);
}

/* ------------------------------------------------------------------ */
/* 3. Grid sampling (steps a1, a2) and prefilter (a3)                  */
/* ------------------------------------------------------------------ */

/* channel kinds: 0 Pauli, 1 London, 2 Coulomb, 3 zero */
/* samples[ix][iy][iz][c] at r = (ix hx, iy hy, z0 + iz hz)  (R7) */
void orc_sample_grid(int n_sub, const double* sub_pos, const double* sub_e, const double* sub_R, const double* sub_q,
                     double alpha, double Lx, double Ly, int Nx, int Ny, double g_cut,
                     int nx, int ny, int nz, double z0, double hz, int nch, const int* kinds, double* samples) {
    long n = (long)nx * ny * nz;
    double hx = Lx / nx, hy = Ly / ny;
    double* pts = (double*)malloc(sizeof(double) * 3 * (size_t)n);
    for (int ix = 0; ix < nx; ++ix) for (int iy = 0; iy < ny; ++iy) for (int iz = 0; iz < nz; ++iz) {
        long p = ((long)ix * ny + iy) * nz + iz;
        pts[3 * p] = ix * hx; pts[3 * p + 1] = iy * hy; pts[3 * p + 2] = z0 + iz * hz;
    }
    double* vp = (double*)malloc(sizeof(double) * (size_t)n);
    double* vl = (double*)malloc(sizeof(double) * (size_t)n);
    double* vc = (double*)malloc(sizeof(double) * (size_t)n);
    int need_m = 0, need_c = 0;
    for (int c = 0; c < nch; ++c) { if (kinds[c] == 0 || kinds[c] == 1) need_m = 1; if (kinds[c] == 2) need_c = 1; }
    if (need_m) orc_morse_points(n_sub, sub_pos, sub_e, sub_R, alpha, Lx, Ly, Nx, Ny, n, pts, vp, vl, NULL, NULL);
    if (need_c) {
        double z_top = -1e300;
        for (int j = 0; j < n_sub; ++j) if (sub_pos[3 * j + 2] > z_top) z_top = sub_pos[3 * j + 2];
        orc_coulomb_points(n_sub, sub_pos, sub_q, Lx, Ly, g_cut, z0 - z_top, n, pts, vc, NULL);
    }
    for (long p = 0; p < n; ++p) for (int c = 0; c < nch; ++c) {
        double v = 0;
        if (kinds[c] == 0) v = vp[p]; else if (kinds[c] == 1) v = vl[p]; else if (kinds[c] == 2) v = vc[p];
        samples[p * nch + c] = v;
    }
    free(pts); free(vp); free(vl); free(vc);
}

/* Dense inverse by Gauss-Jordan with partial pivoting (n <= a few hundred). */
static void dense_inverse(int n, double* A, double* Ai) {
    for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) Ai[i * n + j] = (i == j);
    for (int c = 0; c < n; ++c) {
        int piv = c; double best = fabs(A[c * n + c]);
        for (int r = c + 1; r < n; ++r) if (fabs(A[r * n + c]) > best) { best = fabs(A[r * n + c]); piv = r; }
        if (piv != c) for (int j = 0; j < n; ++j) {
            double t = A[c * n + j]; A[c * n + j] = A[piv * n + j]; A[piv * n + j] = t;
            t = Ai[c * n + j]; Ai[c * n + j] = Ai[piv * n + j]; Ai[piv * n + j] = t;
        }
        double d = 1.0 / A[c * n + c];
        for (int j = 0; j < n; ++j) { A[c * n + j] *= d; Ai[c * n + j] *= d; }
        for (int r = 0; r < n; ++r) if (r != c) {
            double f = A[r * n + c];
            if (f != 0.0) for (int j = 0; j < n; ++j) { A[r * n + j] -= f * A[c * n + j]; Ai[r * n + j] -= f * Ai[c * n + j]; }
        }
    }
}

/* Collocation matrix of the interpolating cubic B-spline on n nodes ("fitted such
 * that the interpolated potential reproduces the reference values at grid nodes"; R2-R4):
 * interior rows (1,4,1)/6; periodic: indices mod n; otherwise not-a-knot end rows
 * (8,-5,4,-1)/6 from the virtual coefficient b_{-1} = 4 b_0 - 6 b_1 + 4 b_2 - b_3.          */
void orc_collocation_matrix(int n, int periodic, double* A) {
    memset(A, 0, sizeof(double) * (size_t)n * n);
    for (int k = 0; k < n; ++k) {
        if (periodic) {
            A[k * n + (k + n - 1) % n] += 1.0 / 6; A[k * n + k] += 4.0 / 6; A[k * n + (k + 1) % n] += 1.0 / 6;
        } else if (k == 0) {
            A[0] = 8.0 / 6; A[1] = -5.0 / 6; A[2] = 4.0 / 6; A[3] = -1.0 / 6;
        } else if (k == n - 1) {
            A[k * n + n - 1] = 8.0 / 6; A[k * n + n - 2] = -5.0 / 6; A[k * n + n - 3] = 4.0 / 6; A[k * n + n - 4] = -1.0 / 6;
        } else {
            A[k * n + k - 1] = 1.0 / 6; A[k * n + k] = 4.0 / 6; A[k * n + k + 1] = 1.0 / 6;
        }
    }
}

/* samples [nx][ny][nz][nch] -> coefficients, in place; axis by axis x, y, z.
 * periodic[3]: 1 cyclic, 0 not-a-knot (GridFF: {1,1,0}). */
void orc_prefilter(int nx, int ny, int nz, int nch, const int* periodic, double* data) {
    int dims[3] = {nx, ny, nz};
    long strides[3] = {(long)ny * nz * nch, (long)nz * nch, (long)nch};
    for (int ax = 0; ax < 3; ++ax) {
        int n = dims[ax];
        double* A = (double*)malloc(sizeof(double) * (size_t)n * n);
        double* Ai = (double*)malloc(sizeof(double) * (size_t)n * n);
        orc_collocation_matrix(n, periodic[ax], A);
        dense_inverse(n, A, Ai);
        int a1 = (ax + 1) % 3, a2 = (ax + 2) % 3;
        long nlines = (long)dims[a1] * dims[a2] * nch;
#pragma omp parallel
        {
            double* f = (double*)malloc(sizeof(double) * (size_t)n);
#pragma omp for schedule(static)
            for (long l = 0; l < nlines; ++l) {
                int c = (int)(l % nch); long r = l / nch;
                int i2 = (int)(r % dims[a2]); int i1 = (int)(r / dims[a2]);
                long base = i1 * strides[a1] + i2 * strides[a2] + c;
                for (int k = 0; k < n; ++k) f[k] = data[base + k * strides[ax]];
                for (int k = 0; k < n; ++k) {
                    double s = 0;
                    for (int j = 0; j < n; ++j) s += Ai[k * n + j] * f[j];
                    data[base + k * strides[ax]] = s;
                }
            }
            free(f);
        }
        free(A); free(Ai);
    }
}

/* ------------------------------------------------------------------ */
/* 4. Tricubic interpolation with analytic gradient (step a5)          */
/* ------------------------------------------------------------------ */

typedef struct {
    int nx, ny, nz, nch;
    double Lx, Ly, hz, z0;      /* z0 = z of node iz = 0 */
    int periodic_xy;            /* 1: GridFF (wrap x,y).  0: all three axes non-periodic (test mode) */
    const double* coef;         /* [nx][ny][nz][nch] */
} orc_grid;

/* One point.  V[c], dV[c][3] per channel.  Returns 0 if the point is above the grid (V=dV=0).
 * PAPER.md:L128-136 (Eq. 5, tensor product over the 4x4x4 block), R5, R6. */
static int interp_point(const orc_grid* g, const double r[3], double* V, double* dV) {
    int nch = g->nch;
    for (int c = 0; c < nch; ++c) { V[c] = 0; dV[3 * c] = dV[3 * c + 1] = dV[3 * c + 2] = 0; }
    double hx = g->Lx / g->nx, hy = g->Ly / g->ny, hz = g->hz;
    double ux, uy, uz = (r[2] - g->z0) / hz;
    int ix, iy, iz;
    if (g->periodic_xy) {
        ux = (r[0] / g->Lx - floor(r[0] / g->Lx)) * g->nx;
        uy = (r[1] / g->Ly - floor(r[1] / g->Ly)) * g->ny;
        ix = (int)floor(ux); iy = (int)floor(uy);
        if (ix >= g->nx) ix = g->nx - 1;           /* ux == nx can only arise from rounding */
        if (iy >= g->ny) iy = g->ny - 1;
    } else {
        ux = r[0] / hx; uy = r[1] / hy;
        ix = (int)floor(ux); iy = (int)floor(uy);
        if (ix < 1) ix = 1;
        if (ix > g->nx - 3) ix = g->nx - 3;
        if (iy < 1) iy = 1;
        if (iy > g->ny - 3) iy = g->ny - 3;
    }
    if (uz >= (double)(g->nz - 2)) return 0;        /* above the stored domain: E = F = 0 */
    iz = (int)floor(uz);
    if (iz < 1) iz = 1;                             /* below: lowest cell's polynomial, t < 0 */
    if (iz > g->nz - 3) iz = g->nz - 3;
    double wx[4], wy[4], wz[4], dwx[4], dwy[4], dwz[4];
    orc_bspline_weights(ux - ix, wx, dwx);
    orc_bspline_weights(uy - iy, wy, dwy);
    orc_bspline_weights(uz - iz, wz, dwz);
    for (int a = 0; a < 4; ++a) {
        int jx = ix - 1 + a; if (g->periodic_xy) jx = ((jx % g->nx) + g->nx) % g->nx;
        for (int b = 0; b < 4; ++b) {
            int jy = iy - 1 + b; if (g->periodic_xy) jy = ((jy % g->ny) + g->ny) % g->ny;
            for (int k = 0; k < 4; ++k) {
                int jz = iz - 1 + k;
                const double* bc = g->coef + (((long)jx * g->ny + jy) * g->nz + jz) * nch;
                double w = wx[a] * wy[b] * wz[k];
                double gxw = dwx[a] * wy[b] * wz[k] / hx;
                double gyw = wx[a] * dwy[b] * wz[k] / hy;
                double gzw = wx[a] * wy[b] * dwz[k] / hz;
                for (int c = 0; c < nch; ++c) {
                    V[c] += w * bc[c];
                    dV[3 * c] += gxw * bc[c]; dV[3 * c + 1] += gyw * bc[c]; dV[3 * c + 2] += gzw * bc[c];
                }
            }
        }
    }
    return 1;
}

/* E_i = sum_c coef_ic V_c(r_i), F_i = -sum_c coef_ic grad V_c  (Eq. 1).
 * Vc_out (optional) [n][nch] raw channel values; dVc_out (optional) [n][nch][3]. */
void orc_interp(const orc_grid* g, long n, const double* pos, const double* coef /*[n][4]*/,
                double* E, double* F, double* Vc_out, double* dVc_out) {
#pragma omp parallel for schedule(static)
    for (long p = 0; p < n; ++p) {
        double V[4], dV[12];
        interp_point(g, pos + 3 * p, V, dV);
        double e = 0, f[3] = {0, 0, 0};
        for (int c = 0; c < g->nch; ++c) {
            double k = coef[4 * p + c];
            e += k * V[c];
            f[0] -= k * dV[3 * c]; f[1] -= k * dV[3 * c + 1]; f[2] -= k * dV[3 * c + 2];
            if (Vc_out) Vc_out[p * g->nch + c] = V[c];
            if (dVc_out) for (int d = 0; d < 3; ++d) dVc_out[(p * g->nch + c) * 3 + d] = dV[3 * c + d];
        }
        if (E) E[p] = e;
        if (F) { F[3 * p] = f[0]; F[3 * p + 1] = f[1]; F[3 * p + 2] = f[2]; }
    }
}

/* Per-atom channel factors, Eq. 4 with e = sqrt(eps) (R9):
 * P_i = e_i exp(2 alpha R_i), L_i = -2 e_i exp(alpha R_i), Q_i = q_i, 0. */
void orc_atom_coefs(int n, const double* e, const double* R, const double* q, double alpha, double* coef) {
    for (int i = 0; i < n; ++i) {
        coef[4 * i] = e[i] * exp(2.0 * alpha * R[i]);
        coef[4 * i + 1] = -2.0 * e[i] * exp(alpha * R[i]);
        coef[4 * i + 2] = q[i];
        coef[4 * i + 3] = 0.0;
    }
}

/* ------------------------------------------------------------------ */
/* 5. Intramolecular force field (step a6; R12)              */
/* ------------------------------------------------------------------ */

typedef struct {
    int n_atoms;
    const double* mass;        /* amu */
    const double* coef;        /* [n][4] channel factors */
    const double* q;           /* e */
    const double* lj_e;        /* sqrt(eps), eV^(1/2) */
    const double* lj_R;        /* Å; R_ij = R_i + R_j */
    int n_bonds;  const int* bond;  const double* bond_k_r0;    /* [.][2] idx, [.][2] k, r0 */
    int n_angles; const int* angle; const double* angle_k_t0;   /* [.][3] i,j(center),k; k, theta0 */
    int n_tors;   const int* tors;  const double* tors_k_n_p0;  /* [.][4]; k, n, phi0 */
    const unsigned char* excl; /* [n][n], 1 = pair excluded from the non-bonded sum */
    /* restart generator (R17) */
    int n_rot; const int* rot_bond /*[.][2]*/; const unsigned char* rot_mask /*[.][n] atoms that move*/;
    const double* ref_pos;     /* [n][3] template conformation */
} orc_topology;

static void cross(const double a[3], const double b[3], double c[3]) {
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}
static double dot(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* Adds forces into F[n][3]; E4 = {bond, angle, torsion, non-bonded}. */
void orc_intramolecular(const orc_topology* T, const double* pos, double* F, double* E4) {
    int n = T->n_atoms;
    double eb = 0, ea = 0, et = 0, en = 0;
    /* bonds: E = 1/2 k (r - r0)^2 */
    for (int b = 0; b < T->n_bonds; ++b) {
        int i = T->bond[2 * b], j = T->bond[2 * b + 1];
        double k = T->bond_k_r0[2 * b], r0 = T->bond_k_r0[2 * b + 1];
        double d[3] = {pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1], pos[3 * i + 2] - pos[3 * j + 2]};
        double r = sqrt(dot(d, d));
        eb += 0.5 * k * (r - r0) * (r - r0);
        double s = -k * (r - r0) / r;
        for (int c = 0; c < 3; ++c) { F[3 * i + c] += s * d[c]; F[3 * j + c] -= s * d[c]; }
    }
    /* angles: E = 1/2 k (theta - theta0)^2, theta = atan2(|a x b|, a.b), a = r_i - r_j, b = r_k - r_j */
    for (int t = 0; t < T->n_angles; ++t) {
        int i = T->angle[3 * t], j = T->angle[3 * t + 1], k = T->angle[3 * t + 2];
        double kk = T->angle_k_t0[2 * t], t0 = T->angle_k_t0[2 * t + 1];
        double a[3], b[3], nn[3], an[3], bn[3];
        for (int c = 0; c < 3; ++c) { a[c] = pos[3 * i + c] - pos[3 * j + c]; b[c] = pos[3 * k + c] - pos[3 * j + c]; }
        cross(a, b, nn);
        double nl = sqrt(dot(nn, nn));
        double th = atan2(nl, dot(a, b));
        ea += 0.5 * kk * (th - t0) * (th - t0);
        double dEdth = kk * (th - t0);
        cross(a, nn, an); cross(b, nn, bn);
        double ca = dEdth / (dot(a, a) * nl), cb = dEdth / (dot(b, b) * nl);
        for (int c = 0; c < 3; ++c) {
            double fi = -ca * an[c];       /* -dE/dth * dth/da,  dth/da = (a x n)/(|a|^2 |n|) */
            double fk = cb * bn[c];        /*  dth/db = -(b x n)/(|b|^2 |n|) */
            F[3 * i + c] += fi; F[3 * k + c] += fk; F[3 * j + c] -= fi + fk;
        }
    }
    /* torsions: E = k [1 + cos(n phi - phi0)], phi = atan2(|b2| b1.(b2 x b3), (b1 x b2).(b2 x b3)) */
    for (int t = 0; t < T->n_tors; ++t) {
        int i = T->tors[4 * t], j = T->tors[4 * t + 1], k = T->tors[4 * t + 2], l = T->tors[4 * t + 3];
        double kk = T->tors_k_n_p0[3 * t], nn = T->tors_k_n_p0[3 * t + 1], p0 = T->tors_k_n_p0[3 * t + 2];
        double b1[3], b2[3], b3[3], n1[3], n2[3];
        for (int c = 0; c < 3; ++c) {
            b1[c] = pos[3 * j + c] - pos[3 * i + c]; b2[c] = pos[3 * k + c] - pos[3 * j + c]; b3[c] = pos[3 * l + c] - pos[3 * k + c];
        }
        cross(b1, b2, n1); cross(b2, b3, n2);
        double b2l = sqrt(dot(b2, b2));
        double phi = atan2(b2l * dot(b1, n2), dot(n1, n2));
        et += kk * (1.0 + cos(nn * phi - p0));
        double dEdphi = -kk * nn * sin(nn * phi - p0);
        /* dphi/dr: end atoms move phi by rotation about b2; inner atoms by lever-arm balance */
        double n1s = dot(n1, n1), n2s = dot(n2, n2);
        double gi[3], gl[3], gj[3], gk[3];
        double p = dot(b1, b2) / (b2l * b2l), q = dot(b3, b2) / (b2l * b2l);
        for (int c = 0; c < 3; ++c) {
            gi[c] = -b2l / n1s * n1[c];
            gl[c] = b2l / n2s * n2[c];
            gj[c] = -gi[c] - p * gi[c] + q * gl[c];
            gk[c] = -gl[c] + p * gi[c] - q * gl[c];
        }
        for (int c = 0; c < 3; ++c) {
            F[3 * i + c] -= dEdphi * gi[c]; F[3 * j + c] -= dEdphi * gj[c];
            F[3 * k + c] -= dEdphi * gk[c]; F[3 * l + c] -= dEdphi * gl[c];
        }
    }
    /* non-bonded: E = e_i e_j [(R/r)^12 - 2 (R/r)^6] + k_e q_i q_j / r over non-excluded i<j, no cut-off */
    if (T->excl) for (int i = 0; i < n; ++i) for (int j = i + 1; j < n; ++j) {
        if (T->excl[i * n + j]) continue;
        double d[3] = {pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1], pos[3 * i + 2] - pos[3 * j + 2]};
        double r2 = dot(d, d), r = sqrt(r2);
        double eps = T->lj_e[i] * T->lj_e[j], R = T->lj_R[i] + T->lj_R[j];
        double s6 = pow(R / r, 6.0), s12 = s6 * s6;
        double qq = ORC_KE * T->q[i] * T->q[j];
        en += eps * (s12 - 2.0 * s6) + qq / r;
        double dEdr = eps * (-12.0 * s12 + 12.0 * s6) / r - qq / r2;
        double s = -dEdr / r;
        for (int c = 0; c < 3; ++c) { F[3 * i + c] += s * d[c]; F[3 * j + c] -= s * d[c]; }
    }
    E4[0] = eb; E4[1] = ea; E4[2] = et; E4[3] = en;
}

/* Total force and the 7 potential-energy terms of one replica:
 * E7 = {grid ch0, grid ch1, grid ch2 (+ ch3 if the grid has a 4th channel), bond, angle, torsion, non-bonded}: the 7 terms sum to the
 * potential whose gradient F is (R22; the paper has three channels).   */
void orc_forces(const orc_grid* g, const orc_topology* T, const double* pos, double* F, double* E7) {
    int n = T->n_atoms;
    for (int i = 0; i < 3 * n; ++i) F[i] = 0;
    for (int c = 0; c < 7; ++c) E7[c] = 0;
    if (g) for (int i = 0; i < n; ++i) {
        double V[4], dV[12];
        interp_point(g, pos + 3 * i, V, dV);
        for (int c = 0; c < g->nch; ++c) {
            double k = T->coef[4 * i + c];
            E7[c < 3 ? c : 2] += k * V[c];
            for (int d = 0; d < 3; ++d) F[3 * i + d] -= k * dV[3 * c + d];
        }
    }
    orc_intramolecular(T, pos, F, E7 + 3);
}

/* ------------------------------------------------------------------ */
/* 6. Philox4x32-10 and the restart generator (step a8; R17) */
/* ------------------------------------------------------------------ */

void orc_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3], k0 = key_in[0], k1 = key_in[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Stream of uniforms in [0,1) with 24 random bits each: u = (x >> 8) 2^-24, exactly representable in
 * fp32 and fp64 alike.  Counter = (block, attempt, restart, replica), key = seed. */
typedef struct { uint32_t ctr[4], key[2], buf[4]; int have; } orc_rng;
static void rng_init(orc_rng* g, uint64_t seed, uint32_t replica, uint32_t restart, uint32_t attempt) {
    g->ctr[0] = 0; g->ctr[1] = attempt; g->ctr[2] = restart; g->ctr[3] = replica;
    g->key[0] = (uint32_t)seed; g->key[1] = (uint32_t)(seed >> 32); g->have = 0;
}
static double rng_uniform(orc_rng* g) {
    if (!g->have) { orc_philox4x32_10(g->ctr, g->key, g->buf); g->ctr[0]++; g->have = 4; }
    uint32_t x = g->buf[4 - g->have]; g->have--;
    return (double)(x >> 8) * (1.0 / 16777216.0);
}

typedef struct {
    int kind;               /* 0 velocity Verlet, 1 FIRE, 2 Langevin (BAOAB) */
    int n_steps; double dt; /* fs */
    double f_tol;           /* eV/Å: FIRE stops when max_i |F_i| < f_tol */
    double dt_max, f_inc, f_dec, a_start, f_a; int n_min;
    int restart;            /* 0: stop when converged; 1: record the minimum and re-seed */
    uint64_t seed;
    double z_ref;           /* top-layer z, for placing restarted molecules */
    double place_z_lo, place_z_hi, place_z_min;  /* centroid height range, lowest-atom floor (3, 6, 2 Å) */
    double clash;           /* reject a conformation with a non-excluded pair closer than clash*(R_i+R_j) */
    double max_step;        /* FIRE: cap on the largest atomic displacement per step, Å (0 = none); R13 */
    /* SURVEY.md §8(f) rows 1-2 */
    double temperature;     /* K, Langevin (kind 2; "1000 steps of Langevin molecular dynamics at ... 300 K") */
    double gamma;           /* friction, 1/fs (kind 2) */
    uint32_t step0;         /* index of the first step of this call in the noise stream (kind 2): 1 x N == k x N/k */
    int n_scan;             /* kind 1: > 0 = driven scan: n_scan times {move the held atoms by scan_dx; relax} */
    uint64_t fixed_mask;    /* bit i: atom i is held (restrained atom of PAPER.md:L178): no force, no velocity, moved only by the scan */
    double scan_dx[3];      /* Å per scan point */
} orc_integrator;

/* New conformation for (replica, restart#): template -> random dihedral about every rotatable bond ->
 * uniform random orientation about the centroid -> centroid at (u Lx, u Ly, z_ref + U(z_lo,z_hi)) ->
 * lift so the lowest atom is >= z_ref + place_z_min.  Up to 16 attempts against the clash test; the 16th is
 * kept regardless.  Returns the number of the accepted attempt (0..15). */
int orc_restart_conformation(const orc_topology* T, const orc_integrator* I, double Lx, double Ly,
                             uint32_t replica, uint32_t restart, double* pos) {
    int n = T->n_atoms;
    for (uint32_t attempt = 0; attempt < 16; ++attempt) {
        orc_rng g; rng_init(&g, I->seed, replica, restart, attempt);
        for (int i = 0; i < 3 * n; ++i) pos[i] = T->ref_pos[i];
        for (int b = 0; b < T->n_rot; ++b) {
            double ang = (2.0 * rng_uniform(&g) - 1.0) * ORC_PI;
            int j0 = T->rot_bond[2 * b], j1 = T->rot_bond[2 * b + 1];
            double o[3] = {pos[3 * j0], pos[3 * j0 + 1], pos[3 * j0 + 2]};
            double ax[3] = {pos[3 * j1] - o[0], pos[3 * j1 + 1] - o[1], pos[3 * j1 + 2] - o[2]};
            double al = sqrt(dot(ax, ax)); ax[0] /= al; ax[1] /= al; ax[2] /= al;
            double c = cos(ang), s = sin(ang);
            for (int i = 0; i < n; ++i) if (T->rot_mask[b * n + i]) {
                double v[3] = {pos[3 * i] - o[0], pos[3 * i + 1] - o[1], pos[3 * i + 2] - o[2]}, kv[3];
                cross(ax, v, kv);
                double kd = dot(ax, v);
                for (int d = 0; d < 3; ++d) pos[3 * i + d] = o[d] + v[d] * c + kv[d] * s + ax[d] * kd * (1.0 - c);  /* Rodrigues */
            }
        }
        /* uniform rotation (Shoemake): q = (sqrt(1-u1) sin 2pi u2, sqrt(1-u1) cos 2pi u2, sqrt(u1) sin 2pi u3, sqrt(u1) cos 2pi u3) */
        double u1 = rng_uniform(&g), u2 = rng_uniform(&g), u3 = rng_uniform(&g);
        double qx = sqrt(1 - u1) * sin(2 * ORC_PI * u2), qy = sqrt(1 - u1) * cos(2 * ORC_PI * u2);
        double qz = sqrt(u1) * sin(2 * ORC_PI * u3), qw = sqrt(u1) * cos(2 * ORC_PI * u3);
        double Rm[9] = {1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - qz * qw), 2 * (qx * qz + qy * qw),
                        2 * (qx * qy + qz * qw), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - qx * qw),
                        2 * (qx * qz - qy * qw), 2 * (qy * qz + qx * qw), 1 - 2 * (qx * qx + qy * qy)};
        double cx = 0, cy = 0, cz = 0;
        for (int i = 0; i < n; ++i) { cx += pos[3 * i]; cy += pos[3 * i + 1]; cz += pos[3 * i + 2]; }
        cx /= n; cy /= n; cz /= n;
        double tx = rng_uniform(&g) * Lx, ty = rng_uniform(&g) * Ly;
        double tz = I->z_ref + I->place_z_lo + (I->place_z_hi - I->place_z_lo) * rng_uniform(&g);
        double zmin = 1e300;
        for (int i = 0; i < n; ++i) {
            double v[3] = {pos[3 * i] - cx, pos[3 * i + 1] - cy, pos[3 * i + 2] - cz};
            pos[3 * i] = tx + Rm[0] * v[0] + Rm[1] * v[1] + Rm[2] * v[2];
            pos[3 * i + 1] = ty + Rm[3] * v[0] + Rm[4] * v[1] + Rm[5] * v[2];
            pos[3 * i + 2] = tz + Rm[6] * v[0] + Rm[7] * v[1] + Rm[8] * v[2];
            if (pos[3 * i + 2] < zmin) zmin = pos[3 * i + 2];
        }
        double lift = I->z_ref + I->place_z_min - zmin;
        if (lift > 0) for (int i = 0; i < n; ++i) pos[3 * i + 2] += lift;
        int clash = 0;
        if (T->excl && I->clash > 0) for (int i = 0; i < n && !clash; ++i) for (int j = i + 1; j < n; ++j) {
            if (T->excl[i * n + j]) continue;
            double d[3] = {pos[3 * i] - pos[3 * j], pos[3 * i + 1] - pos[3 * j + 1], pos[3 * i + 2] - pos[3 * j + 2]};
            double lim = I->clash * (T->lj_R[i] + T->lj_R[j]);
            if (dot(d, d) < lim * lim) { clash = 1; break; }
        }
        if (!clash || attempt == 15) return (int)attempt;
    }
    return 15;
}

/* Three standard normals for (replica, step, atom) of the Langevin thermostat (R18): one Philox4x32-10 block with
 * counter (step, atom, 'Lang', replica) and key = seed; u_k = ((x_k >> 9) + 1/2) 2^-23 in (0,1) (23 random bits: exactly
 * representable in fp32 and fp64 alike); Box-Muller:
 * xi_0 = sqrt(-2 ln u_0) cos 2 pi u_1, xi_1 = sqrt(-2 ln u_0) sin 2 pi u_1, xi_2 = sqrt(-2 ln u_2) cos 2 pi u_3. */
#define ORC_KB 8.617333262e-5       /* eV/K */
void orc_langevin_normals(uint64_t seed, uint32_t replica, uint32_t step, uint32_t atom, double xi[3]) {
    uint32_t ctr[4] = {step, atom, 0x4C616E67u, replica}, key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, o[4];
    orc_philox4x32_10(ctr, key, o);
    double u[4];
    for (int k = 0; k < 4; ++k) u[k] = ((double)(o[k] >> 9) + 0.5) * (1.0 / 8388608.0);
    double r0 = sqrt(-2.0 * log(u[0])), r1 = sqrt(-2.0 * log(u[2]));
    xi[0] = r0 * cos(2.0 * ORC_PI * u[1]);
    xi[1] = r0 * sin(2.0 * ORC_PI * u[1]);
    xi[2] = r1 * cos(2.0 * ORC_PI * u[3]);
}

/* forces with the held atoms' components removed (a held atom takes no part in the dynamics or in the convergence test) */
static void forces_free(const orc_grid* g, const orc_topology* T, const orc_integrator* I, const double* x, double* F, double* E7) {
    orc_forces(g, T, x, F, E7);
    for (int i = 0; i < T->n_atoms; ++i)
        if ((I->fixed_mask >> i) & 1ull) F[3 * i] = F[3 * i + 1] = F[3 * i + 2] = 0.0;
}

/* ------------------------------------------------------------------ */
/* 7. Integrators (steps a7, a8) and outputs (a9)                      */
/* ------------------------------------------------------------------ */

static double kinetic(const orc_topology* T, const double* vel) {
    double k = 0;
    for (int i = 0; i < T->n_atoms; ++i)
        k += 0.5 * T->mass[i] * (vel[3 * i] * vel[3 * i] + vel[3 * i + 1] * vel[3 * i + 1] + vel[3 * i + 2] * vel[3 * i + 2]);
    return k / ORC_ACC;   /* amu Å²/fs² -> eV */
}

/* pos, vel [n_rep][n][3] in/out.  fire [n_rep][4] in/out = {dt, a, steps since last P<=0, restarts done};
 * dt <= 0 on input means "fresh": {I->dt, a_start, 0, 0}.  energy [n_rep][8] = E7 + kinetic at the final
 * state.  status [n_rep][2] = {force evaluations made in this call after the first, converged flag or
 * number of minima recorded}.  minima [cap][4 + 3n] = {replica, restart#, steps, E_total, positions};
 * n_minima counts the records (may exceed cap; excess dropped).  e_trace (optional)
 * [n_rep][n_steps+1] total energy after every force evaluation (velocity Verlet only).            */
void orc_run_replicas(const orc_grid* g, const orc_topology* T, const orc_integrator* I, int n_rep,
                      double* pos, double* vel, double* fire, double* energy, int* status,
                      double* minima, long minima_cap, long* n_minima, double* e_trace, double* scan_out) {
    int n = T->n_atoms;
    long nmin = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < n_rep; ++r) {
        double* x = pos + (long)r * 3 * n;
        double* v = vel + (long)r * 3 * n;
        double* F = (double*)malloc(sizeof(double) * 3 * (size_t)n);
        double E7[7];
        int steps = 0, flag = 0;
        for (int i = 0; i < n; ++i) if ((I->fixed_mask >> i) & 1ull) v[3 * i] = v[3 * i + 1] = v[3 * i + 2] = 0.0;
        if (I->kind == 2) {
            /* Langevin dynamics, BAOAB splitting (Leimkuhler & Matthews 2013; R18):
             *   B: v += dt/2 a(x);  A: x += dt/2 v;  O: v <- c1 v + c2 sqrt(kT/m) xi;  A: x += dt/2 v;  F(x);  B: v += dt/2 a
             *   c1 = exp(-gamma dt), c2 = sqrt(1 - c1^2); the O step is the exact Ornstein-Uhlenbeck solution. */
            const double c1 = exp(-I->gamma * I->dt), c2 = sqrt(1.0 - c1 * c1), kT = ORC_KB * I->temperature;
            forces_free(g, T, I, x, F, E7);
            for (int s = 0; s < I->n_steps; ++s) {
                for (int i = 0; i < n; ++i) {
                    if ((I->fixed_mask >> i) & 1ull) continue;
                    double xi[3]; orc_langevin_normals(I->seed, (uint32_t)r, I->step0 + (uint32_t)s, (uint32_t)i, xi);
                    const double sig = sqrt(kT / T->mass[i] * ORC_ACC);
                    for (int c = 0; c < 3; ++c) {
                        v[3 * i + c] += 0.5 * I->dt * F[3 * i + c] / T->mass[i] * ORC_ACC;
                        x[3 * i + c] += 0.5 * I->dt * v[3 * i + c];
                        v[3 * i + c] = c1 * v[3 * i + c] + c2 * sig * xi[c];
                        x[3 * i + c] += 0.5 * I->dt * v[3 * i + c];
                    }
                }
                forces_free(g, T, I, x, F, E7);
                for (int i = 0; i < n; ++i) for (int c = 0; c < 3; ++c)
                    v[3 * i + c] += 0.5 * I->dt * F[3 * i + c] / T->mass[i] * ORC_ACC;
                ++steps;
            }
        } else if (I->kind == 1 && I->n_scan > 0) {
            /* driven scan (PAPER.md:L178 lift, L184 drag): move the held atoms by scan_dx, relax the others with FIRE (fresh scalars,
             * v = 0) until max |F_i| < f_tol or n_steps iterations, record {E_total, iterations, converged, max |F_i|}; repeat. */
            for (int sc = 0; sc < I->n_scan; ++sc) {
                for (int i = 0; i < n; ++i) if ((I->fixed_mask >> i) & 1ull) for (int c = 0; c < 3; ++c) x[3 * i + c] += I->scan_dx[c];
                for (int i = 0; i < 3 * n; ++i) v[i] = 0;
                double dt = I->dt, a = I->a_start; int npos = 0, it = 0, conv = 0;
                for (it = 0; it < I->n_steps; ++it) {
                    forces_free(g, T, I, x, F, E7);
                    double fmax2 = 0;
                    for (int i = 0; i < n; ++i) {
                        double f2 = F[3 * i] * F[3 * i] + F[3 * i + 1] * F[3 * i + 1] + F[3 * i + 2] * F[3 * i + 2];
                        if (f2 > fmax2) fmax2 = f2;
                    }
                    if (fmax2 < I->f_tol * I->f_tol) { conv = 1; break; }
                    double P = 0, vv = 0, ff = 0;
                    for (int i = 0; i < 3 * n; ++i) { P += F[i] * v[i]; vv += v[i] * v[i]; ff += F[i] * F[i]; }
                    if (P > 0) {
                        double sc2 = a * sqrt(vv) / sqrt(ff);
                        for (int i = 0; i < 3 * n; ++i) v[i] = (1.0 - a) * v[i] + sc2 * F[i];
                        ++npos;
                        if (npos > I->n_min) { dt = fmin(dt * I->f_inc, I->dt_max); a *= I->f_a; }
                    } else {
                        for (int i = 0; i < 3 * n; ++i) v[i] = 0;
                        dt *= I->f_dec; a = I->a_start; npos = 0;
                    }
                    for (int i = 0; i < n; ++i) for (int c = 0; c < 3; ++c)
                        v[3 * i + c] += dt * F[3 * i + c] / T->mass[i] * ORC_ACC;
                    if (I->max_step > 0) {
                        double vmax2 = 0;
                        for (int i = 0; i < n; ++i) {
                            double v2 = v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2];
                            if (v2 > vmax2) vmax2 = v2;
                        }
                        if (dt * sqrt(vmax2) > I->max_step) {
                            double sc2 = I->max_step / (dt * sqrt(vmax2));
                            for (int i = 0; i < 3 * n; ++i) v[i] *= sc2;
                        }
                    }
                    for (int i = 0; i < 3 * n; ++i) x[i] += dt * v[i];
                    ++steps;
                }
                forces_free(g, T, I, x, F, E7);
                double e = 0, fmax2 = 0;
                for (int c = 0; c < 7; ++c) e += E7[c];
                for (int i = 0; i < n; ++i) {
                    double f2 = F[3 * i] * F[3 * i] + F[3 * i + 1] * F[3 * i + 1] + F[3 * i + 2] * F[3 * i + 2];
                    if (f2 > fmax2) fmax2 = f2;
                }
                if (scan_out) {
                    double* o = scan_out + ((long)r * I->n_scan + sc) * 4;
                    o[0] = e; o[1] = it; o[2] = conv; o[3] = sqrt(fmax2);
                }
                flag += conv;
            }
        } else if (I->kind == 0) {
            /* velocity Verlet: v += dt/2 a; x += dt v; F(x); v += dt/2 a     (R13) */
            forces_free(g, T, I, x, F, E7);
            if (e_trace) { double e = kinetic(T, v); for (int c = 0; c < 7; ++c) e += E7[c]; e_trace[(long)r * (I->n_steps + 1)] = e; }
            for (int s = 0; s < I->n_steps; ++s) {
                for (int i = 0; i < n; ++i) for (int c = 0; c < 3; ++c) {
                    v[3 * i + c] += 0.5 * I->dt * F[3 * i + c] / T->mass[i] * ORC_ACC;
                    x[3 * i + c] += I->dt * v[3 * i + c];
                }
                forces_free(g, T, I, x, F, E7);
                for (int i = 0; i < n; ++i) for (int c = 0; c < 3; ++c)
                    v[3 * i + c] += 0.5 * I->dt * F[3 * i + c] / T->mass[i] * ORC_ACC;
                ++steps;
                if (e_trace) { double e = kinetic(T, v); for (int c = 0; c < 7; ++c) e += E7[c]; e_trace[(long)r * (I->n_steps + 1) + s + 1] = e; }
            }
        } else {
            /* FIRE (ref 72), R13.  One loop iteration = one force
             * evaluation followed by either (a) the FIRE velocity update and a semi-implicit Euler step,
             * or (b) when converged in restart mode, recording the minimum and re-seeding (no motion). */
            double dt = fire[4 * r], a = fire[4 * r + 1];
            int npos = (int)fire[4 * r + 2]; int nrestart = (int)fire[4 * r + 3];
            if (dt <= 0) { dt = I->dt; a = I->a_start; npos = 0; nrestart = 0; }
            int stopped = 0;
            for (int s = 0; s < I->n_steps; ++s) {
                forces_free(g, T, I, x, F, E7);
                double fmax2 = 0;
                for (int i = 0; i < n; ++i) {
                    double f2 = F[3 * i] * F[3 * i] + F[3 * i + 1] * F[3 * i + 1] + F[3 * i + 2] * F[3 * i + 2];
                    if (f2 > fmax2) fmax2 = f2;
                }
                if (fmax2 < I->f_tol * I->f_tol) {
                    if (!I->restart) { flag = 1; stopped = 1; break; }
                    long slot;
#pragma omp atomic capture
                    slot = nmin++;
                    if (minima && slot < minima_cap) {
                        double* m = minima + slot * (4 + 3 * n);
                        double e = 0; for (int c = 0; c < 7; ++c) e += E7[c];
                        m[0] = r; m[1] = nrestart; m[2] = steps; m[3] = e;
                        for (int i = 0; i < 3 * n; ++i) m[4 + i] = x[i];
                    }
                    ++flag; ++nrestart;
                    orc_restart_conformation(T, I, g->Lx, g->Ly, (uint32_t)r, (uint32_t)nrestart, x);
                    for (int i = 0; i < 3 * n; ++i) v[i] = 0;
                    dt = I->dt; a = I->a_start; npos = 0;
                    continue;
                }
                double P = 0, vv = 0, ff = 0;
                for (int i = 0; i < 3 * n; ++i) { P += F[i] * v[i]; vv += v[i] * v[i]; ff += F[i] * F[i]; }
                if (P > 0) {
                    double sc = a * sqrt(vv) / sqrt(ff);
                    for (int i = 0; i < 3 * n; ++i) v[i] = (1.0 - a) * v[i] + sc * F[i];
                    ++npos;
                    if (npos > I->n_min) { dt = fmin(dt * I->f_inc, I->dt_max); a *= I->f_a; }
                } else {
                    for (int i = 0; i < 3 * n; ++i) v[i] = 0;
                    dt *= I->f_dec; a = I->a_start; npos = 0;
                }
                for (int i = 0; i < n; ++i) for (int c = 0; c < 3; ++c)
                    v[3 * i + c] += dt * F[3 * i + c] / T->mass[i] * ORC_ACC;
                if (I->max_step > 0) {
                    double vmax2 = 0;
                    for (int i = 0; i < n; ++i) {
                        double v2 = v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2];
                        if (v2 > vmax2) vmax2 = v2;
                    }
                    if (dt * sqrt(vmax2) > I->max_step) {
                        double sc = I->max_step / (dt * sqrt(vmax2));
                        for (int i = 0; i < 3 * n; ++i) v[i] *= sc;
                    }
                }
                for (int i = 0; i < 3 * n; ++i) x[i] += dt * v[i];
                ++steps;
            }
            if (!stopped) {
                /* energies (and, without restart, the converged flag) describe the final state */
                forces_free(g, T, I, x, F, E7);
                if (!I->restart) {
                    double fmax2 = 0;
                    for (int i = 0; i < n; ++i) {
                        double f2 = F[3 * i] * F[3 * i] + F[3 * i + 1] * F[3 * i + 1] + F[3 * i + 2] * F[3 * i + 2];
                        if (f2 > fmax2) fmax2 = f2;
                    }
                    if (fmax2 < I->f_tol * I->f_tol) flag = 1;
                }
            }
            fire[4 * r] = dt; fire[4 * r + 1] = a; fire[4 * r + 2] = npos; fire[4 * r + 3] = nrestart;
        }
        if (energy) { for (int c = 0; c < 7; ++c) energy[8 * r + c] = E7[c]; energy[8 * r + 7] = kinetic(T, v); }
        if (status) { status[2 * r] = steps; status[2 * r + 1] = flag; }
        free(F);
    }
    if (n_minima) *n_minima = nmin;
}

int orc_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}
