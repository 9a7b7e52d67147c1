/*
 * sho_oracle.c -- plain, slow, obviously-correct CPU ORACLE for the SHO projection hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.  It shares no code, header,
 * table or constant with the CUDA library (paper_1905_00480_b200/csrc); neither includes the
 * other.
 *
 * Written from /root/reference/PAPER.md (Baumeister & Tsukamoto, PASC'19, arXiv:1905.00480):
 *   - 1D harmonic-oscillator eigenstates "Hermite polynomials times a Gaussian"
 *       psi_n(x) ~ H_n(x/sigma) exp(-x^2/(2 sigma^2))                    PAPER.md:66-73, eq. (2)-(3)
 *   - 3D product states Psi_{nx ny nz} = psi_nx(x) psi_ny(y) psi_nz(z)    PAPER.md:79-90, eq. (4)-(6)
 *   - truncated basis nx+ny+nz <= numax, N_SHO = (numax+3)(numax+2)(numax+1)/6
 *                                                                         PAPER.md:145-154, eq. (17)-(18)
 *   - projection C_{nx ny nz k} = <nx ny nz|Psi_k> = iiint psi_nx psi_ny psi_nz Psi_k d^3r
 *                                                                         PAPER.md:244-248, eq. (25)-(26)
 *   - non-local action: (1) projection c = <p|Psi>, (3) expansion: add sum_ai d |p>
 *                                                                         PAPER.md:187-190
 *
 * The method reaches exactly (up to summation order) a result with a plain definition -- a finite
 * sum over grid points -- so this oracle IS that definition written out: Hermite polynomials from
 * their explicit textbook sum (NOT the recurrence of eq. 31 that the GPU path uses), the 3D product
 * formed per grid point, a literal triple loop per (atom, band, nx, ny, nz).  No separable
 * reordering, no blocking, no fusion.  OpenMP is used only over independent outputs
 * ((atom,band) pairs in project, bands in add); it never reorders a sum.
 *
 * Readings of the paper where it is silent:
 *   A1  phi_n(u;sigma) = (2^n n! sqrt(pi) sigma)^(-1/2) H_n^phys(u/sigma) exp(-u^2/(2 sigma^2))
 *       (orthonormal; the paper omits the normalisation, north_star fixes it)
 *   A2  grid point i of an axis sits at x_i = i*h; cell is [0, N*h)
 *   A3  region = axis-aligned cube |u_d| <= rcut_sigma*sigma per axis, inclusive, no radial mask:
 *       i_lo = ceil((R_d - rc*sigma)/h), i_hi = floor((R_d + rc*sigma)/h), evaluated in IEEE double
 *       exactly as written (compile with -ffp-contract=off)
 *   A4  periodic axis: loop over the UNWRAPPED index i; j = i mod N (floor-mod), image m = floor(i/N);
 *       a box wider than the cell visits a grid point once per image
 *   A5  isolated axis: psi == 0 outside the grid: clamp [i_lo,i_hi] to [0,N-1]
 *   A6  Bloch: psi(r + L e_d) = exp(2 pi i kfrac_d) psi(r); project multiplies the value read at
 *       image m by exp(2 pi i kfrac_d m), add multiplies by its conjugate.  Projectors stay real.
 *   A7  h^3 volume element in project only; add has none (so add = P^H / h^3)
 *   A8  coefficient order: n=0; for nz in 0..numax: for ny in 0..numax-nz: for nx in 0..numax-nz-ny: n++
 *   A9  layouts: psi [nb][Nz][Ny][Nx] (x fastest), coeff [natoms][nb][N_SHO] (n fastest);
 *       complex data interleaved (re,im)
 *
 * Every function below is pinned by tests/test_oracle_pins.py (-m "not gpu") against things other
 * than itself: printed N_SHO values, scipy's Hermite polynomials, 1D orthonormality, separable ==
 * brute force, the closed-form Gaussian and plane-wave projections (the Gaussian one also through
 * the explicit-pair branch of oracle_project_pairs), the adjoint identity, translation / zero-padding
 * invariances, a hand-written 2x2 product and numpy's matmul for oracle_dmul, Hermiticity of the
 * three-step action.  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_NUMAX_MAX 20

static const double ORACLE_PI = 3.14159265358979323846264338327950288;

/* number of threads the parallel loops below will use (for bench.py's "cores" field) */
int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* eq. (18) */
int oracle_nsho(int numax)
{
    if (numax < 0 || numax > ORACLE_NUMAX_MAX) return -1;
    return (numax + 3) * (numax + 2) * (numax + 1) / 6;
}

/* reading A8: position of (nx,ny,nz) in the coefficient vector, by literal enumeration */
int oracle_index(int nx, int ny, int nz, int numax)
{
    if (nx < 0 || ny < 0 || nz < 0 || nx + ny + nz > numax || numax > ORACLE_NUMAX_MAX) return -1;
    int n = 0;
    for (int kz = 0; kz <= numax; ++kz)
        for (int ky = 0; ky <= numax - kz; ++ky)
            for (int kx = 0; kx <= numax - kz - ky; ++kx) {
                if (kx == nx && ky == ny && kz == nz) return n;
                ++n;
            }
    return -1;
}

static double factorial(int n)
{
    double f = 1.0;
    for (int i = 2; i <= n; ++i) f *= (double)i;
    return f;
}

/* physicists' Hermite polynomial from the explicit textbook sum
 *   H_n(xi) = n! sum_{k=0}^{floor(n/2)} (-1)^k (2 xi)^(n-2k) / (k! (n-2k)!)
 * (the paper's eq. 31 H_n is the monic 2^-n H_n) */
double oracle_hermite_phys(int n, double xi)
{
    double s = 0.0;
    for (int k = 0; 2 * k <= n; ++k) {
        double term = pow(2.0 * xi, (double)(n - 2 * k)) / (factorial(k) * factorial(n - 2 * k));
        s += (k % 2 == 0) ? term : -term;
    }
    return factorial(n) * s;
}

/* reading A1: orthonormal Hermite-Gauss function of width sigma, eq. (3) PAPER.md:70 with the
 * normalisation the paper omits */
double oracle_phi(int n, double u, double sigma)
{
    double xi = u / sigma;
    double norm = 1.0 / sqrt(pow(2.0, (double)n) * factorial(n) * sqrt(ORACLE_PI) * sigma);
    return norm * oracle_hermite_phys(n, xi) * exp(-0.5 * xi * xi);
}

/* floor-mod and floor-div for possibly negative i (reading A4) */
static int floormod(int i, int n) { int r = i % n; return r < 0 ? r + n : r; }
static int floordiv(int i, int n) { return (i - floormod(i, n)) / n; }

/* reading A3/A5: integer box range of one atom on the three axes; returns 1 if the box is empty */
int oracle_box(const int32_t ng[3], double h, const int32_t periodic[3], const double pos[3],
               double sigma, double rcut_sigma, int32_t lo[3], int32_t hi[3])
{
    int empty = 0;
    for (int d = 0; d < 3; ++d) {
        double a = (pos[d] - rcut_sigma * sigma) / h;
        double b = (pos[d] + rcut_sigma * sigma) / h;
        int l = (int)ceil(a);
        int u = (int)floor(b);
        if (!periodic[d]) {
            if (l < 0) l = 0;
            if (u > ng[d] - 1) u = ng[d] - 1;
        }
        lo[d] = l;
        hi[d] = u;
        if (u < l) empty = 1;
    }
    return empty;
}

/* per-atom per-axis table of the 1D function values (explicit formula) over the box,
 * tab[d][n][i-lo]; plus wrapped index and Bloch phase per box index */
typedef struct {
    int lo[3], hi[3], len[3];
    double* phi[3];   /* [ (numax+1) * len ] */
    int* j[3];        /* wrapped grid index  */
    double* wre[3];   /* phase of the image   */
    double* wim[3];
    int empty;
} atom_tab;

static void atom_tab_free(atom_tab* t)
{
    for (int d = 0; d < 3; ++d) { free(t->phi[d]); free(t->j[d]); free(t->wre[d]); free(t->wim[d]); }
}

static void atom_tab_build(atom_tab* t, const int32_t ng[3], double h, const int32_t periodic[3],
                           const double* kfrac, const double pos[3], double sigma, int numax,
                           double rcut_sigma)
{
    int32_t lo[3], hi[3];
    t->empty = oracle_box(ng, h, periodic, pos, sigma, rcut_sigma, lo, hi);
    for (int d = 0; d < 3; ++d) {
        t->lo[d] = lo[d]; t->hi[d] = hi[d];
        int len = hi[d] - lo[d] + 1; if (len < 0) len = 0;
        t->len[d] = len;
        t->phi[d] = (double*)malloc(sizeof(double) * (size_t)(numax + 1) * (size_t)(len > 0 ? len : 1));
        t->j[d]   = (int*)   malloc(sizeof(int)    * (size_t)(len > 0 ? len : 1));
        t->wre[d] = (double*)malloc(sizeof(double) * (size_t)(len > 0 ? len : 1));
        t->wim[d] = (double*)malloc(sizeof(double) * (size_t)(len > 0 ? len : 1));
        for (int q = 0; q < len; ++q) {
            int i = lo[d] + q;
            double u = (double)i * h - pos[d];               /* reading A2: x_i = i*h */
            for (int n = 0; n <= numax; ++n) t->phi[d][(size_t)n * len + q] = oracle_phi(n, u, sigma);
            if (periodic[d]) {
                int m = floordiv(i, ng[d]);
                t->j[d][q] = floormod(i, ng[d]);
                double ang = 2.0 * ORACLE_PI * (kfrac ? kfrac[d] : 0.0) * (double)m;   /* reading A6 */
                t->wre[d][q] = (kfrac && kfrac[d] != 0.0 && m != 0) ? cos(ang) : 1.0;
                t->wim[d][q] = (kfrac && kfrac[d] != 0.0 && m != 0) ? sin(ang) : 0.0;
            } else {
                t->j[d][q] = i; t->wre[d][q] = 1.0; t->wim[d][q] = 0.0;
            }
        }
    }
}

/* one (atom, band) pair of the projection: eq. (25)-(26) discretised with volume element h^3,
 * a literal triple loop per (nx,ny,nz), the 3D product formed at every point */
static void project_pair(const atom_tab* t, const int32_t ng[3], double h, int numax, int is_complex,
                         const double* psi_b /* one band */, double* c /* [N_SHO] or [N_SHO][2] */)
{
    const double h3 = h * h * h;
    const size_t sx = 1, sy = (size_t)ng[0], sz = (size_t)ng[0] * (size_t)ng[1];
    (void)sx;
    int n = 0;
    for (int nz = 0; nz <= numax; ++nz)
        for (int ny = 0; ny <= numax - nz; ++ny)
            for (int nx = 0; nx <= numax - nz - ny; ++nx) {
                double sre = 0.0, sim = 0.0;
                if (!t->empty) {
                    const double* px = t->phi[0] + (size_t)nx * t->len[0];
                    const double* py = t->phi[1] + (size_t)ny * t->len[1];
                    const double* pz = t->phi[2] + (size_t)nz * t->len[2];
                    for (int qz = 0; qz < t->len[2]; ++qz)
                        for (int qy = 0; qy < t->len[1]; ++qy)
                            for (int qx = 0; qx < t->len[0]; ++qx) {
                                double p3 = pz[qz] * py[qy] * px[qx];      /* Phi_n(r - R_a) at this point */
                                size_t j = (size_t)t->j[2][qz] * sz + (size_t)t->j[1][qy] * sy + (size_t)t->j[0][qx];
                                if (!is_complex) {
                                    sre += p3 * psi_b[j];
                                } else {
                                    /* w = w_x w_y w_z, phase of the image this point is read from */
                                    double ar = t->wre[0][qx], ai = t->wim[0][qx];
                                    double br = t->wre[1][qy], bi = t->wim[1][qy];
                                    double cr = t->wre[2][qz], ci = t->wim[2][qz];
                                    double abr = ar * br - ai * bi, abi = ar * bi + ai * br;
                                    double wr = abr * cr - abi * ci, wi = abr * ci + abi * cr;
                                    double vr = psi_b[2 * j], vi = psi_b[2 * j + 1];
                                    sre += p3 * (wr * vr - wi * vi);
                                    sim += p3 * (wr * vi + wi * vr);
                                }
                            }
                }
                if (!is_complex) c[n] = h3 * sre;
                else { c[2 * n] = h3 * sre; c[2 * n + 1] = h3 * sim; }
                ++n;
            }
}

/*
 * Projection of selected (atom, band) pairs.  pair_atom/pair_band == NULL means all pairs in
 * [atom][band] order (npairs must then be natoms*nbands).
 *   psi   [nbands][Nz][Ny][Nx] (x2 doubles if is_complex)
 *   out   [npairs][N_SHO]      (x2 doubles if is_complex)
 * psi_band_ptrs: optional array of per-band pointers (when bands live in separate host buffers);
 *   if non-NULL it overrides psi.
 */
int oracle_project_pairs(const int32_t ng[3], double h, const int32_t periodic[3], const double* kfrac,
                         int natoms, const double* pos, const double* sigma, int numax, double rcut_sigma,
                         int is_complex, int nbands, const double* psi, const double* const* psi_band_ptrs,
                         int64_t npairs, const int32_t* pair_atom, const int32_t* pair_band, double* out)
{
    int nsho = oracle_nsho(numax);
    if (nsho < 0 || natoms < 0 || nbands <= 0 || h <= 0.0) return 1;
    const size_t npts = (size_t)ng[0] * ng[1] * ng[2];
    const size_t cw = is_complex ? 2 : 1;
    int err = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t p = 0; p < npairs; ++p) {
        int a = pair_atom ? pair_atom[p] : (int)(p / nbands);
        int b = pair_band ? pair_band[p] : (int)(p % nbands);
        if (a < 0 || a >= natoms || b < 0 || b >= nbands) { err = 1; continue; }
        atom_tab t;
        atom_tab_build(&t, ng, h, periodic, kfrac, pos + 3 * (size_t)a, sigma[a], numax, rcut_sigma);
        const double* psi_b = psi_band_ptrs ? psi_band_ptrs[b] : psi + (size_t)b * npts * cw;
        project_pair(&t, ng, h, numax, is_complex, psi_b, out + (size_t)p * nsho * cw);
        atom_tab_free(&t);
    }
    return err;
}

/* full projection, coeff [natoms][nbands][N_SHO] */
int oracle_project(const int32_t ng[3], double h, const int32_t periodic[3], const double* kfrac,
                   int natoms, const double* pos, const double* sigma, int numax, double rcut_sigma,
                   int is_complex, int nbands, const double* psi, double* coeff)
{
    return oracle_project_pairs(ng, h, periodic, kfrac, natoms, pos, sigma, numax, rcut_sigma, is_complex,
                                nbands, psi, NULL, (int64_t)natoms * nbands, NULL, NULL, coeff);
}

/*
 * Expansion / add-back, step (3) PAPER.md:190, point-wise definition:
 *   psi[b][j] += sum_a sum_{images i of j inside box a} conj(w(i)) sum_n c[a][b][n] phi_nx phi_ny phi_nz
 * atoms in ascending order; no h^3 (reading A7).
 */
int oracle_add(const int32_t ng[3], double h, const int32_t periodic[3], const double* kfrac,
               int natoms, const double* pos, const double* sigma, int numax, double rcut_sigma,
               int is_complex, int nbands, const double* coeff, double* psi)
{
    int nsho = oracle_nsho(numax);
    if (nsho < 0 || natoms < 0 || nbands <= 0 || h <= 0.0) return 1;
    const size_t npts = (size_t)ng[0] * ng[1] * ng[2];
    const size_t cw = is_complex ? 2 : 1;
    const size_t sy = (size_t)ng[0], sz = (size_t)ng[0] * (size_t)ng[1];
    atom_tab* tabs = (atom_tab*)malloc(sizeof(atom_tab) * (size_t)(natoms > 0 ? natoms : 1));
    for (int a = 0; a < natoms; ++a)
        atom_tab_build(&tabs[a], ng, h, periodic, kfrac, pos + 3 * (size_t)a, sigma[a], numax, rcut_sigma);
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < nbands; ++b) {
        double* psi_b = psi + (size_t)b * npts * cw;
        for (int a = 0; a < natoms; ++a) {
            const atom_tab* t = &tabs[a];
            if (t->empty) continue;
            const double* c = coeff + ((size_t)a * nbands + b) * nsho * cw;
            for (int qz = 0; qz < t->len[2]; ++qz)
                for (int qy = 0; qy < t->len[1]; ++qy)
                    for (int qx = 0; qx < t->len[0]; ++qx) {
                        double vre = 0.0, vim = 0.0;
                        int n = 0;
                        for (int nz = 0; nz <= numax; ++nz)
                            for (int ny = 0; ny <= numax - nz; ++ny)
                                for (int nx = 0; nx <= numax - nz - ny; ++nx) {
                                    double p3 = t->phi[2][(size_t)nz * t->len[2] + qz]
                                              * t->phi[1][(size_t)ny * t->len[1] + qy]
                                              * t->phi[0][(size_t)nx * t->len[0] + qx];
                                    if (!is_complex) vre += c[n] * p3;
                                    else { vre += c[2 * n] * p3; vim += c[2 * n + 1] * p3; }
                                    ++n;
                                }
                        size_t j = (size_t)t->j[2][qz] * sz + (size_t)t->j[1][qy] * sy + (size_t)t->j[0][qx];
                        if (!is_complex) {
                            psi_b[j] += vre;
                        } else {
                            double ar = t->wre[0][qx], ai = t->wim[0][qx];
                            double br = t->wre[1][qy], bi = t->wim[1][qy];
                            double cr = t->wre[2][qz], ci = t->wim[2][qz];
                            double abr = ar * br - ai * bi, abi = ar * bi + ai * br;
                            double wr = abr * cr - abi * ci, wi = abr * ci + abi * cr;
                            /* conj(w) * v */
                            psi_b[2 * j]     += wr * vre + wi * vim;
                            psi_b[2 * j + 1] += wr * vim - wi * vre;
                        }
                    }
        }
    }
    for (int a = 0; a < natoms; ++a) atom_tab_free(&tabs[a]);
    free(tabs);
    return 0;
}

/*
 * The same point-wise definition evaluated only at chosen grid points (for sampled parity at sizes
 * where the full add is too slow): for sample s with wrapped grid index (jx,jy,jz) = pts[s][0..2]
 * and band bands[s],
 *   out[s] = sum_a sum_{images} conj(w) sum_n c[a][b][n] phi_nx phi_ny phi_nz      (the increment only)
 * The images of j on axis d inside box a are i = j + m*N, m = ceil((lo-j)/N) .. floor((hi-j)/N).
 */
int oracle_add_points(const int32_t ng[3], double h, const int32_t periodic[3], const double* kfrac,
                      int natoms, const double* pos, const double* sigma, int numax, double rcut_sigma,
                      int is_complex, int nbands, const double* coeff,
                      int64_t nsamples, const int32_t* pts /* [ns][3] = jx,jy,jz */, const int32_t* bands,
                      double* out /* [ns] (x2 if complex) */)
{
    int nsho = oracle_nsho(numax);
    if (nsho < 0 || natoms < 0 || nbands <= 0 || h <= 0.0) return 1;
    const size_t cw = is_complex ? 2 : 1;
    int32_t* lo = (int32_t*)malloc(sizeof(int32_t) * 3 * (size_t)(natoms > 0 ? natoms : 1));
    int32_t* hi = (int32_t*)malloc(sizeof(int32_t) * 3 * (size_t)(natoms > 0 ? natoms : 1));
    int* empty = (int*)malloc(sizeof(int) * (size_t)(natoms > 0 ? natoms : 1));
    for (int a = 0; a < natoms; ++a)
        empty[a] = oracle_box(ng, h, periodic, pos + 3 * (size_t)a, sigma[a], rcut_sigma, lo + 3 * a, hi + 3 * a);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t s = 0; s < nsamples; ++s) {
        const int32_t* j = pts + 3 * s;
        int b = bands[s];
        double accre = 0.0, accim = 0.0;
        for (int a = 0; a < natoms; ++a) {
            if (empty[a]) continue;
            int m0[3], m1[3], skip = 0;
            for (int d = 0; d < 3; ++d) {
                if (periodic[d]) {
                    m0[d] = (int)ceil(((double)lo[3 * a + d] - (double)j[d]) / (double)ng[d]);
                    m1[d] = (int)floor(((double)hi[3 * a + d] - (double)j[d]) / (double)ng[d]);
                } else {
                    m0[d] = 0;
                    m1[d] = (j[d] >= lo[3 * a + d] && j[d] <= hi[3 * a + d]) ? 0 : -1;
                }
                if (m1[d] < m0[d]) skip = 1;
            }
            if (skip) continue;
            const double* c = coeff + ((size_t)a * nbands + b) * nsho * cw;
            const double* R = pos + 3 * (size_t)a;
            for (int mz = m0[2]; mz <= m1[2]; ++mz)
                for (int my = m0[1]; my <= m1[1]; ++my)
                    for (int mx = m0[0]; mx <= m1[0]; ++mx) {
                        int m[3] = { mx, my, mz };
                        double u[3];
                        for (int d = 0; d < 3; ++d) u[d] = (double)(j[d] + m[d] * ng[d]) * h - R[d];
                        double f[3][ORACLE_NUMAX_MAX + 1];   /* 1D values at this point, explicit formula */
                        for (int d = 0; d < 3; ++d)
                            for (int k = 0; k <= numax; ++k) f[d][k] = oracle_phi(k, u[d], sigma[a]);
                        double vre = 0.0, vim = 0.0;
                        int n = 0;
                        for (int nz = 0; nz <= numax; ++nz)
                            for (int ny = 0; ny <= numax - nz; ++ny)
                                for (int nx = 0; nx <= numax - nz - ny; ++nx) {
                                    double p3 = f[2][nz] * f[1][ny] * f[0][nx];
                                    if (!is_complex) vre += c[n] * p3;
                                    else { vre += c[2 * n] * p3; vim += c[2 * n + 1] * p3; }
                                    ++n;
                                }
                        if (!is_complex) {
                            accre += vre;
                        } else {
                            double ang = 2.0 * ORACLE_PI * (kfrac ? (kfrac[0] * mx + kfrac[1] * my + kfrac[2] * mz) : 0.0);
                            double wr = cos(ang), wi = sin(ang);
                            accre += wr * vre + wi * vim;   /* conj(w) * v */
                            accim += wr * vim - wi * vre;
                        }
                    }
        }
        if (!is_complex) out[s] = accre;
        else { out[2 * s] = accre; out[2 * s + 1] = accim; }
    }
    free(lo); free(hi); free(empty);
    return 0;
}

/*
 * The same point-wise definition for SEVERAL bands of one grid point at once (sampled parity at full
 * size over all bands: the 1D function values of a point do not depend on the band, so they are
 * evaluated once per (point, atom image) and the sum over n runs per selected band):
 *   out[s][k] = sum_a sum_{images} conj(w) sum_n c[a][band_sel[k]][n] phi_nx phi_ny phi_nz
 * Same arithmetic, same order of the sums over atoms, images and n as oracle_add_points.
 */
int oracle_add_points_bands(const int32_t ng[3], double h, const int32_t periodic[3], const double* kfrac,
                            int natoms, const double* pos, const double* sigma, int numax, double rcut_sigma,
                            int is_complex, int nbands, const double* coeff,
                            int64_t nsamples, const int32_t* pts /* [ns][3] = jx,jy,jz */,
                            int nsel, const int32_t* band_sel /* [nsel] */,
                            double* out /* [ns][nsel] (x2 if complex) */)
{
    int nsho = oracle_nsho(numax);
    if (nsho < 0 || natoms < 0 || nbands <= 0 || h <= 0.0 || nsel <= 0) return 1;
    for (int k = 0; k < nsel; ++k)
        if (band_sel[k] < 0 || band_sel[k] >= nbands) return 1;
    const size_t cw = is_complex ? 2 : 1;
    int32_t* lo = (int32_t*)malloc(sizeof(int32_t) * 3 * (size_t)(natoms > 0 ? natoms : 1));
    int32_t* hi = (int32_t*)malloc(sizeof(int32_t) * 3 * (size_t)(natoms > 0 ? natoms : 1));
    int* empty = (int*)malloc(sizeof(int) * (size_t)(natoms > 0 ? natoms : 1));
    for (int a = 0; a < natoms; ++a)
        empty[a] = oracle_box(ng, h, periodic, pos + 3 * (size_t)a, sigma[a], rcut_sigma, lo + 3 * a, hi + 3 * a);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t s = 0; s < nsamples; ++s) {
        const int32_t* j = pts + 3 * s;
        double* o = out + (size_t)s * nsel * cw;
        for (size_t k = 0; k < (size_t)nsel * cw; ++k) o[k] = 0.0;
        for (int a = 0; a < natoms; ++a) {
            if (empty[a]) continue;
            int m0[3], m1[3], skip = 0;
            for (int d = 0; d < 3; ++d) {
                if (periodic[d]) {
                    m0[d] = (int)ceil(((double)lo[3 * a + d] - (double)j[d]) / (double)ng[d]);
                    m1[d] = (int)floor(((double)hi[3 * a + d] - (double)j[d]) / (double)ng[d]);
                } else {
                    m0[d] = 0;
                    m1[d] = (j[d] >= lo[3 * a + d] && j[d] <= hi[3 * a + d]) ? 0 : -1;
                }
                if (m1[d] < m0[d]) skip = 1;
            }
            if (skip) continue;
            const double* R = pos + 3 * (size_t)a;
            for (int mz = m0[2]; mz <= m1[2]; ++mz)
                for (int my = m0[1]; my <= m1[1]; ++my)
                    for (int mx = m0[0]; mx <= m1[0]; ++mx) {
                        int m[3] = { mx, my, mz };
                        double u[3];
                        for (int d = 0; d < 3; ++d) u[d] = (double)(j[d] + m[d] * ng[d]) * h - R[d];
                        double f[3][ORACLE_NUMAX_MAX + 1];   /* 1D values at this point, explicit formula */
                        for (int d = 0; d < 3; ++d)
                            for (int k = 0; k <= numax; ++k) f[d][k] = oracle_phi(k, u[d], sigma[a]);
                        double ang = 2.0 * ORACLE_PI * (kfrac ? (kfrac[0] * mx + kfrac[1] * my + kfrac[2] * mz) : 0.0);
                        double wr = cos(ang), wi = sin(ang);
                        for (int k = 0; k < nsel; ++k) {
                            const double* c = coeff + ((size_t)a * nbands + band_sel[k]) * nsho * cw;
                            double vre = 0.0, vim = 0.0;
                            int n = 0;
                            for (int nz = 0; nz <= numax; ++nz)
                                for (int ny = 0; ny <= numax - nz; ++ny)
                                    for (int nx = 0; nx <= numax - nz - ny; ++nx) {
                                        double p3 = f[2][nz] * f[1][ny] * f[0][nx];
                                        if (!is_complex) vre += c[n] * p3;
                                        else { vre += c[2 * n] * p3; vim += c[2 * n + 1] * p3; }
                                        ++n;
                                    }
                            if (!is_complex) {
                                o[k] += vre;
                            } else {
                                o[2 * k] += wr * vre + wi * vim;       /* conj(w) * v */
                                o[2 * k + 1] += wr * vim - wi * vre;
                            }
                        }
                    }
        }
    }
    free(lo); free(hi); free(empty);
    return 0;
}

/*
 * Step (2) of the non-local action: "Multiplication: d^a_ik = sum_j D^a_ij c^a_jk", with the
 * atomic matrix in the SHO representation, eq. (27)-(28) PAPER.md:252-262: "a real-valued matrix of
 * dimension N_SHO" per atom.
 *   D     [natoms][n][n]   real, row-major: D[a][i][j]
 *   c, d  [natoms][nbands][n] (x2 doubles if is_complex), the layout of the coefficients (reading A9)
 * Plain loops, one output at a time.
 */
int oracle_dmul(int natoms, int nbands, int n, int is_complex, const double* D, const double* c, double* d)
{
    if (natoms < 0 || nbands < 0 || n <= 0) return 1;
    const size_t cw = is_complex ? 2 : 1;
#pragma omp parallel for schedule(static)
    for (int a = 0; a < natoms; ++a)
        for (int b = 0; b < nbands; ++b) {
            const double* cv = c + ((size_t)a * nbands + b) * (size_t)n * cw;
            double* dv = d + ((size_t)a * nbands + b) * (size_t)n * cw;
            for (int i = 0; i < n; ++i) {
                double sre = 0.0, sim = 0.0;
                for (int j = 0; j < n; ++j) {
                    double Dij = D[((size_t)a * n + i) * (size_t)n + j];
                    if (!is_complex) sre += Dij * cv[j];
                    else { sre += Dij * cv[2 * j]; sim += Dij * cv[2 * j + 1]; }
                }
                if (!is_complex) dv[i] = sre;
                else { dv[2 * i] = sre; dv[2 * i + 1] = sim; }
            }
        }
    return 0;
}
