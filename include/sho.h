/*
 * sho.h -- C ABI of libsho: the PAW projection hot path with analytical Spherical-Harmonic-
 * Oscillator (SHO) projectors on one NVIDIA B200 (sm_100a).
 *
 * Method: Baumeister & Tsukamoto, "Analytical PAW Projector Functions for Reduced Bandwidth
 * Requirements", PASC'19 (arXiv:1905.00480).  Citations are PAPER.md:<line>.
 *
 *   projection  (step (1); eq. (25)-(26))
 *       c[a][b][n(nx,ny,nz)] = h^3 * sum_r psi_b(r) phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)
 *   expansion / add-back  (step (3))
 *       psi_b(r) += sum_a sum_n c[a][b][n] phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)
 *   with nx+ny+nz <= numax (eq. (17)-(18)) and phi_n the orthonormal 1D
 *   Hermite-Gauss function of width sigma_a (eq. (3)), sampled ON THE FLY with the
 *   three-term recurrence of eq. (31), PAPER.md:283-286 -- no projector table is read from memory.
 *   sho_project_stored is the paper's "USU" baseline: the same projection
 *   reading pre-sampled 3D projector tables from device memory.
 *
 * Conventions:
 *   - grid point i of axis d sits at x_i = i*h (Bohr); the cell is [0, N_d*h)
 *   - region of atom a: axis-aligned cube |u_d| <= rcut_sigma*sigma_a, inclusive:
 *       i_lo = ceil((R_d - rcut_sigma*sigma)/h), i_hi = floor((R_d + rcut_sigma*sigma)/h)
 *   - periodic axis: indices wrap (j = i mod N); isolated axis: psi == 0 outside, the box is clipped
 *   - Bloch phase: the value read at image m of axis d is multiplied by exp(2 pi i kfrac[d] m) in
 *     project and by its conjugate in add (complex dtypes only)
 *   - coefficient order: n = 0; for nz: for ny: for nx (nx fastest) with nx+ny+nz <= numax
 *   - layouts: psi [nbands][Nz][Ny][Nx] (x fastest); coeff [natoms][nbands][N_SHO] (n fastest);
 *     complex data interleaved (re,im) as in C99 / torch.complex128
 *   - h^3 volume element in project only (so sho_add == adjoint(sho_project) / h^3)
 *
 * Ownership / errors: the caller owns every buffer it passes; the library owns only the opaque
 * handles it returns.  Every function returns a status and never throws or aborts across the
 * boundary; sho_last_error() gives a thread-local detail string.  The DEVICE-pointer hot calls
 * (sho_project, sho_add, sho_project_stored) allocate nothing, are asynchronous on the given CUDA
 * stream and never synchronise the host.  psi must be finite on the whole grid (values just outside
 * a box are multiplied by exact zeros).  There is no CPU fallback: without a CUDA device every call
 * that needs one returns SHO_ERR_CUDA.  A plan belongs to the CUDA device that was current when it was
 * created: every hot call checks that this device is current and returns SHO_ERR_INVALID_ARG otherwise.
 * The only device-side abort is a watchdog: a kernel-internal barrier wait longer than 30 s of wall
 * time (a lost arrival, i.e. a library bug) traps, which the host sees as SHO_ERR_CUDA.
 */
#ifndef SHO_H_
#define SHO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SHO_NUMAX_MAX 15   /* nx+ny+nz <= numax <= 15 (N_SHO <= 816) */

typedef enum {
    SHO_OK = 0,
    SHO_ERR_INVALID_ARG = 1,  /* null pointer, h <= 0, sigma <= 0, numax out of range, dtype mismatch ... */
    SHO_ERR_UNSUPPORTED = 2,  /* valid problem the GPU path does not cover (e.g. periodic box wider than the cell) */
    SHO_ERR_OOM = 3,          /* device allocation failed / tables do not fit */
    SHO_ERR_CUDA = 4          /* CUDA runtime error, or no device */
} sho_status;

/* element type of psi and coeff; arithmetic is IEEE double for all four (fp32 data are widened on
 * load and rounded once on store) */
typedef enum { SHO_R64 = 0, SHO_C128 = 1, SHO_R32 = 2, SHO_C64 = 3 } sho_dtype;

typedef struct sho_plan sho_plan;     /* opaque, library-owned: geometry of one set of atoms on one grid */
typedef struct sho_tables sho_tables; /* opaque, library-owned: pre-sampled 3D projector tables          */
typedef struct sho_tables1d sho_tables1d; /* opaque, library-owned: pre-sampled 1D factor tables          */

/* eq. (18): (numax+1)(numax+2)(numax+3)/6; -1 if numax is outside [0, SHO_NUMAX_MAX] */
int sho_nsho(int numax);
/* position of (nx,ny,nz) in a coefficient vector (order above); -1 if not in the basis */
int sho_index(int nx, int ny, int nz, int numax);

const char* sho_status_string(sho_status s);
const char* sho_last_error(void);

/*
 * Build a plan (set-up, not part of the timed hot path): integer box ranges, wrap segments, the
 * spatially sorted atom order used for L2-friendly scheduling, and the tile -> atom-image lists that
 * let sho_add own each psi tile instead of using atomics.  Uses the current CUDA device.
 *   ng        HOST [3] = Nx, Ny, Nz (each >= 1)
 *   h         grid spacing in Bohr (> 0)
 *   periodic  HOST [3], 1 = periodic, 0 = isolated
 *   kfrac     HOST [3] Bloch phase per wrap = exp(2 pi i kfrac[d]); NULL = all zero.  Must be NULL or
 *             zero for real dtypes.
 *   natoms    >= 0;  pos HOST [natoms][3] (Bohr, any real value on periodic axes);  sigma HOST [natoms] (> 0)
 *   numax     0..SHO_NUMAX_MAX;  rcut_sigma > 0 (the configs use 6.0)
 * Returns SHO_ERR_UNSUPPORTED if a box on a periodic axis is wider than the cell.
 */
sho_status sho_plan_create(sho_plan** out, const int32_t ng[3], double h, const int32_t periodic[3],
                           const double kfrac[3], int32_t natoms, const double* pos, const double* sigma,
                           int32_t numax, double rcut_sigma, sho_dtype dtype);
sho_status sho_plan_destroy(sho_plan* plan);

/*
 * Tuning / test knobs of one plan.  They change launch shapes only, never results (the tests check bit identity).
 *   "project_bands_per_cta"  bands one CTA of sho_project works through with the tables it sampled once, 1..8;
 *                            0 = chosen per launch from the band count and the grid size (default)
 *   "host_chunk_bands"       bands per chunk of the *_host calls, >= 1; 0 = about 128 MB of psi per chunk (default)
 * SHO_ERR_INVALID_ARG for an unknown key or a value out of range.  Set options before the plan is used by hot calls
 * that may run at the same time on other host threads.
 */
sho_status sho_plan_set_option(sho_plan* plan, const char* key, int64_t value);

/* test hook: integer box ranges, HOST lo_hi[natoms][3][2] = (i_lo, i_hi) per axis (unwrapped) */
sho_status sho_plan_boxes(const sho_plan* plan, int32_t* lo_hi);

/* sizes: HOST info[8] = { natoms, N_SHO, numax, dtype, sum over atoms of box points, number of
 * non-empty add tiles, number of (tile, atom-image) pairs, atoms with a non-empty box } */
sho_status sho_plan_info(const sho_plan* plan, int64_t info[8]);

/*
 * Projection, on-the-fly SHO.  psi DEVICE [nbands][Nz][Ny][Nx]; coeff DEVICE [natoms][nbands][N_SHO]
 * (overwritten; atoms with an empty box get zeros).  cuda_stream is a cudaStream_t (NULL = default).
 * Deterministic (fixed summation order, no atomics).  One CTA projects one atom and 1..8 consecutive bands
 * (chosen per launch from the band count and the grid size; sho_plan_set_option "project_bands_per_cta" overrides
 * it -- a test knob, the result does not depend on it).
 */
sho_status sho_project(const sho_plan* plan, const void* psi, int32_t nbands, void* coeff, void* cuda_stream);

/* Expansion / add-back, on-the-fly SHO: psi += A coeff.  coeff DEVICE (read), psi DEVICE (in/out).
 * Deterministic: every psi value is accumulated by exactly one thread, the (atom, image) terms in the
 * fixed order of the plan's tile lists inside FP64 MMA accumulators, then added to psi once: two runs
 * give bit-identical results (the order is not "atoms ascending, one by one"). */
sho_status sho_add(const sho_plan* plan, const void* coeff, int32_t nbands, void* psi, void* cuda_stream);

/*
 * Stored-projector baseline (the paper's "USU" kernels).
 * sho_tables_build samples Phi_n(r - R_a) over every box into device memory (element type = the
 * real type of the plan's dtype).  *bytes_needed is always filled; if the tables do not fit in free
 * device memory the call returns SHO_ERR_OOM and *out = NULL.  Pass out = NULL to query the size only.
 * sho_project_stored adds the partial sums of the box's z segments in a fixed order (bit-reproducible); the small
 * hand-over counters it needs for that live in the tables object.  Calls that share one tables object may come from
 * any stream or host thread: the library chains them on the device (each launch waits for the one before it on
 * that object), so they are safe but do not overlap; use one tables object per stream to overlap them.  One call
 * covers at most 256 groups of 32 real columns per atom, i.e. nbands <= 8192 (real) or 4096 (complex); more bands
 * return SHO_ERR_UNSUPPORTED -- split the call (bands are independent).
 */
sho_status sho_tables_build(const sho_plan* plan, sho_tables** out, size_t* bytes_needed, void* cuda_stream);
sho_status sho_tables_destroy(sho_tables* tables);
sho_status sho_project_stored(const sho_plan* plan, const sho_tables* tables, const void* psi, int32_t nbands,
                              void* coeff, void* cuda_stream);

/*
 * Step (2) of the non-local action: d[a][b][i] = sum_j D[a][i][j] c[a][b][j], with the atomic
 * matrix in the SHO representation (eq. (27)-(28): "a real-valued matrix of dimension
 * N_SHO").  dmat DEVICE fp64 [natoms][N_SHO][N_SHO] row-major (D[a][i][j]; need not be symmetric), coeff_in
 * and coeff_out DEVICE [natoms][nbands][N_SHO] in the plan's dtype; coeff_out may be the same buffer as
 * coeff_in.  Asynchronous on the stream, allocates nothing.
 */
sho_status sho_dmul(const sho_plan* plan, const double* dmat, const void* coeff_in, int32_t nbands, void* coeff_out,
                    void* cuda_stream);

/*
 * Coefficients in the spherical representation (nr, l, m) (f4; eq. (10)-(11)): the unitary
 * transform U between the Cartesian eigenstates Psi_{nx ny nz} and the spherical ones Psi_{nr l m} = R_{nr l}(r/sigma)
 * Y_lm (eq. (7)-(8)).  The paper gives no formula for its elements; sho_umatrix evaluates the overlap
 * integrals exactly (host code, Gauss-Hermite).  Conventions (readings A17-A19): spherical index ordered by
 * nu = l + 2 nr ascending, then nr ascending (l descending), then m = -l..l; REAL spherical harmonics with positive
 * factors (Y_1,-1 ~ y, Y_10 ~ z, Y_11 ~ x); R_{nr l} > 0 at the origin.  U is real orthogonal and vanishes outside
 * the nu-blocks (eq. (11)).
 *   sho_rlm_index  position of (nr, l, m) in that order, -1 if not in the basis
 *   sho_umatrix    u HOST [N_SHO][N_SHO] row-major: u[rlm][sho_index(nx,ny,nz)]
 *   sho_transform  coeff_out[a][b][i] = sum_j umat[i][j] coeff_in[a][b][j] for every atom and band (umat DEVICE fp64
 *                  [N_SHO][N_SHO]; pass U for Cartesian -> spherical, its transpose for the way back; coeff_out may be
 *                  coeff_in).  Runs the batched tensor-core GEMM of sho_dmul with one shared matrix.
 */
int sho_rlm_index(int nr, int l, int m, int numax);
sho_status sho_umatrix(int numax, double* u);
sho_status sho_transform(const sho_plan* plan, const double* umat, const void* coeff_in, int32_t nbands, void* coeff_out,
                         void* cuda_stream);

/*
 * The three steps of PAPER.md:187-190 in one call: c = project(psi); d = D c; psi += add(d), on one stream.
 * psi DEVICE in/out, coeff_work DEVICE [natoms][nbands][N_SHO] caller-owned scratch (holds d on return).
 */
sho_status sho_apply(const sho_plan* plan, const double* dmat, void* psi, int32_t nbands, void* coeff_work,
                     void* cuda_stream);

/*
 * The stored add-back, the paper's "USUadd" (tab. 1): psi += A coeff reading the same
 * pre-sampled 3D tables as sho_project_stored.  A baseline: its results meet in psi by atomicAdd, so it
 * is correct to rounding but not bit-reproducible.
 */
sho_status sho_add_stored(const sho_plan* plan, const sho_tables* tables, const void* coeff, int32_t nbands, void* psi,
                          void* cuda_stream);

/*
 * Stored-1D-table separable variant (sec. 3.4, eq. (22)-(23)): the same separable kernels
 * as sho_project / sho_add, but the 1D factor values phi_n(u) of every atom and box index are read from
 * device memory (pre-sampled by sho_tables1d_build: (n_x + n_y + n_z)(numax + 1) doubles per atom) instead
 * of being generated by the recurrence.  Separates the gain of factorisation from the gain of on-the-fly
 * sampling.  *bytes_needed is always filled; out = NULL queries the size only.
 */
sho_status sho_tables1d_build(const sho_plan* plan, sho_tables1d** out, size_t* bytes_needed, void* cuda_stream);
sho_status sho_tables1d_destroy(sho_tables1d* tables);
sho_status sho_project_stored1d(const sho_plan* plan, const sho_tables1d* tables, const void* psi, int32_t nbands,
                                void* coeff, void* cuda_stream);
sho_status sho_add_stored1d(const sho_plan* plan, const sho_tables1d* tables, const void* coeff, int32_t nbands,
                            void* psi, void* cuda_stream);

/*
 * Band-fastest psi layout psi_bf[Nz][Ny][Nx][nbands] -- the layout of the paper's own kernels, which vectorise
 * over the band index.  The kernels of this library read x-fastest data, so these calls convert
 * chunks of bands into the caller's workspace `work` (DEVICE, work_bytes >= the bytes of one band; an even number
 * of bands per chunk is used when it fits) with a tiled transpose, run the same kernels on the chunk and, for
 * the add-back, accumulate the chunk's increment into psi_bf with the inverse transpose.  coeff keeps the layout
 * [natoms][nbands][N_SHO].  Asynchronous on the stream, allocates nothing.  SHO_ERR_INVALID_ARG if the workspace
 * does not hold one band.
 */
sho_status sho_project_bf(const sho_plan* plan, const void* psi_bf, int32_t nbands, void* coeff, void* work, size_t work_bytes,
                          void* cuda_stream);
sho_status sho_add_bf(const sho_plan* plan, const void* coeff, int32_t nbands, void* psi_bf, void* work, size_t work_bytes,
                      void* cuda_stream);

/*
 * sho_project_bf for callers that cannot bring a workspace.  Same arguments, same result as sho_project_bf, but the
 * chunks of bands are converted in a fixed workspace of SHO_STATIC_WORK_BYTES that is part of the library image
 * instead of one the caller allocates.
 *
 * Who needs this: code that is handed psi and coeff by a host application and has no device memory of its own to
 * lend -- a plug-in inside a DFT program that gave all of the GPU's memory to its own arena at start-up (cudaMalloc
 * then fails), or a routine that is called while the application's other streams are busy (cudaMalloc and cudaFree
 * synchronise the whole device and would stall them).  This call never calls cudaMalloc, cudaFree or any library
 * routine that allocates; the plan it takes was created earlier, at a time when allocating was still possible.
 *
 * Limit: one band of the plan's grid, Nx*Ny*Nz*sizeof(element), must fit in SHO_STATIC_WORK_BYTES (32 MiB: e.g.
 * 128^3 real fp64, the paper's 64^3 grid in every dtype); a larger grid returns SHO_ERR_UNSUPPORTED with the sizes in
 * sho_last_error(), and nothing is launched.  As many bands per chunk as fit are used (the paper's 64^3 fp64
 * grid: 16).
 * Cost: every GPU on which the library's module is loaded holds these 32 MiB until the process exits, whether or
 * not this function is ever called.
 * First call: the first call on each device (with that device current) looks up the device address of the
 * workspace (cudaGetSymbolAddress; this may make the runtime load the library's module) and caches it; make that
 * first call during set-up, before any stream capture begins.
 * Sharing: all calls on one device share the one workspace, which keeps whatever the last call left in it.  This
 * entry point does not depend on those contents (each chunk is fully written before it is read), but two calls
 * whose kernels can overlap on the GPU -- different streams, or different host threads on different streams --
 * race on it and give wrong coefficients: keep all calls on one device on one stream, or order them with events.
 * Asynchronous on the stream otherwise, like sho_project_bf.
 */
#define SHO_STATIC_WORK_BYTES (32u << 20)
sho_status sho_project_bf_static(const sho_plan* plan, const void* psi_bf, int32_t nbands, void* coeff, void* cuda_stream);

/*
 * End-to-end variants with HOST buffers (pinned or pageable): copy in, run the same kernels, copy
 * out, and synchronise the stream before returning.  They use a device workspace owned by the plan
 * (the only hot-path calls that may allocate; it is grown on demand and bounded by the chunk size, not
 * by nbands).  The bands are independent (eq. (25)), so the calls work in chunks of bands
 * (about 128 MB of psi each; sho_plan_set_option "host_chunk_bands" overrides the chunk size)
 * through a ring of three chunk buffers and overlap the H2D copy of the next chunk, the kernels of this
 * one and the D2H copy of the previous one on two copy streams owned by the plan; all of it is ordered
 * after the work already queued on cuda_stream.  If a step fails mid-way the call waits for everything
 * it has queued before it returns the error.
 *   sho_project_host: psi HOST (read), coeff HOST (written)
 *   sho_add_host:     coeff HOST (read), psi HOST (in/out)
 *   sho_apply_host:   dmat HOST fp64 [natoms][N_SHO][N_SHO], psi HOST (in/out): psi is uploaded ONCE,
 *                     project -> D -> add run on the device, psi is downloaded once; the coefficients
 *                     never leave the device
 */
sho_status sho_project_host(sho_plan* plan, const void* psi_host, int32_t nbands, void* coeff_host, void* cuda_stream);
sho_status sho_add_host(sho_plan* plan, const void* coeff_host, int32_t nbands, void* psi_host, void* cuda_stream);
sho_status sho_apply_host(sho_plan* plan, const double* dmat_host, void* psi_host, int32_t nbands, void* cuda_stream);

/* FP64 FMA-pipe micro-benchmark used by bench.py for the roofline denominator: runs `iters` rounds of
 * eight independent DFMA chains per thread on every SM and returns the achieved FLOP/s in *flops_per_s
 * (synchronises).  DMMA.8x8x4 shares that pipe at the same rate. */
sho_status sho_measure_fp64_peak(int32_t iters, double* flops_per_s);

#ifdef __cplusplus
}
#endif
#endif /* SHO_H_ */
