// sho_project.cu -- on-the-fly SHO projection (steps a1-a5 of DESIGN.md), one CTA per (atom, band).
//
//   c[a][b][n(nx,ny,nz)] = h^3 sum_r psi_b(r) phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)
//                                                       eq. (25)-(26); step (1)
//
// Design (B200, sm_100a): the separable contraction runs x -> y -> z, as the paper's eq. (26) is written.
//   a1  every CTA samples the three 1D Hermite-Gauss tables of its atom on the fly (eq. (31)) straight
//       into shared memory, already laid out as FP64 tensor-core fragments; nothing but 80 B of atom
//       parameters is read from HBM for the projectors.
//   a2  psi is read straight from global memory / L2 with 32-byte loads (LDG.256): lane (q,t) of a warp
//       reads 32 contiguous bytes of row q, four lanes cover one 128-byte line, a warp load covers
//       8 rows x 128 B.  The loaded registers ARE the B fragments of the first contraction (K = x,
//       N = 8 rows), so no shared-memory staging or transposition is needed, and the L1 data pipe moves
//       a full line per wavefront (the earlier K = y layout touched 16 lines per 512 B and was bound by
//       that pipe, measured in round 1).  Periodic wrap / isolated clipping are
//       per-lane index arithmetic from two small offset tables.  The loads run one group of G steps
//       ahead of the arithmetic (register double buffer) and the ring runs on across row-block ends and
//       plane ends, so loads stay in flight over the y stage, a5 and its barrier.
//   a3  first-axis (x) contraction: DMMA.8x8x4, M = nx, K = 4 columns, N = 8 rows.  With numax = 8, 9
//       (M = 9, 10) a second, mostly empty MMA row tile would cost 1.6x the algorithmic flops, so the
//       R = 2 remainder rows nx = 8, 9 run as plain DFMAs on the same loaded values instead (template
//       parameter R): per lane a partial over its own columns, reduced once per plane.
//   a4  second-axis (y) contraction: the accumulator fragment of a3 is directly the A fragment of a
//       second DMMA against the phi_ny table (the K order inside an MMA is free).  For R = 2 the six
//       (nx,ny) outputs with nx or ny in {8, 9} are DFMA partials per lane.
//   a5  third axis: each warp owns one z-plane per round; the per-plane T2[nx][ny] meet in shared
//       memory and thread n accumulates c[n] += phi_nz(z) * T2[nx][ny] in a register.  The T2
//       planes go through four mbarrier-guarded buffers, the consumers one round behind the producers (no
//       __syncthreads in the round loop); coalesced store of N_SHO coefficients at the end.
// Bloch phases never touch the inner loop: the x-phase is one accumulator rotation at the wrap column,
// y-phases rotate the a3 accumulators per row, the z-phase (and the last x image) is folded into a5.
#include <algorithm>
#include <cstdlib>

#include "sho_device.cuh"

namespace sho {

constexpr int kProjG = 2;      // loads (of 8 rows x 128 B) per group of the register load ring

struct ProjParams {
    GridDev g;
    const void* psi;
    void* coeff;
    const AtomDev* atoms;
    const int32_t* order;
    const uint32_t* nxyz;
    const double* tab1d;       // stored 1D tables (sho_project_stored1d), or null: sample on the fly
    const long long* tab1d_off;
    int32_t nbands;
    int32_t cnb;               // bands per atom in the coefficient array (>= nbands: a chunk of a wider array)
    int32_t n_work_atoms;      // atoms with a non-empty box (first entries of order[])
    int32_t bands_per_cta;     // consecutive bands one CTA projects with the tables it sampled once
    int32_t kx_cap, yb_cap, nz_cap;    // capacities of the shared tables: x steps, 8-row blocks, planes
    int32_t xalign_span;       // x steps start at a lane-span boundary instead of a 128-byte line (plan statistic)
    int32_t fast;              // 32-byte loads are legal: psi 32-byte aligned and Nx a multiple of the lane span
    long long band_stride;     // elements between bands
};

// per element type: EPL elements of 32 bytes per lane and load; a step covers CWX = 4 EPL columns
template <int DT> struct ProjElem;
template <> struct ProjElem<SHO_C128> { static constexpr int EPL = 2; };
template <> struct ProjElem<SHO_R64>  { static constexpr int EPL = 4; };
template <> struct ProjElem<SHO_C64>  { static constexpr int EPL = 4; };
template <> struct ProjElem<SHO_R32>  { static constexpr int EPL = 8; };

// shared-memory carve-up (doubles unless noted); every block starts 16-byte aligned
template <int MT, int R, int DT>
struct ProjSmem {
    static constexpr int P = Elem<DT>::cplx ? 2 : 1;
    static constexpr int EPL = ProjElem<DT>::EPL;
    static constexpr int CWX = 4 * EPL;
    static constexpr int MP = 8 * MT;                       // nx / ny rows on the MMA
    static constexpr int NV = MP + R;                       // functions sampled per point
    static constexpr int TS = MP * MP + (R ? 8 : 0);        // one part of one plane's T2 (+ the R specials)
    static __host__ __device__ size_t fx(int kx) { return (size_t)kx * EPL * MT * 32; }       // A fragments, x stage
    static __host__ __device__ size_t fxr(int kx) { return R ? (size_t)kx * CWX * 2 : 0; }    // phi_8, phi_9 per column
    static __host__ __device__ size_t fy(int yb) { return (size_t)yb * 2 * MT * 32; }         // B fragments, y stage
    static __host__ __device__ size_t fys(int yb) { return R ? (size_t)yb * 8 * 4 : 0; }      // phi_0,1,8,9 per row
    static __host__ __device__ size_t wy(int yb) { return Elem<DT>::cplx ? (size_t)yb * 8 * 2 : 0; }
    static __host__ __device__ size_t fz(int nz) { return (size_t)nz * NV + (((size_t)nz * NV) & 1); }
    static __host__ __device__ size_t wz(int nz) { return Elem<DT>::cplx ? (size_t)nz * 2 : 0; }
    static __host__ __device__ size_t t2() { return (size_t)4 * kProjWarps * P * TS; }
    static __host__ __device__ size_t ints(int kx, int yb) { return (size_t)yb * 8 + (size_t)(kx + kProjG) * 4 + 4; }
    static __host__ __device__ size_t total_bytes(int kx, int yb, int nz)
    {
        return 8 * (fx(kx) + fxr(kx) + fy(yb) + fys(yb) + wy(yb) + fz(nz) + wz(nz) + t2() + 2 + 4) + 4 * ints(kx, yb) + 16;
    }
};

// position of T2[nx][ny] inside one part of a plane's shared T2 block
template <int MT, int R>
__device__ __forceinline__ int t2_index(int nx, int ny)
{
    constexpr int MP = 8 * MT;
    if (R == 0 || (nx < MP && ny < MP)) return nx * MP + ny;
    if (nx == MP) return MP * MP + ny;            // (8,0) (8,1)
    if (nx == MP + 1) return MP * MP + 2;         // (9,0)
    if (ny == MP) return MP * MP + 3 + 2 * nx;    // (0,8) -> 3, (1,8) -> 5
    return MP * MP + 4;                           // (0,9)
}

// 32 bytes per lane, read-only path (SASS: LDG.E.256.CONSTANT)
__device__ __forceinline__ void ldg256(const double* p, double (&r)[4])
{
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r[0]), "=d"(r[1]), "=d"(r[2]), "=d"(r[3]) : "l"(p));
}
__device__ __forceinline__ void ldg256(const float* p, float (&r)[8])
{
    asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7])
                 : "l"(p));
}

template <int MT, int R, int DT, int G, int MB>
// MB = 1: the CTA projects several bands one after the other (the band loop below); MB = 0: one band, no loop
// three CTAs per SM for real data without remainder rows (80 registers; measured faster), two for complex data and for
// real data with remainder rows (at 80 registers those spill: numax 9 on cfg 4's geometry 40.1 ms against 37.4 with two CTAs)
__global__ void __launch_bounds__(kProjWarps * 32, (DT == SHO_C128 || DT == SHO_C64 || MT == 2 || R > 0) ? 2 : 3) sho_project_kernel(const ProjParams p)
{
    using E = Elem<DT>;
    using S = ProjSmem<MT, R, DT>;
    using real_t = typename E::real_t;
    constexpr bool CPLX = E::cplx;
    constexpr int P = CPLX ? 2 : 1;
    constexpr int EPL = S::EPL, CWX = S::CWX;
    constexpr int RAW = 32 / (int)sizeof(real_t);           // reals per lane and load
    constexpr int MP = S::MP, NV = S::NV, TS = S::TS;
    constexpr int NACC = (MT == 1) ? 1 : (816 + kProjWarps * 32 - 1) / (kProjWarps * 32);   // numax <= 9: N_SHO <= 220

    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* fx = reinterpret_cast<double*>(smem_raw);                 // [step][e][mt][32]  A fragments of the x stage
    double* fxr = fx + S::fx(p.kx_cap);                               // [column][2]        phi_8, phi_9 of the R rows
    double* fy = fxr + S::fxr(p.kx_cap);                              // [block][s][mt][32] B fragments of the y stage
    double* fys = fy + S::fy(p.yb_cap);                               // [row][4]           phi_0, phi_1, phi_8, phi_9
    double* wy = fys + S::fys(p.yb_cap);                              // complex only: [row][2] Bloch phase of the row
    double* fz = wy + S::wy(p.yb_cap);                                // [z][NV]
    double* wz = fz + S::fz(p.nz_cap);                                // complex only: [z][2]
    double* t2s = wz + S::wz(p.nz_cap);                               // [2][W][P][TS]
    double* phx = t2s + S::t2();                                      // x rotation exp(-2 pi i kfrac_x) [re,im]
    uint64_t* t2bar = reinterpret_cast<uint64_t*>(phx + 2);           // [4] one mbarrier per T2 buffer: its 8 planes are written
    int32_t* rowoff = reinterpret_cast<int32_t*>(phx + 2 + 4);            // [padded row] element offset of the row
    int32_t* coloff = rowoff + (size_t)p.yb_cap * 8;                  // [group][t][step in group] element offset of the lane span

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int q = lane >> 2, t = lane & 3;

    // work item: (group of bands_per_cta consecutive bands, atom), band-group-major, atoms in the plan's spatial order
    // (neighbouring CTAs share psi in L2).  The CTA samples its atom's tables once and projects the bands one by one.
    const int bgrp = blockIdx.x / p.n_work_atoms;
    const int a = p.order[blockIdx.x - bgrp * p.n_work_atoms];
    const int b_first = MB ? bgrp * p.bands_per_cta : bgrp;
    const int b_end = MB ? min(b_first + p.bands_per_cta, p.nbands) : b_first + 1;
    const AtomDev at = p.atoms[a];
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int numax = p.g.numax;
    const bool fast = p.fast != 0;

    const int nyl = at.hi[1] - at.lo[1] + 1, nzl = at.hi[2] - at.lo[2] + 1;
    // x: steps of CWX columns (128 bytes per row).  They start at a 128-byte line, or -- when the plan found that this
    // saves more than a tenth of the steps -- at the lane-span boundary (32 bytes) at or before the box: such a step
    // touches two lines per row but the same sectors (cfg 3: 4 steps instead of 4.75 on average, 1.90 -> 1.54 ms;
    // cfg 4: 8 instead of 8.5, but 2 % slower: its L1 data pipe is 89 % busy, so it keeps line-aligned steps)
    const int xalign = p.xalign_span ? EPL : CWX;
    const int xs0 = floordiv(at.lo[0], xalign) * xalign;
    const int KX = (at.hi[0] - xs0 + CWX) / CWX;
    // y: blocks of 8 rows (the N extent of the x-stage MMA)
    const int NYB = (nyl + 7) >> 3;
    // complex data with an x-wrap: the accumulators are rotated by exp(-2 pi i kfrac_x) once, before the first
    // step of the second image; the phase of the last image is folded into wz.  If the image boundary falls
    // inside a step, that step is scheduled twice with complementary column masks in its tables, so the inner
    // loop never looks at single columns.  Schedule: KS steps, step k reads the columns of source step
    // k - (k > kdup); the rotation happens before step krot.
    const bool xphase = CPLX && p.g.has_phase && p.g.periodic[0] && p.g.kfrac[0] != 0.0;
    const bool yphase = CPLX && p.g.has_phase && p.g.periodic[1] && p.g.kfrac[1] != 0.0;
    int xB = INT_MAX, krot = -1, kdup = INT_MAX;
    if (xphase) {
        const int mlo = floordiv(at.lo[0], Nx);
        if (floordiv(at.hi[0], Nx) != mlo) {
            xB = (mlo + 1) * Nx;
            krot = (xB - xs0) / CWX;
            if ((xB - xs0) % CWX != 0) { kdup = krot; krot += 1; }
        }
    }
    const int KS = KX + (kdup != INT_MAX ? 1 : 0);
    // row blocks that hold rows of a y image other than the home cell (the only ones whose phase is not 1)
    int yrot_lo = 0, yrot_hi = -1;
    if (yphase) {
        const int mlo = floordiv(at.lo[1], Ny), mhi = floordiv(at.hi[1], Ny);
        if (mlo != 0 && mhi != 0) { yrot_lo = 0; yrot_hi = NYB - 1; }
        else if (mhi != 0) { yrot_lo = (Ny - at.lo[1]) >> 3; yrot_hi = NYB - 1; }
        else if (mlo != 0) { yrot_lo = 0; yrot_hi = (-at.lo[1] - 1) >> 3; }
    }
    const int KXG = (KS + G - 1) / G;

    // ---------------- a1: sample the 1D tables on the fly, in fragment layout ----------------
    const int nx_items = KS * CWX, ny_items = NYB * 8;
    for (int it = tid; it < nx_items + ny_items + nzl; it += blockDim.x) {
        double v[NV];
        if (it < nx_items) {
            const int k = it / CWX, r = it % CWX, tt = r / EPL, e = r % EPL;      // column r of the step = EPL * t + e
            const int ix = xs0 + CWX * (k - (k > kdup ? 1 : 0)) + r;
            const bool valid = ix >= at.lo[0] && ix <= at.hi[0] &&
                               (kdup == INT_MAX || (k < krot ? ix < xB : ix >= xB));
            if (p.tab1d) stored1d_lookup<NV>(p.tab1d, p.tab1d_off[a], at.lo, at.hi, 0, ix, numax, valid, v);
            else hermite_gauss<NV>(displacement(ix, p.g.h, at.pos[0]), at, p.g.hnorm, numax, valid, v);
            // A fragments [step][mt][e / 2][lane = 4 nx + t][e & 1]: 16-byte loads, lanes 16 bytes apart (no bank conflicts)
#pragma unroll
            for (int n = 0; n < MP; ++n)
                fx[((((size_t)k * MT + (n >> 3)) * (EPL / 2) + (e >> 1)) * 32 + (n & 7) * 4 + tt) * 2 + (e & 1)] = v[n];
            if (R) { fxr[2 * it] = v[MP]; fxr[2 * it + 1] = v[MP + R - 1]; }
        } else if (it < nx_items + ny_items) {
            const int pr = it - nx_items;                        // padded row slot
            int iy = at.lo[1] + pr;
            const bool valid = iy <= at.hi[1];
            if (!valid) iy = at.hi[1];
            if (p.tab1d) stored1d_lookup<NV>(p.tab1d, p.tab1d_off[a], at.lo, at.hi, 1, iy, numax, valid, v);
            else hermite_gauss<NV>(displacement(iy, p.g.h, at.pos[1]), at, p.g.hnorm, numax, valid, v);
            const int yb = pr >> 3, r = pr & 7, tt = r >> 1, s = r & 1;          // row r of the block = 2 t + s
#pragma unroll
            for (int n = 0; n < MP; ++n) fy[(((size_t)yb * 2 + s) * MT + (n >> 3)) * 32 + (n & 7) * 4 + tt] = v[n];
            if (R) { fys[4 * pr] = v[0]; fys[4 * pr + 1] = v[1]; fys[4 * pr + 2] = v[MP]; fys[4 * pr + 3] = v[MP + R - 1]; }
            const int my = p.g.periodic[1] ? floordiv(iy, Ny) : 0;
            const int jy = p.g.periodic[1] ? iy - my * Ny : min(max(iy, 0), Ny - 1);
            rowoff[pr] = jy * Nx;
            if (CPLX) {
                double sn = 0.0, cs = 1.0;
                if (yphase) sincospi(2.0 * p.g.kfrac[1] * (double)my, &sn, &cs);
                wy[2 * pr] = cs; wy[2 * pr + 1] = sn;
            }
        } else {
            const int zi = it - nx_items - ny_items;
            const int iz = at.lo[2] + zi;
            if (p.tab1d) stored1d_lookup<NV>(p.tab1d, p.tab1d_off[a], at.lo, at.hi, 2, iz, numax, true, v);
            else hermite_gauss<NV>(displacement(iz, p.g.h, at.pos[2]), at, p.g.hnorm, numax, true, v);
#pragma unroll
            for (int n = 0; n < NV; ++n) fz[(size_t)zi * NV + n] = v[n];
            if (CPLX) {
                // phase of image m_z, times the phase of the last x image
                double ang = 0.0;
                if (p.g.has_phase) {
                    if (p.g.periodic[2]) ang += p.g.kfrac[2] * (double)floordiv(iz, Nz);
                    if (p.g.periodic[0]) ang += p.g.kfrac[0] * (double)floordiv(at.hi[0], Nx);
                }
                double sn, cs;
                sincospi(2.0 * ang, &sn, &cs);
                wz[2 * zi] = cs; wz[2 * zi + 1] = sn;
            }
        }
    }
    // lane-span offsets of every scheduled step (the steps that pad the last group repeat the last real step)
    for (int it = tid; it < KXG * G * 4; it += blockDim.x) {
        const int k = min(it >> 2, KS - 1), tt = it & 3;
        const int x0 = xs0 + CWX * (k - (k > kdup ? 1 : 0)) + EPL * tt;
        const int off = p.g.periodic[0] ? x0 - floordiv(x0, Nx) * Nx : min(max(x0, 0), max(Nx - EPL, 0));
        coloff[(((it >> 2) / G) * 4 + tt) * G + ((it >> 2) % G)] = off;
    }
    if (CPLX && tid == 0) {
        double sn, cs;
        sincospi(-2.0 * p.g.kfrac[0], &sn, &cs);
        phx[0] = cs; phx[1] = sn;
    }
    if (tid == 0) {
        for (int i = 0; i < 4; ++i) mbar_init(t2bar + i, kProjWarps);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    const size_t plane = (size_t)Ny * Nx;

    // a5 accumulators: thread n owns coefficient(s) n, n + blockDim, ...
    double acc[NACC][P];
    int myt2[NACC], mynz[NACC];
#pragma unroll
    for (int j = 0; j < NACC; ++j) {
        const int n = tid + j * blockDim.x;
        const uint32_t pk = (n < p.g.nsho) ? p.nxyz[n] : 0u;
        myt2[j] = t2_index<MT, R>(pk & 255, (pk >> 8) & 255);
        mynz[j] = (pk >> 16) & 255;
    }
    const int nrounds = (nzl + kProjWarps - 1) / kProjWarps;
    const double h3 = p.g.h * p.g.h * p.g.h;

    // The bands of the group, one after the other.  The T2 buffers and their mbarriers run on across bands: the rounds
    // are numbered through (rbase + round), so buffer and parity continue where the band before stopped.
  for (int b = b_first, rbase = 0; b < b_end; ++b, rbase += nrounds) {
    const real_t* psi_b = reinterpret_cast<const real_t*>(p.psi) + (size_t)b * p.band_stride * P;
#pragma unroll
    for (int j = 0; j < NACC; ++j)
#pragma unroll
        for (int pp = 0; pp < P; ++pp) acc[j][pp] = 0.0;

    // ---- a2 helpers: plane pointer, this lane's row pointer of a row block, one group of loads ----
    auto plane_ptr = [&](int zi) -> const real_t* {
        const int iz = at.lo[2] + zi;
        const int jz = p.g.periodic[2] ? iz - floordiv(iz, Nz) * Nz : iz;
        return psi_b + (size_t)jz * plane * P;
    };
    auto row_ptr = [&](const real_t* pzz, int yb) -> const real_t* { return pzz + (size_t)rowoff[yb * 8 + q] * P; };
    // G consecutive x steps of one row block: lane (q,t) reads columns EPL t .. EPL t + EPL - 1 of row q
    auto load_group = [&](real_t (&raw)[G][RAW], const real_t* rp, int kg) {
        if (fast) {
            int co[G];
            if (G == 2) {
                const int2 c2 = *reinterpret_cast<const int2*>(coloff + (kg * 4 + t) * G);
                co[0] = c2.x; co[G - 1] = c2.y;
            } else {
#pragma unroll
                for (int j = 0; j < G; ++j) co[j] = coloff[(kg * 4 + t) * G + j];
            }
#pragma unroll
            for (int j = 0; j < G; ++j) ldg256(rp + (size_t)co[j] * P, raw[j]);
        } else {
            // unaligned psi or Nx not a multiple of the lane span: element-wise loads, every column wrapped
#pragma unroll
            for (int j = 0; j < G; ++j) {
                const int ks_ = min(kg * G + j, KS - 1);
                const int x0 = xs0 + CWX * (ks_ - (ks_ > kdup ? 1 : 0)) + EPL * t;
#pragma unroll
                for (int e = 0; e < EPL; ++e) {
                    const int ix = x0 + e;
                    const int off = p.g.periodic[0] ? ix - floordiv(ix, Nx) * Nx : min(max(ix, 0), Nx - 1);
#pragma unroll
                    for (int pp = 0; pp < P; ++pp) raw[j][e * P + pp] = __ldg(rp + (size_t)off * P + pp);
                }
            }
        }
    };

    // The load ring: while the G steps in cur are contracted, the next G steps are in flight; the ring
    // runs on across row-block ends (over the y stage) and plane ends (over a5 and its barrier).
    real_t cur[G][RAW];
    const real_t* rp = psi_b;                    // row pointer of the current row block for this lane
#pragma unroll
    for (int j = 0; j < G; ++j)
#pragma unroll
        for (int i = 0; i < RAW; ++i) cur[j][i] = (real_t)0;
    if (warp < nzl) {
        rp = row_ptr(plane_ptr(warp), 0);
        load_group(cur, rp, 0);
    }
    // ---- a5: z contraction of the 8 planes of one round, thread n <- coefficient n ----
    auto a5 = [&](int rnd) {
        const double* t2r = t2s + (size_t)((rbase + rnd) & 3) * kProjWarps * P * TS;
        const int wmax = min(kProjWarps, nzl - rnd * kProjWarps);
#pragma unroll
        for (int j = 0; j < NACC; ++j) {
            const int n = tid + j * blockDim.x;
            if (n < p.g.nsho) {
                for (int w = 0; w < wmax; ++w) {
                    const int z2 = rnd * kProjWarps + w;
                    const double f = fz[(size_t)z2 * NV + mynz[j]];
                    const double* tt = t2r + (size_t)w * P * TS + myt2[j];
                    if (!CPLX) {
                        acc[j][0] = fma(f, tt[0], acc[j][0]);
                    } else {
                        const double re = tt[0], im = tt[TS];
                        const double cr = wz[2 * z2], ci = wz[2 * z2 + 1];
                        acc[j][0] = fma(f, re * cr - im * ci, acc[j][0]);
                        acc[j][P - 1] = fma(f, re * ci + im * cr, acc[j][P - 1]);
                    }
                }
            }
        }
    };

    for (int round = 0; round < nrounds; ++round) {
        const int zi = round * kProjWarps + warp;
        double* t2w = t2s + ((size_t)((rbase + round) & 3) * kProjWarps + warp) * P * TS;
        if (zi < nzl) {
            const real_t* pz = plane_ptr(zi);
            const real_t* pzn = (zi + kProjWarps < nzl) ? plane_ptr(zi + kProjWarps) : pz;

            // T2[part][tx][ty]: tile (1,1) can only hold nx+ny >= 16 > numax and is never needed
            double T2[P][MT][MT][2];
#pragma unroll
            for (int pp = 0; pp < P; ++pp)
#pragma unroll
                for (int tx = 0; tx < MT; ++tx)
#pragma unroll
                    for (int ty = 0; ty < MT; ++ty) T2[pp][tx][ty][0] = T2[pp][tx][ty][1] = 0.0;
            // R specials, per-lane partials: rs = T2[8][0], T2[8][1], T2[9][0]; cs = T2[q][8], T2[q][9]
            double rs[3][P], cs[2][P];
#pragma unroll
            for (int pp = 0; pp < P; ++pp) { rs[0][pp] = rs[1][pp] = rs[2][pp] = 0.0; cs[0][pp] = cs[1][pp] = 0.0; }

            for (int yb = 0; yb < NYB; ++yb) {
                // where the ring goes after this row block: the next block, or block 0 of this warp's next plane
                const real_t* nrp = (yb + 1 < NYB) ? row_ptr(pz, yb + 1) : row_ptr(pzn, 0);

                double C1[MT][2][2];   // [nx tile][re/im, or even/odd column for real data][s]
                double ar[2][2];       // R rows: [nx = 8, 9][re/im], partial over this lane's columns
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) C1[mt][0][0] = C1[mt][0][1] = C1[mt][1][0] = C1[mt][1][1] = 0.0;
                ar[0][0] = ar[0][1] = ar[1][0] = ar[1][1] = 0.0;

                // this lane's table pointers, advanced by a constant per step (no address arithmetic in the loop)
                const double* fxp = fx + (size_t)lane * 2;
                const double* fxrp = fxr + (size_t)t * EPL * 2;
                auto compute_group = [&](const real_t (&buf)[G][RAW], int kg) {
#pragma unroll
                    for (int j = 0; j < G; ++j) {
                        const int k = kg * G + j;
                        if (k < KS) {
                            if (CPLX && k == krot) {
                                // the columns so far belong to the previous x image: rotate what they have summed
                                const double cr = phx[0], ci = phx[1];
#pragma unroll
                                for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                                    for (int s = 0; s < 2; ++s) {
                                        const double re = C1[mt][0][s], im = C1[mt][1][s];
                                        C1[mt][0][s] = re * cr - im * ci;
                                        C1[mt][1][s] = re * ci + im * cr;
                                    }
                                if (R) {
#pragma unroll
                                    for (int i = 0; i < 2; ++i) {
                                        const double re = ar[i][0], im = ar[i][1];
                                        ar[i][0] = re * cr - im * ci;
                                        ar[i][1] = re * ci + im * cr;
                                    }
                                }
                            }
                            // ---- a3: x contraction, EPL K steps of 4 columns ----
                            double afr[MT][EPL];
#pragma unroll
                            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                                for (int eh = 0; eh < EPL / 2; ++eh) {
                                    const double2 a2 = *reinterpret_cast<const double2*>(fxp + (mt * (EPL / 2) + eh) * 64);
                                    afr[mt][2 * eh] = a2.x; afr[mt][2 * eh + 1] = a2.y;
                                }
#pragma unroll
                            for (int e = 0; e < EPL; ++e) {
                                double ve[P];
#pragma unroll
                                for (int pp = 0; pp < P; ++pp) ve[pp] = (double)buf[j][e * P + pp];
#pragma unroll
                                for (int mt = 0; mt < MT; ++mt) {
                                    if (CPLX) {
                                        dmma(C1[mt][0][0], C1[mt][0][1], afr[mt][e], ve[0]);
                                        dmma(C1[mt][1][0], C1[mt][1][1], afr[mt][e], ve[P - 1]);
                                    } else {
                                        dmma(C1[mt][e & 1][0], C1[mt][e & 1][1], afr[mt][e], ve[0]);
                                    }
                                }
                                if (R) {
                                    const double2 f = *reinterpret_cast<const double2*>(fxrp + 2 * e);
#pragma unroll
                                    for (int pp = 0; pp < P; ++pp) {
                                        ar[0][pp] = fma(f.x, ve[pp], ar[0][pp]);
                                        ar[1][pp] = fma(f.y, ve[pp], ar[1][pp]);
                                    }
                                }
                            }
                            fxp += MT * 32 * EPL;
                            fxrp += CWX * 2;
                        }
                    }
                };
                // two register buffers take turns (no copies); only a row block with an odd number of groups ends
                // with the next block's first group in the wrong one
                real_t nxt[G][RAW];
                for (int kg = 0; kg < KXG; kg += 2) {
                    load_group(nxt, (kg == KXG - 1) ? nrp : rp, (kg == KXG - 1) ? 0 : kg + 1);
                    compute_group(cur, kg);
                    if (kg + 1 < KXG) {
                        load_group(cur, (kg + 1 == KXG - 1) ? nrp : rp, (kg + 1 == KXG - 1) ? 0 : kg + 2);
                        compute_group(nxt, kg + 1);
                    } else {
#pragma unroll
                        for (int j = 0; j < G; ++j)
#pragma unroll
                            for (int i = 0; i < RAW; ++i) cur[j][i] = nxt[j][i];
                    }
                }

                // real data: the even / odd column chains meet
                if (!CPLX) {
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) { C1[mt][0][0] += C1[mt][1][0]; C1[mt][0][1] += C1[mt][1][1]; }
                }
                // ---- Bloch phase of each row (complex only): rotate the accumulators ----
                if (yphase && yb >= yrot_lo && yb <= yrot_hi) {       // row blocks of the home image have phase 1
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        const double2 w = *reinterpret_cast<const double2*>(&wy[2 * (8 * yb + 2 * t + s)]);
#pragma unroll
                        for (int mt = 0; mt < MT; ++mt) {
                            const double re = C1[mt][0][s], im = C1[mt][1][s];
                            C1[mt][0][s] = re * w.x - im * w.y;
                            C1[mt][1][s] = re * w.y + im * w.x;
                        }
                    }
                    if (R) {
                        const double2 w = *reinterpret_cast<const double2*>(&wy[2 * (8 * yb + q)]);
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const double re = ar[i][0], im = ar[i][1];
                            ar[i][0] = re * w.x - im * w.y;
                            ar[i][1] = re * w.y + im * w.x;
                        }
                    }
                }
                // ---- a4: y contraction; the a3 accumulators are the A fragments (k = t <-> row 2t + s) ----
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int ty = 0; ty < MT; ++ty) {
                        const double bfr = fy[(((size_t)yb * 2 + s) * MT + ty) * 32 + lane];
#pragma unroll
                        for (int tx = 0; tx < MT; ++tx)
                            if (tx + ty < 2 || MT == 1) {
#pragma unroll
                                for (int pp = 0; pp < P; ++pp) dmma(T2[pp][tx][ty][0], T2[pp][tx][ty][1], C1[tx][pp][s], bfr);
                            }
                    }
                if (R) {
                    // rows nx = 8, 9 against phi_0, phi_1 of this lane's row; columns ny = 8, 9 against the a3
                    // accumulators (rows nx = q; only q = 0, 1 are used)
                    const double2 y0 = *reinterpret_cast<const double2*>(&fys[4 * (8 * yb + q)]);
#pragma unroll
                    for (int pp = 0; pp < P; ++pp) {
                        rs[0][pp] = fma(ar[0][pp], y0.x, rs[0][pp]);
                        rs[1][pp] = fma(ar[0][pp], y0.y, rs[1][pp]);
                        rs[2][pp] = fma(ar[1][pp], y0.x, rs[2][pp]);
                    }
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        const double2 g = *reinterpret_cast<const double2*>(&fys[4 * (8 * yb + 2 * t + s) + 2]);
#pragma unroll
                        for (int pp = 0; pp < P; ++pp) {
                            cs[0][pp] = fma(C1[0][pp][s], g.x, cs[0][pp]);
                            cs[1][pp] = fma(C1[0][pp][s], g.y, cs[1][pp]);
                        }
                    }
                }
                rp = nrp;
            }
            // plane result -> shared, [part][nx][ny] (+ the R specials)
#pragma unroll
            for (int pp = 0; pp < P; ++pp)
#pragma unroll
                for (int tx = 0; tx < MT; ++tx)
#pragma unroll
                    for (int ty = 0; ty < MT; ++ty)
                        if (tx + ty < 2 || MT == 1) {
                            double2 o; o.x = T2[pp][tx][ty][0]; o.y = T2[pp][tx][ty][1];
                            *reinterpret_cast<double2*>(&t2w[(size_t)pp * TS + (8 * tx + q) * MP + 8 * ty + 2 * t]) = o;
                        }
            if (R) {
#pragma unroll
                for (int pp = 0; pp < P; ++pp) {
#pragma unroll
                    for (int i = 0; i < 3; ++i) {
#pragma unroll
                        for (int m = 16; m >= 1; m >>= 1) rs[i][pp] += __shfl_xor_sync(0xffffffffu, rs[i][pp], m);
                    }
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        cs[i][pp] += __shfl_xor_sync(0xffffffffu, cs[i][pp], 1);
                        cs[i][pp] += __shfl_xor_sync(0xffffffffu, cs[i][pp], 2);
                    }
                    double* o = t2w + (size_t)pp * TS + MP * MP;
                    if (lane == 0) { o[0] = rs[0][pp]; o[1] = rs[1][pp]; o[2] = rs[2][pp]; }
                    if (t == 0 && q == 0) { o[3] = cs[0][pp]; o[4] = cs[1][pp]; }
                    if (t == 0 && q == 1) { o[5] = cs[0][pp]; }
                }
            }
        }
        // The planes of this round are handed over through T2 buffer round & 3; its a5 runs one round later,
        // so a warp waits for the others only when it is more than a whole plane ahead of the slowest.  Buffer
        // reuse is safe with four: a5(r-4) precedes arrive(r-2) in every warp, and this warp waited for (r-2).
        __syncwarp();
        if (lane == 0) mbar_arrive(t2bar + ((rbase + round) & 3));
        if (round >= 1) { mbar_wait(t2bar + ((rbase + round - 1) & 3), ((rbase + round - 1) >> 2) & 1); a5(round - 1); }
    }
    if (nrounds >= 1) { mbar_wait(t2bar + ((rbase + nrounds - 1) & 3), ((rbase + nrounds - 1) >> 2) & 1); a5(nrounds - 1); }

    // ---- store: c[a][b][n] = h^3 * acc (reading A7) ----
    real_t* cout = reinterpret_cast<real_t*>(p.coeff) + ((size_t)a * p.cnb + b) * p.g.nsho * P;
#pragma unroll
    for (int j = 0; j < NACC; ++j) {
        const int n = tid + j * blockDim.x;
        if (n < p.g.nsho) {
#pragma unroll
            for (int pp = 0; pp < P; ++pp) cout[(size_t)n * P + pp] = (real_t)(h3 * acc[j][pp]);
        }
    }
  }     // bands of the group
}

template <typename T>
__global__ void sho_zero_empty_kernel(T* coeff, const int32_t* order, int first, int count, int nbands, int nvals, int cnb)
{
    // atoms with an empty box (isolated grid, atom outside): coefficients are exact zeros
    const int a = order[first + blockIdx.x];
    T* c = coeff + (size_t)a * cnb * nvals;
    for (int i = threadIdx.x; i < nbands * nvals; i += blockDim.x) c[i] = (T)0;
    (void)count;
}

template <int MT, int R, int DT, int G>
static sho_status launch_t(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s, int cnb, const sho_tables1d* t1)
{
    using S = ProjSmem<MT, R, DT>;
    constexpr bool CPLX = Elem<DT>::cplx;
    constexpr int EPL = S::EPL, CWX = S::CWX;
    ProjParams p;
    p.g = pl->g;
    p.psi = psi; p.coeff = coeff;
    p.atoms = pl->d_atoms; p.order = pl->d_order; p.nxyz = pl->d_nxyz;
    p.tab1d = t1 ? t1->d_data : nullptr; p.tab1d_off = t1 ? t1->d_atom_off : nullptr;
    p.nbands = nbands;
    p.cnb = cnb;
    p.n_work_atoms = pl->n_nonempty;
    p.xalign_span = pl->proj_xalign_span;
    p.kx_cap = (pl->max_n[0] + 2 * (CWX - 1)) / CWX + 2;     // + the twice-scheduled image-boundary step
    p.yb_cap = (pl->max_n[1] + 7) / 8 + 1;
    p.nz_cap = pl->max_n[2] + 1;
    p.band_stride = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    p.fast = ((reinterpret_cast<uintptr_t>(psi) % 32) == 0) && (pl->g.ng[0] % EPL == 0);
    const size_t smem = S::total_bytes(p.kx_cap, p.yb_cap, p.nz_cap);
    if (smem > 227 * 1024) {
        set_error("sho_project: box of %d x %d x %d points needs %zu bytes of shared memory (> 227 KB)",
                  pl->max_n[0], pl->max_n[1], pl->max_n[2], smem);
        return SHO_ERR_UNSUPPORTED;
    }
    // bands per CTA: the tables of an atom (and the CTA's start-up) are paid once per CTA; with many bands and small
    // boxes (the paper's workload: 1024 bands, 28^3 points) that is a good part of a one-band CTA's life (paper-nu5
    // project 13.6 -> 12.1 ms).  As many bands as leave about 20 full waves of CTAs, at most 8 -- and only while the
    // bands the resident CTAs spread over stay in L2 together (24 MB): CTAs that run at the same time read
    // neighbouring boxes of the same band, and with 7 bands of 113 MB per CTA cfg 5 takes 49.9 instead of 38.3 ms.
    int nsm = 0;
    cudaError_t e0 = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, pl->device);
    if (e0 != cudaSuccess) return cuda_fail(e0, "cudaDeviceGetAttribute(project)");
    const long long per_wave = (long long)std::max(nsm, 1) * ((CPLX || MT == 2 || R > 0) ? 2 : 3);
    const double band_bytes = (double)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2] * elem_size(pl->dtype);
    const long long by_l2 = std::max<long long>(1, (long long)(24.0e6 / band_bytes));
    int bpc = (int)std::min<long long>(std::min<long long>(8, by_l2),
                                             std::max<long long>(1, (long long)pl->n_nonempty * nbands / (20 * per_wave)));
    if (pl->opt_project_bands_per_cta >= 1)                                // sho_plan_set_option: the band loop on small inputs
        bpc = std::min((int)pl->opt_project_bands_per_cta, std::max(nbands, 1));
    p.bands_per_cta = bpc;
    const long long nblocks = (long long)pl->n_nonempty * ((nbands + bpc - 1) / bpc);
    if (nblocks > 0x7fffffffLL) { set_error("sho_project: natoms*nbands too large"); return SHO_ERR_UNSUPPORTED; }
    auto kern = (bpc > 1) ? sho_project_kernel<MT, R, DT, G, 1> : sho_project_kernel<MT, R, DT, G, 0>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(project)");
    if (nblocks > 0) {
        kern<<<(unsigned)nblocks, kProjWarps * 32, smem, s>>>(p);
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "launch sho_project_kernel");
    }
    const int nempty = pl->g.natoms - pl->n_nonempty;
    if (nempty > 0) {
        using real_t = typename Elem<DT>::real_t;
        sho_zero_empty_kernel<real_t><<<nempty, 256, 0, s>>>(reinterpret_cast<real_t*>(coeff), pl->d_order,
                                                              pl->n_nonempty, nempty, nbands,
                                                              pl->g.nsho * (CPLX ? 2 : 1), cnb);
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "launch sho_zero_empty_kernel");
    }
    return SHO_OK;
}

template <int DT, int G>
static sho_status launch_mg(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s, int cnb, const sho_tables1d* t1)
{
    // numax + 1 functions per axis: <= 8 one MMA row tile; 9, 10 one tile + 2 DFMA rows; more: two tiles
    const int M = pl->g.numax + 1;
    if (M <= 8) return launch_t<1, 0, DT, G>(pl, psi, nbands, coeff, s, cnb, t1);
    if (M <= 10) return launch_t<1, 2, DT, G>(pl, psi, nbands, coeff, s, cnb, t1);
    return launch_t<2, 0, DT, G>(pl, psi, nbands, coeff, s, cnb, t1);
}

template <int DT>
static sho_status launch_m(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s, int cnb, const sho_tables1d* t1)
{
    // Loads are issued kProjG = 2 steps at a time (longer prefetch distance); a row block with an odd number of
    // steps then wastes one.  Real data has few, long steps (16 or 32 columns): when more than 6 % of them would
    // be lost, issue them one by one (cfg 3: 4-5 steps per row block, 1.90 vs 2.03 ms; cfg 4: 8, 15.5 vs 16.1 ms).
    if (!Elem<DT>::cplx && pl->proj_odd_steps > 0.06) return launch_mg<DT, 1>(pl, psi, nbands, coeff, s, cnb, t1);
    return launch_mg<DT, kProjG>(pl, psi, nbands, coeff, s, cnb, t1);
}

sho_status launch_project(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s, int cnb, const sho_tables1d* t1)
{
    if (cnb <= 0) cnb = nbands;
    switch (pl->dtype) {
        case SHO_R64:  return launch_m<SHO_R64>(pl, psi, nbands, coeff, s, cnb, t1);
        case SHO_C128: return launch_m<SHO_C128>(pl, psi, nbands, coeff, s, cnb, t1);
        case SHO_R32:  return launch_m<SHO_R32>(pl, psi, nbands, coeff, s, cnb, t1);
        case SHO_C64:  return launch_m<SHO_C64>(pl, psi, nbands, coeff, s, cnb, t1);
    }
    set_error("sho_project: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

}  // namespace sho
