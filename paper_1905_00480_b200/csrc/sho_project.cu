// sho_project.cu -- on-the-fly SHO projection (steps a1-a5 of DESIGN.md), one CTA per (atom, band).
//
//   c[a][b][n(nx,ny,nz)] = h^3 sum_r psi_b(r) phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)
//                                                       eq. (25)-(26); step (1)
//
// Design (B200, sm_100a): the separable contraction runs y -> x -> z.
//   a1  every CTA samples the three 1D Hermite-Gauss tables of its atom on the fly (eq. (31)) straight
//       into shared memory, already laid out as FP64 tensor-core fragments; nothing but 80 B of atom
//       parameters is read from HBM for the projectors.
//   a2  psi is read straight from global memory / L2 with 16-byte loads: a warp load covers 4 rows x
//       128 contiguous bytes, and the loaded registers ARE the B fragments of the first contraction
//       (K = y, N = x contiguous), so no shared-memory staging or transposition is needed.  Periodic
//       wrap / isolated clipping are per-lane index arithmetic.  The loads run one group of G y steps
//       ahead of the arithmetic (register double buffer) and the ring runs on across chunk ends and
//       plane ends, so loads stay in flight over the x stage, a5 and its barrier.
//   a3  first-axis (y) contraction: DMMA.8x8x4, M = ny, K = 4 rows, N = 8 columns.  With numax = 8, 9
//       (M = 9, 10) a second, mostly empty MMA row tile would cost 1.6x the algorithmic flops, so the
//       R = 2 remainder rows ny = 8, 9 run as plain DFMAs on the same loaded values instead (template
//       parameter R): per lane a partial over its own row, reduced once per plane.
//   a4  second-axis (x) contraction: the accumulator fragment of a3 is directly the A fragment of a
//       second DMMA against the phi_nx table (the K order inside an MMA is free).  For R = 2 the six
//       (ny,nx) outputs with ny or nx in {8, 9} are DFMA partials per lane.
//   a5  third axis: each warp owns one z-plane per round; the per-plane T2[ny][nx] meet in shared
//       memory and thread n accumulates c[n] += phi_nz(z) * T2[ny][nx] in a register.  One
//       __syncthreads per round (double-buffered), coalesced store of N_SHO coefficients at the end.
// Bloch phases never touch the inner loop: x-phases rotate the a3 accumulators per column, the y-phase
// is a single accumulator rotation at the wrap row, the z-phase is folded into a5.
#include "sho_device.cuh"

namespace sho {

constexpr int kProjG = 4;      // y steps (of 4 rows x 8/16 columns) per group of the register load ring

struct ProjParams {
    GridDev g;
    const void* psi;
    void* coeff;
    const AtomDev* atoms;
    const int32_t* order;
    const uint32_t* nxyz;
    int32_t nbands;
    int32_t n_work_atoms;      // atoms with a non-empty box (first entries of order[])
    int32_t ky_cap, nxe_cap, nz_cap;   // capacities of the shared tables (from the plan's largest box)
    int32_t vec_ok;            // 16-byte (8-byte for fp32) loads are aligned
    long long band_stride;     // elements between bands
};

// shared-memory carve-up (doubles unless noted); every block starts 16-byte aligned
template <int MT, int R, int DT>
struct ProjSmem {
    static constexpr int P = Elem<DT>::cplx ? 2 : 1;
    static constexpr int MP = 8 * MT;                       // ny / nx rows on the MMA
    static constexpr int NV = MP + R;                       // functions sampled per point
    static constexpr int TS = MP * MP + (R ? 8 : 0);        // one part of one plane's T2 (+ the R specials)
    static __host__ __device__ size_t fy(int ky) { return (size_t)ky * MT * 32; }
    static __host__ __device__ size_t fyr(int ky) { return R ? (size_t)ky * 4 * 2 : 0; }
    static __host__ __device__ size_t fx(int nxe) { return (size_t)nxe * MT * 32; }
    static __host__ __device__ size_t fxs(int nxe) { return R ? (size_t)nxe * 4 * 4 : 0; }
    static __host__ __device__ size_t fz(int nz) { return (size_t)nz * NV + (((size_t)nz * NV) & 1); }
    static __host__ __device__ size_t wz(int nz) { return Elem<DT>::cplx ? (size_t)nz * 2 : 0; }
    static __host__ __device__ size_t t2() { return (size_t)2 * kProjWarps * P * TS; }
    static __host__ __device__ size_t total_bytes(int ky, int nxe, int nz)
    {
        return 8 * (fy(ky) + fyr(ky) + fx(nxe) + fxs(nxe) + fz(nz) + wz(nz) + t2() + 6) + (size_t)(ky + 4) * 4 * 4 + 16;
    }
};

// position of T2[ny][nx] inside one part of a plane's shared T2 block
template <int MT, int R>
__device__ __forceinline__ int t2_index(int ny, int nx)
{
    constexpr int MP = 8 * MT;
    if (R == 0 || (ny < MP && nx < MP)) return ny * MP + nx;
    if (ny == MP) return MP * MP + nx;            // (8,0) (8,1)
    if (ny == MP + 1) return MP * MP + 2;         // (9,0)
    if (nx == MP) return MP * MP + 3 + 2 * ny;    // (0,8) -> 3, (1,8) -> 5
    return MP * MP + 4;                           // (0,9)
}

template <int MT, int R, int DT, int G>
__global__ void __launch_bounds__(kProjWarps * 32, 2) sho_project_kernel(const ProjParams p)
{
    using E = Elem<DT>;
    using S = ProjSmem<MT, R, DT>;
    using real_t = typename E::real_t;
    constexpr bool CPLX = E::cplx;
    constexpr int P = CPLX ? 2 : 1;
    constexpr int MP = S::MP, NV = S::NV, TS = S::TS;
    constexpr int CW = E::cw;                 // columns per chunk (one 16-byte load per lane = 2 MMAs)
    constexpr int XALIGN = CPLX ? 2 : 4;
    constexpr int NACC = (MT == 1) ? 1 : (816 + kProjWarps * 32 - 1) / (kProjWarps * 32);   // numax <= 9: N_SHO <= 220

    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* fy = reinterpret_cast<double*>(smem_raw);                 // [k][mt][32]   A fragments of the y stage
    double* fyr = fy + S::fy(p.ky_cap);                               // [row][2]      phi_8, phi_9 of the R rows
    double* fx = fyr + S::fyr(p.ky_cap);                              // [slot][mt][32] B fragments of the x stage
    double* fxs = fx + S::fx(p.nxe_cap);                              // [column][4]   phi_0, phi_1, phi_8, phi_9
    double* fz = fxs + S::fxs(p.nxe_cap);                             // [z][NV]
    double* wz = fz + S::fz(p.nz_cap);                                // complex only: [z][2]
    double* t2s = wz + S::wz(p.nz_cap);                               // [2][W][P][TS]
    double* phx = t2s + S::t2();                                      // [2 images][re,im] + y rotation [re,im]
    int32_t* rowoff = reinterpret_cast<int32_t*>(phx + 6);            // [padded row] element offset of the row

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int q = lane >> 2, t = lane & 3;

    // work item: band-major, atoms in the plan's spatial order (neighbouring CTAs share psi in L2)
    const int b = blockIdx.x / p.n_work_atoms;
    const int a = p.order[blockIdx.x - b * p.n_work_atoms];
    const AtomDev at = p.atoms[a];
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int numax = p.g.numax;

    const int nzl = at.hi[2] - at.lo[2] + 1;
    // x: chunks of CW columns starting at a sector-aligned column
    const int xs0 = floordiv(at.lo[0], XALIGN) * XALIGN;
    const int XC = (at.hi[0] - xs0 + CW) / CW;
    // y: K steps of 4 rows; complex data with a y-wrap split the rows at the wrap (one accumulator rotation)
    int yB = at.hi[1] + 1;   // first row of the second segment (unwrapped); hi+1 = no split
    if (CPLX && p.g.has_phase && p.g.periodic[1] && p.g.kfrac[1] != 0.0) {
        const int mlo = floordiv(at.lo[1], Ny), mhi = floordiv(at.hi[1], Ny);
        if (mhi != mlo) yB = mhi * Ny;
    }
    const int K0 = (min(yB, at.hi[1] + 1) - at.lo[1] + 3) >> 2;
    const int K1 = (at.hi[1] + 1 - yB + 3) >> 2;          // 0 when there is no split
    const int KY = K0 + (K1 > 0 ? K1 : 0);
    const int krot = (K1 > 0) ? K0 : -1;

    // ---------------- a1: sample the 1D tables on the fly, in fragment layout ----------------
    const int KG = (KY + G - 1) / G;            // groups of G y steps (the load ring's granularity)
    const int ny_items = KG * G * 4, nx_items = XC * CW;
    for (int it = tid; it < ny_items + nx_items + nzl; it += blockDim.x) {
        double v[NV];
        if (it < ny_items) {
            const int pr = it;                                   // padded row slot
            int iy = (pr < K0 * 4) ? at.lo[1] + pr : yB + (pr - K0 * 4);
            const bool valid = (pr < K0 * 4) ? (iy < yB && iy <= at.hi[1]) : (iy <= at.hi[1]);
            if (!valid) iy = at.hi[1];
            const int k = pr >> 2, tt = pr & 3;
            if (k < KY) {
                hermite_gauss<NV>(displacement(iy, p.g.h, at.pos[1]), at, p.g.hnorm, numax, valid, v);
#pragma unroll
                for (int n = 0; n < MP; ++n) fy[((size_t)k * MT + (n >> 3)) * 32 + (n & 7) * 4 + tt] = v[n];
                if (R) { fyr[2 * pr] = v[MP]; fyr[2 * pr + 1] = v[MP + R - 1]; }
            }
            // rows of the steps that pad the last group are never used in arithmetic; they point at a valid row
            int jy = p.g.periodic[1] ? iy - floordiv(iy, Ny) * Ny : min(max(iy, 0), Ny - 1);
            rowoff[((k / G) * 4 + tt) * G + (k % G)] = jy * Nx;      // [group][t][step in group]
        } else if (it < ny_items + nx_items) {
            const int j = it - ny_items;
            const int ix = xs0 + j;
            const bool valid = ix >= at.lo[0] && ix <= at.hi[0];
            hermite_gauss<NV>(displacement(ix, p.g.h, at.pos[0]), at, p.g.hnorm, numax, valid, v);
            const int c = j / CW, r = j % CW;
            int slot, tt;
            if (!CPLX) { tt = r >> 2; slot = (c * 2 + (r & 1)) * 2 + ((r >> 1) & 1); }   // r = 4t + 2s + e
            else       { tt = r >> 1; slot = c * 2 + (r & 1); }                           // r = 2t + s
#pragma unroll
            for (int n = 0; n < MP; ++n) fx[((size_t)slot * MT + (n >> 3)) * 32 + (n & 7) * 4 + tt] = v[n];
            if (R) {
                fxs[4 * j] = v[0]; fxs[4 * j + 1] = v[1]; fxs[4 * j + 2] = v[MP]; fxs[4 * j + 3] = v[MP + R - 1];
            }
        } else {
            const int zi = it - ny_items - nx_items;
            const int iz = at.lo[2] + zi;
            hermite_gauss<NV>(displacement(iz, p.g.h, at.pos[2]), at, p.g.hnorm, numax, true, v);
#pragma unroll
            for (int n = 0; n < NV; ++n) fz[(size_t)zi * NV + n] = v[n];
            if (CPLX) {
                // phase of image m_z, times the overall y factor (phase of the last y segment)
                double ang = 0.0;
                if (p.g.has_phase) {
                    if (p.g.periodic[2]) ang += p.g.kfrac[2] * (double)floordiv(iz, Nz);
                    if (p.g.periodic[1]) ang += p.g.kfrac[1] * (double)floordiv(at.hi[1], Ny);
                }
                double sn, cs;
                sincospi(2.0 * ang, &sn, &cs);
                wz[2 * zi] = cs; wz[2 * zi + 1] = sn;
            }
        }
    }
    if (CPLX && tid == 0) {
        // x phases of the two possible images, and the y rotation exp(-2 pi i kfrac_y)
        const int mlo = p.g.periodic[0] ? floordiv(at.lo[0], Nx) : 0;
        for (int i = 0; i < 2; ++i) {
            double sn, cs;
            sincospi(2.0 * (p.g.has_phase && p.g.periodic[0] ? p.g.kfrac[0] * (double)(mlo + i) : 0.0), &sn, &cs);
            phx[2 * i] = cs; phx[2 * i + 1] = sn;
        }
        double sn, cs;
        sincospi(-2.0 * p.g.kfrac[1], &sn, &cs);
        phx[4] = cs; phx[5] = sn;
    }
    __syncthreads();

    const real_t* psi_b = reinterpret_cast<const real_t*>(p.psi) + (size_t)b * p.band_stride * P;
    const size_t plane = (size_t)Ny * Nx;
    const bool vec = p.vec_ok != 0;
    const int xB = CPLX ? (p.g.periodic[0] ? (floordiv(at.lo[0], Nx) + 1) * Nx : INT_MAX) : 0;
    const bool xphase = CPLX && p.g.has_phase && p.g.periodic[0] && p.g.kfrac[0] != 0.0;

    // a5 accumulators: thread n owns coefficient(s) n, n + blockDim, ...
    double acc[NACC][P];
    int myt2[NACC], mynz[NACC];
#pragma unroll
    for (int j = 0; j < NACC; ++j) {
        const int n = tid + j * blockDim.x;
        const uint32_t pk = (n < p.g.nsho) ? p.nxyz[n] : 0u;
        myt2[j] = t2_index<MT, R>((pk >> 8) & 255, pk & 255);
        mynz[j] = (pk >> 16) & 255;
#pragma unroll
        for (int pp = 0; pp < P; ++pp) acc[j][pp] = 0.0;
    }

    // ---- a2 helpers: plane pointer, this lane's column pointer(s) of a chunk, one group of loads ----
    auto plane_ptr = [&](int zi) -> const real_t* {
        const int iz = at.lo[2] + zi;
        const int jz = p.g.periodic[2] ? iz - floordiv(iz, Nz) * Nz : iz;
        return psi_b + (size_t)jz * plane * P;
    };
    auto col_ptrs = [&](const real_t* pzz, int c, const real_t*& c0, const real_t*& c1, bool& vv) {
        const int ix0 = xs0 + c * CW + (CPLX ? q : 2 * q);
        const int ix1 = ix0 + 1;
        const int off0 = p.g.periodic[0] ? ix0 - floordiv(ix0, Nx) * Nx : min(max(ix0, 0), Nx - 1);
        const int off1 = p.g.periodic[0] ? ix1 - floordiv(ix1, Nx) * Nx : min(max(ix1, 0), Nx - 1);
        c0 = pzz + (size_t)off0 * P;
        c1 = pzz + (size_t)off1 * P;
        vv = vec && (CPLX || off1 == off0 + 1);
    };
    // G consecutive y steps (4 rows each) of one chunk: lane (q,t) reads row 4k+t, column(s) q / 2q, 2q+1
    auto load_group = [&](double (&x0)[G], double (&x1)[G], const real_t* c0, const real_t* c1, bool vv, int kg) {
        int r[G];
        if (G == 4) {
            const int4 r4 = *reinterpret_cast<const int4*>(rowoff + (kg * 4 + t) * G);
            r[0] = r4.x; r[1] = r4.y; r[G - 2] = r4.z; r[G - 1] = r4.w;
        } else {
#pragma unroll
            for (int j = 0; j < G; ++j) r[j] = rowoff[(kg * 4 + t) * G + j];
        }
#pragma unroll
        for (int j = 0; j < G; ++j) {
            const size_t ro = (size_t)r[j] * P;
            if (CPLX) {
                load2(c0 + ro, vec, x0[j], x1[j]);                            // (re, im) of one column
            } else if (vv) {
                load2(c0 + ro, true, x0[j], x1[j]);                           // two adjacent columns
            } else {
                x0[j] = (double)__ldg(c0 + ro); x1[j] = (double)__ldg(c1 + ro);
            }
        }
    };

    // The load ring: while the G steps in cur0/cur1 are contracted, the next G steps are in flight; the
    // ring runs on across chunk ends (over the x stage) and plane ends (over a5 and its barrier).
    const int nrounds = (nzl + kProjWarps - 1) / kProjWarps;
    double cur0[G], cur1[G];
    const real_t *cp0 = psi_b, *cp1 = psi_b;     // column pointer(s) of the current chunk for this lane
    bool cv = false;
#pragma unroll
    for (int j = 0; j < G; ++j) cur0[j] = cur1[j] = 0.0;
    if (warp < nzl) {
        col_ptrs(plane_ptr(warp), 0, cp0, cp1, cv);
        load_group(cur0, cur1, cp0, cp1, cv, 0);
    }
    for (int round = 0; round < nrounds; ++round) {
        const int zi = round * kProjWarps + warp;
        double* t2w = t2s + ((size_t)(round & 1) * kProjWarps + warp) * P * TS;
        if (zi < nzl) {
            const real_t* pz = plane_ptr(zi);
            const real_t* pzn = (zi + kProjWarps < nzl) ? plane_ptr(zi + kProjWarps) : pz;

            // T2[part][ty][tx]: tile (1,1) can only hold ny+nx >= 16 > numax and is never needed
            double T2[P][MT][MT][2];
#pragma unroll
            for (int pp = 0; pp < P; ++pp)
#pragma unroll
                for (int ty = 0; ty < MT; ++ty)
#pragma unroll
                    for (int tx = 0; tx < MT; ++tx) T2[pp][ty][tx][0] = T2[pp][ty][tx][1] = 0.0;
            // R specials, per-lane partials: rs = T2[8][0], T2[8][1], T2[9][0]; cs = T2[q][8], T2[q][9]
            double rs[3][P], cs[2][P];
#pragma unroll
            for (int pp = 0; pp < P; ++pp) { rs[0][pp] = rs[1][pp] = rs[2][pp] = 0.0; cs[0][pp] = cs[1][pp] = 0.0; }

            for (int c = 0; c < XC; ++c) {
                // where the ring goes after this chunk: the next chunk, or chunk 0 of this warp's next plane
                const real_t *np0, *np1;
                bool nv;
                if (c + 1 < XC) col_ptrs(pz, c + 1, np0, np1, nv); else col_ptrs(pzn, 0, np0, np1, nv);

                double C1[MT][2][2];   // [ny tile][e or re/im][s]
                double ar[2][2];       // R rows: [ny = 8, 9][e or re/im], partial over this lane's row t
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) C1[mt][0][0] = C1[mt][0][1] = C1[mt][1][0] = C1[mt][1][1] = 0.0;
                ar[0][0] = ar[0][1] = ar[1][0] = ar[1][1] = 0.0;

                for (int kg = 0; kg < KG; ++kg) {
                    const bool last = (kg == KG - 1);
                    double n0[G], n1[G];
                    load_group(n0, n1, last ? np0 : cp0, last ? np1 : cp1, last ? nv : cv, last ? 0 : kg + 1);
#pragma unroll
                    for (int j = 0; j < G; ++j) {
                        const int k = kg * G + j;
                        if (k < KY) {
                            if (CPLX && k == krot) {
                                const double cr = phx[4], ci = phx[5];
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
                            // ---- a3: y contraction, K = 4 rows ----
                            const double v0 = cur0[j], v1 = cur1[j];
#pragma unroll
                            for (int mt = 0; mt < MT; ++mt) {
                                const double afr = fy[((size_t)k * MT + mt) * 32 + lane];
                                dmma(C1[mt][0][0], C1[mt][0][1], afr, v0);
                                dmma(C1[mt][1][0], C1[mt][1][1], afr, v1);
                            }
                            if (R) {
                                const double2 f = *reinterpret_cast<const double2*>(&fyr[2 * (4 * k + t)]);
                                ar[0][0] = fma(f.x, v0, ar[0][0]); ar[0][1] = fma(f.x, v1, ar[0][1]);
                                ar[1][0] = fma(f.y, v0, ar[1][0]); ar[1][1] = fma(f.y, v1, ar[1][1]);
                            }
                        }
                    }
#pragma unroll
                    for (int j = 0; j < G; ++j) { cur0[j] = n0[j]; cur1[j] = n1[j]; }
                }

                // ---- Bloch phase of each column (complex only): rotate the accumulators ----
                if (xphase) {
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        const int ix = xs0 + c * CW + 2 * t + s;
                        const int im_ = (ix >= xB) ? 1 : 0;
                        const double cr = phx[2 * im_], ci = phx[2 * im_ + 1];
#pragma unroll
                        for (int mt = 0; mt < MT; ++mt) {
                            const double re = C1[mt][0][s], im = C1[mt][1][s];
                            C1[mt][0][s] = re * cr - im * ci;
                            C1[mt][1][s] = re * ci + im * cr;
                        }
                    }
                    if (R) {
                        const int im_ = (xs0 + c * CW + q >= xB) ? 1 : 0;
                        const double cr = phx[2 * im_], ci = phx[2 * im_ + 1];
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            const double re = ar[i][0], im = ar[i][1];
                            ar[i][0] = re * cr - im * ci;
                            ar[i][1] = re * ci + im * cr;
                        }
                    }
                }
                // ---- a4: x contraction; the a3 accumulators are the A fragments ----
                if (!CPLX) {
#pragma unroll
                    for (int e = 0; e < 2; ++e)
#pragma unroll
                        for (int s = 0; s < 2; ++s) {
                            const int slot = (c * 2 + e) * 2 + s;
#pragma unroll
                            for (int tx = 0; tx < MT; ++tx) {
                                const double bfr = fx[((size_t)slot * MT + tx) * 32 + lane];
#pragma unroll
                                for (int ty = 0; ty < MT; ++ty)
                                    if (ty + tx < 2 || MT == 1)
                                        dmma(T2[0][ty][tx][0], T2[0][ty][tx][1], C1[ty][e][s], bfr);
                            }
                        }
                } else {
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        const int slot = c * 2 + s;
#pragma unroll
                        for (int tx = 0; tx < MT; ++tx) {
                            const double bfr = fx[((size_t)slot * MT + tx) * 32 + lane];
#pragma unroll
                            for (int ty = 0; ty < MT; ++ty)
                                if (ty + tx < 2 || MT == 1) {
#pragma unroll
                                    for (int pp = 0; pp < P; ++pp)
                                        dmma(T2[pp][ty][tx][0], T2[pp][ty][tx][1], C1[ty][pp][s], bfr);
                                }
                        }
                    }
                }
                if (R) {
                    // rows ny = 8, 9 against phi_0, phi_1 of this lane's column(s); columns nx = 8, 9
                    // against the a3 accumulators (rows ny = q; only q = 0, 1 are used)
                    if (!CPLX) {
                        const double* fr = fxs + 4 * (size_t)(c * CW + 2 * q);
                        const double2 x0 = *reinterpret_cast<const double2*>(fr);
                        const double2 x1 = *reinterpret_cast<const double2*>(fr + 4);
                        rs[0][0] = fma(ar[0][0], x0.x, fma(ar[0][1], x1.x, rs[0][0]));
                        rs[1][0] = fma(ar[0][0], x0.y, fma(ar[0][1], x1.y, rs[1][0]));
                        rs[2][0] = fma(ar[1][0], x0.x, fma(ar[1][1], x1.x, rs[2][0]));
#pragma unroll
                        for (int e = 0; e < 2; ++e)
#pragma unroll
                            for (int s = 0; s < 2; ++s) {
                                const double2 g =
                                    *reinterpret_cast<const double2*>(fxs + 4 * (size_t)(c * CW + 4 * t + 2 * s + e) + 2);
                                cs[0][0] = fma(C1[0][e][s], g.x, cs[0][0]);
                                cs[1][0] = fma(C1[0][e][s], g.y, cs[1][0]);
                            }
                    } else {
                        const double2 x0 = *reinterpret_cast<const double2*>(fxs + 4 * (size_t)(c * CW + q));
#pragma unroll
                        for (int pp = 0; pp < P; ++pp) {
                            rs[0][pp] = fma(ar[0][pp], x0.x, rs[0][pp]);
                            rs[1][pp] = fma(ar[0][pp], x0.y, rs[1][pp]);
                            rs[2][pp] = fma(ar[1][pp], x0.x, rs[2][pp]);
                        }
#pragma unroll
                        for (int s = 0; s < 2; ++s) {
                            const double2 g = *reinterpret_cast<const double2*>(fxs + 4 * (size_t)(c * CW + 2 * t + s) + 2);
#pragma unroll
                            for (int pp = 0; pp < P; ++pp) {
                                cs[0][pp] = fma(C1[0][pp][s], g.x, cs[0][pp]);
                                cs[1][pp] = fma(C1[0][pp][s], g.y, cs[1][pp]);
                            }
                        }
                    }
                }
                cp0 = np0; cp1 = np1; cv = nv;
            }
            // plane result -> shared, [part][ny][nx] (+ the R specials)
#pragma unroll
            for (int pp = 0; pp < P; ++pp)
#pragma unroll
                for (int ty = 0; ty < MT; ++ty)
#pragma unroll
                    for (int tx = 0; tx < MT; ++tx)
                        if (ty + tx < 2 || MT == 1) {
                            double2 o; o.x = T2[pp][ty][tx][0]; o.y = T2[pp][ty][tx][1];
                            *reinterpret_cast<double2*>(&t2w[(size_t)pp * TS + (8 * ty + q) * MP + 8 * tx + 2 * t]) = o;
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
        __syncthreads();
        // ---- a5: z contraction, thread n <- coefficient n ----
        const double* t2r = t2s + (size_t)(round & 1) * kProjWarps * P * TS;
        const int wmax = min(kProjWarps, nzl - round * kProjWarps);
#pragma unroll
        for (int j = 0; j < NACC; ++j) {
            const int n = tid + j * blockDim.x;
            if (n < p.g.nsho) {
                for (int w = 0; w < wmax; ++w) {
                    const int z2 = round * kProjWarps + w;
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
    }

    // ---- store: c[a][b][n] = h^3 * acc (reading A7) ----
    const double h3 = p.g.h * p.g.h * p.g.h;
    real_t* cout = reinterpret_cast<real_t*>(p.coeff) + ((size_t)a * p.nbands + b) * p.g.nsho * P;
#pragma unroll
    for (int j = 0; j < NACC; ++j) {
        const int n = tid + j * blockDim.x;
        if (n < p.g.nsho) {
#pragma unroll
            for (int pp = 0; pp < P; ++pp) cout[(size_t)n * P + pp] = (real_t)(h3 * acc[j][pp]);
        }
    }
}

template <typename T>
__global__ void sho_zero_empty_kernel(T* coeff, const int32_t* order, int first, int count, int nbands, int nvals)
{
    // atoms with an empty box (isolated grid, atom outside): coefficients are exact zeros
    const int a = order[first + blockIdx.x];
    T* c = coeff + (size_t)a * nbands * nvals;
    for (int i = threadIdx.x; i < nbands * nvals; i += blockDim.x) c[i] = (T)0;
    (void)count;
}


template <int MT, int R, int DT>
static sho_status launch_t(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s)
{
    using S = ProjSmem<MT, R, DT>;
    constexpr bool CPLX = Elem<DT>::cplx;
    constexpr int CW = Elem<DT>::cw;
    ProjParams p;
    p.g = pl->g;
    p.psi = psi; p.coeff = coeff;
    p.atoms = pl->d_atoms; p.order = pl->d_order; p.nxyz = pl->d_nxyz;
    p.nbands = nbands;
    p.n_work_atoms = pl->n_nonempty;
    p.ky_cap = (pl->max_n[1] + 3) / 4 + 2;
    p.nxe_cap = ((pl->max_n[0] + 3 + CW - 1) / CW + 1) * (CPLX ? 2 : 4);
    p.nz_cap = pl->max_n[2] + 1;
    p.band_stride = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    const size_t esz = elem_size(pl->dtype);
    const size_t valign = CPLX ? esz : 2 * esz;      // bytes of one vector load
    p.vec_ok = ((reinterpret_cast<uintptr_t>(psi) % valign) == 0) && (CPLX || (pl->g.ng[0] % 2 == 0));
    const size_t smem = S::total_bytes(p.ky_cap, p.nxe_cap, p.nz_cap);
    if (smem > 227 * 1024) {
        set_error("sho_project: box of %d x %d x %d points needs %zu bytes of shared memory (> 227 KB)",
                  pl->max_n[0], pl->max_n[1], pl->max_n[2], smem);
        return SHO_ERR_UNSUPPORTED;
    }
    auto kern = sho_project_kernel<MT, R, DT, (MT == 1 ? kProjG : 2)>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(project)");
    const long long nblocks = (long long)pl->n_nonempty * nbands;
    if (nblocks > 0x7fffffffLL) { set_error("sho_project: natoms*nbands too large"); return SHO_ERR_UNSUPPORTED; }
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
                                                              pl->g.nsho * (CPLX ? 2 : 1));
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "launch sho_zero_empty_kernel");
    }
    return SHO_OK;
}

template <int DT>
static sho_status launch_m(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s)
{
    // numax + 1 functions per axis: <= 8 one MMA row tile; 9, 10 one tile + 2 DFMA rows; more: two tiles
    const int M = pl->g.numax + 1;
    if (M <= 8) return launch_t<1, 0, DT>(pl, psi, nbands, coeff, s);
    if (M <= 10) return launch_t<1, 2, DT>(pl, psi, nbands, coeff, s);
    return launch_t<2, 0, DT>(pl, psi, nbands, coeff, s);
}

sho_status launch_project(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s)
{
    switch (pl->dtype) {
        case SHO_R64:  return launch_m<SHO_R64>(pl, psi, nbands, coeff, s);
        case SHO_C128: return launch_m<SHO_C128>(pl, psi, nbands, coeff, s);
        case SHO_R32:  return launch_m<SHO_R32>(pl, psi, nbands, coeff, s);
        case SHO_C64:  return launch_m<SHO_C64>(pl, psi, nbands, coeff, s);
    }
    set_error("sho_project: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

}  // namespace sho
