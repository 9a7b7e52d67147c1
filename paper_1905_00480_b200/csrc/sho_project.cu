// sho_project.cu -- on-the-fly SHO projection (steps a1-a5 of DESIGN.md), one CTA per (atom, band).
//
//   c[a][b][n(nx,ny,nz)] = h^3 sum_r psi_b(r) phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)
//                                                       eq. (25)-(26); step (1)
//
// Design (B200, sm_100a): the separable contraction runs y -> x -> z.
//   a1  every CTA samples the three 1D Hermite-Gauss tables of its atom on the fly (eq. (31)) straight
//       into shared memory, already laid out as FP64 tensor-core fragments; nothing but 64 B of atom
//       parameters is read from HBM for the projectors.
//   a2  psi is read straight from global memory / L2 with 16-byte loads: a warp load covers 4 rows x
//       128 contiguous bytes, and the loaded registers ARE the B fragments of the first contraction
//       (K = y, N = x contiguous), so no shared-memory staging or transposition is needed.  Periodic
//       wrap / isolated clipping are per-lane index arithmetic.
//   a3  first-axis (y) contraction: DMMA.8x8x4, M = ny, K = 4 rows, N = 8 columns.
//   a4  second-axis (x) contraction: the accumulator fragment of a3 is directly the A fragment of a
//       second DMMA against the phi_nx table (the K order inside an MMA is free).
//   a5  third axis: each warp owns one z-plane per round; the per-plane [ny][nx] matrices meet in shared
//       memory and thread n accumulates c[n] += phi_nz(z) * T2[ny][nx] in a register.  One
//       __syncthreads per round (double-buffered), coalesced store of N_SHO coefficients at the end.
// Bloch phases never touch the inner loop: x-phases rotate the a3 accumulators per column, the y-phase
// is a single accumulator rotation at the wrap row, the z-phase is folded into a5.
#include "sho_device.cuh"

namespace sho {

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

template <int MT, int DT>
struct ProjSmem {
    // offsets in bytes into dynamic shared memory
    static constexpr int P = Elem<DT>::cplx ? 2 : 1;
    static constexpr int MP = 8 * MT;
    static __host__ __device__ size_t fy_bytes(int ky) { return (size_t)ky * MT * 32 * 8; }
    static __host__ __device__ size_t fx_bytes(int nxe) { return (size_t)nxe * MT * 32 * 8; }
    static __host__ __device__ size_t fz_bytes(int nz) { return (size_t)nz * MP * 8; }
    static __host__ __device__ size_t wz_bytes(int nz) { return Elem<DT>::cplx ? (size_t)nz * 16 : 0; }
    static __host__ __device__ size_t row_bytes(int ky) { return (size_t)ky * 4 * 4; }
    static __host__ __device__ size_t t2_bytes() { return (size_t)2 * kProjWarps * MP * MP * 8 * P; }
    static __host__ __device__ size_t total(int ky, int nxe, int nz)
    {
        return fy_bytes(ky) + fx_bytes(nxe) + fz_bytes(nz) + wz_bytes(nz) + t2_bytes() + row_bytes(ky) + 64;
    }
};

template <int MT, int DT>
__global__ void __launch_bounds__(kProjWarps * 32, 2) sho_project_kernel(const ProjParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    constexpr bool CPLX = E::cplx;
    constexpr int P = CPLX ? 2 : 1;
    constexpr int MP = 8 * MT;
    constexpr int CW = E::cw;                 // columns per chunk (one 16-byte load per lane = 2 MMAs)
    constexpr int NXE_PER_CHUNK = CPLX ? 2 : 4;
    constexpr int XALIGN = CPLX ? 2 : 4;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* fy = reinterpret_cast<double*>(smem_raw);
    double* fx = fy + (size_t)p.ky_cap * MT * 32;
    double* fz = fx + (size_t)p.nxe_cap * MT * 32;
    double* wz = fz + (size_t)p.nz_cap * MP;                          // complex only: [nz][2]
    double* t2s = wz + (CPLX ? (size_t)p.nz_cap * 2 : 0);             // [2][W][P][MP*MP]
    int32_t* rowoff = reinterpret_cast<int32_t*>(t2s + (size_t)2 * kProjWarps * P * MP * MP);
    double* phx = reinterpret_cast<double*>(rowoff + (size_t)p.ky_cap * 4);   // [2 images][re,im] + y rotation [re,im]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int q = lane >> 2, t = lane & 3;

    // work item: band-major, atoms in the plan's spatial order (neighbouring CTAs share psi in L2)
    const int b = blockIdx.x / p.n_work_atoms;
    const int a = p.order[blockIdx.x - b * p.n_work_atoms];
    const AtomDev at = p.atoms[a];
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int numax = p.g.numax;

    const int nxl = at.hi[0] - at.lo[0] + 1, nyl = at.hi[1] - at.lo[1] + 1, nzl = at.hi[2] - at.lo[2] + 1;
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
    const int ny_items = KY * 4, nx_items = XC * CW;
    for (int it = tid; it < ny_items + nx_items + nzl; it += blockDim.x) {
        double v[MP];
        if (it < ny_items) {
            const int pr = it;                                   // padded row slot
            int iy = (pr < K0 * 4) ? at.lo[1] + pr : yB + (pr - K0 * 4);
            const bool valid = (pr < K0 * 4) ? (iy < yB && iy <= at.hi[1]) : (iy <= at.hi[1]);
            if (!valid) iy = at.hi[1];
            hermite_gauss<MP>(displacement(iy, p.g.h, at.pos[1]), at, p.g.hnorm, numax, valid, v);
            const int k = pr >> 2, tt = pr & 3;
#pragma unroll
            for (int n = 0; n < MP; ++n) fy[((size_t)k * MT + (n >> 3)) * 32 + (n & 7) * 4 + tt] = v[n];
            int jy = p.g.periodic[1] ? iy - floordiv(iy, Ny) * Ny : min(max(iy, 0), Ny - 1);
            rowoff[pr] = jy * Nx;
        } else if (it < ny_items + nx_items) {
            const int j = it - ny_items;
            const int ix = xs0 + j;
            const bool valid = ix >= at.lo[0] && ix <= at.hi[0];
            hermite_gauss<MP>(displacement(ix, p.g.h, at.pos[0]), at, p.g.hnorm, numax, valid, v);
            const int c = j / CW, r = j % CW;
            int slot, tt;
            if (!CPLX) { tt = r >> 2; slot = (c * 2 + (r & 1)) * 2 + ((r >> 1) & 1); }   // r = 4t + 2s + e
            else       { tt = r >> 1; slot = c * 2 + (r & 1); }                           // r = 2t + s
#pragma unroll
            for (int n = 0; n < MP; ++n) fx[((size_t)slot * MT + (n >> 3)) * 32 + (n & 7) * 4 + tt] = v[n];
        } else {
            const int zi = it - ny_items - nx_items;
            const int iz = at.lo[2] + zi;
            hermite_gauss<MP>(displacement(iz, p.g.h, at.pos[2]), at, p.g.hnorm, numax, true, v);
#pragma unroll
            for (int n = 0; n < MP; ++n) fz[(size_t)zi * MP + n] = v[n];
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
    constexpr int NACC = (816 + kProjWarps * 32 - 1) / (kProjWarps * 32);
    double acc[NACC][P];
    uint32_t myn[NACC];
#pragma unroll
    for (int j = 0; j < NACC; ++j) {
        const int n = tid + j * blockDim.x;
        myn[j] = (n < p.g.nsho) ? p.nxyz[n] : 0u;
#pragma unroll
        for (int pp = 0; pp < P; ++pp) acc[j][pp] = 0.0;
    }

    const int nrounds = (nzl + kProjWarps - 1) / kProjWarps;
    for (int round = 0; round < nrounds; ++round) {
        const int zi = round * kProjWarps + warp;
        double* t2w = t2s + ((size_t)(round & 1) * kProjWarps + warp) * P * MP * MP;
        if (zi < nzl) {
            const int iz = at.lo[2] + zi;
            const int jz = p.g.periodic[2] ? iz - floordiv(iz, Nz) * Nz : iz;
            const real_t* pz = psi_b + (size_t)jz * plane * P;

            // T2[part][ty][tx]: tile (1,1) can only hold ny+nx >= 16 > numax and is never needed
            double T2[P][MT][MT][2];
#pragma unroll
            for (int pp = 0; pp < P; ++pp)
#pragma unroll
                for (int ty = 0; ty < MT; ++ty)
#pragma unroll
                    for (int tx = 0; tx < MT; ++tx) T2[pp][ty][tx][0] = T2[pp][ty][tx][1] = 0.0;

            for (int c = 0; c < XC; ++c) {
                // ---- a2: per-lane column offset(s) of this chunk (wrap / clip) ----
                int off0, off1;
                {
                    const int ix0 = xs0 + c * CW + (CPLX ? q : 2 * q);
                    const int ix1 = ix0 + 1;
                    off0 = p.g.periodic[0] ? ix0 - floordiv(ix0, Nx) * Nx : min(max(ix0, 0), Nx - 1);
                    off1 = p.g.periodic[0] ? ix1 - floordiv(ix1, Nx) * Nx : min(max(ix1, 0), Nx - 1);
                }
                const bool v2 = vec && (CPLX || off1 == off0 + 1);
                double C1[MT][2][2];   // [ny tile][e or re/im][s]
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) C1[mt][0][0] = C1[mt][0][1] = C1[mt][1][0] = C1[mt][1][1] = 0.0;

                // ---- a3: y contraction, K = 4 rows per step ----
#pragma unroll 4
                for (int k = 0; k < KY; ++k) {
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
                    }
                    const real_t* pr = pz + (size_t)rowoff[4 * k + t] * P;
                    double v0, v1;
                    if (CPLX) {
                        load2(pr + (size_t)off0 * 2, vec, v0, v1);            // (re, im) of one column
                    } else if (v2) {
                        load2(pr + off0, true, v0, v1);                       // two adjacent columns
                    } else {
                        v0 = (double)__ldg(pr + off0); v1 = (double)__ldg(pr + off1);
                    }
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        const double afr = fy[((size_t)k * MT + mt) * 32 + lane];
                        dmma(C1[mt][0][0], C1[mt][0][1], afr, v0);
                        dmma(C1[mt][1][0], C1[mt][1][1], afr, v1);
                    }
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
            }
            // plane result -> shared, [part][ny][nx]
#pragma unroll
            for (int pp = 0; pp < P; ++pp)
#pragma unroll
                for (int ty = 0; ty < MT; ++ty)
#pragma unroll
                    for (int tx = 0; tx < MT; ++tx)
                        if (ty + tx < 2 || MT == 1) {
                            double2 o; o.x = T2[pp][ty][tx][0]; o.y = T2[pp][ty][tx][1];
                            *reinterpret_cast<double2*>(&t2w[(size_t)pp * MP * MP + (8 * ty + q) * MP + 8 * tx + 2 * t]) = o;
                        }
        }
        __syncthreads();
        // ---- a5: z contraction, thread n <- coefficient n ----
        const double* t2r = t2s + (size_t)(round & 1) * kProjWarps * P * MP * MP;
        const int wmax = min(kProjWarps, nzl - round * kProjWarps);
#pragma unroll
        for (int j = 0; j < NACC; ++j) {
            const int n = tid + j * blockDim.x;
            if (n < p.g.nsho) {
                const int nx = myn[j] & 255, ny = (myn[j] >> 8) & 255, nz = (myn[j] >> 16) & 255;
                for (int w = 0; w < wmax; ++w) {
                    const int z2 = round * kProjWarps + w;
                    const double f = fz[(size_t)z2 * MP + nz];
                    const double* tt = t2r + (size_t)w * P * MP * MP + ny * MP + nx;
                    if (!CPLX) {
                        acc[j][0] = fma(f, tt[0], acc[j][0]);
                    } else {
                        const double re = tt[0], im = tt[MP * MP];
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

template <int MT, int DT>
static sho_status launch_t(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s)
{
    using S = ProjSmem<MT, DT>;
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
    const size_t smem = S::total(p.ky_cap, p.nxe_cap, p.nz_cap);
    if (smem > 227 * 1024) {
        set_error("sho_project: box of %d x %d x %d points needs %zu bytes of shared memory (> 227 KB)",
                  pl->max_n[0], pl->max_n[1], pl->max_n[2], smem);
        return SHO_ERR_UNSUPPORTED;
    }
    auto kern = sho_project_kernel<MT, DT>;
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

sho_status launch_project(const sho_plan* pl, const void* psi, int nbands, void* coeff, cudaStream_t s)
{
    const bool two = pl->g.numax >= 8;
    switch (pl->dtype) {
        case SHO_R64:  return two ? launch_t<2, SHO_R64>(pl, psi, nbands, coeff, s)  : launch_t<1, SHO_R64>(pl, psi, nbands, coeff, s);
        case SHO_C128: return two ? launch_t<2, SHO_C128>(pl, psi, nbands, coeff, s) : launch_t<1, SHO_C128>(pl, psi, nbands, coeff, s);
        case SHO_R32:  return two ? launch_t<2, SHO_R32>(pl, psi, nbands, coeff, s)  : launch_t<1, SHO_R32>(pl, psi, nbands, coeff, s);
        case SHO_C64:  return two ? launch_t<2, SHO_C64>(pl, psi, nbands, coeff, s)  : launch_t<1, SHO_C64>(pl, psi, nbands, coeff, s);
    }
    set_error("sho_project: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

}  // namespace sho
