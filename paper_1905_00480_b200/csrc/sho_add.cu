// sho_add.cu -- on-the-fly SHO expansion / add-back (step a6 of DESIGN.md) by OWNERSHIP TILING.
//
//   psi_b(r) += sum_a sum_n c[a][b][n] phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)        step (3)
//
// One CTA owns one psi tile of kAddTX x kAddTY x kAddTZ grid points of one band and keeps it in the
// accumulator registers of its FP64 tensor-core MMAs for the whole kernel; it walks the plan's list
// of (atom, periodic image) pairs whose box touches the tile, in ascending atom order, and finally
// does ONE read-modify-write of the tile.  No atomics, bit-reproducible, psi traffic = read + write
// of every touched tile exactly once.
//
// Per (tile, atom image) the expansion runs z -> x -> y:
//   tables  (CTA-wide, per batch of kAddBatch pairs) the three 1D Hermite-Gauss tables are sampled on
//           the fly (eq. (31)) into shared memory, laid out as DMMA fragments
//   z       T2[z][ny][nx] = conj(w) sum_nz c[n(nx,ny,nz)] phi_nz(z)      (plain FMAs, N_SHO per plane)
//   x       T1[ny][x]     = sum_nx T2[z][ny][nx] phi_nx(x)               DMMA: M = x, K = nx, N = ny
//   y       psi[y][x]    += sum_ny phi_ny(y) T1[ny][x]                   DMMA: M = y, K = ny, N = x
// The accumulator fragment of the x stage is exactly the B fragment of the y stage when column 2t+s of
// the x stage's N tile is assigned ny = 8 nt + 4 s + t: the contracted index is then cut in K steps of
// four consecutive ny, so only ceil((numax+1)/4) steps are issued.
// Warp w of the CTA owns z plane w / 4 and the 8 columns (w % 4) * 8 .. +7 of the tile, all 64 rows.
#include "sho_device.cuh"

namespace sho {

constexpr int kAddBatch = 4;

struct AddParams {
    GridDev g;
    const void* coeff;
    void* psi;
    const AtomDev* atoms;
    const int32_t* tile_ptr;
    const AddEntry* tile_ent;
    const int32_t* tile_list;
    int32_t n_tile_list;
    int32_t nbands;
    int32_t ntile0, ntile1;
    int32_t vec_ok;
    long long band_stride;
};

template <int MT, int DT>
struct AddSmem {
    static constexpr int P = Elem<DT>::cplx ? 2 : 1;
    static constexpr int MP = 8 * MT, KS = 2 * MT;
    static constexpr int FY = (kAddTY / 8) * KS * 32;              // doubles per entry
    static constexpr int FX = (kAddTX / 8) * KS * 32;
    static constexpr int T2 = kAddTZ * P * MT * KS * 32;
    static constexpr int FZ = kAddTZ * MP;
    static constexpr int PH = 2;
    static constexpr int META = 4;                                 // ints
    static constexpr size_t bytes = (size_t)kAddBatch * ((FY + FX + T2 + FZ + PH) * 8 + META * 4);
};

template <int MT, int DT>
__global__ void __launch_bounds__(kAddWarps * 32, 2) sho_add_kernel(const AddParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    using S = AddSmem<MT, DT>;
    constexpr bool CPLX = E::cplx;
    constexpr int P = S::P, MP = S::MP, KSMAX = S::KS;
    constexpr int NB = kAddBatch;
    constexpr int NYT = kAddTY / 8, NXB = kAddTX / 8;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* fyA = reinterpret_cast<double*>(smem_raw);          // [NB][NYT][KS][32]   A fragments of the y stage
    double* fxA = fyA + NB * S::FY;                             // [NB][NXB][KS][32]   A fragments of the x stage
    double* t2B = fxA + NB * S::FX;                             // [NB][TZ][P][MT][KS][32]  B fragments of the x stage
    double* fzs = t2B + NB * S::T2;                             // [NB][TZ][MP]
    double* phs = fzs + NB * S::FZ;                             // [NB][2]  conj(w) of the image
    int32_t* meta = reinterpret_cast<int32_t*>(phs + NB * S::PH);   // [NB][4]  yt_lo, yt_hi, x-block mask, z mask

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int q = lane >> 2, t = lane & 3;
    const int zl = warp / NXB, xb = warp % NXB;

    const int b = blockIdx.x / p.n_tile_list;
    const int tile = p.tile_list[blockIdx.x - b * p.n_tile_list];
    const int tx = tile % p.ntile0, ty = (tile / p.ntile0) % p.ntile1, tz = tile / (p.ntile0 * p.ntile1);
    const int jx0 = tx * kAddTX, jy0 = ty * kAddTY, jz0 = tz * kAddTZ;
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int numax = p.g.numax;
    const int KQ = (numax + 4) >> 2;                            // K steps of four n values that hold n <= numax
    const int ebeg = p.tile_ptr[tile], eend = p.tile_ptr[tile + 1];

    double D[NYT][P][2];
#pragma unroll
    for (int yt = 0; yt < NYT; ++yt)
#pragma unroll
        for (int pp = 0; pp < P; ++pp) D[yt][pp][0] = D[yt][pp][1] = 0.0;

    const real_t* cbase = reinterpret_cast<const real_t*>(p.coeff);

    for (int e0 = ebeg; e0 < eend; e0 += NB) {
        const int nb = min(NB, eend - e0);
        __syncthreads();                                        // the previous batch's tables are no longer read
        // ---------------- tables, phase A: 1D functions (step a1), image phase, overlap ranges ----------------
        constexpr int ITEMS_A = kAddTY + kAddTX + kAddTZ + 1;
        for (int it = tid; it < nb * ITEMS_A; it += blockDim.x) {
            const int i = it / ITEMS_A, r = it - i * ITEMS_A;
            const AddEntry en = p.tile_ent[e0 + i];
            const AtomDev at = p.atoms[en.atom];
            double v[MP];
            if (r < kAddTY) {
                const int jy = jy0 + r, iy = jy + en.m[1] * Ny;
                const bool valid = jy < Ny && iy >= at.lo[1] && iy <= at.hi[1];
                hermite_gauss<MP>(displacement(iy, p.g.h, at.pos[1]), at.sigma, p.g.hnorm, numax, valid, v);
                const int yt = r >> 3, qq = r & 7;
#pragma unroll
                for (int n = 0; n < MP; ++n)   // A[y = qq][k = n & 3] of K step n >> 2
                    fyA[((i * NYT + yt) * KSMAX + (n >> 2)) * 32 + qq * 4 + (n & 3)] = v[n];
            } else if (r < kAddTY + kAddTX) {
                const int cidx = r - kAddTY;
                const int jx = jx0 + cidx, ix = jx + en.m[0] * Nx;
                const bool valid = jx < Nx && ix >= at.lo[0] && ix <= at.hi[0];
                hermite_gauss<MP>(displacement(ix, p.g.h, at.pos[0]), at.sigma, p.g.hnorm, numax, valid, v);
                const int xbb = cidx >> 3, qq = cidx & 7;
#pragma unroll
                for (int n = 0; n < MP; ++n)   // A[x = qq][k = n & 3] of K step n >> 2
                    fxA[((i * NXB + xbb) * KSMAX + (n >> 2)) * 32 + qq * 4 + (n & 3)] = v[n];
            } else if (r < kAddTY + kAddTX + kAddTZ) {
                const int z = r - kAddTY - kAddTX;
                const int jz = jz0 + z, iz = jz + en.m[2] * Nz;
                const bool valid = jz < Nz && iz >= at.lo[2] && iz <= at.hi[2];
                hermite_gauss<MP>(displacement(iz, p.g.h, at.pos[2]), at.sigma, p.g.hnorm, numax, valid, v);
#pragma unroll
                for (int n = 0; n < MP; ++n) fzs[(i * kAddTZ + z) * MP + n] = v[n];
            } else {
                // overlap of the box with the tile, in units the warps can skip
                const int oy = jy0 + en.m[1] * Ny, ox = jx0 + en.m[0] * Nx, oz = jz0 + en.m[2] * Nz;
                const int ylast = min(kAddTY, Ny - jy0) - 1;
                const int ya = max(at.lo[1] - oy, 0), yb = min(at.hi[1] - oy, ylast);
                int xmask = 0, zmask = 0;
                for (int k = 0; k < NXB; ++k) {
                    const int c0 = max(ox + 8 * k, at.lo[0]), c1 = min(min(ox + 8 * k + 7, at.hi[0]), Nx - 1 + en.m[0] * Nx);
                    if (c1 >= c0) xmask |= 1 << k;
                }
                for (int k = 0; k < kAddTZ; ++k) {
                    const int iz = oz + k;
                    if (jz0 + k < Nz && iz >= at.lo[2] && iz <= at.hi[2]) zmask |= 1 << k;
                }
                meta[4 * i + 0] = ya >> 3;
                meta[4 * i + 1] = (yb >= ya) ? (yb >> 3) : -1;
                meta[4 * i + 2] = xmask;
                meta[4 * i + 3] = zmask;
                double sn = 0.0, cs = 1.0;
                if (CPLX && p.g.has_phase)   // conj(w), w = exp(2 pi i k.m)  (reading A6)
                    sincospi(-2.0 * (p.g.kfrac[0] * en.m[0] + p.g.kfrac[1] * en.m[1] + p.g.kfrac[2] * en.m[2]), &sn, &cs);
                phs[2 * i] = cs; phs[2 * i + 1] = sn;
            }
        }
        __syncthreads();
        // ---------------- tables, phase B: z stage, T2 = conj(w) sum_nz c phi_nz(z), as B fragments ----------------
        const int items_b = kAddTZ * MT * KQ * 32;
        for (int it = tid; it < nb * items_b; it += blockDim.x) {
            const int i = it / items_b;
            int r = it - i * items_b;
            const int ln = r & 31; r >>= 5;
            const int ks = r % KQ; r /= KQ;
            const int nt = r % MT, z = r / MT;
            const int qq = ln >> 2, tt = ln & 3;
            const int ny = 8 * nt + 4 * (qq & 1) + (qq >> 1), nx = 4 * ks + tt;   // B[k = tt][col qq]
            double sre = 0.0, sim = 0.0;
            if (ny + nx <= numax && ((meta[4 * i + 3] >> z) & 1)) {
                const AddEntry en = p.tile_ent[e0 + i];
                const real_t* c = cbase + ((size_t)en.atom * p.nbands + b) * p.g.nsho * P;
                const double* fz = fzs + (i * kAddTZ + z) * MP;
                int zoff = 0;
                for (int nz = 0; nz <= numax - ny - nx; ++nz) {
                    const int mrow = numax - nz + 1;                                // rows (ny values) in plane nz
                    const int n = zoff + ny * mrow - (ny * (ny - 1)) / 2 + nx;      // reading A8
                    if (!CPLX) sre = fma((double)__ldg(c + n), fz[nz], sre);
                    else {
                        sre = fma((double)__ldg(c + 2 * n), fz[nz], sre);
                        sim = fma((double)__ldg(c + 2 * n + 1), fz[nz], sim);
                    }
                    zoff += mrow * (mrow + 1) / 2;
                }
            }
            double* dst = t2B + ((((size_t)(i * kAddTZ + z) * P) * MT + nt) * KSMAX + ks) * 32 + ln;
            if (!CPLX) dst[0] = sre;
            else {
                const double cr = phs[2 * i], ci = phs[2 * i + 1];
                dst[0] = sre * cr - sim * ci;
                dst[(size_t)MT * KSMAX * 32] = sre * ci + sim * cr;
            }
        }
        __syncthreads();
        // ---------------- x and y stages on the tensor cores ----------------
        for (int i = 0; i < nb; ++i) {
            const int ytlo = meta[4 * i + 0], ythi = meta[4 * i + 1];
            if (!((meta[4 * i + 2] >> xb) & 1) || !((meta[4 * i + 3] >> zl) & 1) || ythi < ytlo) continue;
            double D1[MT][P][2];
#pragma unroll
            for (int nt = 0; nt < MT; ++nt)
#pragma unroll
                for (int pp = 0; pp < P; ++pp) D1[nt][pp][0] = D1[nt][pp][1] = 0.0;
#pragma unroll
            for (int nt = 0; nt < MT; ++nt)
#pragma unroll
                for (int ks = 0; ks < KSMAX; ++ks)
                    if (ks < KQ && 8 * nt + 4 * ks <= numax) {
                        const double a = fxA[((i * NXB + xb) * KSMAX + ks) * 32 + lane];
#pragma unroll
                        for (int pp = 0; pp < P; ++pp) {
                            const double bb = t2B[((((size_t)(i * kAddTZ + zl) * P + pp) * MT + nt) * KSMAX + ks) * 32 + lane];
                            dmma(D1[nt][pp][0], D1[nt][pp][1], a, bb);
                        }
                    }
#pragma unroll
            for (int yt = 0; yt < NYT; ++yt)
                if (yt >= ytlo && yt <= ythi) {
#pragma unroll
                    for (int kk = 0; kk < KSMAX; ++kk)
                        if (kk < KQ) {
                            const double a = fyA[((i * NYT + yt) * KSMAX + kk) * 32 + lane];
#pragma unroll
                            for (int pp = 0; pp < P; ++pp) dmma(D[yt][pp][0], D[yt][pp][1], a, D1[kk >> 1][pp][kk & 1]);
                        }
                }
        }
    }

    // ---------------- one read-modify-write of the owned tile ----------------
    const int jz = jz0 + zl;
    if (jz < Nz) {
        real_t* pb = reinterpret_cast<real_t*>(p.psi) + ((size_t)b * p.band_stride + (size_t)jz * Ny * Nx) * P;
        const int jx = jx0 + xb * 8 + 2 * t;
#pragma unroll
        for (int yt = 0; yt < NYT; ++yt) {
            const int jy = jy0 + 8 * yt + q;
            if (jy < Ny && jx < Nx) {
                real_t* pp_ = pb + ((size_t)jy * Nx + jx) * P;
                if (!CPLX) {
                    if (p.vec_ok && jx + 1 < Nx) {
                        double v0, v1;
                        load2_rw(pp_, v0, v1);
                        store2(pp_, v0 + D[yt][0][0], v1 + D[yt][0][1]);
                    } else {
                        pp_[0] = (real_t)((double)pp_[0] + D[yt][0][0]);
                        if (jx + 1 < Nx) pp_[1] = (real_t)((double)pp_[1] + D[yt][0][1]);
                    }
                } else {
#pragma unroll
                    for (int s = 0; s < 2; ++s)
                        if (jx + s < Nx) {
                            real_t* pc = pp_ + 2 * s;
                            if (p.vec_ok) {
                                double v0, v1;
                                load2_rw(pc, v0, v1);
                                store2(pc, v0 + D[yt][0][s], v1 + D[yt][P - 1][s]);
                            } else {
                                pc[0] = (real_t)((double)pc[0] + D[yt][0][s]);
                                pc[1] = (real_t)((double)pc[1] + D[yt][P - 1][s]);
                            }
                        }
                }
            }
        }
    }
}

template <int MT, int DT>
static sho_status launch_t(const sho_plan* pl, const void* coeff, int nbands, void* psi, cudaStream_t s)
{
    using S = AddSmem<MT, DT>;
    constexpr bool CPLX = Elem<DT>::cplx;
    AddParams p;
    p.g = pl->g;
    p.coeff = coeff; p.psi = psi;
    p.atoms = pl->d_atoms;
    p.tile_ptr = pl->d_tile_ptr; p.tile_ent = pl->d_tile_ent; p.tile_list = pl->d_tile_list;
    p.n_tile_list = pl->n_tile_list;
    p.nbands = nbands;
    p.ntile0 = pl->ntile[0]; p.ntile1 = pl->ntile[1];
    p.band_stride = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    const size_t esz = elem_size(pl->dtype);
    const size_t valign = CPLX ? esz : 2 * esz;
    p.vec_ok = ((reinterpret_cast<uintptr_t>(psi) % valign) == 0) && (CPLX || (pl->g.ng[0] % 2 == 0));
    auto kern = sho_add_kernel<MT, DT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::bytes);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(add)");
    const long long nblocks = (long long)pl->n_tile_list * nbands;
    if (nblocks > 0x7fffffffLL) { set_error("sho_add: tiles*nbands too large"); return SHO_ERR_UNSUPPORTED; }
    kern<<<(unsigned)nblocks, kAddWarps * 32, S::bytes, s>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launch sho_add_kernel");
    return SHO_OK;
}

sho_status launch_add(const sho_plan* pl, const void* coeff, int nbands, void* psi, cudaStream_t s)
{
    const bool two = pl->g.numax >= 8;
    switch (pl->dtype) {
        case SHO_R64:  return two ? launch_t<2, SHO_R64>(pl, coeff, nbands, psi, s)  : launch_t<1, SHO_R64>(pl, coeff, nbands, psi, s);
        case SHO_C128: return two ? launch_t<2, SHO_C128>(pl, coeff, nbands, psi, s) : launch_t<1, SHO_C128>(pl, coeff, nbands, psi, s);
        case SHO_R32:  return two ? launch_t<2, SHO_R32>(pl, coeff, nbands, psi, s)  : launch_t<1, SHO_R32>(pl, coeff, nbands, psi, s);
        case SHO_C64:  return two ? launch_t<2, SHO_C64>(pl, coeff, nbands, psi, s)  : launch_t<1, SHO_C64>(pl, coeff, nbands, psi, s);
    }
    set_error("sho_add: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

}  // namespace sho
