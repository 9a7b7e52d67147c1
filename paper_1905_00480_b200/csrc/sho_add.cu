// sho_add.cu -- on-the-fly SHO expansion / add-back (step a6 of DESIGN.md) by OWNERSHIP TILING.
//
//   psi_b(r) += sum_a sum_n c[a][b][n] phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)        step (3)
//
// One CTA owns one psi tile of kAddTX x kAddTY x kAddTZ = 8 x 64 x 16 grid points of one band and keeps
// it in the accumulator registers of its FP64 tensor-core MMAs for the whole kernel; it walks the plan's
// list of (atom, periodic image) pairs whose box touches the tile, in ascending atom order, and finally
// does ONE read-modify-write of the tile.  No atomics, bit-reproducible, psi traffic = read + write of
// every touched tile exactly once.  Warp w owns z plane w of the tile (64 rows x 8 columns).
//
// Per batch of (tile, atom image) pairs:
//   tables  (CTA-wide) the three 1D Hermite-Gauss tables of every pair are sampled on the fly (eq. (31),
//           PAPER.md:283-286) into shared memory, x and y laid out as DMMA A fragments; the pair's
//           coefficients c[a][b][:] are staged next to them with coalesced loads
// then every warp, for every pair of the batch that touches its plane, expands z -> x -> y:
//   z       T2[ny][nx] = conj(w) sum_nz c[n(nx,ny,nz)] phi_nz(z)         plain FMAs, each lane computes
//                                                                       exactly the B-fragment entries it needs
//   x       T1[x][ny]  = sum_nx phi_nx(x) T2[ny][nx]                     DMMA: M = x, K = nx, N = ny
//   y       psi[y][x] += sum_ny phi_ny(y) T1[x][ny]                      DMMA: M = y, K = ny, N = x
// The accumulator fragment of the x stage is exactly the B fragment of the y stage when column 2t+s of
// the x stage's N tile is assigned ny = 8 nt + 4 s + t: the contracted index is then cut in K steps of
// four consecutive ny, so only ceil((numax+1)/4) steps are issued.
#include "sho_device.cuh"

namespace sho {

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
    int32_t batch;             // pairs per batch (shared-memory slots)
    long long band_stride;
};

template <int MT, int DT>
struct AddSmem {
    static constexpr int P = Elem<DT>::cplx ? 2 : 1;
    static constexpr int MP = 8 * MT, KS = 2 * MT;
    static constexpr int FY = (kAddTY / 8) * KS * 32;              // doubles per pair
    static constexpr int FX = KS * 32;
    static constexpr int FZ = kAddTZ * MP;
    static constexpr int HEAD = 4;                                 // conj(w) re, im; 4 ints of overlap ranges
    static __host__ __device__ int slot_doubles(int nsho) { return FY + FX + FZ + HEAD + ((nsho * P + 1) & ~1); }
};

template <int MT, int DT>
__global__ void __launch_bounds__(kAddWarps * 32, 1) sho_add_kernel(const AddParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    using S = AddSmem<MT, DT>;
    constexpr bool CPLX = E::cplx;
    constexpr int P = S::P, MP = S::MP, KSMAX = S::KS;
    constexpr int NYT = kAddTY / 8;
    static_assert(kAddTX == 8, "one 8-column block per tile");

    extern __shared__ __align__(16) double smem[];
    const int nsho = p.g.nsho;
    const int SLOT = S::slot_doubles(nsho);
    // slot layout: [FY fyA][FX fxA][FZ fzs][2 phase][4 ints meta][nsho*P coefficients]

    const int tid = threadIdx.x, lane = tid & 31, zl = tid >> 5;
    const int q = lane >> 2, t = lane & 3;

    const int b = blockIdx.x / p.n_tile_list;
    const int tile = p.tile_list[blockIdx.x - b * p.n_tile_list];
    const int tx = tile % p.ntile0, ty = (tile / p.ntile0) % p.ntile1, tz = tile / (p.ntile0 * p.ntile1);
    const int jx0 = tx * kAddTX, jy0 = ty * kAddTY, jz0 = tz * kAddTZ;
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int numax = p.g.numax;
    const int KQ = (numax + 4) >> 2;                            // K steps of four n values that hold n <= numax
    const int ebeg = p.tile_ptr[tile], eend = p.tile_ptr[tile + 1];
    const int NB = p.batch;

    double D[NYT][P][2];
#pragma unroll
    for (int yt = 0; yt < NYT; ++yt)
#pragma unroll
        for (int pp = 0; pp < P; ++pp) D[yt][pp][0] = D[yt][pp][1] = 0.0;

    const real_t* cbase = reinterpret_cast<const real_t*>(p.coeff);
    // (ny, nx) of the B-fragment entries this lane computes in the z stage: B[k = t][col = q]
    const int ny_l = 4 * (q & 1) + (q >> 1);                    // + 8 nt

    for (int e0 = ebeg; e0 < eend; e0 += NB) {
        const int nb = min(NB, eend - e0);
        __syncthreads();                                        // the previous batch's tables are no longer read
        // ---------------- tables: 1D functions (step a1), image phase, overlap ranges ----------------
        constexpr int ITEMS = kAddTY + kAddTX + kAddTZ + 1;
        for (int it = tid; it < nb * ITEMS; it += blockDim.x) {
            const int i = it / ITEMS, r = it - i * ITEMS;
            const AddEntry en = p.tile_ent[e0 + i];
            const AtomDev at = p.atoms[en.atom];
            double* slot = smem + (size_t)i * SLOT;
            double v[MP];
            if (r < kAddTY) {
                const int jy = jy0 + r, iy = jy + en.m[1] * Ny;
                const bool valid = jy < Ny && iy >= at.lo[1] && iy <= at.hi[1];
                hermite_gauss<MP>(displacement(iy, p.g.h, at.pos[1]), at, p.g.hnorm, numax, valid, v);
                double* fyA = slot + ((r >> 3) * KSMAX) * 32 + (r & 7) * 4;
#pragma unroll
                for (int n = 0; n < MP; ++n)   // A[y = r & 7][k = n & 3] of K step n >> 2
                    fyA[(n >> 2) * 32 + (n & 3)] = v[n];
            } else if (r < kAddTY + kAddTX) {
                const int cidx = r - kAddTY;
                const int jx = jx0 + cidx, ix = jx + en.m[0] * Nx;
                const bool valid = jx < Nx && ix >= at.lo[0] && ix <= at.hi[0];
                hermite_gauss<MP>(displacement(ix, p.g.h, at.pos[0]), at, p.g.hnorm, numax, valid, v);
                double* fxA = slot + S::FY + cidx * 4;
#pragma unroll
                for (int n = 0; n < MP; ++n)   // A[x = cidx][k = n & 3] of K step n >> 2
                    fxA[(n >> 2) * 32 + (n & 3)] = v[n];
            } else if (r < kAddTY + kAddTX + kAddTZ) {
                const int z = r - kAddTY - kAddTX;
                const int jz = jz0 + z, iz = jz + en.m[2] * Nz;
                const bool valid = jz < Nz && iz >= at.lo[2] && iz <= at.hi[2];
                hermite_gauss<MP>(displacement(iz, p.g.h, at.pos[2]), at, p.g.hnorm, numax, valid, v);
                double* fzs = slot + S::FY + S::FX + z * MP;
#pragma unroll
                for (int n = 0; n < MP; ++n) fzs[n] = v[n];
            } else {
                // overlap of the box with the tile, in units the warps can skip
                const int oy = jy0 + en.m[1] * Ny, oz = jz0 + en.m[2] * Nz;
                const int ylast = min(kAddTY, Ny - jy0) - 1;
                const int ya = max(at.lo[1] - oy, 0), yb = min(at.hi[1] - oy, ylast);
                int zmask = 0;
                for (int k = 0; k < kAddTZ; ++k) {
                    const int iz = oz + k;
                    if (jz0 + k < Nz && iz >= at.lo[2] && iz <= at.hi[2]) zmask |= 1 << k;
                }
                double* head = slot + S::FY + S::FX + S::FZ;
                double sn = 0.0, cs = 1.0;
                if (CPLX && p.g.has_phase)   // conj(w), w = exp(2 pi i k.m)  (reading A6)
                    sincospi(-2.0 * (p.g.kfrac[0] * en.m[0] + p.g.kfrac[1] * en.m[1] + p.g.kfrac[2] * en.m[2]), &sn, &cs);
                head[0] = cs; head[1] = sn;
                int32_t* meta = reinterpret_cast<int32_t*>(head + 2);
                meta[0] = ya >> 3;
                meta[1] = (yb >= ya) ? (yb >> 3) : -1;
                meta[2] = zmask;
                meta[3] = en.atom;
            }
        }
        // coefficients of the batch, coalesced: c[atom][b][0 .. nsho) -> shared (as doubles)
        for (int i = 0; i < nb; ++i) {
            const int atom = p.tile_ent[e0 + i].atom;
            const real_t* c = cbase + ((size_t)atom * p.nbands + b) * nsho * P;
            double* cs = smem + (size_t)i * SLOT + S::FY + S::FX + S::FZ + S::HEAD;
            for (int n = tid; n < nsho * P; n += blockDim.x) cs[n] = (double)__ldg(c + n);
        }
        __syncthreads();
        // ---------------- z, x and y stages: every warp on its own plane ----------------
        for (int i = 0; i < nb; ++i) {
            const double* slot = smem + (size_t)i * SLOT;
            const double* head = slot + S::FY + S::FX + S::FZ;
            const int32_t* meta = reinterpret_cast<const int32_t*>(head + 2);
            const int ytlo = meta[0], ythi = meta[1];
            if (!((meta[2] >> zl) & 1) || ythi < ytlo) continue;
            const double* fz = slot + S::FY + S::FX + zl * MP;
            const double* cs = head + S::HEAD;
            const double wr = head[0], wi = head[1];

            double D1[MT][P][2];
#pragma unroll
            for (int nt = 0; nt < MT; ++nt)
#pragma unroll
                for (int pp = 0; pp < P; ++pp) D1[nt][pp][0] = D1[nt][pp][1] = 0.0;
#pragma unroll
            for (int nt = 0; nt < MT; ++nt) {
                const int ny = 8 * nt + ny_l;
#pragma unroll
                for (int ks = 0; ks < KSMAX; ++ks) {
                    if (ks < KQ && 8 * nt + 4 * ks <= numax) {          // warp-uniform: the block holds some ny+nx <= numax
                        const int nx = 4 * ks + t;
                        const int lim = numax - ny - nx;                // nz <= lim
                        const int base = ny * (numax + 1) - (ny * (ny - 1)) / 2 + nx;   // reading A8, minus the nz part
                        double sre = 0.0, sim = 0.0;
#pragma unroll
                        for (int nz = 0; nz < MP; ++nz) {
                            if (nz <= lim) {
                                const int n = base + p.g.zoff[nz] - ny * nz;
                                const double f = fz[nz];
                                if (!CPLX) sre = fma(cs[n], f, sre);
                                else { sre = fma(cs[2 * n], f, sre); sim = fma(cs[2 * n + 1], f, sim); }
                            }
                        }
                        const double a = slot[S::FY + ks * 32 + lane];
                        if (!CPLX) dmma(D1[nt][0][0], D1[nt][0][1], a, sre);
                        else {
                            dmma(D1[nt][0][0], D1[nt][0][1], a, sre * wr - sim * wi);
                            dmma(D1[nt][P - 1][0], D1[nt][P - 1][1], a, sre * wi + sim * wr);
                        }
                    }
                }
            }
#pragma unroll
            for (int yt = 0; yt < NYT; ++yt)
                if (yt >= ytlo && yt <= ythi) {
#pragma unroll
                    for (int kk = 0; kk < KSMAX; ++kk)
                        if (kk < KQ) {
                            const double a = slot[(yt * KSMAX + kk) * 32 + lane];
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
        const int jx = jx0 + 2 * t;
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
    const size_t slot_bytes = (size_t)S::slot_doubles(pl->g.nsho) * 8;
    p.batch = (int)std::max<size_t>(1, std::min<size_t>(11, (200 * 1024) / slot_bytes));
    const size_t smem = slot_bytes * p.batch;
    auto kern = sho_add_kernel<MT, DT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(add)");
    const long long nblocks = (long long)pl->n_tile_list * nbands;
    if (nblocks > 0x7fffffffLL) { set_error("sho_add: tiles*nbands too large"); return SHO_ERR_UNSUPPORTED; }
    kern<<<(unsigned)nblocks, kAddWarps * 32, smem, s>>>(p);
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
