// sho_add.cu -- on-the-fly SHO expansion / add-back (step a6 of DESIGN.md) by OWNERSHIP TILING.
//
//   psi_b(r) += sum_a sum_n c[a][b][n] phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)        step (3)
//
// One CTA owns one psi tile of kAddTX x kAddTY x kAddTZ = 8 x 64 x 8 grid points of one band and keeps
// it in the accumulator registers of its FP64 tensor-core MMAs for the whole kernel; it walks the plan's
// list of (atom, periodic image) pairs whose box touches the tile, in ascending atom order, and finally
// does ONE read-modify-write of the tile.  No atomics, bit-reproducible, psi traffic = read + write of
// every touched tile exactly once.  Warp w owns z plane w of the tile (64 rows x 8 columns); two CTAs
// share an SM so that one computes while the other samples its tables.
//
// Per batch of (tile, atom image) pairs, all three expansion stages run on DMMA.8x8x4:
//   tables  (CTA-wide) the three 1D Hermite-Gauss tables of every pair are sampled on the fly (eq. (31),
//           PAPER.md:283-286) into shared memory in MMA fragment order; the pair's coefficients
//           c[a][b][:] are read once (coalesced), multiplied by the conjugate Bloch phase of the image
//           and scattered into the A fragments of the z stage
//   z       (CTA-wide, tasks spread over the warps)
//           T2[z][(ny,nx)] = sum_nz c[n(nx,ny,nz)] phi_nz(z)         M = (ny,nx) pairs sorted by ny+nx, so
//                                                                   that row tile mt needs only nz <=
//                                                                   numax - s_min(mt); K = nz; N = 8 planes
//   then every warp, for every pair of the batch that touches its plane:
//   x       T1[x][ny]  = sum_nx phi_nx(x) T2[z][(ny,nx)]             M = x, K = nx, N = ny
//   y       psi[y][x] += sum_ny phi_ny(y) T1[x][ny]                  M = y, K = ny, N = x
// The accumulator fragment of the x stage is exactly the B fragment of the y stage when column 2t+s of
// the x stage's N tile is assigned ny = 8 nt + 4 s + t: the contracted index is then cut in K steps of
// four consecutive ny, so only ceil((numax+1)/4) steps are issued.
#include "sho_device.cuh"

namespace sho {

struct AddParams {
    GridDev g;
    AddZTiles zt;
    const void* coeff;
    void* psi;
    const AtomDev* atoms;
    const int32_t* tile_ptr;
    const AddEntry* tile_ent;
    const int32_t* tile_list;
    const uint16_t* cainv;
    int32_t n_tile_list;
    int32_t nbands;
    int32_t ntile0, ntile1;
    int32_t vec_ok;
    int32_t batch;             // pairs per batch (shared-memory slots)
    int32_t npp;               // row stride of T2 (doubles): 8 nmt + 2, = 2 mod 8 and != 0 mod 16 (bank spread)
    int32_t slot;              // doubles per pair slot
    long long band_stride;
};

constexpr int kAddPoints = kAddTY + kAddTX + kAddTZ;    // 1D sample points per pair: 8 y blocks, 1 x block, 1 z block

// slot layout (doubles): [F: 10 blocks x KQ x 32][CA: nblk x P x 32][T2: P x 8 x npp][head: 2]
template <int KQ, int DT>
struct AddSmem {
    static constexpr int P = Elem<DT>::cplx ? 2 : 1;
    static constexpr int F = (kAddPoints / 8) * KQ * 32;
    static __host__ __device__ int ca(int) { return F; }
    static __host__ __device__ int t2(int nblk) { return F + nblk * P * 32; }
    static __host__ __device__ int head(int nblk, int npp) { return t2(nblk) + P * kAddTZ * npp; }
    static __host__ __device__ int slot_doubles(int nblk, int npp) { return head(nblk, npp) + 2; }
};

// phi_0..phi_{NV-1} as in sho_device.cuh::hermite_gauss, from the scalars of one atom
template <int NV>
__device__ __forceinline__ void hermite_gauss_s(double u, double inv_sigma, double pref, const double* __restrict__ hnorm,
                                                int numax, double (&out)[NV])
{
    const double xi = u * inv_sigma;
    const double g = exp(-0.5 * xi * xi) * pref;
    double hm = 0.0, hc = 1.0;
#pragma unroll
    for (int n = 0; n < NV; ++n) {
        out[n] = (n <= numax) ? hc * g * hnorm[n < SHO_NUMAX_MAX ? n : SHO_NUMAX_MAX] : 0.0;
        const double hn = xi * hc - (0.5 * (double)n) * hm;
        hm = hc;
        hc = hn;
    }
}

template <int KQ, int DT>
__global__ void __launch_bounds__(kAddWarps * 32, 2) sho_add_kernel(const AddParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    using S = AddSmem<KQ, DT>;
    constexpr bool CPLX = E::cplx;
    constexpr int P = S::P;
    constexpr int NV = 4 * KQ;                 // sampled functions per point (numax + 1 rounded up to 4)
    constexpr int NT = (KQ + 1) / 2;           // ny tiles of 8 in the x stage
    constexpr int NYT = kAddTY / 8;
    static_assert(kAddTX == 8 && kAddTZ == 8 && kAddWarps == 8, "one 8x8 MMA block per x / z extent");

    extern __shared__ __align__(16) double smem[];
    const int nsho = p.g.nsho;
    const int SLOT = p.slot;
    const int nblk = p.zt.nblk, nmt = p.zt.nmt, npp = p.npp;
    const int CA = S::ca(nblk), T2 = S::t2(nblk), HEAD = S::head(nblk, npp);

    const int tid = threadIdx.x, lane = tid & 31, zl = tid >> 5;
    const int q = lane >> 2, t = lane & 3;

    const int b = blockIdx.x / p.n_tile_list;
    const int tile = p.tile_list[blockIdx.x - b * p.n_tile_list];
    const int tx = tile % p.ntile0, ty = (tile / p.ntile0) % p.ntile1, tz = tile / (p.ntile0 * p.ntile1);
    const int jx0 = tx * kAddTX, jy0 = ty * kAddTY, jz0 = tz * kAddTZ;
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int numax = p.g.numax;
    const int ebeg = p.tile_ptr[tile], eend = p.tile_ptr[tile + 1];
    const int NB = p.batch;

    // zero the slots once: the padding entries of the z-stage A fragments and the zero column of T2 stay zero
    for (int i = tid; i < NB * SLOT; i += blockDim.x) smem[i] = 0.0;

    double D[NYT][P][2];
#pragma unroll
    for (int yt = 0; yt < NYT; ++yt)
#pragma unroll
        for (int pp = 0; pp < P; ++pp) D[yt][pp][0] = D[yt][pp][1] = 0.0;

    // x stage, B fragment B[k = nx][col = ny]: this lane reads T2[(ny,nx)] with nx = 4 ks + t and
    // ny = 8 nt + 4 (q & 1) + (q >> 1); pairs outside the basis read the zero column
    int t2off[NT][KQ];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int ks = 0; ks < KQ; ++ks) {
            const int ny = 8 * nt + 4 * (q & 1) + (q >> 1), nx = 4 * ks + t, s = ny + nx;
            t2off[nt][ks] = (s <= numax) ? (s * (s + 1)) / 2 + nx : 8 * nmt;
        }

    const real_t* cbase = reinterpret_cast<const real_t*>(p.coeff);

    for (int e0 = ebeg; e0 < eend; e0 += NB) {
        const int nb = min(NB, eend - e0);
        __syncthreads();                                        // the previous batch's tables are no longer read
        // ---------------- tables: 1D functions (step a1) in fragment order ----------------
        for (int it = tid; it < nb * kAddPoints; it += blockDim.x) {
            const int i = it / kAddPoints, r = it - i * kAddPoints;
            const AddEntry* en = p.tile_ent + e0 + i;
            const AtomDev* at = p.atoms + en->atom;
            const int d = r < kAddTY ? 1 : (r < kAddTY + kAddTX ? 0 : 2);
            const int N = p.g.ng[d];
            const int j = (d == 1 ? jy0 + r : (d == 0 ? jx0 : jz0) + (r & 7));
            const int iu = j + (int)en->m[d] * N;
            const bool valid = j < N && iu >= at->lo[d] && iu <= at->hi[d];
            double v[NV];
            if (valid) {
                hermite_gauss_s<NV>(displacement(iu, p.g.h, at->pos[d]), at->inv_sigma, at->pref, p.g.hnorm, numax, v);
            } else {
#pragma unroll
                for (int n = 0; n < NV; ++n) v[n] = 0.0;
            }
            // block r >> 3 (y: 0..7, x: 8, z: 9), point r & 7: element [k = n & 3] of K step n >> 2
            double* dst = smem + (size_t)i * SLOT + ((r >> 3) * KQ) * 32 + (r & 7) * 4;
#pragma unroll
            for (int kk = 0; kk < KQ; ++kk) {
                double2 a, c;
                a.x = v[4 * kk]; a.y = v[4 * kk + 1]; c.x = v[4 * kk + 2]; c.y = v[4 * kk + 3];
                *reinterpret_cast<double2*>(dst + kk * 32) = a;
                *reinterpret_cast<double2*>(dst + kk * 32 + 2) = c;
            }
        }
        if (tid < nb) {
            const AddEntry* en = p.tile_ent + e0 + tid;
            int32_t* meta = reinterpret_cast<int32_t*>(smem + (size_t)tid * SLOT + HEAD);
            meta[0] = en->ytlo; meta[1] = en->ythi; meta[2] = en->zmask; meta[3] = en->atom;
        }
        // coefficients of the batch: coalesced read, conjugate image phase, scatter into the z-stage A fragments
        for (int i = 0; i < nb; ++i) {
            const AddEntry* en = p.tile_ent + e0 + i;
            const real_t* c = cbase + ((size_t)en->atom * p.nbands + b) * nsho * P;
            double* ca = smem + (size_t)i * SLOT + CA;
            const double wr = en->wr, wi = en->wi;
            for (int n = tid; n < nsho; n += blockDim.x) {
                const int o = p.cainv[n];
                double* dst = ca + (o >> 5) * (32 * P) + (o & 31);
                if (!CPLX) {
                    dst[0] = (double)__ldg(c + n);
                } else {
                    double re, im;
                    load2(c + 2 * (size_t)n, p.vec_ok != 0, re, im);
                    dst[0] = re * wr - im * wi;
                    dst[32] = re * wi + im * wr;
                }
            }
        }
        __syncthreads();
        // ---------------- z stage: T2[z][(ny,nx)] for the 8 planes of the tile ----------------
        for (int task = zl; task < nb * nmt; task += kAddWarps) {
            const int i = task / nmt, mt = task - i * nmt;
            double* slot = smem + (size_t)i * SLOT;
            const int blk0 = p.zt.blk0[mt], nks = p.zt.nks[mt];
            double d[P][2];
#pragma unroll
            for (int pp = 0; pp < P; ++pp) d[pp][0] = d[pp][1] = 0.0;
            for (int ks = 0; ks < nks; ++ks) {
                const double bfr = slot[(9 * KQ + ks) * 32 + lane];            // B[k = nz][col = plane]
                const double* ap = slot + CA + (size_t)(blk0 + ks) * (32 * P) + lane;
#pragma unroll
                for (int pp = 0; pp < P; ++pp) dmma(d[pp][0], d[pp][1], ap[32 * pp], bfr);
            }
#pragma unroll
            for (int pp = 0; pp < P; ++pp) {
                double* o = slot + T2 + ((size_t)pp * kAddTZ + 2 * t) * npp + 8 * mt + q;
                o[0] = d[pp][0];
                o[npp] = d[pp][1];
            }
        }
        __syncthreads();
        // ---------------- x and y stages: every warp on its own plane ----------------
        for (int i = 0; i < nb; ++i) {
            const double* slot = smem + (size_t)i * SLOT;
            const int32_t* meta = reinterpret_cast<const int32_t*>(slot + HEAD);
            const int ytlo = meta[0], ythi = meta[1];
            if (!((meta[2] >> zl) & 1)) continue;
            const double* t2p = slot + T2 + (size_t)zl * npp;

            double D1[NT][P][2];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int pp = 0; pp < P; ++pp) D1[nt][pp][0] = D1[nt][pp][1] = 0.0;
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int ks = 0; ks < KQ; ++ks)
                    if (8 * nt + 4 * ks <= numax) {                     // warp-uniform: the block holds some ny+nx <= numax
                        const double a = slot[(8 * KQ + ks) * 32 + lane];
#pragma unroll
                        for (int pp = 0; pp < P; ++pp)
                            dmma(D1[nt][pp][0], D1[nt][pp][1], a, t2p[(size_t)pp * kAddTZ * npp + t2off[nt][ks]]);
                    }
#pragma unroll
            for (int yt = 0; yt < NYT; ++yt)
                if (yt >= ytlo && yt <= ythi) {
#pragma unroll
                    for (int kk = 0; kk < KQ; ++kk) {
                        const double a = slot[(yt * KQ + kk) * 32 + lane];
#pragma unroll
                        for (int pp = 0; pp < P; ++pp) dmma(D[yt][pp][0], D[yt][pp][1], a, D1[kk >> 1][pp][kk & 1]);
                    }
                }
        }
    }

    // ---------------- one read-modify-write of the owned tile ----------------
    const int jz = jz0 + zl;
    if (jz < Nz && eend > ebeg) {
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

template <int KQ, int DT>
static sho_status launch_t(const sho_plan* pl, const void* coeff, int nbands, void* psi, cudaStream_t s)
{
    using S = AddSmem<KQ, DT>;
    constexpr bool CPLX = Elem<DT>::cplx;
    AddParams p;
    p.g = pl->g;
    p.zt = pl->ztiles;
    p.coeff = coeff; p.psi = psi;
    p.atoms = pl->d_atoms;
    p.tile_ptr = pl->d_tile_ptr; p.tile_ent = pl->d_tile_ent; p.tile_list = pl->d_tile_list;
    p.cainv = pl->d_cainv;
    p.n_tile_list = pl->n_tile_list;
    p.nbands = nbands;
    p.ntile0 = pl->ntile[0]; p.ntile1 = pl->ntile[1];
    p.band_stride = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    const size_t esz = elem_size(pl->dtype);
    const size_t valign = CPLX ? esz : 2 * esz;
    p.vec_ok = ((reinterpret_cast<uintptr_t>(psi) % valign) == 0) && (CPLX || (pl->g.ng[0] % 2 == 0));
    if (CPLX && (reinterpret_cast<uintptr_t>(coeff) % esz) != 0) p.vec_ok = 0;
    p.npp = 8 * pl->ztiles.nmt + 2;
    p.slot = S::slot_doubles(pl->ztiles.nblk, p.npp);
    const size_t slot_bytes = (size_t)p.slot * 8;
    const size_t budget = 112 * 1024;                        // two CTAs per SM
    p.batch = (int)std::max<size_t>(1, std::min<size_t>(16, budget / slot_bytes));
    const size_t smem = slot_bytes * p.batch;
    auto kern = sho_add_kernel<KQ, DT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(add)");
    const long long nblocks = (long long)pl->n_tile_list * nbands;
    if (nblocks > 0x7fffffffLL) { set_error("sho_add: tiles*nbands too large"); return SHO_ERR_UNSUPPORTED; }
    kern<<<(unsigned)nblocks, kAddWarps * 32, smem, s>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launch sho_add_kernel");
    return SHO_OK;
}

template <int DT>
static sho_status launch_kq(const sho_plan* pl, const void* coeff, int nbands, void* psi, cudaStream_t s)
{
    switch ((pl->g.numax + 4) >> 2) {          // K steps of four n values that hold n <= numax
        case 1: return launch_t<1, DT>(pl, coeff, nbands, psi, s);
        case 2: return launch_t<2, DT>(pl, coeff, nbands, psi, s);
        case 3: return launch_t<3, DT>(pl, coeff, nbands, psi, s);
        default: return launch_t<4, DT>(pl, coeff, nbands, psi, s);
    }
}

sho_status launch_add(const sho_plan* pl, const void* coeff, int nbands, void* psi, cudaStream_t s)
{
    switch (pl->dtype) {
        case SHO_R64:  return launch_kq<SHO_R64>(pl, coeff, nbands, psi, s);
        case SHO_C128: return launch_kq<SHO_C128>(pl, coeff, nbands, psi, s);
        case SHO_R32:  return launch_kq<SHO_R32>(pl, coeff, nbands, psi, s);
        case SHO_C64:  return launch_kq<SHO_C64>(pl, coeff, nbands, psi, s);
    }
    set_error("sho_add: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

}  // namespace sho
