// sho_add.cu -- on-the-fly SHO expansion / add-back (step a6 of DESIGN.md) by OWNERSHIP TILING.
//
//   psi_b(r) += sum_a sum_n c[a][b][n] phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)        step (3)
//
// One CTA owns one psi tile of kAddTX x kAddTY x kAddTZ = 8 x 64 x 8 grid points of one band and keeps
// it in the accumulator registers of its FP64 tensor-core MMAs for the whole kernel; it walks the plan's
// list of (atom, periodic image) pairs whose box touches the tile, in ascending atom order, and finally
// does ONE read-modify-write of the tile.  No atomics, bit-reproducible, psi traffic = read + write of
// every touched tile exactly once.  Warp w owns z plane w of the tile (64 rows x 8 columns); two CTAs
// share an SM.
//
// The pair list is consumed in groups of NG pairs by a software pipeline with ONE barrier per step; in
// step s every warp runs, back to back and without waiting for the other warps,
//   E(s+1)  cp.async of the 96-byte records of the next group (atom parameters included: no pointer chase)
//   C(s)    issue the global loads of the group's coefficients c[a][b][:] (consumed at the end of the step)
//   XY(s-2) the x and y stages of the group whose tables and T2 are complete, on its own z plane:
//             x   T1[x][ny]  = sum_nx phi_nx(x) T2[z][(ny,nx)]       M = x, K = nx, N = ny
//             y   psi[y][x] += sum_ny phi_ny(y) T1[x][ny]            M = y, K = ny, N = x
//           The accumulator fragment of the x stage is exactly the B fragment of the y stage when column
//           2t+s of the x stage's N tile is assigned ny = 8 nt + 4 s + t.
//   Z(s-1)  its share of the z stage of the previous group
//             T2[z][(ny,nx)] = sum_nz c[n(nx,ny,nz)] phi_nz(z)       M = (ny,nx) pairs sorted by ny+nx, so that
//                                                                   row tile mt needs only nz <= numax -
//                                                                   s_min(mt); K = nz; N = 8 planes
//   T(s)    its share of the group's three 1D Hermite-Gauss tables, sampled on the fly (eq. (31),
//           PAPER.md:283-286) into shared memory in MMA fragment order, and the scatter of the (now arrived)
//           coefficients, times the conjugate Bloch phase of the image, into the A fragments of the z stage
// so the latency-bound stages (E, C, T) of one warp overlap the tensor-core stages of the others.  All
// three expansion stages run on DMMA.8x8x4.  Ring depths: x/y tables 3, everything else 2.
#include <algorithm>
#include <cstring>

#include "sho_device.cuh"

namespace sho {

constexpr int kAddZTMax = 6;       // z-stage tasks one warp can own per step

struct AddZTask { int32_t ca, fz, t2, w; };     // offsets inside a ring slot; w = nks | mt << 8 | pair << 16 (nks = 0: none)

struct AddParams {
    GridDev g;
    const void* coeff;
    void* psi;
    const int32_t* tile_ptr;
    const AddEntry* tile_ent;
    const int32_t* tile_list;
    const uint16_t* cainv;
    const uint16_t* t2pos;
    int32_t n_tile_list;
    int32_t nbands;
    int32_t ntile0, ntile1;
    int32_t vec_ok;
    int32_t ng;                // pairs per pipeline step (NG)
    int32_t npp;               // columns per plane of T2: 8 nmt + 2; column 8 nmt holds zeros
    int32_t nblk, nmt;         // K blocks of the z-stage A fragments per pair; row tiles of the z stage
    int32_t zt;                // z-stage tasks per warp and step (<= kAddZTMax)
    int32_t t_first;           // first thread that samples table points (the T stage runs on the last warps)
    long long band_stride;
    double hz[SHO_NUMAX_MAX + 1];                  // sqrt(2^n / n!) for n <= numax, 0 beyond (padding functions vanish)
    AddZTask ztask[kAddWarps][kAddZTMax];          // balanced against the T stage on the host (launch_t)
};

constexpr int kAddPoints = kAddTY + kAddTX + kAddTZ;    // 1D sample points per pair: 8 y blocks, 1 x block, 1 z block

// shared-memory carve-up (doubles): [FXY: 3 NG x 9 KQ 32][FZ: 2 NG x KQ 32][CA: 2 NG x nblk 32 P][T2: 2 NG x 8 npp P]
// then [ENT: 2 NG records][META: 3 NG int32][ZPOS: 8 nmt uint16].  CA and T2 keep the real and imaginary
// parts of complex data side by side, so one 16-byte access moves both.
template <int KQ, int DT>
struct AddSmem {
    static constexpr int P = Elem<DT>::cplx ? 2 : 1;
    static constexpr int FXYS = 9 * KQ * 32;
    static constexpr int FZS = KQ * 32;
    static constexpr int CPT = (KQ == 4) ? 4 : 2;            // coefficients a thread holds in flight per step
    static __host__ __device__ int cas(int nblk) { return nblk * 32 * P; }
    static __host__ __device__ int t2s(int npp) { return kAddTZ * npp * P; }
    static __host__ __device__ size_t bytes(int ng, int nblk, int nmt)
    {
        const int npp = 8 * nmt + 2;
        size_t b = 8 * (size_t)ng * (3 * FXYS + 2 * FZS + 2 * cas(nblk) + 2 * t2s(npp));
        b += (size_t)2 * ng * sizeof(AddEntry) + (size_t)3 * ng * 4 + (size_t)8 * nmt * 2;
        return (b + 15) & ~(size_t)15;
    }
};

// one real (P = 1) or one complex (P = 2) value as a single shared-memory access
template <int P> struct PartVec;
template <> struct PartVec<1> { double x; __device__ double re() const { return x; } __device__ double im() const { return 0.0; } };
template <> struct __align__(16) PartVec<2> { double x, y; __device__ double re() const { return x; } __device__ double im() const { return y; } };

// H_n(xi) exp(-xi^2/2) (sqrt(pi) sigma)^(-1/2) scale[n], n < NV, by the paper's monic recurrence (eq. (31),
// PAPER.md:283-284) carried on p_n = H_n g; scale[n] = sqrt(2^n/n!) makes the functions orthonormal (reading A1)
template <int NV>
__device__ __forceinline__ void hermite_gauss_s(double u, double inv_sigma, double pref, const double* __restrict__ scale,
                                                double (&out)[NV])
{
    const double xi = u * inv_sigma;
    double pm = 0.0, pc = exp(-0.5 * xi * xi) * pref;
#pragma unroll
    for (int n = 0; n < NV; ++n) {
        out[n] = pc * scale[n];
        const double pn = xi * pc - (0.5 * (double)n) * pm;
        pm = pc;
        pc = pn;
    }
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// coefficient loads that stay where they are issued (start of the step), read-only path
__device__ __forceinline__ void ldg_pinned(const double* p, bool vec, double& re, double& im)
{
    if (vec) asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(re), "=d"(im) : "l"(p));
    else { asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(re) : "l"(p)); asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(im) : "l"(p + 1)); }
}
__device__ __forceinline__ void ldg_pinned(const float* p, bool vec, double& re, double& im)
{
    float a, b;
    if (vec) asm volatile("ld.global.nc.v2.f32 {%0,%1}, [%2];" : "=f"(a), "=f"(b) : "l"(p));
    else { asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(a) : "l"(p)); asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(b) : "l"(p + 1)); }
    re = (double)a; im = (double)b;
}
__device__ __forceinline__ void ldg_pinned(const double* p, double& re)
{
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(re) : "l"(p));
}
__device__ __forceinline__ void ldg_pinned(const float* p, double& re)
{
    float a;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(a) : "l"(p));
    re = (double)a;
}

template <int KQ, int DT>
__global__ void __launch_bounds__(kAddWarps * 32, 2) sho_add_kernel(const __grid_constant__ AddParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    using S = AddSmem<KQ, DT>;
    constexpr bool CPLX = E::cplx;
    constexpr int P = S::P;
    using PV = PartVec<P>;
    constexpr int NV = 4 * KQ;                 // sampled functions per point (numax + 1 rounded up to 4)
    constexpr int NT = (KQ + 1) / 2;           // ny tiles of 8 in the x stage
    constexpr int NYT = kAddTY / 8;
    constexpr int FXYS = S::FXYS, FZS = S::FZS, CPT = S::CPT;
    constexpr int NTHR = kAddWarps * 32;
    static_assert(kAddTX == 8 && kAddTZ == 8 && kAddWarps == 8, "one 8x8 MMA block per x / z extent");

    extern __shared__ __align__(16) double smem[];
    const int nsho = p.g.nsho;
    const int NG = p.ng;
    const int npp = p.npp;
    const int CAS = S::cas(p.nblk), T2S = S::t2s(npp);    // doubles per pair
    double* FXY = smem;                                   // [3][NG][FXYS]  y blocks 0..7, x block 8
    double* FZ = FXY + (size_t)3 * NG * FXYS;             // [2][NG][FZS]
    double* CA = FZ + (size_t)2 * NG * FZS;               // [2][NG][nblk][32][P]   A fragments of the z stage
    double* T2 = CA + (size_t)2 * NG * CAS;               // [2][NG][8][npp][P]
    AddEntry* ENT = reinterpret_cast<AddEntry*>(T2 + (size_t)2 * NG * T2S);      // [2][NG]
    int32_t* META = reinterpret_cast<int32_t*>(ENT + 2 * NG);                    // [3][NG] zmask | ytlo << 8 | ythi << 16
    uint16_t* ZPOS = reinterpret_cast<uint16_t*>(META + 3 * NG);                 // [8 nmt] T2 column of z-stage row

    const int tid = threadIdx.x, lane = tid & 31, zl = tid >> 5;
    const int q = lane >> 2, t = lane & 3;

    const int b = blockIdx.x / p.n_tile_list;
    const int tile = p.tile_list[blockIdx.x - b * p.n_tile_list];
    const int tx = tile % p.ntile0, ty = (tile / p.ntile0) % p.ntile1, tz = tile / (p.ntile0 * p.ntile1);
    const int jx0 = tx * kAddTX, jy0 = ty * kAddTY, jz0 = tz * kAddTZ;
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int ebeg = p.tile_ptr[tile], eend = p.tile_ptr[tile + 1];
    const int npairs = eend - ebeg;
    const int nG = (npairs + NG - 1) / NG;

    // E: records of group g -> ENT[g & 1], six 16-byte pieces each
    auto fetch_entries = [&](int g) {
        if (tid < NG * 6) {
            const int i = tid / 6, piece = tid - 6 * i;
            const int e = g * NG + i;
            if (e < npairs)
                cp_async16(reinterpret_cast<char*>(ENT + (g & 1) * NG + i) + 16 * piece,
                           reinterpret_cast<const char*>(p.tile_ent + ebeg + e) + 16 * piece);
        }
    };
    fetch_entries(0);

    // zero CA and T2 once: the padding entries of the z-stage A fragments and the zero column of T2 stay zero
    for (int i = tid; i < 2 * NG * (CAS + T2S); i += NTHR) CA[i] = 0.0;
    for (int i = tid; i < 8 * p.nmt; i += NTHR) ZPOS[i] = p.t2pos[256 + i];

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
        for (int ks = 0; ks < KQ; ++ks) t2off[nt][ks] = p.t2pos[16 * (8 * nt + 4 * (q & 1) + (q >> 1)) + 4 * ks + t];

    // this thread's share of a group's coefficients: slot k = coefficient cn[k] of pair ci[k] -> CA element co[k]
    int ci[CPT], co[CPT];
    const real_t* cptr[CPT];
    const real_t* cbase = reinterpret_cast<const real_t*>(p.coeff) + (size_t)b * nsho * P;
#pragma unroll
    for (int k = 0; k < CPT; ++k) {
        const int idx = tid + k * NTHR;
        ci[k] = -1; co[k] = 0; cptr[k] = cbase;
        if (idx < NG * nsho) {
            ci[k] = idx / nsho;
            const int n = idx - ci[k] * nsho;
            cptr[k] = cbase + (size_t)n * P;
            co[k] = ci[k] * (CAS / P) + p.cainv[n];
        }
    }
    const size_t catom = (size_t)p.nbands * nsho * P;
    const bool cvec = p.vec_ok != 0;

    // this thread's table points: point r of pair ti (T stage runs on the last warps, the z stage mostly on the first)
    const int tpt = tid - p.t_first;

    cp_async_wait_all();
    __syncthreads();

    int r3 = 0;                                             // s mod 3
    for (int s = 0; s < nG + 2; ++s) {
        const int r2 = s & 1;
        const int r3m2 = (r3 == 0) ? 1 : (r3 == 1 ? 2 : 0);  // (s - 2) mod 3
        // ---------------- E(s+1) ----------------
        if (s + 1 < nG) fetch_entries(s + 1);
        // ---------------- C(s): issue the coefficient loads ----------------
        double creg[CPT][P];
        if (s < nG) {
#pragma unroll
            for (int k = 0; k < CPT; ++k) {
#pragma unroll
                for (int pp = 0; pp < P; ++pp) creg[k][pp] = 0.0;
                if (ci[k] >= 0 && s * NG + ci[k] < npairs) {
                    const real_t* c = cptr[k] + (size_t)ENT[r2 * NG + ci[k]].atom * catom;
                    if (CPLX) ldg_pinned(c, cvec, creg[k][0], creg[k][P - 1]);
                    else ldg_pinned(c, creg[k][0]);
                }
            }
        }
        // ---------------- XY(s-2): every warp on its own plane ----------------
        if (s >= 2) {
            const int32_t* meta_r = META + r3m2 * NG;
            const double* fxy = FXY + (size_t)r3m2 * NG * FXYS + lane;
            const PV* t2p = reinterpret_cast<const PV*>(T2 + (size_t)r2 * NG * T2S) + zl * npp;
            for (int i = 0; i < NG; ++i, fxy += FXYS, t2p += kAddTZ * npp) {
                const int meta = meta_r[i];
                if (!((meta >> zl) & 1)) continue;
                const int ytlo = (meta >> 8) & 0xff, ythi = (meta >> 16) & 0xff;

                double D1[NT][P][2];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                    for (int pp = 0; pp < P; ++pp) D1[nt][pp][0] = D1[nt][pp][1] = 0.0;
#pragma unroll
                for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                    for (int ks = 0; ks < KQ; ++ks)
                        if (8 * nt + 4 * ks <= 4 * KQ - 4) {               // the block holds some ny+nx <= numax (numax >= 4 KQ - 4)
                            const double a = fxy[(8 * KQ + ks) * 32];
                            const PV bv = t2p[t2off[nt][ks]];
                            dmma(D1[nt][0][0], D1[nt][0][1], a, bv.re());
                            if (CPLX) dmma(D1[nt][P - 1][0], D1[nt][P - 1][1], a, bv.im());
                        }
#pragma unroll
                for (int yt = 0; yt < NYT; ++yt)
                    if (yt >= ytlo && yt <= ythi) {
#pragma unroll
                        for (int kk = 0; kk < KQ; ++kk) {
                            const double a = fxy[(yt * KQ + kk) * 32];
#pragma unroll
                            for (int pp = 0; pp < P; ++pp) dmma(D[yt][pp][0], D[yt][pp][1], a, D1[kk >> 1][pp][kk & 1]);
                        }
                    }
            }
        }
        // ---------------- Z(s-1): T2[z][(ny,nx)] for the 8 planes of the tile ----------------
        if (s >= 1 && s - 1 < nG) {
            const int r2m1 = r2 ^ 1;
            const int cnt = min(NG, npairs - (s - 1) * NG);
            const double* fz_r = FZ + (size_t)r2m1 * NG * FZS + lane;
            const PV* ca_r = reinterpret_cast<const PV*>(CA + (size_t)r2m1 * NG * CAS) + lane;
            PV* t2_r = reinterpret_cast<PV*>(T2 + (size_t)r2m1 * NG * T2S) + 2 * t * npp;
            for (int k = 0; k < p.zt; ++k) {
                const AddZTask zd = p.ztask[zl][k];
                const int nks = zd.w & 0xff, mt = (zd.w >> 8) & 0xff;
                if (nks == 0 || (zd.w >> 16) >= cnt) continue;
                const double* fz = fz_r + zd.fz;
                const PV* ap = ca_r + zd.ca;
                double d[P][2];
#pragma unroll
                for (int pp = 0; pp < P; ++pp) d[pp][0] = d[pp][1] = 0.0;
#pragma unroll
                for (int ks = 0; ks < KQ; ++ks)
                    if (ks < nks) {
                        const double bfr = fz[ks * 32];                          // B[k = nz][col = plane]
                        const PV av = ap[ks * 32];
                        dmma(d[0][0], d[0][1], av.re(), bfr);
                        if (CPLX) dmma(d[P - 1][0], d[P - 1][1], av.im(), bfr);
                    }
                PV* o = t2_r + zd.t2 + ZPOS[8 * mt + q];
                PV o0, o1;
                o0.x = d[0][0]; o1.x = d[0][1];
                if constexpr (CPLX) { o0.y = d[1][0]; o1.y = d[1][1]; }
                o[0] = o0;
                o[npp] = o1;
            }
        }
        // ---------------- T(s): 1D functions (step a1) in fragment order; scatter of C(s) ----------------
        if (s < nG) {
            for (int it = tpt; it >= 0 && it < NG * kAddPoints; it += NTHR) {
                const int i = it / kAddPoints, r = it - i * kAddPoints;
                if (s * NG + i >= npairs) break;
                const AddEntry* en = ENT + r2 * NG + i;
                const int d = r < kAddTY ? 1 : (r < kAddTY + kAddTX ? 0 : 2);
                const int N = p.g.ng[d];
                const int j = (d == 1 ? jy0 + r : (d == 0 ? jx0 : jz0) + (r & 7));
                const int iu = j + (int)en->m[d] * N;
                const bool valid = j < N && iu >= en->lo[d] && iu <= en->hi[d];
                double v[NV];
                if (valid) {
                    hermite_gauss_s<NV>(displacement(iu, p.g.h, en->pos[d]), en->inv_sigma, en->pref, p.hz, v);
                } else {
#pragma unroll
                    for (int n = 0; n < NV; ++n) v[n] = 0.0;
                }
                // block r >> 3 (y: 0..7, x: 8, z: own ring), point r & 7: element [k = n & 3] of K step n >> 2
                double* dst = (d == 2) ? FZ + (size_t)(r2 * NG + i) * FZS + (r & 7) * 4
                                       : FXY + (size_t)(r3 * NG + i) * FXYS + ((r >> 3) * KQ) * 32 + (r & 7) * 4;
#pragma unroll
                for (int kk = 0; kk < KQ; ++kk) {
                    double2 a, c;
                    a.x = v[4 * kk]; a.y = v[4 * kk + 1]; c.x = v[4 * kk + 2]; c.y = v[4 * kk + 3];
                    *reinterpret_cast<double2*>(dst + kk * 32) = a;
                    *reinterpret_cast<double2*>(dst + kk * 32 + 2) = c;
                }
            }
            if (tid < NG) {
                const AddEntry* en = ENT + r2 * NG + tid;
                META[r3 * NG + tid] = (s * NG + tid < npairs)
                                          ? ((int)en->zmask | ((int)en->ytlo << 8) | ((int)en->ythi << 16)) : 0;
            }
            // coefficients of the group: conjugate image phase, scatter into the z-stage A fragments
            PV* ca = reinterpret_cast<PV*>(CA + (size_t)r2 * NG * CAS);
#pragma unroll
            for (int k = 0; k < CPT; ++k)
                if (ci[k] >= 0 && s * NG + ci[k] < npairs) {
                    PV o;
                    if constexpr (!CPLX) {
                        o.x = creg[k][0];
                    } else {
                        const AddEntry* en = ENT + r2 * NG + ci[k];
                        const double wr = en->wr, wi = en->wi;
                        const double re = creg[k][0], im = creg[k][P - 1];
                        o.x = re * wr - im * wi;
                        o.y = re * wi + im * wr;
                    }
                    ca[co[k]] = o;
                }
        }
        cp_async_wait_all();
        __syncthreads();
        r3 = (r3 == 2) ? 0 : r3 + 1;
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
    constexpr int P = S::P;
    AddParams p;
    std::memset(&p, 0, sizeof(p));
    p.g = pl->g;
    p.coeff = coeff; p.psi = psi;
    p.tile_ptr = pl->d_tile_ptr; p.tile_ent = pl->d_tile_ent; p.tile_list = pl->d_tile_list;
    p.cainv = pl->d_cainv; p.t2pos = pl->d_t2pos;
    p.n_tile_list = pl->n_tile_list;
    p.nbands = nbands;
    p.ntile0 = pl->ntile[0]; p.ntile1 = pl->ntile[1];
    p.band_stride = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    const size_t esz = elem_size(pl->dtype);
    const size_t valign = CPLX ? esz : 2 * esz;
    p.vec_ok = ((reinterpret_cast<uintptr_t>(psi) % valign) == 0) && (CPLX || (pl->g.ng[0] % 2 == 0));
    if (CPLX && (reinterpret_cast<uintptr_t>(coeff) % esz) != 0) p.vec_ok = 0;
    const AddZTiles& zt = pl->ztiles;
    p.nblk = zt.nblk; p.nmt = zt.nmt;
    p.npp = 8 * zt.nmt + 2;
    for (int n = 0; n <= SHO_NUMAX_MAX; ++n) p.hz[n] = (n <= pl->g.numax) ? pl->g.hnorm[n] : 0.0;
    // pairs per pipeline step: as many as fit two CTAs per SM and CPT coefficients per thread (at most 4)
    const size_t budget = 112 * 1024;
    int ng = 1;
    while (ng < 4 && S::bytes(ng + 1, zt.nblk, zt.nmt) <= budget &&
           (ng + 1) * pl->g.nsho <= S::CPT * kAddWarps * 32) ++ng;
    p.ng = ng;
    const size_t smem = S::bytes(ng, zt.nblk, zt.nmt);
    if (smem > 227 * 1024 || pl->g.nsho > S::CPT * kAddWarps * 32) {
        set_error("sho_add: numax = %d needs %zu bytes of shared memory (> 227 KB)", pl->g.numax, smem);
        return SHO_ERR_UNSUPPORTED;
    }
    // The T stage (ng * 80 table points, one per thread) runs on the last warps; the z-stage tasks (pair, row
    // tile) go to the least loaded warp, a table point batch counting as kTCost K steps of the z stage.
    {
        const int npts = ng * kAddPoints;
        const int nthr = kAddWarps * 32;
        p.t_first = std::max(0, nthr - ((npts + 31) / 32) * 32);
        if (npts > nthr) p.t_first = 0;
        const int kTCost = 10;
        int load[kAddWarps], cnt[kAddWarps];
        for (int w = 0; w < kAddWarps; ++w) {
            const int lo = std::max(w * 32, p.t_first), hi = std::min((w + 1) * 32, p.t_first + npts);
            load[w] = (hi > lo) ? kTCost * ((npts + nthr - 1) / nthr) : 0;
            cnt[w] = 0;
        }
        for (int i = 0; i < ng; ++i)
            for (int mt = 0; mt < zt.nmt; ++mt) {
                int best = -1;
                for (int w = 0; w < kAddWarps; ++w)
                    if (cnt[w] < kAddZTMax && (best < 0 || load[w] < load[best])) best = w;
                if (best < 0) { set_error("sho_add: z-stage task table overflow"); return SHO_ERR_UNSUPPORTED; }
                AddZTask& zk = p.ztask[best][cnt[best]++];
                zk.ca = i * (S::cas(zt.nblk) / P) + zt.blk0[mt] * 32;
                zk.fz = i * S::FZS;
                zk.t2 = i * (S::t2s(p.npp) / P);
                zk.w = zt.nks[mt] | (mt << 8) | (i << 16);
                load[best] += 1 + zt.nks[mt];
            }
        p.zt = 0;
        for (int w = 0; w < kAddWarps; ++w) p.zt = std::max(p.zt, cnt[w]);
    }
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
