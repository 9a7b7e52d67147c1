// sho_add.cu -- on-the-fly SHO expansion / add-back (step a6 of DESIGN.md) by OWNERSHIP TILING.
//
//   psi_b(r) += sum_a sum_n c[a][b][n] phi_nx(x-X_a) phi_ny(y-Y_a) phi_nz(z-Z_a)        step (3)
//
// One CTA owns one psi tile of kAddTX x kAddTY x kAddTZ = 8 x 64 x 8 grid points of TWO real channels (the
// real and imaginary part of one complex band -- the projectors are real, so the two parts are independent
// real problems -- or two real bands) and keeps it in the accumulator registers of FP64 tensor-core MMAs
// for the whole kernel; it walks the plan's list of (atom, periodic image) pairs whose box touches the
// tile and finally does ONE read-modify-write of the tile.  No atomics, bit-reproducible, psi traffic =
// read + write of every touched tile exactly once.
//
// The CTA is persistent and warp-specialised; the two roles are coupled only by an mbarrier ring, never by a
// CTA barrier:
//   producer warps (8)  warp w builds pairs w, w + 8, ... entirely on its own: the pair's record and its
//                 coefficients c[a][b][:] (cp.async, each lane copying exactly the A-fragment elements it will
//                 feed to the z-stage MMAs), the three 1D Hermite-Gauss tables sampled on the fly (eq. (31),
//                 PAPER.md:283-286) into shared memory in MMA fragment order (shared by both channels), then the
//                 z stage   T2[z][(ny,nx)] = sum_nz c[n(nx,ny,nz)] phi_nz(z)    M = (ny,nx) pairs sorted by
//                 ny+nx (row tile mt needs only nz <= numax - s_min(mt)), K = nz, N = the 8 planes,
//                 with the conjugate Bloch phase of the image applied to the A elements
//   XY warps (8 complex / 16 real)  a warp owns 64 rows x 8 columns of one plane (both channels for complex
//                 data, one channel for real data):
//                 x stage   T1[x][ny]  = sum_nx phi_nx(x) T2[z][(ny,nx)]        M = x, K = nx, N = ny
//                 y stage   psi[y][x] += sum_ny phi_ny(y) T1[x][ny]             M = y, K = ny, N = x
//                 The accumulator fragment of the x stage is exactly the B fragment of the y stage when
//                 column 2t+s of the x stage's N tile is assigned ny = 8 nt + 4 s + t.
// All three expansion stages run on DMMA.8x8x4.  The producers run up to RD pairs ahead of the XY warps, so
// their latency-bound work (exp, recurrences, L2 round trips) hides behind the tensor-core work.
#include <algorithm>
#include <cstring>

#include "sho_device.cuh"

namespace sho {

constexpr int kAddPWarps = 8;               // producer warps, one pair each at a time
// XY warps: complex data 8 (one z plane, both channels each), real data 16 ((plane, channel))
__host__ __device__ constexpr int add_xy_warps(bool cplx) { return cplx ? kAddTZ : 2 * kAddTZ; }
__host__ __device__ constexpr int add_threads(bool cplx) { return (add_xy_warps(cplx) + kAddPWarps) * 32; }

struct AddParams {
    GridDev g;
    AddZTiles zt;
    const void* coeff;
    void* psi;
    const int4* tile_info;     // per listed tile: (tile, first entry, entries, 0)
    const AddEntry* tile_ent;
    const double* tab1d;       // stored 1D tables (sho_add_stored1d), or null: sample on the fly
    const long long* tab1d_off;
    const uint16_t* cidx;      // [nblk][32] coefficient index held by lane 4 q + t of z-stage K block (0xffff: none)
    const uint16_t* t2pos;
    int32_t n_tile_list;
    int32_t nitems;            // work items = listed tiles x band chunks (one complex band or two real bands)
    int32_t nbands;
    int32_t cnb;               // bands per atom in the coefficient array (>= nbands: a chunk of a wider array)
    int32_t ntile0, ntile1;
    int32_t vec_ok;
    int32_t rd;                // ring depth (pairs in flight between producers and XY warps)
    int32_t npw;               // producer warps in use (<= kAddPWarps; each needs a ring slot, a staging buffer)
    int32_t nblk;              // K blocks of the z-stage A fragments
    int32_t npp;               // columns per plane of T2: 8 nmt + 2; column 8 nmt holds zeros
    long long band_stride;
    double hz[SHO_NUMAX_MAX + 1];                  // sqrt(2^n / n!) for n <= numax, 0 beyond (padding functions vanish)
};

// shared-memory carve-up (doubles): [FXY: RD x 9 KQ 32][T2: RD x 2 x 8 npp][FZ: npw x KQ 32][STG: npw x stg]
// [EXPT: 64][ENT: npw x 2 records] then [META: RD int32][ZPOS: 8 nmt uint16][CIDX: 32 nblk uint16][mbarriers: full RD, empty RD]
template <int KQ>
struct AddSmem {
    static constexpr int FXYS = 9 * KQ * 32;
    static constexpr int FZS = KQ * 32;
    static __host__ __device__ constexpr int t2s(int npp) { return 2 * kAddTZ * npp; }
    // z-stage A fragments of one pair in the element type of the data: [K block][lane][channel]
    static __host__ __device__ constexpr int stg(int nblk, int real_bytes) { return ((64 * nblk * real_bytes + 15) / 16) * 2; }
    static __host__ __device__ constexpr size_t bytes(int rd, int npw, int nmt, int nblk, int real_bytes, bool cplx)
    {
        const int npp = 8 * nmt + 2;
        size_t b = 8 * ((size_t)rd * (FXYS + t2s(npp)) + (size_t)npw * (FZS + stg(nblk, real_bytes)) + 64);
        b += (size_t)npw * 2 * sizeof(AddEntry);
        b += (size_t)rd * 4 + (size_t)8 * nmt * 2 + (size_t)32 * nblk * 2;
        b = (b + 7) & ~(size_t)7;
        return b + (size_t)2 * rd * 8 + 16;
    }
    // producer warps and ring depth: every producer warp fills a slot of its own while the XY warps drain others, so
    // rd > npw; as many of both as fit in the shared memory of one CTA per SM
    static constexpr size_t kBudget = 224 * 1024;
    static __host__ __device__ constexpr int pick_npw(int nmt, int nblk, int real_bytes, bool cplx)
    {
        int npw = kAddPWarps;
        while (npw > 1 && bytes(npw + 2, npw, nmt, nblk, real_bytes, cplx) > kBudget) --npw;
        return npw;
    }
    static __host__ __device__ constexpr int pick_rd(int npw, int nmt, int nblk, int real_bytes, bool cplx)
    {
        int rd = npw + 2;
        while (rd < 2 * npw + 2 && bytes(rd + 1, npw, nmt, nblk, real_bytes, cplx) <= kBudget) ++rd;
        return rd;
    }
};

// Row tiles and K blocks of the z stage for a given numax, as sho_plan_create lays them out (AddZTiles): known at compile
// time in the kernel variants that are instantiated for one numax (template parameter NX), where they turn ring depth,
// table strides and loop bounds into constants -- the XY warps otherwise re-load them from the parameter bank per pair
__host__ __device__ constexpr int add_nmt(int numax) { return ((numax + 1) * (numax + 2) / 2 + 7) / 8; }
__host__ __device__ constexpr int add_nks(int numax, int mt)       // K steps of row tile mt: nz <= numax - s_min(mt)
{
    int sm = 0;
    while ((sm + 1) * (sm + 2) / 2 <= 8 * mt) ++sm;
    return (numax - sm) / 4 + 1;
}
__host__ __device__ constexpr int add_nblk(int numax)
{
    int blk = 0;
    for (int mt = 0; mt < add_nmt(numax); ++mt) {
        int sm = 0;
        while ((sm + 1) * (sm + 2) / 2 <= 8 * mt) ++sm;
        blk += (numax - sm) / 4 + 1;
    }
    return blk;
}

// exp(x), x <= 0, in 11 FP64-pipe instructions (the library routine takes about 28; the producer warps share the
// FP64 pipe with the DMMAs of the XY warps, so every instruction there waits its turn):
//   x = (64 k + j) ln2/64 + r,  |r| <= ln2/128,   exp(x) = 2^k 2^(j/64) exp(r),
// 2^(j/64) from a 64-entry table in shared memory, exp(r) by its Taylor polynomial of degree 5 (remainder
// r^6/720 < 4e-17), 2^k by an integer add on the exponent field.  Relative error <= 4e-16 (checked against 60-digit
// arithmetic on 2e5 arguments in [-700, 0]).
__device__ __forceinline__ double exp_neg(double x, const double* __restrict__ tab)
{
    x = fmax(x, -700.0);
    const double magic = 6755399441055744.0;                                   // 1.5 * 2^52: rounds to an integer in the low word
    const double tn = fma(x, 92.33248261689366, magic);                    // 64 / ln2
    const int n = __double2loint(tn);
    const double fn = tn - magic;
    double r = fma(fn, -0.010830424695996044, x);                              // ln2/64, high 34 bits (0x1.62e42fef8p-7): exact product
    r = fma(fn, -2.5310172166650877e-13, r);                                   // ln2/64, the rest
    double q = fma(r, 8.3333333333333332e-3, 4.1666666666666664e-2);
    q = fma(q, r, 1.6666666666666666e-1);
    q = fma(q, r, 0.5);
    q = fma(q, r, 1.0);
    q = fma(q, r, 1.0);
    const double tj = tab[n & 63];
    const int hi = __double2hiint(tj) + ((n >> 6) << 20);
    return q * __hiloint2double(hi, __double2loint(tj));
}

// H_n(xi) exp(-xi^2/2) (sqrt(pi) sigma)^(-1/2) scale[n], n < NV, by the paper's monic recurrence (eq. (31),
// PAPER.md:283-284) carried on p_n = H_n g; scale[n] = sqrt(2^n/n!) makes the functions orthonormal (reading A1)
// NC <= NV functions are computed, the rest are zeros (NC = 10 when numax <= 9 is known at compile time)
template <int NV, int NC>
__device__ __forceinline__ void hermite_gauss_s(double u, double inv_sigma, double pref, const double* __restrict__ scale,
                                                const double* __restrict__ exptab, double (&out)[NV])
{
    const double xi = u * inv_sigma;
    double pm = 0.0, pc = exp_neg(-0.5 * xi * xi, exptab) * pref;
#pragma unroll
    for (int n = 0; n < NV; ++n) {
        if (n >= NC) { out[n] = 0.0; continue; }
        out[n] = pc * scale[n];
        if (n + 1 < NC) {
            const double pn = xi * pc - (0.5 * (double)n) * pm;
            pm = pc;
            pc = pn;
        }
    }
}

// asynchronous global -> shared copy of 4, 8 or 16 bytes (both addresses aligned to the size); with
// take == false nothing is read and the destination is filled with zeros
__device__ __forceinline__ void cp_async(void* smem_dst, const void* gmem_src, int bytes, bool take = true)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    const int n = take ? bytes : 0;
    if (bytes == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gmem_src), "r"(n) : "memory");
    else if (bytes == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(gmem_src), "r"(n) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;\n" ::"r"(d), "l"(gmem_src), "r"(n) : "memory");
}

// z stage of two row tiles (N0 >= N1 K steps; N1 = 0: one tile) as straight-line code: every operand is
// loaded first, the MMAs of the two tiles and the two channels alternate (four accumulator chains)
template <int N0, int N1, bool CPLX, typename real_t>
__device__ __forceinline__ void add_zpair(const real_t* __restrict__ a0p, const real_t* __restrict__ a1p,
                                          const double* __restrict__ fz, bool phased, double wr, double wi,
                                          double (&d)[2][2][2])
{
    double bz[N0], a[2][N0][2];
#pragma unroll
    for (int ks = 0; ks < N0; ++ks) {
        bz[ks] = fz[ks * 32];                                                    // B[k = nz][col = plane]
        load2_rw(a0p + ks * 64, a[0][ks][0], a[0][ks][1]);
        if (ks < N1) load2_rw(a1p + ks * 64, a[1][ks][0], a[1][ks][1]);
    }
    if (CPLX && phased) {                                                        // conjugate Bloch phase of the image
#pragma unroll
        for (int ks = 0; ks < N0; ++ks)
#pragma unroll
            for (int u = 0; u < 2; ++u)
                if (u == 0 || ks < N1) {
                    const double re = a[u][ks][0], im = a[u][ks][1];
                    a[u][ks][0] = re * wr - im * wi;
                    a[u][ks][1] = re * wi + im * wr;
                }
    }
#pragma unroll
    for (int ks = 0; ks < N0; ++ks) {
        dmma(d[0][0][0], d[0][0][1], a[0][ks][0], bz[ks]);
        dmma(d[0][1][0], d[0][1][1], a[0][ks][1], bz[ks]);
        if (ks < N1) {
            dmma(d[1][0][0], d[1][0][1], a[1][ks][0], bz[ks]);
            dmma(d[1][1][0], d[1][1][1], a[1][ks][1], bz[ks]);
        }
    }
}

// The whole z stage of a pair for a numax known at compile time: row tiles MT0, MT0 + 1, ... two at a time, their K-step
// counts and K-block offsets constants, no jump table
template <int NX, int MT0, int BLK, bool CPLX, typename real_t>
__device__ __forceinline__ void add_ztiles(const real_t* __restrict__ stg_lane, const double* __restrict__ fzl, bool phased,
                                           double wr, double wi, double* __restrict__ t2, const uint16_t* __restrict__ zpos,
                                           int q, int npp)
{
    if constexpr (MT0 < add_nmt(NX)) {
        constexpr int N0 = add_nks(NX, MT0);
        constexpr int N1 = (MT0 + 1 < add_nmt(NX)) ? add_nks(NX, MT0 + 1 < add_nmt(NX) ? MT0 + 1 : MT0) : 0;
        double d[2][2][2];
#pragma unroll
        for (int u = 0; u < 2; ++u) d[u][0][0] = d[u][0][1] = d[u][1][0] = d[u][1][1] = 0.0;
        add_zpair<N0, N1, CPLX>(stg_lane + (size_t)BLK * 64, stg_lane + (size_t)(BLK + N0) * 64, fzl, phased, wr, wi, d);
#pragma unroll
        for (int u = 0; u < 2; ++u)
            if (u == 0 || N1 > 0) {
                double* o = t2 + zpos[8 * (MT0 + u) + q];
                o[0] = d[u][0][0]; o[npp] = d[u][0][1];
                o[(size_t)kAddTZ * npp] = d[u][1][0]; o[(size_t)kAddTZ * npp + npp] = d[u][1][1];
            }
        add_ztiles<NX, MT0 + 2, BLK + N0 + N1, CPLX>(stg_lane, fzl, phased, wr, wi, t2, zpos, q, npp);
    }
}

// MIX (numax = 8, 9 only): the third K step of the y stage holds just ny = 8, 9, and the x stage spends one MMA per
// channel on the three pairs (ny, nx) = (8,0), (8,1), (9,0) and another on (0,8), (0,9), (1,8).  With MIX the free
// half of that y K step carries ny = 0, 1 a second time -- A fragment (phi_8, phi_9, phi_0, phi_1)(y) -- against the
// partial x sums over nx = 8, 9 only, and ONE x-stage MMA with the A fragment (phi_0, phi_1, phi_8, phi_9)(x) yields
// its four B columns: T1[x][8], T1[x][9] (from nx = 0, 1) and the nx = 8, 9 parts of T1[x][0], T1[x][1].  Three
// x-stage MMAs per plane and channel instead of four, two shared-memory loads fewer; nothing else changes.
// NX: the numax this variant is compiled for (5, 7, 8, 9: the configs' and the paper's), or -1: any numax with this KQ,
// sizes at run time.  With NX the z stage is straight-line code (add_ztiles) instead of a loop over a jump table.
template <int KQ, int DT, int NX>
__global__ void __launch_bounds__(add_threads(Elem<DT>::cplx), 1) sho_add_kernel(const __grid_constant__ AddParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    using S = AddSmem<KQ>;
    constexpr bool CPLX = E::cplx;
    constexpr int P = CPLX ? 2 : 1;
    constexpr int NV = 4 * KQ;                 // sampled functions per point (numax + 1 rounded up to 4)
    constexpr int NT = (KQ + 1) / 2;           // ny tiles of 8 in the x stage
    constexpr int NYT = kAddTY / 8;
    constexpr int FXYS = S::FXYS, FZS = S::FZS;
    constexpr int MTC = (KQ <= 2) ? 4 : 3;     // z-stage row tiles whose coefficients a producer lane holds at once
    static_assert(kAddTX == 8 && kAddTZ == 8, "one 8x8 MMA block per x / z extent");
    constexpr bool MIX = (NX == 8 || NX == 9);
    constexpr bool EX = NX >= 0;
    static_assert(!EX || ((NX + 4) >> 2) == KQ, "NX and KQ disagree");
    constexpr int C_NMT = EX ? add_nmt(EX ? NX : 0) : 0, C_NBLK = EX ? add_nblk(EX ? NX : 0) : 0;
    constexpr int C_RB = (int)sizeof(real_t);
    constexpr int C_NPW = EX ? S::pick_npw(C_NMT, C_NBLK, C_RB, CPLX) : 0;
    constexpr int C_RD = EX ? S::pick_rd(EX ? C_NPW : 1, C_NMT, C_NBLK, C_RB, CPLX) : 0;
    constexpr int kAddXYWarps = add_xy_warps(CPLX), kAddThreads = add_threads(CPLX);

    extern __shared__ __align__(16) double smem[];
    const int nsho = p.g.nsho;
    const int RD = EX ? C_RD : p.rd;
    const int npp = EX ? 8 * C_NMT + 2 : p.npp;
    const int nmt = EX ? C_NMT : p.zt.nmt;
    const int nblk = EX ? C_NBLK : p.nblk;
    const int T2S = S::t2s(npp);
    double* FXY = smem;                                   // [RD][9 KQ][32]     y blocks 0..7, x block 8
    double* T2 = FXY + (size_t)RD * FXYS;                 // [RD][2][8][npp]
    const int NPW = EX ? C_NPW : p.npw;
    const int STGS = S::stg(nblk, (int)sizeof(real_t));
    double* FZ = T2 + (size_t)RD * T2S;                   // [npw][KQ][32]
    double* STG = FZ + (size_t)NPW * FZS;                 // [npw][STGS]   z-stage A fragments of the pair in production, element type of the data
    double* EXPT = STG + (size_t)NPW * STGS;              // [64]  2^(j/64), see exp_neg
    AddEntry* ENTW = reinterpret_cast<AddEntry*>(EXPT + 64);                     // [npw][2]  this and the next record
    int32_t* META = reinterpret_cast<int32_t*>(ENTW + 2 * NPW);                  // [RD] zmask | ytlo << 8 | ythi << 16
    uint16_t* ZPOS = reinterpret_cast<uint16_t*>(META + RD);                     // [8 nmt] T2 column of z-stage row
    uint16_t* CIDX = ZPOS + 8 * nmt;                                             // [nblk][32] coefficient of an A-fragment element
    uint64_t* full = reinterpret_cast<uint64_t*>((reinterpret_cast<uintptr_t>(CIDX + 32 * nblk) + 7) & ~(uintptr_t)7);   // [RD] 1 producer warp
    uint64_t* empty = full + RD;                                                 // [RD] 16 XY warps

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int q = lane >> 2, t = lane & 3;

    // The CTA is persistent: it takes work items blockIdx.x, blockIdx.x + gridDim.x, ... (item = band chunk x
    // listed tile, tile fastest; a chunk is one complex band or two real bands) and the ring runs on across
    // them, so the producers fill it for the next tile while the XY warps write the finished one back.
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    struct Item { int b0, jx0, jy0, jz0, ebeg, npairs; };
    auto item_info = [&](int item) -> int4 {          // (tile, first entry, entries, chunk)
        const int chunk = item / p.n_tile_list;
        int4 v = __ldg(p.tile_info + (item - chunk * p.n_tile_list));
        v.w = chunk;
        return v;
    };
    auto decode = [&](const int4& v) -> Item {
        Item it;
        it.b0 = CPLX ? v.w : 2 * v.w;
        const int tile = v.x;
        const int tx = tile % p.ntile0, ty = (tile / p.ntile0) % p.ntile1, tz = tile / (p.ntile0 * p.ntile1);
        it.jx0 = tx * kAddTX; it.jy0 = ty * kAddTY; it.jz0 = tz * kAddTZ;
        it.ebeg = v.y; it.npairs = v.z;
        return it;
    };

    // zero T2 once: its zero column stays zero (z-stage rows past the last pair write zeros there)
    for (int i = tid; i < RD * T2S; i += kAddThreads) T2[i] = 0.0;
    for (int i = tid; i < 8 * nmt; i += kAddThreads) ZPOS[i] = p.t2pos[256 + i];
    for (int i = tid; i < 32 * nblk; i += kAddThreads) CIDX[i] = p.cidx[i];
    if (tid < 64) EXPT[tid] = exp2((double)tid * (1.0 / 64.0));
    if (tid == 0) {
        for (int i = 0; i < RD; ++i) { mbar_init(full + i, 1); mbar_init(empty + i, kAddXYWarps); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    if (warp < kAddXYWarps) {
      // Two mappings of the XY warps (measured): complex data runs 8 warps, one z plane of both channels each (64
      // accumulator registers, 128 registers per thread); real data runs 16 warps, (plane, channel).
      if constexpr (CPLX) {
        // =============================== XY warps ===============================
        // warp = z plane: its 64 rows x 8 columns of BOTH channels (64 accumulator registers), so that one
        // A-fragment load feeds two MMAs, two accumulator chains alternate and the write-back needs no exchange
        const int plane = warp;
        // x stage, B fragment B[k = nx][col = ny]: this lane reads T2[(ny,nx)] with nx = 4 ks + t and
        // ny = 8 nt + 4 (q & 1) + (q >> 1); pairs outside the basis read the zero column
        int t2off[NT][KQ];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int ks = 0; ks < KQ; ++ks) t2off[nt][ks] = p.t2pos[16 * (8 * nt + 4 * (q & 1) + (q >> 1)) + 4 * ks + t];
        // MIX: B fragment of the one mixed x-stage MMA, B[k = t][column q]: columns 0, 2 <- (8, nx = t), (9, nx = t) for t < 2;
        // columns 4, 6 <- (0, nx = 6 + t), (1, nx = 6 + t) for t >= 2; everything else reads the zero column
        const int t2off_mix = !MIX ? 0 : (int)p.t2pos[(q == 0 && t < 2) ? 16 * 8 + t : (q == 2 && t < 2) ? 16 * 9 + t :
                                                       (q == 4 && t >= 2) ? 6 + t : (q == 6 && t >= 2) ? 16 + 6 + t : 255];

        int slot = 0, ph = 0;
        const double* fxy = FXY + lane;
        const double* t2p = T2 + (size_t)plane * npp;                       // channel 1: + kAddTZ * npp
        int4 info_next = item_info(blockIdx.x);
        for (int item = blockIdx.x; item < p.nitems; item += gridDim.x) {
            const Item it = decode(info_next);
            if (item + (int)gridDim.x < p.nitems) info_next = item_info(item + gridDim.x);   // arrives during this item
            const int npairs = it.npairs;
            const bool two = CPLX || (it.b0 + 1 < p.nbands);                // second channel exists
            const int jz = it.jz0 + plane;
            const int row0 = it.jy0;
            real_t* pb = reinterpret_cast<real_t*>(p.psi) + ((size_t)it.b0 * p.band_stride + (size_t)jz * Ny * Nx) * P;
            // the owned rows are read once, at the end of the item: ask L2 for their lines now
            if (jz < Nz) {
                constexpr int kLineElems = 128 / (int)(sizeof(real_t) * P);           // tile columns per 128-byte line
                for (int r = lane; r < kAddTY * ((kAddTX + kLineElems - 1) / kLineElems); r += 32) {
                    const int row = r % kAddTY, seg = r / kAddTY;
                    if (row0 + row < Ny && it.jx0 + seg * kLineElems < Nx) {
                        const real_t* a = pb + ((size_t)(row0 + row) * Nx + it.jx0 + seg * kLineElems) * P;
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
                        if (!CPLX && two) asm volatile("prefetch.global.L2 [%0];" ::"l"(a + p.band_stride));
                    }
                }
            }
            double D[NYT][2][2];                                            // [block][channel][column]
#pragma unroll
            for (int yt = 0; yt < NYT; ++yt) D[yt][0][0] = D[yt][0][1] = D[yt][1][0] = D[yt][1][1] = 0.0;

            for (int g = 0; g < npairs; ++g) {
                mbar_wait(full + slot, ph);
                const int meta = META[slot];
                const int ytlo = (meta >> 8) & 0xff, ythi = (meta >> 16) & 0xff;       // the touched 8-row blocks
                if ((meta >> plane) & 1) {
                    double D1[NT][2][2];
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) D1[nt][0][0] = D1[nt][0][1] = D1[nt][1][0] = D1[nt][1][1] = 0.0;
#pragma unroll
                    for (int ks = 0; ks < KQ; ++ks)
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt)
                            if (MIX ? (nt == 0 && ks < 2) || (nt == 1 && ks == 2) : 8 * nt + 4 * ks <= 4 * KQ - 4) {   // the block holds some ny+nx <= numax (numax >= 4 KQ - 4)
                                const double a = fxy[(8 * KQ + ks) * 32];
                                const int o = (MIX && nt == 1) ? t2off_mix : t2off[nt][ks];
                                dmma(D1[nt][0][0], D1[nt][0][1], a, t2p[o]);
                                dmma(D1[nt][1][0], D1[nt][1][1], a, t2p[(size_t)kAddTZ * npp + o]);
                            }
                    // A predicated-off DMMA still takes its 16 cycles of the pipe (measured), and the compiler
                    // predicates a short "if": enter the unrolled blocks by a jump and leave them by a branch instead.
                    // the A fragments of a block are loaded while the MMAs of the block before it issue (two register
                    // sets take turns; the last block's look-ahead load is harmless: block 8 of the slot is the x block)
#define SHO_ADD_YBLOCK(YT, CUR, NXT)                                                                    \
    {                                                                                                   \
        _Pragma("unroll") for (int kk = 0; kk < KQ; ++kk) NXT[kk] = fxy[((YT + 1) * KQ + kk) * 32];     \
        _Pragma("unroll") for (int kk = 0; kk < KQ; ++kk) {                                             \
            dmma(D[YT][0][0], D[YT][0][1], CUR[kk], D1[kk >> 1][0][kk & 1]);                            \
            dmma(D[YT][1][0], D[YT][1][1], CUR[kk], D1[kk >> 1][1][kk & 1]);                            \
        }                                                                                               \
    }
                    double aA[KQ], aB[KQ];
#pragma unroll
                    for (int kk = 0; kk < KQ; ++kk) aA[kk] = aB[kk] = fxy[(ytlo * KQ + kk) * 32];
                    switch (ytlo) {
                        case 0: SHO_ADD_YBLOCK(0, aA, aB) if (ythi == 0) break;
                        case 1: SHO_ADD_YBLOCK(1, aB, aA) if (ythi == 1) break;
                        case 2: SHO_ADD_YBLOCK(2, aA, aB) if (ythi == 2) break;
                        case 3: SHO_ADD_YBLOCK(3, aB, aA) if (ythi == 3) break;
                        case 4: SHO_ADD_YBLOCK(4, aA, aB) if (ythi == 4) break;
                        case 5: SHO_ADD_YBLOCK(5, aB, aA) if (ythi == 5) break;
                        case 6: SHO_ADD_YBLOCK(6, aA, aB) if (ythi == 6) break;
                        case 7: SHO_ADD_YBLOCK(7, aB, aA)
                        default: break;
                    }
#undef SHO_ADD_YBLOCK
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + slot);
                fxy += FXYS; t2p += T2S;
                if (++slot == RD) { slot = 0; ph ^= 1; fxy = FXY + lane; t2p = T2 + (size_t)plane * npp; }
            }

            // ---------------- one read-modify-write of the owned rows ----------------
            if (jz < Nz) {
                const int jx = it.jx0 + 2 * t;
#pragma unroll
                for (int yt = 0; yt < NYT; ++yt) {
                    const int jy = row0 + 8 * yt + q;
                    if (jy < Ny && jx < Nx) {
                        if (CPLX) {
                            real_t* pc = pb + ((size_t)jy * Nx + jx) * 2;
#pragma unroll
                            for (int sx = 0; sx < 2; ++sx)
                                if (jx + sx < Nx) {
                                    if (p.vec_ok) {
                                        double v0, v1;
                                        load2_rw(pc + 2 * sx, v0, v1);
                                        store2(pc + 2 * sx, v0 + D[yt][0][sx], v1 + D[yt][1][sx]);
                                    } else {
                                        pc[2 * sx] = (real_t)((double)pc[2 * sx] + D[yt][0][sx]);
                                        pc[2 * sx + 1] = (real_t)((double)pc[2 * sx + 1] + D[yt][1][sx]);
                                    }
                                }
                        } else {
#pragma unroll
                            for (int c = 0; c < 2; ++c)
                                if (c == 0 || two) {
                                    real_t* pp_ = pb + (size_t)c * p.band_stride + ((size_t)jy * Nx + jx);
                                    if (p.vec_ok && jx + 1 < Nx) {
                                        double v0, v1;
                                        load2_rw(pp_, v0, v1);
                                        store2(pp_, v0 + D[yt][c][0], v1 + D[yt][c][1]);
                                    } else {
                                        pp_[0] = (real_t)((double)pp_[0] + D[yt][c][0]);
                                        if (jx + 1 < Nx) pp_[1] = (real_t)((double)pp_[1] + D[yt][c][1]);
                                    }
                                }
                        }
                    }
                }
            }
        }
      } else {
        // =============================== XY warps ===============================
        const int plane = warp & 7, ch = warp >> 3;
        // x stage, B fragment B[k = nx][col = ny]: this lane reads T2[(ny,nx)] with nx = 4 ks + t and
        // ny = 8 nt + 4 (q & 1) + (q >> 1); pairs outside the basis read the zero column
        int t2off[NT][KQ];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int ks = 0; ks < KQ; ++ks) t2off[nt][ks] = p.t2pos[16 * (8 * nt + 4 * (q & 1) + (q >> 1)) + 4 * ks + t];
        // MIX: B fragment of the one mixed x-stage MMA, B[k = t][column q]: columns 0, 2 <- (8, nx = t), (9, nx = t) for t < 2;
        // columns 4, 6 <- (0, nx = 6 + t), (1, nx = 6 + t) for t >= 2; everything else reads the zero column
        const int t2off_mix = !MIX ? 0 : (int)p.t2pos[(q == 0 && t < 2) ? 16 * 8 + t : (q == 2 && t < 2) ? 16 * 9 + t :
                                                       (q == 4 && t >= 2) ? 6 + t : (q == 6 && t >= 2) ? 16 + 6 + t : 255];

        int slot = 0, ph = 0;
        const double* fxy = FXY + lane;
        const double* t2p = T2 + (size_t)(ch * kAddTZ + plane) * npp;
        int4 info_next = item_info(blockIdx.x);
        for (int item = blockIdx.x; item < p.nitems; item += gridDim.x) {
            const Item it = decode(info_next);
            if (item + (int)gridDim.x < p.nitems) info_next = item_info(item + gridDim.x);   // arrives during this item
            const int npairs = it.npairs;
            const bool active = CPLX || (it.b0 + ch < p.nbands);
            const int jz = it.jz0 + plane;
            real_t* pb = reinterpret_cast<real_t*>(p.psi) +
                         (CPLX ? ((size_t)it.b0 * p.band_stride + (size_t)jz * Ny * Nx) * 2
                               : ((size_t)(it.b0 + ch) * p.band_stride + (size_t)jz * Ny * Nx));
            // the owned rows are read once, at the end of the item: ask L2 for their lines now
            if (active && jz < Nz && (!CPLX || ch == 0)) {
                constexpr int kLineElems = 128 / (int)(sizeof(real_t) * P);           // tile columns per 128-byte line
                for (int r = lane; r < kAddTY * ((kAddTX + kLineElems - 1) / kLineElems); r += 32) {
                    const int row = r % kAddTY, seg = r / kAddTY;
                    if (it.jy0 + row < Ny && it.jx0 + seg * kLineElems < Nx)
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(pb + ((size_t)(it.jy0 + row) * Nx + it.jx0 + seg * kLineElems) * P));
                }
            }
            double D[NYT][2];
#pragma unroll
            for (int yt = 0; yt < NYT; ++yt) D[yt][0] = D[yt][1] = 0.0;

            for (int g = 0; g < npairs; ++g) {
                mbar_wait(full + slot, ph);
                const int meta = META[slot];
                if (active && ((meta >> plane) & 1)) {
                    const int ytlo = (meta >> 8) & 0xff, ythi = (meta >> 16) & 0xff;
                    double D1[NT][2];
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) D1[nt][0] = D1[nt][1] = 0.0;
                    // independent accumulators next to each other: a dependent DMMA issues 26 cycles after its source
#pragma unroll
                    for (int ks = 0; ks < KQ; ++ks)
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt)
                            if (MIX ? (nt == 0 && ks < 2) || (nt == 1 && ks == 2) : 8 * nt + 4 * ks <= 4 * KQ - 4)   // the block holds some ny+nx <= numax
                                dmma(D1[nt][0], D1[nt][1], fxy[(8 * KQ + ks) * 32], t2p[(MIX && nt == 1) ? t2off_mix : t2off[nt][ks]]);
                    // The touched 8-row blocks are ytlo..ythi.  A predicated-off DMMA still takes its 16 cycles of
                    // the pipe (measured), and the compiler predicates a short "if": enter the unrolled blocks by
                    // a jump and leave them by a branch instead.
#define SHO_ADD_YBLOCK(YT)                                                                              \
    {                                                                                                   \
        double a_[KQ];                                                                                  \
        _Pragma("unroll") for (int kk = 0; kk < KQ; ++kk) a_[kk] = fxy[((YT) * KQ + kk) * 32];          \
        _Pragma("unroll") for (int kk = 0; kk < KQ; ++kk) dmma(D[YT][0], D[YT][1], a_[kk], D1[kk >> 1][kk & 1]); \
    }
                    switch (ytlo) {
                        case 0: SHO_ADD_YBLOCK(0) if (ythi == 0) break;
                        case 1: SHO_ADD_YBLOCK(1) if (ythi == 1) break;
                        case 2: SHO_ADD_YBLOCK(2) if (ythi == 2) break;
                        case 3: SHO_ADD_YBLOCK(3) if (ythi == 3) break;
                        case 4: SHO_ADD_YBLOCK(4) if (ythi == 4) break;
                        case 5: SHO_ADD_YBLOCK(5) if (ythi == 5) break;
                        case 6: SHO_ADD_YBLOCK(6) if (ythi == 6) break;
                        case 7: SHO_ADD_YBLOCK(7)
                        default: break;
                    }
#undef SHO_ADD_YBLOCK
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty + slot);
                fxy += FXYS; t2p += T2S;
                if (++slot == RD) { slot = 0; ph ^= 1; fxy = FXY + lane; t2p = T2 + (size_t)(ch * kAddTZ + plane) * npp; }
            }

            // ---------------- one read-modify-write of the owned rows ----------------
            if (active && jz < Nz) {
                const int jx = it.jx0 + 2 * t;
#pragma unroll
                for (int yt = 0; yt < NYT; ++yt) {
                    const int jy = it.jy0 + 8 * yt + q;
                    if (jy < Ny && jx < Nx) {
                        real_t* pp_ = pb + ((size_t)jy * Nx + jx);
                        if (p.vec_ok && jx + 1 < Nx) {
                            double v0, v1;
                            load2_rw(pp_, v0, v1);
                            store2(pp_, v0 + D[yt][0], v1 + D[yt][1]);
                        } else {
                            pp_[0] = (real_t)((double)pp_[0] + D[yt][0]);
                            if (jx + 1 < Nx) pp_[1] = (real_t)((double)pp_[1] + D[yt][1]);
                        }
                    }
                }
            }
        }
      }
    } else {
        // =============================== producer warps ===============================
        // Warp pw produces pairs pw, pw + NPW, ... on its own: tables, coefficients, z stage.  Its latency per
        // pair may be NPW times the XY warps' time per pair before they starve.  Global latency never sits on
        // that path: the pair's raw coefficients are copied to shared memory by cp.async while the tables are
        // sampled, and the record of the warp's next pair while this one is produced.
        // The pairs of all of this CTA's work items form one stream; warp pw takes elements pw, pw + NPW, ...
        const int pw = warp - kAddXYWarps;
        if (pw < NPW) {
        double* fzw = FZ + (size_t)pw * FZS;
        real_t* stg = reinterpret_cast<real_t*>(STG + (size_t)pw * STGS);
        AddEntry* entw = ENTW + 2 * pw;
        const size_t catom = (size_t)p.cnb * nsho * P;
        // copy granule: one complex coefficient when its alignment is known, else one real number
        const int gran = (CPLX && p.vec_ok) ? 2 : 1;       // reals per cp.async
        // stream cursor: (citem, ci) is the work item that holds stream element cbase_s .. cbase_s + ci.z - 1;
        // the record of the item after it is already on its way (pf)
        const int grid = (int)gridDim.x;
        int citem = blockIdx.x, cbase_s = 0;
        int4 ci = item_info(citem);
        int4 pf = (citem + grid < p.nitems) ? item_info(citem + grid) : make_int4(0, 0, 0, 0);
        auto seek = [&](int gs) -> bool {
            while (citem < p.nitems && gs >= cbase_s + ci.z) {
                cbase_s += ci.z;
                citem += grid;
                ci = pf;
                if (citem + grid < p.nitems) pf = item_info(citem + grid);
            }
            return citem < p.nitems;
        };
        auto fetch_entry = [&](int gs, int buf) {        // the cursor stands on stream element gs
            if (lane < 6)
                cp_async(reinterpret_cast<char*>(entw + buf) + 16 * lane,
                         reinterpret_cast<const char*>(p.tile_ent + ci.y + (gs - cbase_s)) + 16 * lane, 16);
        };
        // K steps per row tile of the z stage, 2 bits each (nks - 1), kept in registers (<= 17 tiles)
        unsigned long long nks_packed = 0;
        for (int mt = 0; mt < nmt; ++mt) nks_packed |= (unsigned long long)(p.zt.nks[mt] - 1) << (2 * mt);
        // numax 8, 9: this lane's coefficient index per K block stays in registers (cfg 5: 47.83 -> 47.53 ms; no gain for numax 7)
        constexpr bool CREG = EX && KQ == 3;
        int cidx_r[CREG ? C_NBLK : 1];
#pragma unroll
        for (int blk = 0; blk < (CREG ? C_NBLK : 1); ++blk) cidx_r[blk] = CREG ? (int)CIDX[blk * 32 + lane] : 0;
        int G = pw;
        bool more = seek(G);
        if (more) fetch_entry(G, 0);
        int4 cur = ci;
        int slot = pw % RD, k = pw / RD, ebuf = 0;
        for (; more; G += NPW, ebuf ^= 1) {
            asm volatile("cp.async.wait_all;\n" ::: "memory");           // this pair's record (issued one iteration ago)
            __syncwarp();
            const AddEntry* en = entw + ebuf;
            const Item it = decode(cur);
            const int jx0 = it.jx0, jy0 = it.jy0, jz0 = it.jz0;
            const real_t* cbase = reinterpret_cast<const real_t*>(p.coeff) + (size_t)it.b0 * nsho * P;
            const bool two = CPLX || (it.b0 + 1 < p.nbands);      // second channel exists
            // ---- coefficients of the pair -> A fragments of the z stage.  Every coefficient sits in exactly one
            // fragment element: the lane copies its own (cp.async gather, zero fill for the padding elements) ----
            {
                const real_t* c = cbase + (size_t)en->atom * catom;
#pragma unroll
                for (int blk = 0; blk < (CREG ? C_NBLK : 1) * (CREG ? 1 : nblk); ++blk) {
                    const int n = CREG ? cidx_r[CREG ? blk : 0] : (int)CIDX[blk * 32 + lane];
                    const bool has = n != 0xffff;
                    const real_t* src = c + (has ? (size_t)n * P : 0);
                    real_t* dst = stg + (size_t)(blk * 32 + lane) * 2;
                    if (CPLX && gran == 2) cp_async(dst, src, 2 * (int)sizeof(real_t), has);
                    else {
                        cp_async(dst, src, (int)sizeof(real_t), has);
                        cp_async(dst + 1, src + (CPLX ? 1 : nsho), (int)sizeof(real_t), has && two);
                    }
                }
            }
            asm volatile("cp.async.commit_group;\n" ::: "memory");
            more = seek(G + NPW);                                    // the cursor moves on to this warp's next pair
            if (more) fetch_entry(G + NPW, ebuf ^ 1);                // not waited for before the next iteration
            asm volatile("cp.async.commit_group;\n" ::: "memory");
            cur = ci;
            const double inv_sigma = en->inv_sigma, pref = en->pref;
            const int ytlo = en->ytlo, ythi = en->ythi;
            if (k >= 1) mbar_wait(empty + slot, (k - 1) & 1);        // the slot's previous pair has been consumed
            double* fxy_s = FXY + (size_t)slot * FXYS;
            // ---- 1D functions (step a1) in fragment order: block (y: 0..7, x: 8; z: this warp's own buffer), point
            // r & 7 holds element [k = n & 3] of K step n >> 2.  Points of the pair: 8 z planes, 8 x columns, then
            // the rows of the 8-row blocks the box touches (the others are never read); 32 points per pass ----
            {
                const int npts = 16 + 8 * (ythi - ytlo + 1);
                for (int i = lane; i < npts; i += 32) {
                    const int d = i < 8 ? 2 : (i < 16 ? 0 : 1);
                    const int r = (d == 1) ? 8 * ytlo + i - 16 : (i & 7);            // row of the tile / point of the block
                    const int j = (d == 1 ? jy0 : (d == 2 ? jz0 : jx0)) + r;
                    const int N = p.g.ng[d];
                    const int iu = j + (int)en->m[d] * N;
                    const bool valid = j < N && iu >= en->lo[d] && iu <= en->hi[d];
                    double v[NV];
                    if (valid && p.tab1d) {
                        stored1d_lookup<NV>(p.tab1d, p.tab1d_off[en->atom], en->lo, en->hi, d, iu, p.g.numax, true, v);
                    } else if (valid) {
                        hermite_gauss_s<NV, (EX ? NX + 1 : NV)>(displacement(iu, p.g.h, en->pos[d]), inv_sigma, pref, p.hz, EXPT, v);
                    } else {
#pragma unroll
                        for (int n = 0; n < NV; ++n) v[n] = 0.0;
                    }
                    double* dst = (d == 2) ? fzw + r * 4
                                           : fxy_s + ((d == 0 ? 8 : (r >> 3)) * KQ) * 32 + (r & 7) * 4;
#pragma unroll
                    for (int kk = 0; kk < KQ; ++kk) {
                        double2 a, c;
                        a.x = v[4 * kk]; a.y = v[4 * kk + 1]; c.x = v[4 * kk + 2]; c.y = v[4 * kk + 3];
                        if (MIX && kk == 2 && d == 1) { c.x = v[0]; c.y = v[1]; }                     // y: (phi_8, phi_9, phi_0, phi_1)
                        if (MIX && kk == 2 && d == 0) { c = a; a.x = v[0]; a.y = v[1]; }              // x: (phi_0, phi_1, phi_8, phi_9)
                        *reinterpret_cast<double2*>(dst + kk * 32) = a;
                        *reinterpret_cast<double2*>(dst + kk * 32 + 2) = c;
                    }
                }
            }
            if (lane == 0) META[slot] = (int)en->zmask | (ytlo << 8) | (ythi << 16);
            asm volatile("cp.async.wait_group 1;\n" ::: "memory");     // the coefficients; the next record may still fly
            __syncwarp();
            // ---- z stage: T2[z][(ny,nx)] for the 8 planes; two row tiles in flight ----
            {
                const double wr = en->wr, wi = en->wi;
                const bool phased = !(wr == 1.0 && wi == 0.0);                  // warp-uniform; most images have none
                double* t2 = T2 + (size_t)slot * T2S + (size_t)(2 * t) * npp;
                if constexpr (EX) {
                    add_ztiles<(EX ? NX : 0), 0, 0, CPLX>(stg + (size_t)lane * 2, fzw + lane, phased, wr, wi, t2, ZPOS, q, npp);
                } else {
                int blk_run = 0;                     // first K block of row tile mt0 (the tiles' blocks are consecutive)
                for (int mt0 = 0; mt0 < nmt; mt0 += 2) {
                    double d[2][2][2];
                    int nks[2];
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        nks[u] = (mt0 + u < nmt) ? (int)((nks_packed >> (2 * (mt0 + u))) & 3) + 1 : 0;
                        d[u][0][0] = d[u][0][1] = d[u][1][0] = d[u][1][1] = 0.0;
                    }
                    const int blk_u[2] = { blk_run, blk_run + nks[0] };
                    blk_run += nks[0] + nks[1];
                    // one straight-line variant per (K steps of the first tile, of the second): entered by a jump,
                    // so no MMA is predicated (a predicated-off DMMA still costs its pipe time)
                    const real_t* a0p = stg + (size_t)(blk_u[0] * 32 + lane) * 2;
                    const real_t* a1p = stg + (size_t)(blk_u[1] * 32 + lane) * 2;
                    const double* fzl = fzw + lane;
#define SHO_ZCASE(N0, N1) case (N0) * 8 + (N1): if constexpr ((N0) <= KQ) add_zpair<N0, N1, CPLX>(a0p, a1p, fzl, phased, wr, wi, d); break;
                    switch (nks[0] * 8 + nks[1]) {
                        SHO_ZCASE(1, 0) SHO_ZCASE(1, 1)
                        SHO_ZCASE(2, 0) SHO_ZCASE(2, 1) SHO_ZCASE(2, 2)
                        SHO_ZCASE(3, 0) SHO_ZCASE(3, 1) SHO_ZCASE(3, 2) SHO_ZCASE(3, 3)
                        SHO_ZCASE(4, 0) SHO_ZCASE(4, 1) SHO_ZCASE(4, 2) SHO_ZCASE(4, 3) SHO_ZCASE(4, 4)
                        default: break;
                    }
#undef SHO_ZCASE
#pragma unroll
                    for (int u = 0; u < 2; ++u)
                        if (nks[u] > 0) {
                            double* o = t2 + ZPOS[8 * (mt0 + u) + q];
                            o[0] = d[u][0][0]; o[npp] = d[u][0][1];
                            o[(size_t)kAddTZ * npp] = d[u][1][0]; o[(size_t)kAddTZ * npp + npp] = d[u][1][1];
                        }
                }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(full + slot);
            slot += NPW;
            while (slot >= RD) { slot -= RD; ++k; }
        }
        }
    }
}

template <int KQ, int DT, int NX>
static sho_status launch_t(const sho_plan* pl, const void* coeff, int nbands, void* psi, cudaStream_t s, int cnb, const sho_tables1d* t1)
{
    using S = AddSmem<KQ>;
    constexpr bool CPLX = Elem<DT>::cplx;
    AddParams p;
    std::memset(&p, 0, sizeof(p));
    p.g = pl->g;
    p.zt = pl->ztiles;
    p.coeff = coeff; p.psi = psi;
    p.tile_info = pl->d_tile_info; p.tile_ent = pl->d_tile_ent;
    p.tab1d = t1 ? t1->d_data : nullptr; p.tab1d_off = t1 ? t1->d_atom_off : nullptr;
    p.cidx = pl->d_cidx; p.t2pos = pl->d_t2pos;
    p.n_tile_list = pl->n_tile_list;
    p.nbands = nbands;
    p.cnb = cnb;
    p.ntile0 = pl->ntile[0]; p.ntile1 = pl->ntile[1];
    p.band_stride = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    const size_t esz = elem_size(pl->dtype);
    const size_t valign = CPLX ? esz : 2 * esz;
    p.vec_ok = ((reinterpret_cast<uintptr_t>(psi) % valign) == 0) && (CPLX || (pl->g.ng[0] % 2 == 0));
    if (CPLX && (reinterpret_cast<uintptr_t>(coeff) % esz) != 0) p.vec_ok = 0;
    const AddZTiles& zt = pl->ztiles;
    p.npp = 8 * zt.nmt + 2;
    for (int n = 0; n <= SHO_NUMAX_MAX; ++n) p.hz[n] = (n <= pl->g.numax) ? pl->g.hnorm[n] : 0.0;
    // producer warps and ring depth: every producer warp fills a slot of its own while the XY warps drain
    // others, so rd > npw; as many of both as fit in the shared memory of one CTA per SM
    p.nblk = zt.nblk;
    const int rb = (int)(esz / (CPLX ? 2 : 1));
    const int npw = S::pick_npw(zt.nmt, zt.nblk, rb, CPLX);
    const int rd = S::pick_rd(npw, zt.nmt, zt.nblk, rb, CPLX);
    p.npw = npw; p.rd = rd;
    if (NX >= 0 && (zt.nmt != add_nmt(NX >= 0 ? NX : 0) || zt.nblk != add_nblk(NX >= 0 ? NX : 0) || pl->g.numax != NX)) {
        set_error("sho_add: internal: the plan's z-stage layout differs from the compiled one for numax = %d", NX);
        return SHO_ERR_UNSUPPORTED;
    }
    const size_t smem = S::bytes(rd, npw, zt.nmt, zt.nblk, rb, CPLX);
    if (smem > 227 * 1024) {
        set_error("sho_add: numax = %d needs %zu bytes of shared memory (> 227 KB)", pl->g.numax, smem);
        return SHO_ERR_UNSUPPORTED;
    }
    auto kern = sho_add_kernel<KQ, DT, NX>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(add)");
    const int nchunk = CPLX ? nbands : (nbands + 1) / 2;
    const long long nitems = (long long)pl->n_tile_list * nchunk;
    if (nitems > 0x7fffffffLL) { set_error("sho_add: tiles*nbands too large"); return SHO_ERR_UNSUPPORTED; }
    p.nitems = (int)nitems;
    int nsm = 0;
    e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, pl->device);
    if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute(add)");
    const unsigned grid = (unsigned)std::min<long long>(nitems, std::max(nsm, 1));     // persistent: one CTA per SM
    kern<<<grid, add_threads(CPLX), smem, s>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launch sho_add_kernel");
    return SHO_OK;
}

template <int DT>
static sho_status launch_kq(const sho_plan* pl, const void* coeff, int nbands, void* psi, cudaStream_t s, int cnb, const sho_tables1d* t1)
{
    switch ((pl->g.numax + 4) >> 2) {          // K steps of four n values that hold n <= numax
        case 1: return launch_t<1, DT, -1>(pl, coeff, nbands, psi, s, cnb, t1);
        case 2: return pl->g.numax == 7 ? launch_t<2, DT, 7>(pl, coeff, nbands, psi, s, cnb, t1)
                     : pl->g.numax == 5 ? launch_t<2, DT, 5>(pl, coeff, nbands, psi, s, cnb, t1)
                                        : launch_t<2, DT, -1>(pl, coeff, nbands, psi, s, cnb, t1);
        case 3: return pl->g.numax == 9 ? launch_t<3, DT, 9>(pl, coeff, nbands, psi, s, cnb, t1)
                     : pl->g.numax == 8 ? launch_t<3, DT, 8>(pl, coeff, nbands, psi, s, cnb, t1)
                                        : launch_t<3, DT, -1>(pl, coeff, nbands, psi, s, cnb, t1);
        default: return launch_t<4, DT, -1>(pl, coeff, nbands, psi, s, cnb, t1);
    }
}

sho_status launch_add(const sho_plan* pl, const void* coeff, int nbands, void* psi, cudaStream_t s, int cnb, const sho_tables1d* t1)
{
    if (cnb <= 0) cnb = nbands;
    switch (pl->dtype) {
        case SHO_R64:  return launch_kq<SHO_R64>(pl, coeff, nbands, psi, s, cnb, t1);
        case SHO_C128: return launch_kq<SHO_C128>(pl, coeff, nbands, psi, s, cnb, t1);
        case SHO_R32:  return launch_kq<SHO_R32>(pl, coeff, nbands, psi, s, cnb, t1);
        case SHO_C64:  return launch_kq<SHO_C64>(pl, coeff, nbands, psi, s, cnb, t1);
    }
    set_error("sho_add: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

}  // namespace sho
