// sho_dmul.cu -- step (2) of the non-local action: "Multiplication: d^a_ik = sum_j D^a_ij c^a_jk" with the
// atomic matrix in the SHO representation, eq. (27)-(28) PAPER.md:252-262: "a real-valued matrix of dimension N_SHO".
//
//   d[a][b][i] = sum_j D[a][i][j] c[a][b][j]        D real fp64 [natoms][N_SHO][N_SHO], c and d in the plan's dtype
//
// A batched small GEMM on the FP64 tensor cores: per atom M = i (N_SHO rows of D), K = j, N = the real columns of
// c (bands x re/im).  One CTA owns one (atom, chunk of 32 real columns): it stages its columns of c in shared memory
// as B fragments (widened to fp64), then each warp streams row tiles of D (A fragments straight from global memory:
// lane (q,t) reads D[8 mt + q][4 ks + t], four lanes cover 32 contiguous bytes of a row) against them and writes
// its 8 x 32 block of d.  Because the CTA has read all of its columns before it writes any, d may alias c (in place).
// Cost: 2 N_SHO^2 flops per (atom, real column) -- 1.3e10 flop at cfg 5 against 6.7e11 of one projection -- and D is
// read once per column chunk (cfg 5: 396 MB x 4 chunks, from L2 after the first).
#include "sho_device.cuh"

namespace sho {

constexpr int kDmWarps = 8;
constexpr int kDmCols = 32;             // real columns per CTA (4 N tiles)

struct DmulParams {
    const double* dmat;
    const void* cin;
    void* cout;
    int32_t nsho, nbands, natoms, ncolchunks;
    long long dstride;         // doubles between the matrices of two atoms (0: one matrix for all atoms, sho_transform)
};

template <int DT>
__global__ void __launch_bounds__(kDmWarps * 32) sho_dmul_kernel(const DmulParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    constexpr int P = E::cplx ? 2 : 1;
    constexpr int NT = kDmCols / 8;
    extern __shared__ __align__(16) double bs[];          // [ks][nt][32] B fragments: lane (q,t) holds c[j = 4 ks + t][col 8 nt + q]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int q = lane >> 2, t = lane & 3;
    const int a = blockIdx.x / p.ncolchunks, cc = blockIdx.x - a * p.ncolchunks;
    const int n = p.nsho, KS = (n + 3) >> 2, MT = (n + 7) >> 3;
    const int ncols = p.nbands * P;                        // real columns of this atom
    const int col0 = cc * kDmCols;
    const real_t* cin = reinterpret_cast<const real_t*>(p.cin) + (size_t)a * p.nbands * n * P;
    real_t* cout = reinterpret_cast<real_t*>(p.cout) + (size_t)a * p.nbands * n * P;
    // column col = band * P + part: element (j, col) sits at cin[(band * n + j) * P + part]
    for (int e = tid; e < KS * 4 * kDmCols; e += blockDim.x) {
        const int j = e % (KS * 4), cl = e / (KS * 4);
        const int col = col0 + cl;
        double v = 0.0;
        if (j < n && col < ncols) v = (double)cin[((size_t)(col / P) * n + j) * P + (col % P)];
        bs[((j >> 2) * NT + (cl >> 3)) * 32 + (cl & 7) * 4 + (j & 3)] = v;
    }
    __syncthreads();
    const double* D = p.dmat + (size_t)a * p.dstride;
    for (int mt = warp; mt < MT; mt += kDmWarps) {
        const int i = 8 * mt + q;
        const double* drow = D + (size_t)min(i, n - 1) * n;
        double acc[NT][2];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) acc[nt][0] = acc[nt][1] = 0.0;
#pragma unroll 4
        for (int ks = 0; ks < KS; ++ks) {
            const int j = 4 * ks + t;
            const double av = (i < n && j < n) ? __ldg(drow + j) : 0.0;
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma(acc[nt][0], acc[nt][1], av, bs[(ks * NT + nt) * 32 + lane]);
        }
        if (i < n) {
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const int col = col0 + 8 * nt + 2 * t + s;
                    if (col < ncols) cout[((size_t)(col / P) * n + i) * P + (col % P)] = (real_t)acc[nt][s];
                }
        }
    }
}

template <int DT>
static sho_status launch_t(const sho_plan* pl, const double* dmat, const void* cin, int nbands, void* cout, cudaStream_t s, bool shared)
{
    constexpr int P = Elem<DT>::cplx ? 2 : 1;
    DmulParams p;
    p.dmat = dmat; p.cin = cin; p.cout = cout;
    p.nsho = pl->g.nsho; p.nbands = nbands; p.natoms = pl->g.natoms;
    p.ncolchunks = (nbands * P + kDmCols - 1) / kDmCols;
    p.dstride = shared ? 0 : (long long)pl->g.nsho * pl->g.nsho;
    const long long nblocks = (long long)pl->g.natoms * p.ncolchunks;
    if (nblocks > 0x7fffffffLL) { set_error("sho_dmul: natoms*nbands too large"); return SHO_ERR_UNSUPPORTED; }
    if (nblocks == 0) return SHO_OK;
    const size_t smem = (size_t)((pl->g.nsho + 3) / 4) * (kDmCols / 8) * 32 * sizeof(double);
    auto kern = sho_dmul_kernel<DT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(dmul)");
    kern<<<(unsigned)nblocks, kDmWarps * 32, smem, s>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launch sho_dmul_kernel");
    return SHO_OK;
}

sho_status launch_dmul(const sho_plan* pl, const double* dmat, const void* cin, int nbands, void* cout, cudaStream_t s, bool shared)
{
    switch (pl->dtype) {
        case SHO_R64:  return launch_t<SHO_R64>(pl, dmat, cin, nbands, cout, s, shared);
        case SHO_C128: return launch_t<SHO_C128>(pl, dmat, cin, nbands, cout, s, shared);
        case SHO_R32:  return launch_t<SHO_R32>(pl, dmat, cin, nbands, cout, s, shared);
        case SHO_C64:  return launch_t<SHO_C64>(pl, dmat, cin, nbands, cout, s, shared);
    }
    set_error("sho_dmul: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

}  // namespace sho
