// sho_layout.cu -- the band-fastest psi layout of the paper's own kernels ("This index is used for vectorization
// over warps of 32 GPU-threads"): psi_bf[Nz][Ny][Nx][nbands].  The kernels of this library want the
// x-fastest layout psi[nbands][Nz][Ny][Nx], so the *_bf entry points of the ABI convert a
// chunk of bands at a time into a caller-provided workspace with the two tiled transposes below (32 x 32 elements
// through shared memory, both sides coalesced):
//   to_x_fastest:    xf[b - b0][r] = bf[r][b]                 b0 <= b < b0 + nb
//   from_x_fastest:  bf[r][b]     += xf[b - b0][r]            (accumulating: the add-back of a chunk)
// Pure data movement, HBM-bound: 2 x sizeof(elem) bytes per value each way.
#include "sho_device.cuh"

namespace sho {

template <typename T> struct AddElem { static __device__ __forceinline__ T add(T a, T b) { return a + b; } };
template <> struct AddElem<double2> { static __device__ __forceinline__ double2 add(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); } };
template <> struct AddElem<float2> { static __device__ __forceinline__ float2 add(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); } };

template <typename T, bool TO_XF>
__global__ void __launch_bounds__(256) sho_transpose_kernel(const T* __restrict__ src, T* __restrict__ dst, long long npts, int nbands,
                                                            int b0, int nb)
{
    __shared__ T tile[32][33];
    const long long r0 = (long long)blockIdx.x * 32;
    const int c0 = blockIdx.y * 32;                      // band offset inside the chunk
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    if (TO_XF) {
        // read bf[r][b0 + c] (c fastest), write xf[c][r] (r fastest)
        for (int i = ty; i < 32; i += 8) {
            const long long r = r0 + i;
            const int c = c0 + tx;
            if (r < npts && c < nb) tile[i][tx] = src[r * nbands + b0 + c];
        }
        __syncthreads();
        for (int i = ty; i < 32; i += 8) {
            const int c = c0 + i;
            const long long r = r0 + tx;
            if (r < npts && c < nb) dst[(long long)c * npts + r] = tile[tx][i];
        }
    } else {
        // read xf[c][r] (r fastest), accumulate into bf[r][b0 + c] (c fastest)
        for (int i = ty; i < 32; i += 8) {
            const int c = c0 + i;
            const long long r = r0 + tx;
            if (r < npts && c < nb) tile[tx][i] = src[(long long)c * npts + r];
        }
        __syncthreads();
        for (int i = ty; i < 32; i += 8) {
            const long long r = r0 + i;
            const int c = c0 + tx;
            if (r < npts && c < nb) {
                T* d = dst + r * nbands + b0 + c;
                *d = AddElem<T>::add(*d, tile[i][tx]);
            }
        }
    }
}

template <typename T, bool TO_XF>
static sho_status launch_tr(const sho_plan* pl, const void* src, int nbands, int b0, int nb, void* dst, cudaStream_t s)
{
    const long long npts = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    if (npts == 0 || nb == 0) return SHO_OK;
    dim3 grid((unsigned)((npts + 31) / 32), (unsigned)((nb + 31) / 32));
    sho_transpose_kernel<T, TO_XF><<<grid, 256, 0, s>>>(static_cast<const T*>(src), static_cast<T*>(dst), npts, nbands, b0, nb);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launch sho_transpose_kernel");
    return SHO_OK;
}

template <bool TO_XF>
static sho_status launch_any(const sho_plan* pl, const void* src, int nbands, int b0, int nb, void* dst, cudaStream_t s)
{
    switch (pl->dtype) {
        case SHO_R64:  return launch_tr<double, TO_XF>(pl, src, nbands, b0, nb, dst, s);
        case SHO_C128: return launch_tr<double2, TO_XF>(pl, src, nbands, b0, nb, dst, s);
        case SHO_R32:  return launch_tr<float, TO_XF>(pl, src, nbands, b0, nb, dst, s);
        case SHO_C64:  return launch_tr<float2, TO_XF>(pl, src, nbands, b0, nb, dst, s);
    }
    set_error("sho layout: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

sho_status launch_to_x_fastest(const sho_plan* pl, const void* psi_bf, int nbands, int b0, int nb, void* psi_xf, cudaStream_t s)
{
    return launch_any<true>(pl, psi_bf, nbands, b0, nb, psi_xf, s);
}

sho_status launch_from_x_fastest(const sho_plan* pl, const void* psi_xf, int nbands, int b0, int nb, void* psi_bf, cudaStream_t s)
{
    return launch_any<false>(pl, psi_xf, nbands, b0, nb, psi_bf, s);
}

}  // namespace sho
