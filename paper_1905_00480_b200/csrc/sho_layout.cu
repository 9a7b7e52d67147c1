// sho_layout.cu -- the band-fastest psi layout of the paper's own kernels ("This index is used for vectorization
// over warps of 32 GPU-threads"): psi_bf[Nz][Ny][Nx][nbands].  The kernels of this library want the
// x-fastest layout psi[nbands][Nz][Ny][Nx], so the *_bf entry points of the ABI convert a
// chunk of bands at a time into a caller-provided workspace with the two tiled transposes below (32 x 32 elements
// through shared memory, both sides coalesced):
//   to_x_fastest:    xf[b - b0][r] = bf[r][b]                 b0 <= b < b0 + nb
//   from_x_fastest:  bf[r][b]     += xf[b - b0][r]            (accumulating: the add-back of a chunk)
// Pure data movement, HBM-bound: 2 x sizeof(elem) bytes per value each way.
#include <algorithm>
#include <mutex>

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

// ---- sho_project_bf_static: the band-fastest projection for callers that have no device memory to lend -----------
// sho_project_bf converts psi chunk by chunk into a workspace the CALLER must bring.  A caller that lives inside
// somebody else's program often cannot: a plug-in of a DFT code that handed the whole HBM to its own arena at
// start-up (a later cudaMalloc fails there), or a routine called in the middle of that program's stream work (a
// cudaMalloc there synchronises the whole device and stalls every other stream).  Such a caller owns psi and coeff
// and nothing else.  For it the library keeps ONE fixed workspace of SHO_STATIC_WORK_BYTES in its own image: the
// file-scope device array below.  It exists on every GPU that loads libsho, from the moment the module is loaded
// until the process exits, and costs that GPU 32 MiB whether or not the entry point is ever called.
//
// g_static_work is a device symbol.  In host code its name is only a stand-in of the host compiler, not an address
// the GPU understands: handing `g_static_work` itself to a kernel would fault (or, where the GPU can reach host
// memory, quietly read and write the wrong bytes).  The host therefore asks the runtime for the real address with
// cudaGetSymbolAddress, once per device and with that device current, and passes that pointer to the transpose and
// projection kernels like any other workspace.
namespace sho {

static __device__ __align__(256) unsigned char g_static_work[SHO_STATIC_WORK_BYTES];

constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mutex;
static void* g_static_ptr[kStaticMaxDevices] = {};       // device address of g_static_work on device i, once known

// device must be the current device.  The first call per device may load the module (that is when the driver
// places the array); later calls only read the cached address.
static sho_status static_work_address(int device, void** ptr)
{
    if (device < 0 || device >= kStaticMaxDevices) {
        set_error("sho_project_bf_static: CUDA device %d is outside the %d devices this entry point keeps an address for",
                  device, kStaticMaxDevices);
        return SHO_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[device]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_static_work);
        if (e != cudaSuccess) return cuda_fail(e, "sho_project_bf_static: cudaGetSymbolAddress of the built-in workspace");
        if (!p) { set_error("sho_project_bf_static: the built-in workspace has no device address"); return SHO_ERR_CUDA; }
        g_static_ptr[device] = p;
    }
    *ptr = g_static_ptr[device];
    return SHO_OK;
}

}  // namespace sho

extern "C" sho_status sho_project_bf_static(const sho_plan* plan, const void* psi_bf, int32_t nbands, void* coeff,
                                            void* cuda_stream)
{
    using namespace sho;
    if (plan && plan->g.natoms == 0 && psi_bf && nbands > 0) return SHO_OK;      // coeff is empty (may be null)
    if (!plan || !psi_bf || !coeff) { set_error("sho_project_bf_static: null argument"); return SHO_ERR_INVALID_ARG; }
    if (nbands <= 0) { set_error("sho_project_bf_static: nbands must be > 0"); return SHO_ERR_INVALID_ARG; }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "sho_project_bf_static");
    if (dev != plan->device) {
        set_error("sho_project_bf_static: the plan belongs to CUDA device %d but device %d is current", plan->device, dev);
        return SHO_ERR_INVALID_ARG;
    }
    // the size limit: the workspace must hold at least one band of the plan's grid
    const size_t esz = elem_size(plan->dtype);
    const size_t band_bytes = (size_t)plan->g.ng[0] * plan->g.ng[1] * plan->g.ng[2] * esz;
    if (band_bytes > (size_t)SHO_STATIC_WORK_BYTES) {
        set_error("sho_project_bf_static: one band of this %d x %d x %d grid is %zu bytes, more than the built-in workspace of "
                  "%zu bytes (SHO_STATIC_WORK_BYTES); use sho_project_bf with a workspace of your own",
                  plan->g.ng[0], plan->g.ng[1], plan->g.ng[2], band_bytes, (size_t)SHO_STATIC_WORK_BYTES);
        return SHO_ERR_UNSUPPORTED;
    }
    void* work = nullptr;
    sho_status st = static_work_address(dev, &work);
    if (st != SHO_OK) return st;
    // bands per chunk: as many as fit, an even number when more than one does (the rule of sho_project_bf)
    size_t n = band_bytes ? (size_t)SHO_STATIC_WORK_BYTES / band_bytes : (size_t)nbands;
    if (n > 1) n -= n & 1;
    const int cb = (int)std::min<size_t>(n, (size_t)nbands);
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t row = (size_t)plan->g.nsho * esz;
    // Nothing in the workspace has to start at zero: the transpose writes every element of the chunk before the
    // projection reads it, and what an earlier call left behind past the chunk is never read.
    for (int b0 = 0; b0 < nbands; b0 += cb) {
        const int nb = std::min(cb, nbands - b0);
        if ((st = launch_to_x_fastest(plan, psi_bf, nbands, b0, nb, work, s)) != SHO_OK) return st;
        if ((st = launch_project(plan, work, nb, static_cast<char*>(coeff) + (size_t)b0 * row, s, nbands)) != SHO_OK) return st;
    }
    return SHO_OK;
}
