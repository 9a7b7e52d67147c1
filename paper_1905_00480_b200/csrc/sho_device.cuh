// sho_device.cuh -- device helpers: the on-the-fly 1D Hermite-Gauss sampler (eq. (31)),
// the FP64 tensor-core MMA wrapper, typed loads/stores.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sho_internal.h"

namespace sho {

// D(8x8) += A(8x4) * B(4x8), FP64 tensor core (SASS: DMMA.8x8x4).  Fragment layout, lane = 4*q + t:
//   a = A[row q][col t],  b = B[row t][col q],  d0,d1 = D[row q][col 2t, 2t+1]
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// ---- mbarrier (shared::cta) ----
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}
// Wait until the phase with this parity has completed.  try_wait suspends the thread for a hardware-chosen
// time slice, so the loop is not a hot spin.  A wait that lasts longer than kMbarTimeoutNs of wall time (a
// lost arrival: a bug, not a slow run -- compute-sanitizer or a debugger stretch a wait by far less) traps
// instead of hanging the GPU; the host then sees SHO_ERR_CUDA from the next runtime call on that context.
constexpr unsigned long long kMbarTimeoutNs = 30ull * 1000000000ull;
__device__ __forceinline__ unsigned long long global_timer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t a, int parity)
{
    uint32_t done;
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.b32 %0, 1, 0, p;\n}\n"
                 : "=r"(done) : "r"(a), "r"((uint32_t)parity) : "memory");
    return done != 0;
}
static __device__ __noinline__ void mbar_wait_slow(uint32_t a, int parity)
{
    const unsigned long long t0 = global_timer_ns();
    for (;;) {
#pragma unroll 1
        for (int spin = 0; spin < 4096; ++spin)          // a compact loop: unrolled, this cold path was 280 instructions
            if (mbar_try_wait(a, parity)) return;
        if (global_timer_ns() - t0 > kMbarTimeoutNs) __trap();
    }
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, int parity)
{
    const uint32_t a = (uint32_t)__cvta_generic_to_shared(bar);
    if (mbar_try_wait(a, parity)) return;
    if (mbar_try_wait(a, parity)) return;
    mbar_wait_slow(a, parity);
}

__device__ __forceinline__ int floordiv(int i, int n)
{
    int q = i / n;
    return (i % n < 0) ? q - 1 : q;
}

// Orthonormal Hermite-Gauss functions phi_0..phi_{NMAX-1} of width sigma at displacement u (step a1):
// the paper's monic three-term recurrence, eq. (31) PAPER.md:283-284,
//     H_0 = 1, H_1 = xi, H_{n+1} = xi H_n - (n/2) H_{n-1},
// times the Gaussian of eq. (3) PAPER.md:70 and the normalisation the paper leaves to the D matrices
// (PAPER.md:286): phi_n = sqrt(2^n/n!) (sqrt(pi) sigma)^(-1/2) H_n(xi) exp(-xi^2/2), xi = u/sigma.
// Entries with n > numax (or valid == false) are written as exact zeros.
template <int NMAX>
__device__ __forceinline__ void hermite_gauss(double u, const AtomDev& at, const double* __restrict__ hnorm, int numax,
                                              bool valid, double (&out)[NMAX])
{
    const double xi = u * at.inv_sigma;
    const double g = valid ? exp(-0.5 * xi * xi) * at.pref : 0.0;
    double hm = 0.0, hc = 1.0;
#pragma unroll
    for (int n = 0; n < NMAX; ++n) {
        out[n] = (n <= numax) ? hc * g * hnorm[n < SHO_NUMAX_MAX ? n : SHO_NUMAX_MAX] : 0.0;
        const double hn = xi * hc - (0.5 * (double)n) * hm;
        hm = hc;
        hc = hn;
    }
}

// The stored-1D-table variant (f3: the factor matrices v[x], v[y], v[z] of eq. (22)-(23) read from
// memory instead of being generated): per atom the rows phi_0..phi_numax of every box index of the x, then y, then z
// axis, M = numax + 1 doubles per index.  Returns the M values of axis d at unwrapped index i (zeros beyond numax or
// when !valid).
template <int NMAX>
__device__ __forceinline__ void stored1d_lookup(const double* __restrict__ tab, long long atom_off, const int32_t (&lo)[3],
                                                const int32_t (&hi)[3], int d, int i, int numax, bool valid, double (&out)[NMAX])
{
    const int M = numax + 1;
    long long base = atom_off;
    if (d >= 1) base += (long long)(hi[0] - lo[0] + 1) * M;
    if (d >= 2) base += (long long)(hi[1] - lo[1] + 1) * M;
    const double* row = tab + base + (long long)(i - lo[d]) * M;
#pragma unroll
    for (int n = 0; n < NMAX; ++n) out[n] = (valid && n <= numax) ? __ldg(row + n) : 0.0;
}

// unwrapped index -> displacement from the atom, written as the paper's grid convention x_i = i*h
// (no FMA contraction, so box-edge values match a plain evaluation)
__device__ __forceinline__ double displacement(int i, double h, double pos) { return __dsub_rn(__dmul_rn((double)i, h), pos); }

// ---- typed access: element type -> two fp64 lanes per 16/8-byte load -------------------------------
template <int DT> struct Elem;
template <> struct Elem<SHO_R64>  { using real_t = double; static constexpr bool cplx = false; static constexpr int cw = 16; };
template <> struct Elem<SHO_R32>  { using real_t = float;  static constexpr bool cplx = false; static constexpr int cw = 16; };
template <> struct Elem<SHO_C128> { using real_t = double; static constexpr bool cplx = true;  static constexpr int cw = 8; };
template <> struct Elem<SHO_C64>  { using real_t = float;  static constexpr bool cplx = true;  static constexpr int cw = 8; };

__device__ __forceinline__ void load2(const double* p, bool vec, double& v0, double& v1)
{
    if (vec) { const double2 v = __ldg(reinterpret_cast<const double2*>(p)); v0 = v.x; v1 = v.y; }
    else { v0 = __ldg(p); v1 = __ldg(p + 1); }
}
__device__ __forceinline__ void load2(const float* p, bool vec, double& v0, double& v1)
{
    if (vec) { const float2 v = __ldg(reinterpret_cast<const float2*>(p)); v0 = (double)v.x; v1 = (double)v.y; }
    else { v0 = (double)__ldg(p); v1 = (double)__ldg(p + 1); }
}

// plain (coherent) two-element load and store for the read-modify-write of sho_add; p is 2-element aligned
__device__ __forceinline__ void load2_rw(const double* p, double& v0, double& v1)
{
    const double2 v = *reinterpret_cast<const double2*>(p); v0 = v.x; v1 = v.y;
}
__device__ __forceinline__ void load2_rw(const float* p, double& v0, double& v1)
{
    const float2 v = *reinterpret_cast<const float2*>(p); v0 = (double)v.x; v1 = (double)v.y;
}
__device__ __forceinline__ void store2(double* p, double v0, double v1)
{
    double2 v; v.x = v0; v.y = v1; *reinterpret_cast<double2*>(p) = v;
}
__device__ __forceinline__ void store2(float* p, double v0, double v1)
{
    float2 v; v.x = (float)v0; v.y = (float)v1; *reinterpret_cast<float2*>(p) = v;
}

}  // namespace sho
