// sho_stored.cu -- the stored-projector BASELINE (step a7 of DESIGN.md): the paper's "USU" scheme
// on B200.  The 3D projector values Phi_n(r - R_a) = phi_nz phi_ny phi_nx are
// sampled ONCE over every atom's box into device memory (sho_tables_build, set-up) and the projection
//     c[a][b][n] = h^3 sum_r T[a][n][r] w(r) psi_b(r)
// then streams those tables from HBM: a tall-skinny GEMM per atom, M = n (N_SHO), N = bands, K = box
// points, on the FP64 tensor cores.  This kernel exists to measure what the on-the-fly scheme saves:
// its HBM traffic is the table bytes (cfg 3: 53 GB), and it needs N_SHO / (numax+1) times the flops.
//
// Table layout (private to the library): per atom, per z plane of the box, per K step of 4 plane
// points (x fastest, padded to a multiple of 4 with zeros), per M tile of 8 coefficients, the 32
// values of one DMMA A fragment: lane 4q+t holds T[n = 8 mt + q][point 4k + t].  A warp's load of one
// fragment is one contiguous 256-byte (fp64) line, read exactly once per band group.
#include "sho_device.cuh"

namespace sho {

constexpr int kStoWarps = 8;
constexpr int kStoPlanes = 8;       // z planes of the box per CTA (K split; the partial sums are added in segment order)
constexpr int kStoCols = 32;        // real columns (bands x re/im) per CTA
constexpr int kStoKC = 32;          // K steps staged in shared memory at a time (128 points)
constexpr int kStoKStride = (kStoCols / 8) * 32 + 4;   // padded stride of one K step in shared memory

__host__ __device__ inline int sto_mtiles(int nsho) { return (nsho + 7) / 8; }

// ------------------------------------------------------------------------------------------------
// table builder: one CTA per (atom, box plane)
template <typename real_t>
__global__ void __launch_bounds__(256) sho_tables_kernel(GridDev g, const AtomDev* atoms, const int64_t* atom_off,
                                                        const int32_t* plane_atom, const int32_t* plane_qz,
                                                        const uint32_t* nxyz, real_t* data)
{
    extern __shared__ double sm[];                  // [nxl + nyl][M] 1D tables, then fz[M]
    const int a = plane_atom[blockIdx.x], qz = plane_qz[blockIdx.x];
    const AtomDev at = atoms[a];
    const int M = g.numax + 1;
    const int nxl = at.hi[0] - at.lo[0] + 1, nyl = at.hi[1] - at.lo[1] + 1;
    double* fx = sm; double* fy = fx + (size_t)nxl * M; double* fz = fy + (size_t)nyl * M;
    for (int it = threadIdx.x; it < nxl + nyl + 1; it += blockDim.x) {
        double v[SHO_NUMAX_MAX + 1];
        const int d = it < nxl ? 0 : it < nxl + nyl ? 1 : 2;
        const int i = d == 0 ? at.lo[0] + it : d == 1 ? at.lo[1] + it - nxl : at.lo[2] + qz;
        hermite_gauss<SHO_NUMAX_MAX + 1>(displacement(i, g.h, at.pos[d]), at, g.hnorm, g.numax, true, v);
        double* dst = d == 0 ? fx + (size_t)it * M : d == 1 ? fy + (size_t)(it - nxl) * M : fz;
        for (int n = 0; n < M; ++n) dst[n] = v[n];
    }
    __syncthreads();
    const int npl = nxl * nyl, KP = (npl + 3) >> 2, MTILES = sto_mtiles(g.nsho);
    real_t* out = data + atom_off[a] + (size_t)qz * KP * MTILES * 32;
    const size_t total = (size_t)KP * MTILES * 32;
    for (size_t e = threadIdx.x; e < total; e += blockDim.x) {
        const int ln = (int)(e & 31);
        const size_t km = e >> 5;
        const int mt = (int)(km % MTILES), k = (int)(km / MTILES);
        const int n = 8 * mt + (ln >> 2), r = 4 * k + (ln & 3);
        double val = 0.0;
        if (n < g.nsho && r < npl) {
            const uint32_t c = nxyz[n];
            const int qy = r / nxl, qx = r - qy * nxl;
            val = fz[(c >> 16) & 255] * fy[(size_t)qy * M + ((c >> 8) & 255)] * fx[(size_t)qx * M + (c & 255)];
        }
        out[e] = (real_t)val;
    }
}

// ------------------------------------------------------------------------------------------------
struct StoParams {
    GridDev g;
    const void* psi;
    void* coeff;
    const void* data;
    const AtomDev* atoms;
    const int64_t* atom_off;
    const int32_t* seg_atom;     // [nseg]
    const int32_t* seg_qz0;      // [nseg] first box plane of the segment
    int32_t nseg;
    int32_t nbands;
    long long band_stride;
    int* turn;                   // [natoms][ngroups] turnstile of the stored projection's K segments
    int32_t ngroups;
};

template <int MTW, int DT>
__global__ void __launch_bounds__(kStoWarps * 32, 2) sho_project_stored_kernel(const StoParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    constexpr bool CPLX = E::cplx;
    constexpr int P = CPLX ? 2 : 1;
    constexpr int NT = kStoCols / 8;
    __shared__ __align__(16) double bs[kStoKC * kStoKStride];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int q = lane >> 2, t = lane & 3;
    // Work item (K segment, column group) = block index.  The turnstile at the end of the kernel (segment k waits for
    // k - 1 of the same atom, i.e. for the block before this one) relies on blocks being dispatched in index order, which
    // holds on this hardware but is not a CUDA guarantee; the wait therefore carries the 30 s watchdog and traps rather
    // than hangs if that ever fails.  Handing out work by an atomicAdd ticket at CTA start makes the order hold by
    // construction and was measured: cfg 3 19.65 ms against 18.57 ms with the ticket on a cache line of its
    // own (the cause was not isolated; the placement of neighbouring segments on the SMs changes), so the block index stays.
    const int seg = blockIdx.x % p.nseg, bg = blockIdx.x / p.nseg;
    const int a = p.seg_atom[seg], qz0 = p.seg_qz0[seg];
    const AtomDev at = p.atoms[a];
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int nxl = at.hi[0] - at.lo[0] + 1, nyl = at.hi[1] - at.lo[1] + 1, nzl = at.hi[2] - at.lo[2] + 1;
    const int npl = nxl * nyl, KP = (npl + 3) >> 2, MTILES = sto_mtiles(p.g.nsho);
    const int band0 = bg * (kStoCols / P);
    const int nbl = min(kStoCols / P, p.nbands - band0);      // bands of this group
    const real_t* tab = reinterpret_cast<const real_t*>(p.data) + p.atom_off[a];
    const real_t* psi = reinterpret_cast<const real_t*>(p.psi);

    double D[MTW][NT][2];
#pragma unroll
    for (int i = 0; i < MTW; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) D[i][j][0] = D[i][j][1] = 0.0;

    const int qz1 = min(qz0 + kStoPlanes, nzl);
    for (int qz = qz0; qz < qz1; ++qz) {
        const int iz = at.lo[2] + qz;
        const int mz = p.g.periodic[2] ? floordiv(iz, Nz) : 0;
        const int jz = iz - mz * Nz;
        const real_t* tpl = tab + (size_t)qz * KP * MTILES * 32;
        for (int k0 = 0; k0 < KP; k0 += kStoKC) {
            const int kc = min(kStoKC, KP - k0);
            __syncthreads();
            // ---- stage psi (wrap, Bloch phase) as B fragments: B[k = point 4k+t][col = band (x re/im)].  A thread
            // keeps one point of the chunk (its grid offset and phase are computed once) and walks the bands ----
            for (int rr = tid; rr < kc * 4; rr += blockDim.x) {
                const int r = 4 * k0 + rr;
                const bool inside = r < npl;
                size_t j = 0;
                double cs = 1.0, sn = 0.0;
                if (inside) {
                    const int qy = r / nxl, qx = r - qy * nxl;
                    const int ix = at.lo[0] + qx, iy = at.lo[1] + qy;
                    const int mx = p.g.periodic[0] ? floordiv(ix, Nx) : 0, my = p.g.periodic[1] ? floordiv(iy, Ny) : 0;
                    j = ((size_t)jz * Ny + (iy - my * Ny)) * Nx + (ix - mx * Nx);
                    if (CPLX && p.g.has_phase && (mx | my | mz))
                        sincospi(2.0 * (p.g.kfrac[0] * mx + p.g.kfrac[1] * my + p.g.kfrac[2] * mz), &sn, &cs);
                }
                const int kk = rr >> 2, tt = rr & 3;
                double* dst = bs + kk * kStoKStride + tt;
                const real_t* src = psi + ((size_t)band0 * p.band_stride + j) * P;
                constexpr int NB = kStoCols / P;
                for (int bl0 = 0; bl0 < NB; bl0 += 8) {
                    double v0[8], v1[8];
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        v0[u] = v1[u] = 0.0;
                        if (inside && bl0 + u < nbl) {
                            const real_t* sp = src + (size_t)(bl0 + u) * p.band_stride * P;
                            v0[u] = (double)__ldg(sp);
                            if (CPLX) v1[u] = (double)__ldg(sp + 1);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        if (!CPLX) {
                            const int col = bl0 + u;
                            dst[(col >> 3) * 32 + (col & 7) * 4] = v0[u];
                        } else {
                            const int col = (bl0 + u) * 2;
                            dst[(col >> 3) * 32 + (col & 7) * 4] = v0[u] * cs - v1[u] * sn;
                            dst[((col + 1) >> 3) * 32 + ((col + 1) & 7) * 4] = v0[u] * sn + v1[u] * cs;
                        }
                    }
                }
            }
            __syncthreads();
            // ---- stream the table fragments, K = 4 points per step ----
#pragma unroll 8
            for (int kk = 0; kk < kc; ++kk) {
                double afr[MTW];
#pragma unroll
                for (int i = 0; i < MTW; ++i) {
                    const int mt = warp + i * kStoWarps;
                    afr[i] = (mt < MTILES) ? (double)__ldcs(tpl + ((size_t)(k0 + kk) * MTILES + mt) * 32 + lane) : 0.0;
                }
#pragma unroll
                for (int j = 0; j < NT; ++j) {
                    const double bfr = bs[kk * kStoKStride + j * 32 + lane];
#pragma unroll
                    for (int i = 0; i < MTW; ++i) dmma(D[i][j][0], D[i][j][1], afr[i], bfr);
                }
            }
        }
    }
    // ---- the partial sums of the K segments of one (atom, column group) are added to c in segment order: segment k
    // waits until k - 1 has published its sum (a turnstile counter per (atom, group), zeroed by the launcher; the CTA
    // of segment k - 1 has the block index before this one, so it is already running or done), then does a plain
    // read-modify-write.  The wait has the same 30 s watchdog as the mbarrier waits: a lost hand-over traps.  Fixed summation order, no atomics on the data: bit-reproducible.  (fp32 data: each
    // segment's sum is rounded to fp32 when it is added -- the one place where this baseline does not round once.)
    const double h3 = p.g.h * p.g.h * p.g.h;
    real_t* cout = reinterpret_cast<real_t*>(p.coeff);
    const int kseg = qz0 / kStoPlanes;
    int* turn = p.turn + (size_t)a * p.ngroups + bg;
    __syncthreads();
    if (kseg > 0) {
        if (tid == 0) {
            const unsigned long long t0 = global_timer_ns();
            unsigned spins = 0;
            while (atomicAdd(turn, 0) != kseg) {
                __nanosleep(64);
                if ((++spins & 4095u) == 0 && global_timer_ns() - t0 > kMbarTimeoutNs) __trap();
            }
            __threadfence();
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < MTW; ++i) {
        const int n = 8 * (warp + i * kStoWarps) + q;
        if (n < p.g.nsho) {
#pragma unroll
            for (int j = 0; j < NT; ++j)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const int col = 8 * j + 2 * t + s;
                    const int bl = col / P, pp = col - bl * P;
                    if (bl < nbl) {
                        real_t* o = cout + (((size_t)a * p.nbands + band0 + bl) * p.g.nsho + n) * P + pp;
                        const double prev = (kseg > 0) ? (double)__ldcg(o) : 0.0;
                        *o = (real_t)(prev + h3 * D[i][j][s]);
                    }
                }
        }
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) atomicExch(turn, kseg + 1);
}

// ------------------------------------------------------------------------------------------------
sho_status tables_build(const sho_plan* pl, sho_tables** out, size_t* bytes_needed, cudaStream_t s)
{
    const int MTILES = sto_mtiles(pl->g.nsho);
    const size_t rsz = (pl->dtype == SHO_R64 || pl->dtype == SHO_C128) ? 8 : 4;
    std::vector<int64_t> off(pl->atoms.size() + 1, 0);
    std::vector<int32_t> plane_atom, plane_qz, seg_atom, seg_qz0;
    size_t max_sm = 0;
    for (size_t a = 0; a < pl->atoms.size(); ++a) {
        const AtomDev& at = pl->atoms[a];
        const int nxl = at.hi[0] - at.lo[0] + 1, nyl = at.hi[1] - at.lo[1] + 1, nzl = at.hi[2] - at.lo[2] + 1;
        int64_t n = 0;
        if (nxl > 0 && nyl > 0 && nzl > 0) {
            const int64_t KP = ((int64_t)nxl * nyl + 3) / 4;
            n = (int64_t)nzl * KP * MTILES * 32;
            max_sm = std::max(max_sm, (size_t)(nxl + nyl + 1) * (pl->g.numax + 1) * 8);
        }
        off[a + 1] = off[a] + n;
    }
    *bytes_needed = (size_t)off.back() * rsz;
    if (!out) return SHO_OK;
    *out = nullptr;
    if (pl->g.numax > 9) { set_error("sho_tables_build: the stored baseline covers numax <= 9"); return SHO_ERR_UNSUPPORTED; }
    if (max_sm > 200 * 1024) { set_error("sho_tables_build: box too large for the table builder"); return SHO_ERR_UNSUPPORTED; }
    size_t free_b = 0, total_b = 0;
    cudaError_t e = cudaMemGetInfo(&free_b, &total_b);
    if (e != cudaSuccess) return cuda_fail(e, "sho_tables_build: cudaMemGetInfo");
    if (*bytes_needed + (64u << 20) > free_b) {
        set_error("sho_tables_build: tables need %zu bytes, %zu bytes of device memory are free", *bytes_needed, free_b);
        return SHO_ERR_OOM;
    }
    // work lists in the plan's spatial atom order (neighbouring CTAs share psi in L2)
    for (int32_t oi = 0; oi < pl->n_nonempty; ++oi) {
        const int32_t a = pl->order[oi];
        const AtomDev& at = pl->atoms[a];
        const int nzl = at.hi[2] - at.lo[2] + 1;
        for (int qz = 0; qz < nzl; ++qz) { plane_atom.push_back(a); plane_qz.push_back(qz); }
        for (int qz = 0; qz < nzl; qz += kStoPlanes) { seg_atom.push_back(a); seg_qz0.push_back(qz); }
    }
    sho_tables* t = new (std::nothrow) sho_tables();
    if (!t) { set_error("sho_tables_build: host allocation failed"); return SHO_ERR_OOM; }
    t->plan = pl; t->plan_serial = pl->serial; t->d_turn = nullptr; t->last_launch = nullptr; t->turn_count = (size_t)std::max<size_t>(pl->atoms.size(), 1) * 256; t->d_data = nullptr; t->d_atom_off = nullptr; t->d_seg_atom = nullptr; t->d_seg_qz0 = nullptr;
    t->atom_off = off; t->bytes = *bytes_needed; t->nseg = (int32_t)seg_atom.size();
    int32_t *d_pa = nullptr, *d_pq = nullptr;
    auto fail = [&](sho_status st) { if (t->last_launch) cudaEventDestroy(t->last_launch);
                                     cudaFree(d_pa); cudaFree(d_pq); cudaFree(t->d_turn); cudaFree(t->d_seg_atom); cudaFree(t->d_seg_qz0);
                                     cudaFree(t->d_data); cudaFree(t->d_atom_off); delete t; return st; };
    auto up = [&](void** dst, const void* src, size_t bytes) -> cudaError_t {
        cudaError_t ee = cudaMalloc(dst, std::max<size_t>(bytes, 16));
        if (ee == cudaSuccess && bytes) ee = cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice);
        return ee;
    };
    if ((e = cudaMalloc(&t->d_data, std::max<size_t>(t->bytes, 16))) != cudaSuccess) {
        cudaGetLastError();
        set_error("sho_tables_build: cudaMalloc of %zu bytes failed", t->bytes);
        return fail(SHO_ERR_OOM);
    }
    if ((e = cudaMalloc(&t->d_turn, t->turn_count * sizeof(int))) != cudaSuccess) return fail(cuda_fail(e, "sho_tables_build: turnstile"));
    if ((e = cudaEventCreateWithFlags(&t->last_launch, cudaEventDisableTiming)) != cudaSuccess) return fail(cuda_fail(e, "sho_tables_build: event"));
    if ((e = up((void**)&t->d_atom_off, off.data(), off.size() * 8)) != cudaSuccess ||
        (e = up((void**)&t->d_seg_atom, seg_atom.data(), seg_atom.size() * 4)) != cudaSuccess ||
        (e = up((void**)&t->d_seg_qz0, seg_qz0.data(), seg_qz0.size() * 4)) != cudaSuccess ||
        (e = up((void**)&d_pa, plane_atom.data(), plane_atom.size() * 4)) != cudaSuccess ||
        (e = up((void**)&d_pq, plane_qz.data(), plane_qz.size() * 4)) != cudaSuccess)
        return fail(cuda_fail(e, "sho_tables_build: upload"));
    if (!plane_atom.empty()) {
        if (rsz == 8) {
            cudaFuncSetAttribute(sho_tables_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_sm);
            sho_tables_kernel<double><<<(unsigned)plane_atom.size(), 256, max_sm, s>>>(pl->g, pl->d_atoms, t->d_atom_off, d_pa, d_pq,
                                                                                      pl->d_nxyz, (double*)t->d_data);
        } else {
            cudaFuncSetAttribute(sho_tables_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)max_sm);
            sho_tables_kernel<float><<<(unsigned)plane_atom.size(), 256, max_sm, s>>>(pl->g, pl->d_atoms, t->d_atom_off, d_pa, d_pq,
                                                                                     pl->d_nxyz, (float*)t->d_data);
        }
        if ((e = cudaGetLastError()) != cudaSuccess) return fail(cuda_fail(e, "launch sho_tables_kernel"));
    }
    if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return fail(cuda_fail(e, "sho_tables_build: synchronize"));
    cudaFree(d_pa); cudaFree(d_pq);
    *out = t;
    return SHO_OK;
}

template <int MTW, int DT>
static sho_status launch_t(const sho_plan* pl, const sho_tables* tb, const void* psi, int nbands, void* coeff, cudaStream_t s)
{
    constexpr int P = Elem<DT>::cplx ? 2 : 1;
    StoParams p;
    p.g = pl->g; p.psi = psi; p.coeff = coeff; p.data = tb->d_data;
    p.atoms = pl->d_atoms; p.atom_off = tb->d_atom_off; p.seg_atom = tb->d_seg_atom; p.seg_qz0 = tb->d_seg_qz0;
    p.nseg = tb->nseg; p.nbands = nbands;
    p.band_stride = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    const int ngroups = (nbands * P + kStoCols - 1) / kStoCols;
    if ((size_t)pl->g.natoms * ngroups > tb->turn_count) {
        set_error("sho_project_stored: %d bands need more turnstile counters than the tables hold (at most %zu column groups per atom)",
                  nbands, pl->g.natoms ? tb->turn_count / (size_t)pl->g.natoms : (size_t)0);
        return SHO_ERR_UNSUPPORTED;
    }
    const long long nblocks = (long long)tb->nseg * ngroups;
    if (nblocks > 0x7fffffffLL) { set_error("sho_project_stored: grid too large"); return SHO_ERR_UNSUPPORTED; }
    // The turnstile counters are per-launch state that lives in the tables object.  Launches that share
    // one tables object -- from any stream, from any host thread -- are therefore chained on the device: each waits
    // for the event recorded behind the one before it (a no-op on the first launch and within one stream), and the
    // host side of the chain is held under the object's mutex.  Without this a second launch's memset could clear
    // the counters under a running kernel (wrong sums or an endless wait).
    std::lock_guard<std::mutex> chain(tb->launch_mutex);
    cudaError_t e = cudaStreamWaitEvent(s, tb->last_launch, 0);
    // atoms with an empty box have no segment: their coefficients are the zeros written here
    if (e == cudaSuccess) e = cudaMemsetAsync(coeff, 0, (size_t)pl->g.natoms * nbands * pl->g.nsho * elem_size(pl->dtype), s);
    if (e == cudaSuccess) e = cudaMemsetAsync(tb->d_turn, 0, (size_t)pl->g.natoms * ngroups * sizeof(int), s);
    if (e != cudaSuccess) return cuda_fail(e, "sho_project_stored: memset");
    p.turn = tb->d_turn; p.ngroups = ngroups;
    if (nblocks > 0) {
        sho_project_stored_kernel<MTW, DT><<<(unsigned)nblocks, kStoWarps * 32, 0, s>>>(p);
        if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, "launch sho_project_stored_kernel");
    }
    if ((e = cudaEventRecord(tb->last_launch, s)) != cudaSuccess) return cuda_fail(e, "sho_project_stored: event record");
    return SHO_OK;
}

template <int DT>
static sho_status launch_d(const sho_plan* pl, const sho_tables* tb, const void* psi, int nbands, void* coeff, cudaStream_t s)
{
    const int mtw = (sto_mtiles(pl->g.nsho) + kStoWarps - 1) / kStoWarps;
    if (mtw <= 1) return launch_t<1, DT>(pl, tb, psi, nbands, coeff, s);
    if (mtw <= 2) return launch_t<2, DT>(pl, tb, psi, nbands, coeff, s);
    if (mtw <= 4) return launch_t<4, DT>(pl, tb, psi, nbands, coeff, s);
    set_error("sho_project_stored: numax too large for the stored baseline");
    return SHO_ERR_UNSUPPORTED;
}

sho_status launch_project_stored(const sho_plan* pl, const sho_tables* tb, const void* psi, int nbands, void* coeff,
                                 cudaStream_t s)
{
    switch (pl->dtype) {
        case SHO_R64:  return launch_d<SHO_R64>(pl, tb, psi, nbands, coeff, s);
        case SHO_C128: return launch_d<SHO_C128>(pl, tb, psi, nbands, coeff, s);
        case SHO_R32:  return launch_d<SHO_R32>(pl, tb, psi, nbands, coeff, s);
        case SHO_C64:  return launch_d<SHO_C64>(pl, tb, psi, nbands, coeff, s);
    }
    set_error("sho_project_stored: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

// ------------------------------------------------------------------------------------------------
// Stored add-back (the paper's "USUadd", tab. 1): the expansion of step (3), PAPER.md:190,
//     psi_b(r) += conj(w(r)) sum_n T[a][n][r] c[a][b][n]
// reading the same pre-sampled 3D tables.  Per (atom, 8 box planes, 32 real columns) a GEMM M = box points,
// K = n (N_SHO), N = columns on the FP64 tensor cores; the table fragments are read with the transposed lane
// mapping (lane (q,t) takes T[n = 4 ks + t][point 8 pt + q]: two runs of 128 contiguous bytes per warp).  The boxes
// of different atoms overlap and this baseline does what a stored-projector code does: it adds its results to psi
// with atomicAdd (so, unlike sho_add, it is not bit-reproducible).
template <int DT>
__global__ void __launch_bounds__(kStoWarps * 32, 2) sho_add_stored_kernel(const StoParams p)
{
    using E = Elem<DT>;
    using real_t = typename E::real_t;
    constexpr bool CPLX = E::cplx;
    constexpr int P = CPLX ? 2 : 1;
    constexpr int NT = kStoCols / 8;
    extern __shared__ __align__(16) double cs[];          // [ks][nt][32] B fragments: lane (q,t) holds c[n = 4 ks + t][col 8 nt + q]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int q = lane >> 2, t = lane & 3;
    const int seg = blockIdx.x % p.nseg, bg = blockIdx.x / p.nseg;
    const int a = p.seg_atom[seg], qz0 = p.seg_qz0[seg];
    const AtomDev at = p.atoms[a];
    const int Nx = p.g.ng[0], Ny = p.g.ng[1], Nz = p.g.ng[2];
    const int nxl = at.hi[0] - at.lo[0] + 1, nyl = at.hi[1] - at.lo[1] + 1, nzl = at.hi[2] - at.lo[2] + 1;
    const int npl = nxl * nyl, KP = (npl + 3) >> 2, MTILES = sto_mtiles(p.g.nsho);
    const int n = p.g.nsho, KS = (n + 3) >> 2;
    const int band0 = bg * (kStoCols / P);
    const int ncols = min(kStoCols, (p.nbands - band0) * P);
    const real_t* tab = reinterpret_cast<const real_t*>(p.data) + p.atom_off[a];
    const real_t* cin = reinterpret_cast<const real_t*>(p.coeff) + ((size_t)a * p.nbands + band0) * n * P;
    real_t* psi = reinterpret_cast<real_t*>(const_cast<void*>(p.psi));
    for (int e = tid; e < KS * 4 * kStoCols; e += blockDim.x) {
        const int j = e % (KS * 4), cl = e / (KS * 4);
        double v = 0.0;
        if (j < n && cl < ncols) v = (double)cin[((size_t)(cl / P) * n + j) * P + (cl % P)];
        cs[((j >> 2) * NT + (cl >> 3)) * 32 + (cl & 7) * 4 + (j & 3)] = v;
    }
    __syncthreads();
    const int qz1 = min(qz0 + kStoPlanes, nzl);
    const int NPT = (npl + 7) >> 3;                          // groups of 8 points per plane
    for (int work = warp; work < (qz1 - qz0) * NPT; work += kStoWarps) {
        const int qz = qz0 + work / NPT, pt = work % NPT;
        const real_t* tpl = tab + (size_t)qz * KP * MTILES * 32;
        double D[NT][2];
#pragma unroll
        for (int j = 0; j < NT; ++j) D[j][0] = D[j][1] = 0.0;
        // A[point 8 pt + q][n = 4 ks + t] = T[n][point]: element (n, r) of the plane sits at ((r >> 2) MTILES + (n >> 3)) 32 + (n & 7) 4 + (r & 3)
        const int r = 8 * pt + q;
        const size_t rbase = (size_t)(r >> 2) * MTILES * 32 + (r & 3);
        const bool rin = (r >> 2) < KP;
#pragma unroll 4
        for (int ks = 0; ks < KS; ++ks) {
            const int nn = 4 * ks + t;
            const double av = (rin && nn < 8 * MTILES) ? (double)__ldcs(tpl + rbase + (size_t)(nn >> 3) * 32 + (nn & 7) * 4) : 0.0;
#pragma unroll
            for (int j = 0; j < NT; ++j) dmma(D[j][0], D[j][1], av, cs[(ks * NT + j) * 32 + lane]);
        }
        // this lane holds point r (row q) x columns 8 j + 2 t, 2 t + 1
        if (r < npl) {
            const int iz = at.lo[2] + qz;
            const int mz = p.g.periodic[2] ? floordiv(iz, Nz) : 0;
            const int qy = r / nxl, qx = r - qy * nxl;
            const int ix = at.lo[0] + qx, iy = at.lo[1] + qy;
            const int mx = p.g.periodic[0] ? floordiv(ix, Nx) : 0, my = p.g.periodic[1] ? floordiv(iy, Ny) : 0;
            const size_t jpt = ((size_t)(iz - mz * Nz) * Ny + (iy - my * Ny)) * Nx + (ix - mx * Nx);
            double cw = 1.0, sw = 0.0;
            if (CPLX && p.g.has_phase && (mx | my | mz))
                sincospi(-2.0 * (p.g.kfrac[0] * mx + p.g.kfrac[1] * my + p.g.kfrac[2] * mz), &sw, &cw);      // conj(w)
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                const int col = 8 * j + 2 * t;
                if (col >= ncols) continue;
                if (CPLX) {      // columns (2t, 2t+1) = (re, im) of one band
                    real_t* o = psi + ((size_t)(band0 + col / 2) * p.band_stride + jpt) * 2;
                    atomicAdd(o, (real_t)(D[j][0] * cw - D[j][1] * sw));
                    atomicAdd(o + 1, (real_t)(D[j][0] * sw + D[j][1] * cw));
                } else {
                    atomicAdd(psi + (size_t)(band0 + col) * p.band_stride + jpt, (real_t)D[j][0]);
                    if (col + 1 < ncols) atomicAdd(psi + (size_t)(band0 + col + 1) * p.band_stride + jpt, (real_t)D[j][1]);
                }
            }
        }
    }
}

template <int DT>
static sho_status launch_add_t(const sho_plan* pl, const sho_tables* tb, const void* coeff, int nbands, void* psi, cudaStream_t s)
{
    constexpr int P = Elem<DT>::cplx ? 2 : 1;
    StoParams p;
    p.g = pl->g; p.psi = psi; p.coeff = const_cast<void*>(coeff); p.data = tb->d_data;
    p.atoms = pl->d_atoms; p.atom_off = tb->d_atom_off; p.seg_atom = tb->d_seg_atom; p.seg_qz0 = tb->d_seg_qz0;
    p.nseg = tb->nseg; p.nbands = nbands; p.turn = nullptr; p.ngroups = 0;
    p.band_stride = (long long)pl->g.ng[0] * pl->g.ng[1] * pl->g.ng[2];
    const int ngroups = (nbands * P + kStoCols - 1) / kStoCols;
    const long long nblocks = (long long)tb->nseg * ngroups;
    if (nblocks > 0x7fffffffLL) { set_error("sho_add_stored: grid too large"); return SHO_ERR_UNSUPPORTED; }
    if (nblocks == 0) return SHO_OK;
    const size_t smem = (size_t)((pl->g.nsho + 3) / 4) * (kStoCols / 8) * 32 * sizeof(double);
    auto kern = sho_add_stored_kernel<DT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(add_stored)");
    kern<<<(unsigned)nblocks, kStoWarps * 32, smem, s>>>(p);
    if ((e = cudaGetLastError()) != cudaSuccess) return cuda_fail(e, "launch sho_add_stored_kernel");
    return SHO_OK;
}

sho_status launch_add_stored(const sho_plan* pl, const sho_tables* tb, const void* coeff, int nbands, void* psi, cudaStream_t s)
{
    switch (pl->dtype) {
        case SHO_R64:  return launch_add_t<SHO_R64>(pl, tb, coeff, nbands, psi, s);
        case SHO_C128: return launch_add_t<SHO_C128>(pl, tb, coeff, nbands, psi, s);
        case SHO_R32:  return launch_add_t<SHO_R32>(pl, tb, coeff, nbands, psi, s);
        case SHO_C64:  return launch_add_t<SHO_C64>(pl, tb, coeff, nbands, psi, s);
    }
    set_error("sho_add_stored: bad dtype");
    return SHO_ERR_INVALID_ARG;
}

// ------------------------------------------------------------------------------------------------
// stored 1D tables (f3): the separable scheme with its factor matrices read from memory (sho_device.cuh::stored1d_lookup)
__global__ void sho_tables1d_kernel(GridDev g, const AtomDev* atoms, const long long* atom_off, int natoms, double* data)
{
    const int a = blockIdx.x;
    const AtomDev at = atoms[a];
    const int M = g.numax + 1;
    const int n0 = max(at.hi[0] - at.lo[0] + 1, 0), n1 = max(at.hi[1] - at.lo[1] + 1, 0), n2 = max(at.hi[2] - at.lo[2] + 1, 0);
    if (n0 == 0 || n1 == 0 || n2 == 0) return;
    for (int it = threadIdx.x; it < n0 + n1 + n2; it += blockDim.x) {
        const int d = it < n0 ? 0 : it < n0 + n1 ? 1 : 2;
        const int i = at.lo[d] + (d == 0 ? it : d == 1 ? it - n0 : it - n0 - n1);
        double v[SHO_NUMAX_MAX + 1];
        hermite_gauss<SHO_NUMAX_MAX + 1>(displacement(i, g.h, at.pos[d]), at, g.hnorm, g.numax, true, v);
        double* dst = data + atom_off[a] + (size_t)it * M;
        for (int n = 0; n < M; ++n) dst[n] = v[n];
    }
    (void)natoms;
}

sho_status tables1d_build(const sho_plan* pl, sho_tables1d** out, size_t* bytes_needed, cudaStream_t s)
{
    const int M = pl->g.numax + 1;
    std::vector<long long> off(pl->atoms.size() + 1, 0);
    for (size_t a = 0; a < pl->atoms.size(); ++a) {
        const AtomDev& at = pl->atoms[a];
        long long n = 0;
        if (at.hi[0] >= at.lo[0] && at.hi[1] >= at.lo[1] && at.hi[2] >= at.lo[2])
            n = (long long)((at.hi[0] - at.lo[0] + 1) + (at.hi[1] - at.lo[1] + 1) + (at.hi[2] - at.lo[2] + 1)) * M;
        off[a + 1] = off[a] + n;
    }
    *bytes_needed = (size_t)off.back() * sizeof(double);
    if (!out) return SHO_OK;
    *out = nullptr;
    sho_tables1d* t = new (std::nothrow) sho_tables1d();
    if (!t) { set_error("sho_tables1d_build: host allocation failed"); return SHO_ERR_OOM; }
    t->plan = pl; t->plan_serial = pl->serial; t->d_data = nullptr; t->d_atom_off = nullptr; t->bytes = *bytes_needed;
    cudaError_t e = cudaMalloc(&t->d_data, std::max<size_t>(t->bytes, 16));
    if (e == cudaSuccess) e = cudaMalloc(&t->d_atom_off, off.size() * sizeof(long long));
    if (e == cudaSuccess) e = cudaMemcpy(t->d_atom_off, off.data(), off.size() * sizeof(long long), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaGetLastError();
        cudaFree(t->d_data); cudaFree(t->d_atom_off); delete t;
        set_error("sho_tables1d_build: cannot allocate %zu bytes", *bytes_needed);
        return SHO_ERR_OOM;
    }
    if (!pl->atoms.empty()) {
        sho_tables1d_kernel<<<(unsigned)pl->atoms.size(), 128, 0, s>>>(pl->g, pl->d_atoms, t->d_atom_off, (int)pl->atoms.size(), t->d_data);
        if ((e = cudaGetLastError()) == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { cudaFree(t->d_data); cudaFree(t->d_atom_off); delete t; return cuda_fail(e, "sho_tables1d_build"); }
    }
    *out = t;
    return SHO_OK;
}

}  // namespace sho
