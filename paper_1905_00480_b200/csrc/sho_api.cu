// sho_api.cu -- the C ABI of libsho (include/sho.h): argument validation, the plan (step a0 of
// integer box ranges, spatial atom order, tile -> atom-image lists for the ownership-tiled
// add), the HOST-buffer end-to-end variants and the FP64 micro-benchmark.  All arithmetic of the hot
// path lives in the kernels (sho_project.cu, sho_add.cu, sho_stored.cu).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "sho_internal.h"

namespace sho {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

sho_status cuda_fail(cudaError_t e, const char* what)
{
    set_error("%s: %s", what, cudaGetErrorString(e));
    return (e == cudaErrorMemoryAllocation) ? SHO_ERR_OOM : SHO_ERR_CUDA;
}

static int floordiv_h(int i, int n)
{
    int q = i / n;
    return (i % n < 0) ? q - 1 : q;
}

template <typename T>
static sho_status upload(T** dst, const std::vector<T>& src, const char* what)
{
    *dst = nullptr;
    const size_t bytes = sizeof(T) * std::max<size_t>(src.size(), 1);
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(dst), bytes);
    if (e != cudaSuccess) return cuda_fail(e, what);
    if (!src.empty()) {
        e = cudaMemcpy(*dst, src.data(), sizeof(T) * src.size(), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return cuda_fail(e, what);
    }
    return SHO_OK;
}

static void plan_free_device(sho_plan* p)
{
    cudaFree(p->d_atoms); cudaFree(p->d_order); cudaFree(p->d_nxyz);
    cudaFree(p->d_tile_ptr); cudaFree(p->d_tile_ent); cudaFree(p->d_tile_list); cudaFree(p->d_tile_info); cudaFree(p->d_cainv); cudaFree(p->d_t2pos); cudaFree(p->d_cidx);
    cudaFree(p->ws_psi); cudaFree(p->ws_c); cudaFree(p->ws_d);
    if (p->s_in) cudaStreamDestroy(p->s_in);
    if (p->s_out) cudaStreamDestroy(p->s_out);
    p->s_in = nullptr; p->s_out = nullptr;
    p->d_atoms = nullptr; p->d_order = nullptr; p->d_nxyz = nullptr; p->d_cainv = nullptr; p->d_t2pos = nullptr; p->d_cidx = nullptr;
    p->d_tile_ptr = nullptr; p->d_tile_ent = nullptr; p->d_tile_list = nullptr; p->d_tile_info = nullptr;
    p->ws_psi = nullptr; p->ws_c = nullptr; p->ws_d = nullptr;
}

}  // namespace sho

using namespace sho;

extern "C" {

int sho_nsho(int numax)
{
    if (numax < 0 || numax > SHO_NUMAX_MAX) return -1;
    return (numax + 1) * (numax + 2) * (numax + 3) / 6;
}

// closed form of the enumeration "for nz: for ny: for nx" (reading A8): entries before plane nz, then
// before row ny inside that plane, then nx
int sho_index(int nx, int ny, int nz, int numax)
{
    if (numax < 0 || numax > SHO_NUMAX_MAX || nx < 0 || ny < 0 || nz < 0 || nx + ny + nz > numax) return -1;
    int n = 0;
    for (int kz = 0; kz < nz; ++kz) { const int m = numax - kz + 1; n += m * (m + 1) / 2; }
    for (int ky = 0; ky < ny; ++ky) n += numax - nz - ky + 1;
    return n + nx;
}

const char* sho_status_string(sho_status s)
{
    switch (s) {
        case SHO_OK: return "SHO_OK";
        case SHO_ERR_INVALID_ARG: return "SHO_ERR_INVALID_ARG";
        case SHO_ERR_UNSUPPORTED: return "SHO_ERR_UNSUPPORTED";
        case SHO_ERR_OOM: return "SHO_ERR_OOM";
        case SHO_ERR_CUDA: return "SHO_ERR_CUDA";
    }
    return "SHO_ERR_?";
}

const char* sho_last_error(void) { return g_err; }

sho_status sho_plan_create(sho_plan** out, const int32_t ng[3], double h, const int32_t periodic[3],
                           const double kfrac[3], int32_t natoms, const double* pos, const double* sigma,
                           int32_t numax, double rcut_sigma, sho_dtype dtype)
{
    if (out) *out = nullptr;
    if (!out || !ng || !periodic) { set_error("sho_plan_create: null argument"); return SHO_ERR_INVALID_ARG; }
    if (natoms < 0 || (natoms > 0 && (!pos || !sigma))) { set_error("sho_plan_create: bad natoms / null pos, sigma"); return SHO_ERR_INVALID_ARG; }
    if (!(h > 0.0) || !std::isfinite(h)) { set_error("sho_plan_create: h must be > 0"); return SHO_ERR_INVALID_ARG; }
    if (!(rcut_sigma > 0.0) || !std::isfinite(rcut_sigma)) { set_error("sho_plan_create: rcut_sigma must be > 0"); return SHO_ERR_INVALID_ARG; }
    if (numax < 0 || numax > SHO_NUMAX_MAX) { set_error("sho_plan_create: numax must be in [0, %d]", SHO_NUMAX_MAX); return SHO_ERR_INVALID_ARG; }
    if (dtype != SHO_R64 && dtype != SHO_C128 && dtype != SHO_R32 && dtype != SHO_C64) { set_error("sho_plan_create: bad dtype"); return SHO_ERR_INVALID_ARG; }
    for (int d = 0; d < 3; ++d) {
        if (ng[d] < 1) { set_error("sho_plan_create: grid dims must be >= 1"); return SHO_ERR_INVALID_ARG; }
        if (kfrac && kfrac[d] != 0.0 && !is_complex(dtype)) { set_error("sho_plan_create: kfrac != 0 needs a complex dtype"); return SHO_ERR_INVALID_ARG; }
        if (kfrac && !std::isfinite(kfrac[d])) { set_error("sho_plan_create: kfrac not finite"); return SHO_ERR_INVALID_ARG; }
    }
    if ((double)ng[0] * ng[1] * ng[2] > 2.0e9) { set_error("sho_plan_create: more than 2e9 grid points per band"); return SHO_ERR_UNSUPPORTED; }
    for (int a = 0; a < natoms; ++a) {
        if (!(sigma[a] > 0.0) || !std::isfinite(sigma[a])) { set_error("sho_plan_create: sigma[%d] must be > 0", a); return SHO_ERR_INVALID_ARG; }
        for (int d = 0; d < 3; ++d)
            if (!std::isfinite(pos[3 * a + d])) { set_error("sho_plan_create: pos[%d] not finite", a); return SHO_ERR_INVALID_ARG; }
    }

    sho_plan* p = new (std::nothrow) sho_plan();
    if (!p) { set_error("sho_plan_create: host allocation failed"); return SHO_ERR_OOM; }
    p->d_atoms = nullptr; p->d_order = nullptr; p->d_nxyz = nullptr;
    p->d_tile_ptr = nullptr; p->d_tile_ent = nullptr; p->d_tile_list = nullptr; p->d_tile_info = nullptr; p->d_cainv = nullptr; p->d_t2pos = nullptr; p->d_cidx = nullptr;
    p->ws_psi = nullptr; p->ws_c = nullptr; p->ws_d = nullptr; p->ws_psi_bytes = 0; p->ws_c_bytes = 0; p->ws_d_bytes = 0;
    p->s_in = nullptr; p->s_out = nullptr;
    p->opt_project_bands_per_cta = 0; p->opt_host_chunk_bands = 0;
    p->rcut_sigma = rcut_sigma;
    p->dtype = dtype;
    {
        static std::atomic<uint64_t> next_serial{1};
        p->serial = next_serial.fetch_add(1);
    }
    std::memset(&p->g, 0, sizeof(p->g));
    GridDev& g = p->g;
    for (int d = 0; d < 3; ++d) {
        g.ng[d] = ng[d];
        g.periodic[d] = periodic[d] ? 1 : 0;
        g.kfrac[d] = (kfrac && is_complex(dtype) && periodic[d]) ? kfrac[d] : 0.0;
    }
    g.h = h;
    g.numax = numax;
    g.nsho = sho_nsho(numax);
    g.natoms = natoms;
    g.has_phase = (g.kfrac[0] != 0.0 || g.kfrac[1] != 0.0 || g.kfrac[2] != 0.0) ? 1 : 0;
    {   // sqrt(2^n / n!): turns the monic recurrence of eq. (31) into the orthonormal functions (reading A1)
        double r = 1.0;
        for (int n = 0; n <= SHO_NUMAX_MAX; ++n) {
            if (n > 0) r *= 2.0 / (double)n;
            g.hnorm[n] = std::sqrt(r);
        }
    }

    for (int nz = 0, run = 0; nz <= SHO_NUMAX_MAX; ++nz) {
        g.zoff[nz] = run;
        const int m = numax - nz + 1;
        if (m > 0) run += m * (m + 1) / 2;
    }

    // ---- integer box ranges (reading A3/A5), evaluated in IEEE double exactly as written ----
    p->atoms.resize(natoms);
    p->max_n[0] = p->max_n[1] = p->max_n[2] = 0;
    p->sum_box = 0;
    std::vector<int32_t> nonempty, empty;
    for (int a = 0; a < natoms; ++a) {
        AtomDev& at = p->atoms[a];
        std::memset(&at, 0, sizeof(at));
        at.sigma = sigma[a];
        at.inv_sigma = 1.0 / sigma[a];
        at.pref = 1.0 / std::sqrt(1.7724538509055160273 * sigma[a]);     // (sqrt(pi) sigma)^(-1/2)
        bool is_empty = false;
        int64_t npts = 1;
        for (int d = 0; d < 3; ++d) {
            at.pos[d] = pos[3 * a + d];
            volatile double r = rcut_sigma * sigma[a];
            volatile double lo_x = pos[3 * a + d] - r;
            volatile double hi_x = pos[3 * a + d] + r;
            const double lo_f = std::ceil(lo_x / h), hi_f = std::floor(hi_x / h);
            if (std::fabs(lo_f) > 1.0e9 || std::fabs(hi_f) > 1.0e9) {
                set_error("sho_plan_create: atom %d box index out of the 32-bit range", a);
                delete p;
                return SHO_ERR_INVALID_ARG;
            }
            int lo = (int)lo_f, hi = (int)hi_f;
            if (!g.periodic[d]) { lo = std::max(lo, 0); hi = std::min(hi, ng[d] - 1); }
            else if (hi - lo + 1 > ng[d]) {
                set_error("sho_plan_create: atom %d: box of %d points is wider than the periodic cell (%d) on axis %d",
                          a, hi - lo + 1, ng[d], d);
                delete p;
                return SHO_ERR_UNSUPPORTED;
            }
            if (g.periodic[d] && (std::abs(floordiv_h(lo, ng[d])) > 32000 || std::abs(floordiv_h(hi, ng[d])) > 32000)) {
                set_error("sho_plan_create: atom %d is more than 32000 cells away from the home cell on axis %d", a, d);
                delete p;
                return SHO_ERR_UNSUPPORTED;
            }
            at.lo[d] = lo; at.hi[d] = hi;
            if (hi < lo) is_empty = true;
            npts *= std::max(hi - lo + 1, 0);
        }
        if (is_empty) { empty.push_back(a); continue; }
        nonempty.push_back(a);
        p->sum_box += npts;
        for (int d = 0; d < 3; ++d) p->max_n[d] = std::max(p->max_n[d], at.hi[d] - at.lo[d] + 1);
    }

    // ---- spatial order: z-slab major, so CTAs that run together read neighbouring psi from L2 ----
    {
        auto cell = [&](int a, int d) {
            const AtomDev& at = p->atoms[a];
            const int mid = (at.lo[d] + at.hi[d]) / 2;
            const int j = g.periodic[d] ? mid - floordiv_h(mid, g.ng[d]) * g.ng[d] : mid;
            return j / 16;
        };
        std::stable_sort(nonempty.begin(), nonempty.end(), [&](int a, int b) {
            const int za = cell(a, 2), zb = cell(b, 2);
            if (za != zb) return za < zb;
            const int ya = cell(a, 1), yb = cell(b, 1);
            if (ya != yb) return ya < yb;
            return cell(a, 0) < cell(b, 0);
        });
    }
    p->n_nonempty = (int32_t)nonempty.size();
    {   // x load steps of the project kernel per row block (one 128-byte line per row and step, real data)
        // steps of cwx columns (real data; complex data: half of that) from a 128-byte line or from a 32-byte lane span
        const int cwx = (dtype == SHO_R32) ? 32 : (is_complex(dtype) ? (dtype == SHO_C64 ? 16 : 8) : 16), epl = cwx / 4;
        int64_t steps[2] = { 0, 0 }, odd[2] = { 0, 0 };
        for (int a : nonempty) {
            const AtomDev& at = p->atoms[(size_t)a];
            for (int v = 0; v < 2; ++v) {
                const int al = v ? epl : cwx;
                const int xs0 = floordiv_h(at.lo[0], al) * al;
                const int ks = (at.hi[0] - xs0 + cwx) / cwx;
                steps[v] += ks; odd[v] += ks & 1;
            }
        }
        p->proj_xalign_span = (steps[1] * 10 < steps[0] * 9) ? 1 : 0;
        const int v = p->proj_xalign_span;
        p->proj_odd_steps = steps[v] ? (double)odd[v] / (double)steps[v] : 0.0;
    }
    p->order = nonempty;
    p->order.insert(p->order.end(), empty.begin(), empty.end());

    // ---- (nx,ny,nz) of every coefficient, packed (reading A8) ----
    std::vector<uint32_t> nxyz;
    for (int nz = 0; nz <= numax; ++nz)
        for (int ny = 0; ny <= numax - nz; ++ny)
            for (int nx = 0; nx <= numax - nz - ny; ++nx) nxyz.push_back((uint32_t)nx | ((uint32_t)ny << 8) | ((uint32_t)nz << 16));

    // ---- add tiling: for every psi tile the (atom, image) pairs whose box touches it, atoms ascending ----
    const int T[3] = { kAddTX, kAddTY, kAddTZ };
    for (int d = 0; d < 3; ++d) p->ntile[d] = (ng[d] + T[d] - 1) / T[d];
    p->ntiles = (int64_t)p->ntile[0] * p->ntile[1] * p->ntile[2];
    std::vector<int32_t> tile_ptr((size_t)p->ntiles + 1, 0);
    std::vector<AddEntry> tile_ent;
    {
        struct AxisHit { int32_t tile, m; };
        auto axis_hits = [&](const AtomDev& at, int d, std::vector<AxisHit>& hits) {
            hits.clear();
            const int N = g.ng[d];
            const int m0 = g.periodic[d] ? floordiv_h(at.lo[d], N) : 0;
            const int m1 = g.periodic[d] ? floordiv_h(at.hi[d], N) : 0;
            for (int m = m0; m <= m1; ++m)
                for (int t = 0; t < p->ntile[d]; ++t) {
                    const int a0 = t * T[d] + m * N, a1 = std::min((t + 1) * T[d], N) - 1 + m * N;
                    if (a1 >= at.lo[d] && a0 <= at.hi[d]) hits.push_back({ t, m });
                }
        };
        std::vector<AxisHit> hx, hy, hz;
        for (int pass = 0; pass < 2; ++pass) {
            std::vector<int32_t> fill;
            if (pass == 1) {
                int64_t run = 0;
                for (int64_t t = 0; t < p->ntiles; ++t) { const int32_t c = tile_ptr[t + 1]; tile_ptr[t] = (int32_t)run; run += c; }
                // tile_ptr[t] now = start of tile t; counts were stored at [t+1]
                if (run > 0x7fffffffLL) { set_error("sho_plan_create: too many (tile, atom) pairs"); delete p; return SHO_ERR_UNSUPPORTED; }
                tile_ptr[p->ntiles] = (int32_t)run;
                tile_ent.resize((size_t)run);
                fill.assign(tile_ptr.begin(), tile_ptr.end() - 1);
            }
            for (int a = 0; a < natoms; ++a) {
                const AtomDev& at = p->atoms[a];
                if (at.hi[0] < at.lo[0] || at.hi[1] < at.lo[1] || at.hi[2] < at.lo[2]) continue;
                axis_hits(at, 0, hx); axis_hits(at, 1, hy); axis_hits(at, 2, hz);
                for (const AxisHit& z : hz)
                    for (const AxisHit& y : hy)
                        for (const AxisHit& x : hx) {
                            const int64_t t = ((int64_t)z.tile * p->ntile[1] + y.tile) * p->ntile[0] + x.tile;
                            if (pass == 0) tile_ptr[t + 1] += 1;
                            else {
                                AddEntry e;
                                std::memset(&e, 0, sizeof(e));
                                e.atom = a; e.m[0] = (int16_t)x.m; e.m[1] = (int16_t)y.m; e.m[2] = (int16_t)z.m;
                                for (int d = 0; d < 3; ++d) { e.pos[d] = at.pos[d]; e.lo[d] = at.lo[d]; e.hi[d] = at.hi[d]; }
                                e.inv_sigma = at.inv_sigma; e.pref = at.pref;
                                // overlap of the box with the tile, in the units the warps can skip
                                const int oy = y.tile * kAddTY + y.m * g.ng[1], oz = z.tile * kAddTZ + z.m * g.ng[2];
                                const int ylast = std::min(kAddTY, g.ng[1] - y.tile * kAddTY) - 1;
                                const int ya = std::max(at.lo[1] - oy, 0), yb = std::min(at.hi[1] - oy, ylast);
                                e.ytlo = (int8_t)(ya >> 3); e.ythi = (int8_t)(yb >> 3);
                                unsigned zm = 0;
                                for (int k = 0; k < kAddTZ; ++k) {
                                    const int iz = oz + k;
                                    if (z.tile * kAddTZ + k < g.ng[2] && iz >= at.lo[2] && iz <= at.hi[2]) zm |= 1u << k;
                                }
                                e.zmask = (uint8_t)zm;
                                // conj(w), w = exp(2 pi i kfrac.m)  (reading A6)
                                const double ang = -2.0 * 3.14159265358979323846 *
                                                   (g.kfrac[0] * x.m + g.kfrac[1] * y.m + g.kfrac[2] * z.m);
                                e.wr = g.has_phase ? std::cos(ang) : 1.0;
                                e.wi = g.has_phase ? std::sin(ang) : 0.0;
                                tile_ent[(size_t)fill[t]++] = e;
                            }
                        }
            }
            if (pass == 0 && p->ntiles > 0) {
                // keep counts at [t+1]; the prefix sum happens at the start of pass 1
            }
        }
    }
    p->npairs = (int64_t)tile_ent.size();
    std::vector<int32_t> tile_list;
    for (int64_t t = 0; t < p->ntiles; ++t)
        if (tile_ptr[t + 1] > tile_ptr[t]) tile_list.push_back((int32_t)t);
    p->n_tile_list = (int32_t)tile_list.size();
    std::vector<int4> tile_info;
    for (int32_t t : tile_list) tile_info.push_back(make_int4(t, tile_ptr[(size_t)t], tile_ptr[(size_t)t + 1] - tile_ptr[(size_t)t], 0));

    // ---- z stage of the add as an MMA: (ny,nx) pairs sorted by s = ny+nx, row tiles of 8 ----
    std::vector<uint16_t> cainv((size_t)g.nsho, 0);
    {
        AddZTiles& zt = p->ztiles;
        std::memset(&zt, 0, sizeof(zt));
        const int npair = (numax + 1) * (numax + 2) / 2;
        zt.nmt = (npair + 7) / 8;
        int blk = 0;
        for (int mt = 0; mt < zt.nmt; ++mt) {
            int s = 0;                                         // s of the first pair of the tile = smallest s
            while ((s + 1) * (s + 2) / 2 <= 8 * mt) ++s;
            zt.blk0[mt] = (int8_t)blk;
            zt.nks[mt] = (int8_t)((numax - s) / 4 + 1);
            blk += zt.nks[mt];
        }
        zt.nblk = blk;
        for (int nz = 0, n = 0; nz <= numax; ++nz)
            for (int ny = 0; ny <= numax - nz; ++ny)
                for (int nx = 0; nx <= numax - nz - ny; ++nx, ++n) {
                    const int s = ny + nx, pi = s * (s + 1) / 2 + nx;
                    const int b = zt.blk0[pi >> 3] + (nz >> 2);
                    cainv[(size_t)n] = (uint16_t)(b * 32 + 4 * (pi & 7) + (nz & 3));
                }
    }

    // ---- columns of the add's T2[z][column]: the x stage reads pair (ny,nx) as the B fragment of block
    // (nt,ks) with ny = 8 nt + 4 (q & 1) + (q >> 1), nx = 4 ks + t on lane 4 q + t; the pairs of a block
    // get consecutive columns in lane order, so that a warp's read is one contiguous, conflict-free run
    std::vector<uint16_t> t2pos((size_t)256 + 8 * p->ztiles.nmt, 0);
    {
        const int zero_col = 8 * p->ztiles.nmt;
        for (auto& v : t2pos) v = (uint16_t)zero_col;
        const int KQ = (numax + 4) >> 2, NT = (KQ + 1) / 2;
        int col = 0;
        for (int nt = 0; nt < NT; ++nt)
            for (int ks = 0; ks < KQ; ++ks)
                for (int lane = 0; lane < 32; ++lane) {
                    const int q = lane >> 2, t = lane & 3;
                    const int ny = 8 * nt + 4 * (q & 1) + (q >> 1), nx = 4 * ks + t;
                    if (ny + nx <= numax) t2pos[(size_t)16 * ny + nx] = (uint16_t)col++;
                }
        // z-stage row 8 mt + q = pair index s (s + 1) / 2 + nx with s = ny + nx (rows past the last pair hold zeros)
        for (int s = 0; s <= numax; ++s)
            for (int nx = 0; nx <= s; ++nx) t2pos[(size_t)256 + s * (s + 1) / 2 + nx] = t2pos[(size_t)16 * (s - nx) + nx];
    }

    // ---- inverse of cainv: the coefficient that lane 4 q + t holds in K block blk of the z-stage A fragments ----
    std::vector<uint16_t> cidx((size_t)std::max(p->ztiles.nblk, 1) * 32, (uint16_t)0xffff);
    for (int n = 0; n < g.nsho; ++n) cidx[cainv[(size_t)n]] = (uint16_t)n;

    // ---- device mirrors ----
    cudaError_t e = cudaGetDevice(&p->device);
    if (e != cudaSuccess) { sho_status s = cuda_fail(e, "sho_plan_create: cudaGetDevice (no CUDA device?)"); delete p; return s; }
    sho_status st;
    if ((st = upload(&p->d_atoms, p->atoms, "sho_plan_create: atoms")) != SHO_OK ||
        (st = upload(&p->d_order, p->order, "sho_plan_create: order")) != SHO_OK ||
        (st = upload(&p->d_nxyz, nxyz, "sho_plan_create: nxyz")) != SHO_OK ||
        (st = upload(&p->d_tile_ptr, tile_ptr, "sho_plan_create: tile_ptr")) != SHO_OK ||
        (st = upload(&p->d_tile_ent, tile_ent, "sho_plan_create: tile_ent")) != SHO_OK ||
        (st = upload(&p->d_tile_list, tile_list, "sho_plan_create: tile_list")) != SHO_OK ||
        (st = upload(&p->d_tile_info, tile_info, "sho_plan_create: tile_info")) != SHO_OK ||
        (st = upload(&p->d_cainv, cainv, "sho_plan_create: cainv")) != SHO_OK ||
        (st = upload(&p->d_t2pos, t2pos, "sho_plan_create: t2pos")) != SHO_OK ||
        (st = upload(&p->d_cidx, cidx, "sho_plan_create: cidx")) != SHO_OK) {
        plan_free_device(p);
        delete p;
        return st;
    }
    *out = p;
    return SHO_OK;
}

sho_status sho_plan_destroy(sho_plan* plan)
{
    if (!plan) return SHO_OK;
    plan_free_device(plan);
    delete plan;
    return SHO_OK;
}

sho_status sho_plan_boxes(const sho_plan* plan, int32_t* lo_hi)
{
    if (!plan || !lo_hi) { set_error("sho_plan_boxes: null argument"); return SHO_ERR_INVALID_ARG; }
    for (size_t a = 0; a < plan->atoms.size(); ++a)
        for (int d = 0; d < 3; ++d) {
            lo_hi[(a * 3 + d) * 2 + 0] = plan->atoms[a].lo[d];
            lo_hi[(a * 3 + d) * 2 + 1] = plan->atoms[a].hi[d];
        }
    return SHO_OK;
}

sho_status sho_plan_info(const sho_plan* plan, int64_t info[8])
{
    if (!plan || !info) { set_error("sho_plan_info: null argument"); return SHO_ERR_INVALID_ARG; }
    info[0] = plan->g.natoms; info[1] = plan->g.nsho; info[2] = plan->g.numax; info[3] = (int64_t)plan->dtype;
    info[4] = plan->sum_box; info[5] = plan->n_tile_list; info[6] = plan->npairs; info[7] = plan->n_nonempty;
    return SHO_OK;
}

static sho_status check_hot(const char* fn, const sho_plan* plan, const void* a, const void* b, int32_t nbands)
{
    if (!plan || !a || !b) { set_error("%s: null argument", fn); return SHO_ERR_INVALID_ARG; }
    if (nbands <= 0) { set_error("%s: nbands must be > 0", fn); return SHO_ERR_INVALID_ARG; }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, fn);
    if (dev != plan->device) {
        set_error("%s: the plan belongs to CUDA device %d but device %d is current", fn, plan->device, dev);
        return SHO_ERR_INVALID_ARG;
    }
    return SHO_OK;
}

sho_status sho_plan_set_option(sho_plan* plan, const char* key, int64_t value)
{
    if (!plan || !key) { set_error("sho_plan_set_option: null argument"); return SHO_ERR_INVALID_ARG; }
    if (std::strcmp(key, "project_bands_per_cta") == 0) {
        if (value < 0 || value > 8) { set_error("sho_plan_set_option: project_bands_per_cta must be 0 (automatic) or 1..8"); return SHO_ERR_INVALID_ARG; }
        plan->opt_project_bands_per_cta = (int32_t)value;
        return SHO_OK;
    }
    if (std::strcmp(key, "host_chunk_bands") == 0) {
        if (value < 0 || value > 0x7fffffff) { set_error("sho_plan_set_option: host_chunk_bands must be 0 (automatic) or >= 1"); return SHO_ERR_INVALID_ARG; }
        plan->opt_host_chunk_bands = (int32_t)value;
        return SHO_OK;
    }
    set_error("sho_plan_set_option: unknown key '%s'", key);
    return SHO_ERR_INVALID_ARG;
}

sho_status sho_project(const sho_plan* plan, const void* psi, int32_t nbands, void* coeff, void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi && nbands > 0) return SHO_OK;   // coeff is empty (may be null)
    sho_status st = check_hot("sho_project", plan, psi, coeff, nbands);
    if (st != SHO_OK) return st;
    return launch_project(plan, psi, nbands, coeff, static_cast<cudaStream_t>(cuda_stream));
}

sho_status sho_add(const sho_plan* plan, const void* coeff, int32_t nbands, void* psi, void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi && nbands > 0) return SHO_OK;   // coeff is empty (may be null)
    sho_status st = check_hot("sho_add", plan, coeff, psi, nbands);
    if (st != SHO_OK) return st;
    if (plan->n_tile_list == 0) return SHO_OK;
    return launch_add(plan, coeff, nbands, psi, static_cast<cudaStream_t>(cuda_stream));
}

sho_status sho_tables_build(const sho_plan* plan, sho_tables** out, size_t* bytes_needed, void* cuda_stream)
{
    if (out) *out = nullptr;
    if (!plan || !bytes_needed) { set_error("sho_tables_build: null argument"); return SHO_ERR_INVALID_ARG; }
    return tables_build(plan, out, bytes_needed, static_cast<cudaStream_t>(cuda_stream));
}

sho_status sho_tables_destroy(sho_tables* t)
{
    if (!t) return SHO_OK;
    cudaFree(t->d_data);
    cudaFree(t->d_atom_off);
    cudaFree(t->d_seg_atom);
    cudaFree(t->d_seg_qz0);
    cudaFree(t->d_turn);
    if (t->last_launch) cudaEventDestroy(t->last_launch);
    delete t;
    return SHO_OK;
}

sho_status sho_project_stored(const sho_plan* plan, const sho_tables* tables, const void* psi, int32_t nbands,
                              void* coeff, void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi && nbands > 0 && tables && tables->plan == plan && tables->plan_serial == plan->serial) return SHO_OK;
    sho_status st = check_hot("sho_project_stored", plan, psi, coeff, nbands);
    if (st != SHO_OK) return st;
    if (!tables || tables->plan != plan || tables->plan_serial != plan->serial) { set_error("sho_project_stored: tables do not belong to this plan"); return SHO_ERR_INVALID_ARG; }
    return launch_project_stored(plan, tables, psi, nbands, coeff, static_cast<cudaStream_t>(cuda_stream));
}

// ---- step (2) and the three-step non-local action ------------------------------------------------
sho_status sho_dmul(const sho_plan* plan, const double* dmat, const void* coeff_in, int32_t nbands, void* coeff_out,
                    void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && nbands > 0) return SHO_OK;
    sho_status st = check_hot("sho_dmul", plan, coeff_in, coeff_out, nbands);
    if (st != SHO_OK) return st;
    if (!dmat) { set_error("sho_dmul: null argument"); return SHO_ERR_INVALID_ARG; }
    return launch_dmul(plan, dmat, coeff_in, nbands, coeff_out, static_cast<cudaStream_t>(cuda_stream));
}

sho_status sho_transform(const sho_plan* plan, const double* umat, const void* coeff_in, int32_t nbands, void* coeff_out,
                         void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && nbands > 0) return SHO_OK;
    sho_status st = check_hot("sho_transform", plan, coeff_in, coeff_out, nbands);
    if (st != SHO_OK) return st;
    if (!umat) { set_error("sho_transform: null argument"); return SHO_ERR_INVALID_ARG; }
    return launch_dmul(plan, umat, coeff_in, nbands, coeff_out, static_cast<cudaStream_t>(cuda_stream), true);
}

sho_status sho_apply(const sho_plan* plan, const double* dmat, void* psi, int32_t nbands, void* coeff_work, void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi && nbands > 0) return SHO_OK;
    sho_status st = check_hot("sho_apply", plan, psi, coeff_work, nbands);
    if (st != SHO_OK) return st;
    if (!dmat) { set_error("sho_apply: null argument"); return SHO_ERR_INVALID_ARG; }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    if ((st = launch_project(plan, psi, nbands, coeff_work, s)) != SHO_OK) return st;
    if ((st = launch_dmul(plan, dmat, coeff_work, nbands, coeff_work, s)) != SHO_OK) return st;
    if (plan->n_tile_list == 0) return SHO_OK;
    return launch_add(plan, coeff_work, nbands, psi, s);
}

// ---- stored variants beyond the 3D projection (f3) ---------------------------------------------------
sho_status sho_add_stored(const sho_plan* plan, const sho_tables* tables, const void* coeff, int32_t nbands, void* psi,
                          void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi && nbands > 0 && tables && tables->plan == plan && tables->plan_serial == plan->serial) return SHO_OK;
    sho_status st = check_hot("sho_add_stored", plan, coeff, psi, nbands);
    if (st != SHO_OK) return st;
    if (!tables || tables->plan != plan || tables->plan_serial != plan->serial) { set_error("sho_add_stored: tables do not belong to this plan"); return SHO_ERR_INVALID_ARG; }
    return launch_add_stored(plan, tables, coeff, nbands, psi, static_cast<cudaStream_t>(cuda_stream));
}

sho_status sho_tables1d_build(const sho_plan* plan, sho_tables1d** out, size_t* bytes_needed, void* cuda_stream)
{
    if (out) *out = nullptr;
    if (!plan || !bytes_needed) { set_error("sho_tables1d_build: null argument"); return SHO_ERR_INVALID_ARG; }
    return tables1d_build(plan, out, bytes_needed, static_cast<cudaStream_t>(cuda_stream));
}

sho_status sho_tables1d_destroy(sho_tables1d* t)
{
    if (!t) return SHO_OK;
    cudaFree(t->d_data);
    cudaFree(t->d_atom_off);
    delete t;
    return SHO_OK;
}

static sho_status check_t1(const char* fn, const sho_plan* plan, const sho_tables1d* t)
{
    if (!t || t->plan != plan || t->plan_serial != plan->serial) { set_error("%s: tables do not belong to this plan", fn); return SHO_ERR_INVALID_ARG; }
    return SHO_OK;
}

sho_status sho_project_stored1d(const sho_plan* plan, const sho_tables1d* tables, const void* psi, int32_t nbands, void* coeff,
                                void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi && nbands > 0) return SHO_OK;
    sho_status st = check_hot("sho_project_stored1d", plan, psi, coeff, nbands);
    if (st != SHO_OK || (st = check_t1("sho_project_stored1d", plan, tables)) != SHO_OK) return st;
    return launch_project(plan, psi, nbands, coeff, static_cast<cudaStream_t>(cuda_stream), 0, tables);
}

sho_status sho_add_stored1d(const sho_plan* plan, const sho_tables1d* tables, const void* coeff, int32_t nbands, void* psi,
                            void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi && nbands > 0) return SHO_OK;
    sho_status st = check_hot("sho_add_stored1d", plan, coeff, psi, nbands);
    if (st != SHO_OK || (st = check_t1("sho_add_stored1d", plan, tables)) != SHO_OK) return st;
    if (plan->n_tile_list == 0) return SHO_OK;
    return launch_add(plan, coeff, nbands, psi, static_cast<cudaStream_t>(cuda_stream), 0, tables);
}

// ---- band-fastest psi layout (the paper's own layout) ---------------------------------
static sho_status bf_chunk(const char* fn, const sho_plan* plan, int32_t nbands, size_t work_bytes, int* cb)
{
    const size_t band_bytes = (size_t)plan->g.ng[0] * plan->g.ng[1] * plan->g.ng[2] * elem_size(plan->dtype);
    size_t n = band_bytes ? work_bytes / band_bytes : (size_t)nbands;
    if (n > 1) n -= n & 1;                       // an even number of bands: the add kernel pairs real bands
    if (n < 1) {
        set_error("%s: the workspace of %zu bytes does not hold one band (%zu bytes)", fn, work_bytes, band_bytes);
        return SHO_ERR_INVALID_ARG;
    }
    *cb = (int)std::min<size_t>(n, (size_t)nbands);
    return SHO_OK;
}

sho_status sho_project_bf(const sho_plan* plan, const void* psi_bf, int32_t nbands, void* coeff, void* work, size_t work_bytes,
                          void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi_bf && nbands > 0) return SHO_OK;
    sho_status st = check_hot("sho_project_bf", plan, psi_bf, coeff, nbands);
    if (st != SHO_OK) return st;
    if (!work) { set_error("sho_project_bf: null workspace"); return SHO_ERR_INVALID_ARG; }
    int cb = 0;
    if ((st = bf_chunk("sho_project_bf", plan, nbands, work_bytes, &cb)) != SHO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t row = (size_t)plan->g.nsho * elem_size(plan->dtype);
    for (int b0 = 0; b0 < nbands; b0 += cb) {
        const int nb = std::min(cb, nbands - b0);
        if ((st = launch_to_x_fastest(plan, psi_bf, nbands, b0, nb, work, s)) != SHO_OK) return st;
        if ((st = launch_project(plan, work, nb, static_cast<char*>(coeff) + (size_t)b0 * row, s, nbands)) != SHO_OK) return st;
    }
    return SHO_OK;
}

sho_status sho_add_bf(const sho_plan* plan, const void* coeff, int32_t nbands, void* psi_bf, void* work, size_t work_bytes,
                      void* cuda_stream)
{
    if (plan && plan->g.natoms == 0 && psi_bf && nbands > 0) return SHO_OK;
    sho_status st = check_hot("sho_add_bf", plan, coeff, psi_bf, nbands);
    if (st != SHO_OK) return st;
    if (!work) { set_error("sho_add_bf: null workspace"); return SHO_ERR_INVALID_ARG; }
    if (plan->n_tile_list == 0) return SHO_OK;
    int cb = 0;
    if ((st = bf_chunk("sho_add_bf", plan, nbands, work_bytes, &cb)) != SHO_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t band_bytes = (size_t)plan->g.ng[0] * plan->g.ng[1] * plan->g.ng[2] * elem_size(plan->dtype);
    const size_t row = (size_t)plan->g.nsho * elem_size(plan->dtype);
    for (int b0 = 0; b0 < nbands; b0 += cb) {
        const int nb = std::min(cb, nbands - b0);
        // the chunk's increment A c is built in the (zeroed) workspace, then accumulated into psi_bf in one pass
        cudaError_t e = cudaMemsetAsync(work, 0, band_bytes * nb, s);
        if (e != cudaSuccess) return cuda_fail(e, "sho_add_bf: memset");
        if ((st = launch_add(plan, static_cast<const char*>(coeff) + (size_t)b0 * row, nb, work, s, nbands)) != SHO_OK) return st;
        if ((st = launch_from_x_fastest(plan, work, nbands, b0, nb, psi_bf, s)) != SHO_OK) return st;
    }
    return SHO_OK;
}

// ---- HOST-buffer end-to-end variants ------------------------------------------------------------
static sho_status ws_reserve(void** ws, size_t* have, size_t need, const char* what)
{
    if (*have >= need) return SHO_OK;
    cudaFree(*ws);
    *ws = nullptr; *have = 0;
    cudaError_t e = cudaMalloc(ws, need);
    if (e != cudaSuccess) { cudaGetLastError(); set_error("%s: cannot allocate %zu bytes of device workspace", what, need); return SHO_ERR_OOM; }
    *have = need;
    return SHO_OK;
}

// bands per chunk: about 128 MB of psi (the first upload and the last download are not overlapped with anything, so
// small chunks win: cfg 5 end to end 177 / 165 / 160 / 158 ms with 8 / 4 / 2 / 1 bands of 113 MB per chunk), an even
// number (the add kernel pairs real bands), at most 64 chunks
static int host_chunk_bands(const sho_plan* plan, int nbands)
{
    if (plan->opt_host_chunk_bands > 0) return std::min(plan->opt_host_chunk_bands, nbands);   // sho_plan_set_option
    const double band_bytes = (double)plan->g.ng[0] * plan->g.ng[1] * plan->g.ng[2] * elem_size(plan->dtype);
    int cb = (int)std::max(1.0, std::floor(128.0e6 / band_bytes));
    cb = std::max(cb, (nbands + 63) / 64);
    if (cb > 1) cb += cb & 1;
    return std::min(cb, nbands);
}

// The bands are independent, so the host-buffer calls pipeline them in chunks through a ring of kHostRing chunk
// buffers on the device (the workspace is bounded by the chunk size, not by nbands): the H2D copy of chunk i+1, the
// kernels of chunk i and the D2H copy of chunk i-1 run at the same time on three streams (PCIe is full duplex).  A
// ring slot is reused only after the D2H copy (hence the kernels) of the chunk that used it last has finished.  A
// chunk's coefficients [natoms][chunk][N_SHO] are a 2D sub-array of the caller's [natoms][nbands][N_SHO].
constexpr int kHostRing = 3;
enum HostMode { kHostProject, kHostAdd, kHostApply };

static sho_status host_run(sho_plan* plan, HostMode mode, const char* fn, void* psi_host, void* coeff_host,
                           const double* dmat_dev, int32_t nbands, cudaStream_t s)
{
    const size_t esz = elem_size(plan->dtype);
    const size_t band_bytes = (size_t)plan->g.ng[0] * plan->g.ng[1] * plan->g.ng[2] * esz;
    const size_t row_bytes = (size_t)plan->g.nsho * esz;                     // coefficients of one (atom, band)
    const int cb = host_chunk_bands(plan, nbands);
    const int nchunks = (nbands + cb - 1) / cb;
    const int nring = std::min(nchunks, kHostRing);
    const size_t psi_slot = band_bytes * cb, c_slot = std::max<size_t>((size_t)plan->g.natoms * cb * row_bytes, 16);
    sho_status st;
    if ((st = ws_reserve(&plan->ws_psi, &plan->ws_psi_bytes, psi_slot * nring, fn)) != SHO_OK) return st;
    if ((st = ws_reserve(&plan->ws_c, &plan->ws_c_bytes, c_slot * nring, fn)) != SHO_OK) return st;
    if (!plan->s_in && cudaStreamCreateWithFlags(&plan->s_in, cudaStreamNonBlocking) != cudaSuccess) return cuda_fail(cudaGetLastError(), fn);
    if (!plan->s_out && cudaStreamCreateWithFlags(&plan->s_out, cudaStreamNonBlocking) != cudaSuccess) return cuda_fail(cudaGetLastError(), fn);
    cudaStream_t s_in = plan->s_in, s_out = plan->s_out;
    std::vector<cudaEvent_t> events;
    // Every ordering edge between the three streams is an event.  A failed event call would silently drop an edge
    // (the streams would then race on the chunk buffers), so the first failure is kept in ev_err and ends the call.
    cudaError_t ev_err = cudaSuccess;
    auto note = [&](cudaError_t r) { if (r != cudaSuccess && ev_err == cudaSuccess) ev_err = r; return r == cudaSuccess; };
    auto mark = [&](cudaStream_t signaller) -> cudaEvent_t {                            // an event behind what signaller has queued
        cudaEvent_t ev = nullptr;
        if (!note(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming))) return nullptr;
        events.push_back(ev);
        if (!note(cudaEventRecord(ev, signaller))) return nullptr;
        return ev;
    };
    // waiter continues after what signaller has queued (the caller's stream may be the default stream, handle 0)
    auto after = [&](cudaStream_t waiter, cudaStream_t signaller) {
        cudaEvent_t ev = mark(signaller);
        if (ev) note(cudaStreamWaitEvent(waiter, ev, 0));
    };
    // on any failure: let everything that was queued finish before the caller gets its buffers back
    auto finish = [&](sho_status status) {
        cudaStreamSynchronize(s_in); cudaStreamSynchronize(s); cudaStreamSynchronize(s_out);
        for (cudaEvent_t e : events) cudaEventDestroy(e);
        return status;
    };
    auto edge_lost = [&]() { return finish(cuda_fail(ev_err, fn)); };
    after(s_in, s);                         // the copies start after what the caller queued on its stream
    after(s_out, s);
    if (ev_err != cudaSuccess) return edge_lost();
    cudaEvent_t slot_free[kHostRing] = { nullptr, nullptr, nullptr };
    cudaError_t e = cudaSuccess;
    for (int i = 0, b0 = 0; b0 < nbands; ++i, b0 += cb) {
        const int nb = std::min(cb, nbands - b0), slot = i % nring;
        char* d_psi = static_cast<char*>(plan->ws_psi) + (size_t)slot * psi_slot;
        char* d_c = static_cast<char*>(plan->ws_c) + (size_t)slot * c_slot;                 // [natoms][nb][N_SHO]
        char* h_psi = static_cast<char*>(psi_host) + (size_t)b0 * band_bytes;
        char* h_c = coeff_host ? static_cast<char*>(coeff_host) + (size_t)b0 * row_bytes : nullptr;
        if (slot_free[slot] && !note(cudaStreamWaitEvent(s_in, slot_free[slot], 0))) return edge_lost();
        if (mode == kHostAdd && plan->g.natoms > 0) {
            e = cudaMemcpy2DAsync(d_c, (size_t)nb * row_bytes, h_c, (size_t)nbands * row_bytes, (size_t)nb * row_bytes,
                                  (size_t)plan->g.natoms, cudaMemcpyHostToDevice, s_in);
            if (e != cudaSuccess) return finish(cuda_fail(e, fn));
        }
        e = cudaMemcpyAsync(d_psi, h_psi, band_bytes * nb, cudaMemcpyHostToDevice, s_in);
        if (e != cudaSuccess) return finish(cuda_fail(e, fn));
        after(s, s_in);
        if (ev_err != cudaSuccess) return edge_lost();
        if (plan->g.natoms > 0) {
            if (mode == kHostProject) st = launch_project(plan, d_psi, nb, d_c, s);
            else if (mode == kHostAdd) st = plan->n_tile_list ? launch_add(plan, d_c, nb, d_psi, s) : SHO_OK;
            else {
                st = launch_project(plan, d_psi, nb, d_c, s);
                if (st == SHO_OK) st = launch_dmul(plan, dmat_dev, d_c, nb, d_c, s);
                if (st == SHO_OK && plan->n_tile_list) st = launch_add(plan, d_c, nb, d_psi, s);
            }
            if (st != SHO_OK) return finish(st);
        }
        after(s_out, s);
        if (ev_err != cudaSuccess) return edge_lost();
        if (mode == kHostProject) {
            if (plan->g.natoms > 0)
                e = cudaMemcpy2DAsync(h_c, (size_t)nbands * row_bytes, d_c, (size_t)nb * row_bytes, (size_t)nb * row_bytes,
                                      (size_t)plan->g.natoms, cudaMemcpyDeviceToHost, s_out);
        } else {
            e = cudaMemcpyAsync(h_psi, d_psi, band_bytes * nb, cudaMemcpyDeviceToHost, s_out);
        }
        if (e != cudaSuccess) return finish(cuda_fail(e, fn));
        slot_free[slot] = mark(s_out);
        if (ev_err != cudaSuccess) return edge_lost();
    }
    after(s, s_out);
    if (ev_err != cudaSuccess) return edge_lost();
    e = cudaStreamSynchronize(s);
    for (cudaEvent_t ev : events) cudaEventDestroy(ev);
    if (e != cudaSuccess) return cuda_fail(e, fn);
    return SHO_OK;
}

sho_status sho_project_host(sho_plan* plan, const void* psi_host, int32_t nbands, void* coeff_host, void* cuda_stream)
{
    sho_status st = check_hot("sho_project_host", plan, psi_host, coeff_host, nbands);
    if (st != SHO_OK) return st;
    return host_run(plan, kHostProject, "sho_project_host", const_cast<void*>(psi_host), coeff_host, nullptr, nbands,
                    static_cast<cudaStream_t>(cuda_stream));
}

sho_status sho_add_host(sho_plan* plan, const void* coeff_host, int32_t nbands, void* psi_host, void* cuda_stream)
{
    sho_status st = check_hot("sho_add_host", plan, coeff_host, psi_host, nbands);
    if (st != SHO_OK) return st;
    if (plan->g.natoms == 0 || plan->n_tile_list == 0) return SHO_OK;
    return host_run(plan, kHostAdd, "sho_add_host", psi_host, const_cast<void*>(coeff_host), nullptr, nbands,
                    static_cast<cudaStream_t>(cuda_stream));
}

sho_status sho_apply_host(sho_plan* plan, const double* dmat_host, void* psi_host, int32_t nbands, void* cuda_stream)
{
    sho_status st = check_hot("sho_apply_host", plan, dmat_host ? (const void*)dmat_host : psi_host, psi_host, nbands);
    if (st != SHO_OK) return st;
    if (plan->g.natoms == 0 || plan->n_tile_list == 0) return SHO_OK;
    if (!dmat_host) { set_error("sho_apply_host: null argument"); return SHO_ERR_INVALID_ARG; }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t d_bytes = (size_t)plan->g.natoms * plan->g.nsho * plan->g.nsho * sizeof(double);
    if ((st = ws_reserve(&plan->ws_d, &plan->ws_d_bytes, d_bytes, "sho_apply_host")) != SHO_OK) return st;
    cudaError_t e = cudaMemcpyAsync(plan->ws_d, dmat_host, d_bytes, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(e, "sho_apply_host: H2D of the atomic matrices");
    return host_run(plan, kHostApply, "sho_apply_host", psi_host, nullptr, static_cast<const double*>(plan->ws_d), nbands, s);
}

}  // extern "C"

// ---- FP64 pipe micro-benchmark (roofline denominator measured in the same run) ------------------
namespace sho {
__global__ void __launch_bounds__(512) fp64_peak_kernel(double* out, int iters, double s)
{
    double a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = fma(a[i], s, s);
    }
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) r += a[i];
    if (r == 12345.678) out[0] = r;   // never true; keeps the chain alive
}
}  // namespace sho

extern "C" sho_status sho_measure_fp64_peak(int32_t iters, double* flops_per_s)
{
    if (!flops_per_s || iters <= 0) { set_error("sho_measure_fp64_peak: bad argument"); return SHO_ERR_INVALID_ARG; }
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "sho_measure_fp64_peak: cudaGetDevice");
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    double* d = nullptr;
    if ((e = cudaMalloc(&d, 8)) != cudaSuccess) return cuda_fail(e, "sho_measure_fp64_peak: cudaMalloc");
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = 2 * sms, threads = 512;
    sho::fp64_peak_kernel<<<blocks, threads>>>(d, iters, 0.999);   // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0);
        sho::fp64_peak_kernel<<<blocks, threads>>>(d, iters, 0.999);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double fl = 2.0 * 8.0 * (double)iters * blocks * threads / (ms * 1e-3);
        best = std::max(best, fl);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e, "sho_measure_fp64_peak");
    *flops_per_s = best;
    return SHO_OK;
}
