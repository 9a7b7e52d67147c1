// sho_internal.h -- host-side plan object and kernel parameter blocks shared by the .cu files of
// libsho.  Not part of the ABI (include/sho.h is).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/sho.h"

namespace sho {

constexpr int kProjWarps = 8;          // warps per CTA in the project kernel (one z-plane each per round)
constexpr int kAddTX = 8, kAddTY = 64, kAddTZ = 8;    // psi tile owned by one CTA of the add kernel
constexpr int kAddWarps = kAddTZ;                     // one z plane (64 rows x 8 columns) per warp
constexpr int kAddMaxMT = 17;                         // (ny,nx) pairs of numax = 15: 136 = 17 MMA row tiles

// one atom as the kernels see it (80 bytes)
struct AtomDev {
    double pos[3];
    double sigma;
    double inv_sigma;   // 1 / sigma
    double pref;        // (sqrt(pi) sigma)^(-1/2): normalisation of phi_0 (reading A1)
    int32_t lo[3];   // unwrapped inclusive box range per axis (reading A3); lo > hi on any axis: empty
    int32_t hi[3];
    int32_t pad[2];
};

// one (atom image) that overlaps an add tile: unwrapped index i = j + m*N on each axis.  Self-contained
// (the atom's parameters are copied in) so that the add kernel fetches one 96-byte record per pair with
// cp.async and never chases a pointer; 16-byte aligned
struct AddEntry {
    double pos[3];
    double inv_sigma;    // 1 / sigma
    double pref;         // (sqrt(pi) sigma)^(-1/2)
    double wr, wi;       // conj(exp(2 pi i kfrac.m)): Bloch phase of the image, conjugated (reading A6)
    int32_t atom;
    int32_t lo[3], hi[3];   // the atom's unwrapped inclusive box range
    int16_t m[3];
    uint8_t zmask;       // planes of the tile inside the box (bit k = plane k)
    int8_t ytlo, ythi;   // first / last 8-row block of the tile that the box touches
    uint8_t pad[3];
};
static_assert(sizeof(AddEntry) == 96, "AddEntry is fetched as six 16-byte cp.async pieces");

// the (ny,nx) pairs with ny+nx <= numax, sorted by s = ny+nx (pair index s(s+1)/2 + nx), cut in MMA row
// tiles of 8: tile mt needs nz <= numax - s_min(mt), i.e. nks[mt] K steps of 4, stored from block blk0[mt]
struct AddZTiles {
    int32_t nmt;         // row tiles
    int32_t nblk;        // sum of nks
    int8_t blk0[kAddMaxMT];
    int8_t nks[kAddMaxMT];
};

struct GridDev {
    int32_t ng[3];
    int32_t periodic[3];
    double h;
    double kfrac[3];
    double hnorm[SHO_NUMAX_MAX + 1];   // sqrt(2^n / n!): scale of the monic recurrence of eq. (31)
    int32_t zoff[SHO_NUMAX_MAX + 1];   // coefficients before plane nz of the (nx,ny,nz) enumeration (reading A8)
    int32_t numax;
    int32_t nsho;
    int32_t natoms;
    int32_t has_phase;                 // complex dtype and some kfrac != 0 on a periodic axis
};

}  // namespace sho

struct sho_plan {
    sho::GridDev g;
    double rcut_sigma;
    sho_dtype dtype;
    int device;
    uint64_t serial;                       // unique per plan (a new plan at a recycled address is a different plan)
    std::vector<sho::AtomDev> atoms;       // host copy, original order
    std::vector<int32_t> order;            // spatially sorted atom indices (non-empty boxes first)
    int32_t n_nonempty;
    int32_t max_n[3];                      // largest box extent per axis
    int64_t sum_box;                       // sum over atoms of box points
    int32_t proj_xalign_span;              // project: x steps start at a 32-byte lane span instead of a 128-byte line (saves > 10 % of them)
    double proj_odd_steps;                 // real data: share of x load steps lost if they are issued in pairs (see launch_project)
    // device mirrors
    sho::AtomDev* d_atoms;
    int32_t* d_order;
    uint32_t* d_nxyz;                      // [nsho] packed nx | ny<<8 | nz<<16
    // add tiling
    int32_t ntile[3];
    int64_t ntiles;
    int64_t npairs;
    int32_t* d_tile_ptr;                   // [ntiles+1]
    sho::AddEntry* d_tile_ent;             // [npairs]
    int32_t* d_tile_list;                  // tiles with at least one entry
    int4* d_tile_info;                     // per listed tile: (tile, first entry, entries, 0): one 16-byte load per work item
    int32_t n_tile_list;
    sho::AddZTiles ztiles;
    uint16_t* d_cainv;                     // [nsho] coefficient n -> slot (block*32 + 4 q + t) of the z-stage A fragments
    uint16_t* d_cidx;                      // [nblk][32] inverse of cainv (0xffff: padding element)
    uint16_t* d_t2pos;                     // [256 + 8 nmt]: column of T2 that holds pair (ny,nx) (index 16 ny + nx; the zero
                                           // column for ny+nx > numax), then the column of z-stage row 8 mt + q
    // workspace for the *_host calls
    void* ws_psi; size_t ws_psi_bytes;
    void* ws_c;   size_t ws_c_bytes;
    void* ws_d;   size_t ws_d_bytes;       // atomic matrices of sho_apply_host
    cudaStream_t s_in, s_out;              // copy streams of the *_host calls (created on first use)
    // sho_plan_set_option (0 = automatic)
    int32_t opt_project_bands_per_cta;
    int32_t opt_host_chunk_bands;
};

struct sho_tables {
    const sho_plan* plan;
    uint64_t plan_serial;
    void* d_data;                          // fragment-ordered tables, see sho_stored.cu
    int64_t* d_atom_off;                   // [natoms+1] offsets in elements
    int32_t* d_seg_atom;                   // K segments (atom, first box plane) = the CTAs of the stored kernel
    int32_t* d_seg_qz0;
    int32_t nseg;
    int* d_turn;                           // [turn_count] turnstile counters of sho_project_stored (256 column groups per atom)
    size_t turn_count;
    cudaEvent_t last_launch;               // recorded behind every sho_project_stored launch; the next launch waits for it
    mutable std::mutex launch_mutex;       // host side of that chain (the ABI hands the object out as const)
    std::vector<int64_t> atom_off;
    size_t bytes;
};

struct sho_tables1d {
    const sho_plan* plan;
    uint64_t plan_serial;
    double* d_data;                        // per atom: x rows, y rows, z rows; M = numax + 1 doubles per box index
    long long* d_atom_off;                 // [natoms] first element of the atom
    size_t bytes;
};

namespace sho {

void set_error(const char* fmt, ...);
sho_status cuda_fail(cudaError_t e, const char* what);
inline size_t elem_size(sho_dtype t) { return t == SHO_R64 ? 8 : t == SHO_C128 ? 16 : t == SHO_R32 ? 4 : 8; }
inline bool is_complex(sho_dtype t) { return t == SHO_C128 || t == SHO_C64; }

// launchers (defined next to their kernels)
// cnb: bands per atom in the coefficient array when the launch covers a chunk of a wider array (0: nbands)
sho_status launch_project(const sho_plan* p, const void* psi, int nbands, void* coeff, cudaStream_t s, int cnb = 0,
                          const sho_tables1d* t1 = nullptr);
sho_status launch_add(const sho_plan* p, const void* coeff, int nbands, void* psi, cudaStream_t s, int cnb = 0,
                      const sho_tables1d* t1 = nullptr);
sho_status tables1d_build(const sho_plan* p, sho_tables1d** out, size_t* bytes_needed, cudaStream_t s);
sho_status launch_add_stored(const sho_plan* p, const sho_tables* t, const void* coeff, int nbands, void* psi, cudaStream_t s);
sho_status launch_to_x_fastest(const sho_plan* p, const void* psi_bf, int nbands, int b0, int nb, void* psi_xf, cudaStream_t s);
sho_status launch_from_x_fastest(const sho_plan* p, const void* psi_xf, int nbands, int b0, int nb, void* psi_bf, cudaStream_t s);
// shared: dmat is ONE [N_SHO][N_SHO] matrix applied to every atom (sho_transform) instead of one per atom
sho_status launch_dmul(const sho_plan* p, const double* dmat, const void* cin, int nbands, void* cout, cudaStream_t s, bool shared = false);
sho_status launch_project_stored(const sho_plan* p, const sho_tables* t, const void* psi, int nbands, void* coeff,
                                 cudaStream_t s);
sho_status tables_build(const sho_plan* p, sho_tables** out, size_t* bytes_needed, cudaStream_t s);

}  // namespace sho
