// md_internal.cuh -- shared declarations of libmd_b200 (host handle, device parameter block, workspace map).
// Product code: shares nothing with oracle/.  Citations as in include/md_b200.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "md_b200.h"

#define MD_TILE 32            // particles per list tile (one warp)
#define MD_MAX_PATCH 8

// Device error bits latched in DevCtrl::err
#define MD_DEVERR_CAPACITY 1
#define MD_DEVERR_FENE 2

// Device-resident control block (first bytes of the workspace).
struct DevCtrl {
    int rebuild;                 // skin criterion tripped (S:A5); consumed by the gated build kernels
    int err;                     // MD_DEVERR_* bits
    unsigned int n_edges;        // E = 1/2 sum |L_i|
    int max_seen;                // max |L_i| at the last build
    unsigned long long n_full;   // sum |L_i|
    int n_rebuilds;              // builds triggered by the skin criterion inside md_integrate
    int pad0;
    unsigned int scan_total;     // scratch for the scan kernels
    int pad[7];
};

// Parameter block passed by value to every kernel.
struct DevParams {
    int N, ntiles, cap, capg;          // capg = cap/4 (int4 groups per list row)
    float Lx, Ly, Lz, hLx, hLy, hLz;   // box and half box (fp32, exactly the fp32 box of the fixtures)
    double dLx, dLy, dLz;              // same values in double (S:Q7)
    double rv2d, rc2d;                 // (rcut+skin)^2 and rcut^2 formed in double (S:O0, S:Q5)
    double cscale_x, cscale_y, cscale_z;   // cells per unit length, n_k / L_k
    int ncx, ncy, ncz, ncell;
    float rc2, band_abs;               // fp32 cutoff and the half-width of the fp64-recheck band |d2 - rc2| (S:H10)
    float half_skin2;                  // (skin/2)^2
    // pair potential
    int kind;
    float eps, sig2, mass, inv_mass;
    float c48, c24, c4, vshift;        // 48 eps, 24 eps, 4 eps, V_c
    float lj_a, lj_b, lj_c, lj_d;      // 48 eps sigma^12, 24 eps sigma^6, 4 eps sigma^12, 4 eps sigma^6
    // WCA core of the patchy potential
    float core_rc2, core_vshift;
    // FENE
    float fene_K, fene_R02, fene_invR02;
    int chain_len;
    // patches
    int n_patches;
    float pdir[MD_MAX_PATCH][3];
    float eps_patch, inv_2sr2, inv_sr2, inv_w2, sigma, inv_inertia;
};

// All device pointers carved from the caller's workspace.
struct DevBuffers {
    DevCtrl* ctrl;
    int* cell_of;          // [N]
    int* cell_count;       // [ncell+1]
    int* cell_start;       // [ncell+1]
    int* cell_rank;        // [ncell] linear cell -> storage rank (Hilbert or identity)
    int* items_tmp;        // [N]
    int* items;            // [N] slots sorted by cell rank, ascending slot inside a cell
    int* ids;              // [N] slot -> original id
    int* ids_tmp;          // [N]
    int* slot_of_id;       // [N]
    float4* tmp4;          // [N] permutation scratch
    float4* pos_ref;       // [N]
    int* nl_count;         // [Npad]
    int* nl_full;          // [ntiles*32*cap] tile-transposed full list
    int2* tile_info;       // [ntiles] (kmax | needs_image << 30, kmin over the tile's live lanes)
    int* half_count;       // [N]
    unsigned int* edge_off;// [N+1]
    int2* edges;           // [ecap]
    unsigned int* in_off;  // [N+1]   segmented scatter: incoming-edge index
    unsigned int* in_edge; // [ecap]
    float4* edge_f;        // [ecap]  per-edge force (fx,fy,fz,V)
    float4* edge_ti;       // [ecap]  per-edge torque on i (patchy)
    float4* edge_tj;       // [ecap]  per-edge torque on j (patchy)
    unsigned int* scan_blk;// [scan blocks]
    double* e_part;        // [e_blocks*3]
    double* e_out;         // [3]
    float4* stage4;        // [N] staging for md_step_host un-permute
};

struct md_system {
    DevParams P;
    DevBuffers B;
    cudaStream_t stream;
    int64_t N;
    size_t ecap;
    double rcut, skin;
    md_potential pot;
    int order;
    bool rigid;
    float4 *pos, *vel, *force, *quat, *angmom, *torque;
    bool bound, cells_valid, lists_valid, forces_valid, seg_valid;
    int64_t launches;
    int sticky;              // sticky md_status (CUDA errors)
    char errmsg[512];
    void* workspace;
    size_t workspace_bytes;
    int* h_cell_rank;        // host copy (built at create)
};

// ---- kernel launch entry points (defined in the .cu files) ----
void md_launch_build_cells(md_system* s, bool gated);
void md_launch_build_verlet(md_system* s, bool gated);
void md_launch_seg_index(md_system* s, bool gated);
void md_launch_build_end(md_system* s, bool gated);
void md_launch_forces(md_system* s, int strategy, int scatter);
void md_launch_kick_drift(md_system* s, float dt);
void md_launch_kick(md_system* s, float dt);
void md_launch_energy(md_system* s);
void md_launch_unpermute(md_system* s, const float4* src, float4* dst);   // dst[ids[s]] = src[s]

#define MD_ERRBUF(s, ...) snprintf((s)->errmsg, sizeof((s)->errmsg), __VA_ARGS__)
