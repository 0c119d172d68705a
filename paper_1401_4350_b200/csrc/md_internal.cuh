// md_internal.cuh -- shared declarations of libmd_b200 (host handle, device parameter block, workspace map).
// Product code: shares nothing with oracle/.  Citations as in include/md_b200.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "md_b200.h"

#define MD_TILE 32            // particles per list tile (one warp)
#define MD_MAX_PATCH 8
#define MD_GRAPH_STEPS 16       // steps per launch of the multi-step graph of md_integrate
#define MD_CLUSTER 16           // owners per cluster of MD_SCATTER_CLUSTER (one 16-bit mask per (cluster, j) unit)

// Device error bits latched in DevCtrl::err
#define MD_DEVERR_CAPACITY 1
#define MD_DEVERR_FENE 2
#define MD_DEVERR_STAGE 4     // a block's staged neighbourhood / segment table exceeds its capacity

// ---- shared-memory staged path (md_staged.cu) ----
#define MD_TB 256             // particles per block (consecutive slots of the cell-sorted storage)
#define MD_NCAND 8192         // candidate cells per block before sort + unique (27 x non-empty own cells <= 27 x MD_TB)
#define MD_UMAX 4096          // distinct cells in a block's neighbourhood
#define MD_SEGMAX 1024        // contiguous slot segments per block
// BlkInfo flags
#define MD_BLK_WRAP 1         // some listed pair of the block crosses a periodic face
#define MD_BLK_SHIFT_OK 2     // ... and the shift-down transform of the staged coordinates reproduces every minimum image
#define MD_BLK_AXIS_SHIFT 4   // bits 2..4: axes (x, y, z) the transform applies to
#define MD_BLK_SH4 256         // row entries of the block are byte offsets (local index << 4): its neighbourhood has <= 4096 entries

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
    int max_stage;               // largest staged neighbourhood (particles) over the blocks at the last staged build
    int max_seg;                 // largest segment count
    int pad1;
    unsigned long long n_in;     // E_in: listed pairs inside the cutoff at the current positions (md_stats_ex)
    unsigned long long n_units;  // (cluster, j) units of the cluster list (MD_SCATTER_CLUSTER)
    unsigned long long n_cl_pairs; // sum of their popcounts = E
    unsigned int cl_cursor;      // next free slot of cl_units (rounds of 32)
    int pad2[5];
};

// per-block header of the staged path
struct BlkInfo {
    int nseg;        // contiguous slot segments to stage
    int M;           // staged particles (the dummy entry sits at local index M)
    int own_base;    // local index of the block's first own particle
    int flags;       // MD_BLK_*
};

// Parameter block passed by value to every kernel.
struct DevParams {
    int N, ntiles, cap, capg;          // capg = cap/4 (int4 groups per list row)
    int n_active;                      // original ids >= n_active are ghosts of a space decomposition: not integrated, not in the energy (md_set_active)
    float Lx, Ly, Lz, hLx, hLy, hLz;   // box and half box (fp32, exactly the fp32 box of the fixtures)
    double dLx, dLy, dLz;              // same values in double (S:Q7)
    double rv2d, rc2d;                 // (rcut+skin)^2 and rcut^2 formed in double (S:O0, S:Q5)
    double cscale_x, cscale_y, cscale_z;   // cells per unit length, n_k / L_k
    int ncx, ncy, ncz, ncell;
    float rc2, band_abs;               // fp32 cutoff and the half-width of the fp64-recheck band |d2 - rc2| (S:H10)
    float half_skin2;                  // (skin/2)^2
    float rv2, band_rv;                // fp32 list radius^2 and its fp64-recheck band (S:Q6)
    int nblk, stage_cap, rcap, mask_words;   // mask_words: 32-bit candidate-mask words per stencil cell (build scratch)
    int use_masks;                     // staged build: candidate masks (1) or index lists (0, few particles per cell)
    int row_schedule;                  // staged build: 1 = rows ordered by bank column (pass B buckets), 0 = scan order (MD_OPT_ROW_SCHEDULE)
    int build_direct;                  // staged build, dense cells: 1 = rows emitted from the hit words (MD_OPT_BUILD_DIRECT)
    float skinf;
    float shift_margin;                // r_v + skin: see k_build_staged step 7c
    // pair potential
    int kind;
    float eps, sig2, mass, inv_mass;
    float c48, c24, c4, vshift;        // 48 eps, 24 eps, 4 eps, V_c
    float lj_a, lj_b, lj_c, lj_d;      // 48 eps sigma^12, 24 eps sigma^6, 4 eps sigma^12, 4 eps sigma^6
    float2 k_nrc2, k_na, k_b, k_c, k_nd, k_nvs;   // duplicated constants of the packed (f32x2) LJ visit: -rc2, -lj_a, lj_b, lj_c, -lj_d, -vshift
    // WCA core of the patchy potential
    float core_rc2, core_vshift;
    // FENE
    float fene_K, fene_R02, fene_invR02;
    int chain_len;
    // patches
    int n_patches;
    int tetra;                         // the patch set is config 4's tetrahedron in its canonical order: packed fast path (md_pair.cuh)
    float pdir[MD_MAX_PATCH][3];
    float eps_patch, inv_2sr2, inv_sr2, inv_w2, sigma, inv_inertia;
    // MD_POT_PATCHY_PP (the paper's own patchy model, S:8(f2)): runs on the rigid-body kernels with kind == MD_POT_PATCHY
    int pp_model, pp_core_half, pp_half_n;   // flag; core_exponent / 2; patch_exponent / 2
    float pp_radius, pp_inv_w2, pp_rc2, pp_core_n, pp_n;
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
    float4* tmp4;          // [3 or 6][Npad] permutation scratch, one plane per bound state array
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
    // staged path
    int* cell_lin;         // [ncell] storage rank -> linear cell index (inverse of cell_rank)
    unsigned short* rows;  // [nblk][rcap/4][MD_TB] x 4 u16: Verlet rows of block-local indices, block-transposed chunks of 4
    unsigned short* rows_tmp; // [2][nblk][rcap + 2][MD_TB] build scratch: neighbours sorted by bank column; list form: scan order
    unsigned int* cmask;      // [nblk][27 * mask_words][MD_TB] build scratch: per stencil cell, bitmask of the candidates inside r_v
    int* row_count;        // [Npad] |L_i|
    int* lo_count;         // [Npad] neighbours with slot < i
    BlkInfo* blk;          // [nblk]
    int2* seg;             // [nblk*MD_SEGMAX] (first slot, first local index)
    // cluster list of MD_SCATTER_CLUSTER (md_cluster.cu)
    uint2* cl_units;       // [ucap] (j | image << 31, 16-bit owner mask), per cluster `rounds` x 32 lanes
    int2* cl_info;         // [ceil(N / MD_CLUSTER)] (first unit, rounds)
    // mixed precision (S:8(f3)): fp64 copies of the integrated state, two 16-byte planes per array so that the
    // reordering moves them like any other plane: [0] pos (x,y) [1] pos (z,-) [2] vel (x,y) [3] vel (z,-)
    // [4] angmom (x,y) [5] angmom (z,-) [6] quat (w,x) [7] quat (y,z)
    float4* shadow[8];     // each [Npad]; [4..7] only for rigid bodies
};

struct md_system {
    DevParams P;
    DevBuffers B;
    cudaStream_t stream;
    int64_t N;
    int64_t N_capacity;      // N at creation: md_resize may not exceed it (the workspace was carved for it)
    size_t ecap;
    size_t ucap;             // capacity of cl_units
    double rcut, skin;
    md_potential pot;
    int order;
    bool rigid;
    float4 *pos, *vel, *force, *quat, *angmom, *torque;
    bool bound, cells_valid, lists_valid, forces_valid, seg_valid;
    bool staged_valid, legacy_valid;   // which list representations describe the current build
    bool cluster_valid;                // the (cluster, j) unit list of MD_SCATTER_CLUSTER describes the current build
    int stage_limit;         // MD_OPT_STAGE_LIMIT: cap on the staged launch capacity (0 = none; tests of the unstaged path)
    bool no_graph, debug;    // MD_OPT_NO_GRAPH, MD_OPT_DEBUG
    bool fuse_steps;         // MD_OPT_FUSE_STEPS: fused step tails in the multi-step graphs (default on)
    int device, sm_count;    // the device the handle was created on and its SM count (cudaDeviceProp)
    size_t smem_optin, smem_per_sm;   // largest opt-in dynamic shared memory per block / shared memory per SM of that device
    int build_carve;         // shared-memory carveout k_build_staged was last configured with on this device (-1 = none)
    long long n_edges_host;  // E at the last synchronising call (0 before the first): picks the EDGE slice width
    int stage_launch;        // staged-particle capacity the force kernels are launched with (from the last synchronised build)
    int64_t launches;
    int sticky;              // sticky md_status (CUDA errors)
    char errmsg[512];
    void* workspace;
    size_t workspace_bytes;
    int* h_cell_rank;        // host copy (built at create)
    // one velocity-Verlet step as an executable CUDA graph: kick+drift, rebuild inside a conditional IF node that the
    // device-side skin flag drives, forces, kick (md_api.cu build_step_graph)
    cudaEvent_t ev_in, ev_vel;               // md_step_host: ordering of the velocity upload on aux_stream
    cudaGraphExec_t step_exec, multi_exec;   // one step / MD_GRAPH_STEPS steps per launch
    cudaGraphExec_t oct_exec, quad_exec, pair_exec;    // 8, 4 and 2 steps per launch: the tail of a call, with the fused closing kicks of the multi-step form
    int oct_nodes, quad_nodes, pair_nodes;
    cudaStream_t cap_stream, aux_stream; // internal capture streams: main sequence, conditional body
    int step_strategy, step_variant, step_stage, step_nodes, multi_nodes;   // *_nodes: kernels per launch outside the IF body
    float step_dt;
    int precision;                       // md_precision
    bool shadow_valid;                   // the fp64 copies describe the bound fp32 arrays
    double dt_d, step_dt_d;              // time step of the running / captured md_integrate in fp64 (mixed precision)
    bool graphs_off;                     // graph construction failed once: plain launches from then on
    // thermostat (reading QT of P:53): applied by md_integrate after every thermo_n-th step since md_set_thermostat
    int64_t thermo_n, thermo_steps;      // 0 = off; steps integrated since md_set_thermostat
    double thermo_T, thermo_pt, thermo_pr;
    unsigned long long thermo_seed;
};

// ---- kernel launch entry points (defined in the .cu files) ----
void md_launch_build_cells(md_system* s, bool gated);
void md_launch_build_verlet(md_system* s, bool gated, const float4* pos_src);   // explicit (global-slot) lists
void md_launch_edge_offsets(md_system* s, bool gated);   // edge_off = exclusive scan of half_count
void md_launch_seg_index(md_system* s, bool gated);
void md_launch_build_end(md_system* s, bool gated);
void md_launch_forces(md_system* s, int strategy, int scatter);
void md_launch_kick_drift(md_system* s, float dt, bool pre);   // pre: also the previous step's closing half kick
void md_launch_kick(md_system* s, float dt);
void md_launch_thermostat(md_system* s, double T, double p_t, double p_r, unsigned long long seed, unsigned int call);   // reading QT
void md_launch_shadow_init(md_system* s);   // fp64 copies <- bound fp32 arrays
void md_launch_energy(md_system* s);
void md_launch_set_cond(md_system* s, unsigned long long cond_handle);   // conditional value = rebuild flag
void md_launch_unpermute(md_system* s, const float4* src, float4* dst);   // dst[ids[s]] = src[s]
void md_launch_permute_in(md_system* s, const float4* src, float4* dst);  // dst[s] = src[ids[s]]
void md_launch_iota_ids(md_system* s);                                    // ids[s] = slot_of_id[s] = s
void md_launch_count_in_cutoff(md_system* s);                             // ctrl->n_in from the explicit edge list
void md_staged_configure(md_system* s);                                   // per-device kernel attributes of md_staged.cu
int md_staged_threads_per_particle(const md_system* s);                   // NS the staged LJ launch would use (0: rigid)
bool md_run_probe(md_system* s, int kind, double* value);                 // md_probe.cu
void md_drop_graphs(md_system* s);                                        // the captured step graphs (md_api.cu)
// cluster list (md_cluster.cu)
void md_cluster_configure(md_system* s);
bool md_launch_build_cluster(md_system* s, bool gated, const float4* pos_src);
void md_launch_edge_cluster(md_system* s);                                // force / torque zeroed by the caller
// staged path (md_staged.cu)
void md_launch_build_staged(md_system* s, bool gated);
void md_launch_edges_from_rows(md_system* s);     // explicit (i, j) edge list from the staged rows (export / legacy EDGE variants)
// Fused step tail of the staged LJ / FENE VERTEX kernel (inner steps of the multi-step graphs): instead of storing the force the
// thread applies the closing half kick of its step and the opening half kick + drift of the next one (the arithmetic of
// k_kick_drift<false, true>, same roundings), writes the new position to ANOTHER array -- other blocks still read the old
// ones -- and runs the skin check.  vel == nullptr: off (the force is stored).
struct FuseArgs { float4* vel; float4* pos_next; float dt; };
bool md_launch_forces_staged(md_system* s, bool energy, FuseArgs fuse = FuseArgs{ nullptr, nullptr, 0.0f });   // VERTEX on the staged rows; energy = false: force.w is not needed
void md_launch_kick_drift_to(md_system* s, float dt, float4* pos_out);   // fp32, point particles: opening half kick + drift, new positions to pos_out
size_t md_staged_smem_bytes(const md_system* s, int stage_entries);

#define MD_ERRBUF(s, ...) snprintf((s)->errmsg, sizeof((s)->errmsg), __VA_ARGS__)
