/*
 * md_b200.h -- C ABI of libmd_b200.so: the short-range force hot path of arXiv 1401.4350
 * ("A comparison between parallelization approaches in molecular dynamics simulations on GPUs")
 * written for one NVIDIA B200 (sm_100a).
 *
 * Citations: P:<n> = PAPER.md line n of the paper text; B:<n> = BASELINE.json line n;
 *            S:<x> = SURVEY.md section 8 item x; D:<x> = DESIGN.md section x.
 *
 * The library implements, as hand-written CUDA kernels only (no CPU fallback, no library kernels):
 *   - the "standard cell algorithm" + Verlet lists L_i of radius r_v = r_c + r_s
 *   - VERTEX: one thread per particle loops over L_i, every pair computed twice, no atomics
 *   - EDGE:   one thread per potentially interacting pair, F_ij = -F_ji, scatter to both
 *   - velocity-Verlet NVE with a skin-triggered rebuild, energies                          (B:5)
 *
 * Conventions
 *   Units        reduced LJ units, epsilon = sigma = m = k_B = 1 in all configs (B:7).
 *   Memory       the CALLER owns all device memory: six state arrays and one workspace blob sized by
 *                md_workspace_bytes().  The library never allocates device memory; md_destroy frees
 *                only the host handle.  "device" / "host" is stated for every pointer below.
 *   State layout float4 per particle (16-byte aligned device pointers), S:A1:
 *                  pos   = (x, y, z, unused)        vel    = (vx, vy, vz, unused)
 *                  force = (fx, fy, fz, pe_i)       pe_i = half of every pair/bond energy of i
 *                  quat  = (w, x, y, z) unit        angmom = (Lx, Ly, Lz, unused) space frame
 *                  torque= (tx, ty, tz, unused)     space frame
 *                The arrays are borrowed from md_bind_state() until md_destroy().  When an order
 *                other than MD_ORDER_NONE is set, md_build_cells() PERMUTES them in place: slot s
 *                then holds the particle whose original id is ids[s] (md_get_ids).
 *   Stream       every call enqueues on the CUDA stream given to md_create and returns without
 *                synchronising, except md_energy, md_stats, md_stats_ex, md_get_pairs, md_get_ids,
 *                md_get_state_double, md_step_host, md_probe, and md_build_verlet when a storage order is set
 *                (it reads the size of the largest staged neighbourhood back); they synchronise that stream.
 *   Errors       every function returns an md_status (0 = success, negative = failure); the
 *                text is available from md_last_error().  Device-detected conditions (neighbour
 *                capacity overflow, FENE bond >= R0) are latched in a device flag, reported ONCE by
 *                the next synchronising call and cleared by it: after md_bind_state / a rebuild with valid
 *                data the handle works again.  Only MD_ERR_CUDA is sticky.  No partial results are defined
 *                after a failure.
 *   Box          box[k] must be exactly representable in fp32 ((double)(float)box[k] == box[k]): the fp32
 *                minimum image and the fp64 list / cutoff predicates (S:O0) then use the same box (S:Q7).
 *   Determinism  MD_VERTEX and MD_SCATTER_SEGMENTED are run-to-run bitwise reproducible; the
 *                atomic scatter variants and MD_VERTEX_N3 are not.
 */
#ifndef MD_B200_H
#define MD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct md_system md_system; /* opaque host handle */

typedef enum {
    MD_OK = 0,
    MD_ERR_INVALID = -1,  /* bad argument or geometry (box too small for r_v, N <= 0, ...) */
    MD_ERR_STATE = -2,    /* call order: forces before lists, no state bound, ...            */
    MD_ERR_CAPACITY = -3, /* a particle has more than max_neigh Verlet neighbours            */
    MD_ERR_CUDA = -4,     /* CUDA runtime error (sticky)                                     */
    MD_ERR_NUMERIC = -5   /* FENE bond length >= R0                                          */
} md_status;

typedef enum { MD_POT_LJ = 0, MD_POT_FENE_WCA = 1, MD_POT_PATCHY = 2, MD_POT_PATCHY_PP = 3 } md_pot_kind;
typedef enum {
    MD_VERTEX = 0,   /* one thread per particle, every pair evaluated twice, no atomics                        */
    MD_EDGE = 1,     /* one thread per pair of the Verlet list, scatter to both particles                      */
    MD_VERTEX_N3 = 2 /* one thread per particle over its HALF list (j-side of every pair), Newton's third law:
                        own sum in registers, -f added atomically into one of m private force copies per particle,
                        copies combined afterwards.  Third argument of md_forces / md_integrate = m (1..64, 0 = 12;
                        P:71 "insensitive ... as long as m > 10"); MD_ERR_INVALID if m * N exceeds the edge capacity
                        N * max_neigh / 2 (the copies live in the workspace's per-edge scratch).                    */
} md_strategy;
/* EDGE scatter alternatives (B:5, S:A7); third argument of md_forces / md_integrate / md_step_host when strategy == MD_EDGE. */
typedef enum {
    MD_SCATTER_RED = 0,      /* red.global.add.f32, one per component                           */
    MD_SCATTER_RED_V4 = 1,   /* red.global.add.v4.f32, one per particle and output array        */
    MD_SCATTER_WARP = 2,     /* runs of equal owner i combined by warp shuffles, then one red.v4 */
    MD_SCATTER_SEGMENTED = 3, /* per-edge store + atomic-free segmented reduction        */
    MD_SCATTER_CLUSTER = 4   /* j side aggregated BEFORE L2: the half list of 16 consecutive owners is stored as
                                (j, 16-bit owner mask) units; one lane walks the pairs of a unit with the j side in
                                registers (one red.v4 per unit) and the owner side in lane-private shared-memory rows
                                (16 red.v4 per cluster).  Needs N < 2^31 only; fastest with an order set       */
} md_scatter;
/* VERTEX gather alternatives (B:5 "neighbour positions staged through shared memory or L2-resident gathers"):
 * passed as the third argument of md_forces / md_integrate / md_step_host when strategy == MD_VERTEX. */
typedef enum {
    MD_GATHER_AUTO = 0, /* SMEM when the storage is cell-sorted (an order is set), else L2 */
    MD_GATHER_L2 = 1,   /* one thread per particle, neighbour positions gathered from L1/L2 by global slot */
    MD_GATHER_SMEM = 2  /* one thread per particle, the block's neighbourhood staged in shared memory by bulk TMA copies,
                           16-bit block-local list entries ordered at build time for conflict-free 128-bit gathers */
} md_gather;
typedef enum { MD_ORDER_NONE = 0, MD_ORDER_CELL = 1, MD_ORDER_HILBERT = 2 } md_order;
/* P:59 (S:8(f3)): MD_PREC_F32 = fp32 state and integration (B:7, the default); MD_PREC_MIXED = the paper's production
 * mode, "mixed precision": positions, velocities (and angular momenta, quaternions) integrated in fp64, forces and
 * torques computed in fp32 from the rounded positions. */
typedef enum { MD_PREC_F32 = 0, MD_PREC_MIXED = 1 } md_precision;

/* Pair potential and rigid-body parameters.
 *   MD_POT_LJ        Eq. (1), cut at rcut and energy-shifted by V(rcut) if shift_energy.
 *   MD_POT_FENE_WCA  B:9: WCA (LJ cut at rcut = 2^(1/6) sigma, shifted by +epsilon) on all pairs, plus
 *                    FENE bonds U = -1/2 K R0^2 ln(1 - r^2/R0^2) between ids (i, i+1) inside chains of
 *                    chain_len consecutive ids.
 *   MD_POT_PATCHY    B:10: WCA core cut at rcut_core plus n_patches x n_patches patch terms
 *                    -eps_patch exp(-(r-sigma)^2/(2 patch_sigma_r^2)) exp(-(1-cos th_i)/patch_sigma_ang^2)
 *                    exp(-(1-cos th_j)/patch_sigma_ang^2), truncated (not shifted) at rcut.
 *   MD_POT_PATCHY_PP the paper's own patchy model, Eqs. (2)-(4) P:103-113 (S:8(f2), reading S:Q1 -- Eq. (4) is garbled in
 *                    the source, parity unpinned): V = epsilon (sigma/r)^core_exponent - eps_patch sum_a sum_b
 *                    exp[-1/2 (r_ab / patch_sigma_r)^patch_exponent], r_ab = distance between patch a of i and patch b of
 *                    j, patches at patch_radius * patch_dir from the centres, only patch pairs with r_ab < rcut_patch
 *                    (P:117), truncated not shifted.  Both exponents even integers <= 400; rcut >= 2 patch_radius +
 *                    rcut_patch; rcut_core and patch_sigma_ang are ignored but must be valid (> 0, rcut_core <= rcut). */
typedef struct {
    int32_t kind; /* md_pot_kind */
    float epsilon, sigma, mass;
    int32_t shift_energy;
    float fene_K, fene_R0;
    int32_t chain_len;
    int32_t n_patches; /* <= 8 */
    float patch_dir[8][3]; /* body-frame unit vectors */
    float eps_patch, patch_sigma_r, patch_sigma_ang;
    float rcut_core;
    float inertia; /* scalar moment of inertia of the spherical top (S:O7) */
    float patch_radius, patch_exponent, core_exponent, rcut_patch; /* MD_POT_PATCHY_PP only */
} md_potential;

/* Behaviour switches of a handle (no environment variables are read by the library, S:8(b)). */
typedef enum {
    MD_OPT_STAGE_LIMIT = 0, /* cap (staged particles, 0 = none) on the launch capacity of the shared-memory staged VERTEX
                               kernels: blocks with a larger neighbourhood take the unstaged path (tests of that path) */
    MD_OPT_NO_GRAPH = 1,    /* != 0: md_integrate launches its kernels one by one instead of replaying CUDA graphs
                               (profilers then list every kernel); same results bit for bit                          */
    MD_OPT_DEBUG = 2,       /* != 0: step-graph construction failures are printed on stderr                         */
    MD_OPT_ROW_SCHEDULE = 3, /* staged Verlet rows: 1 (default) = entries ordered at build time by shared-memory bank column
                               so that the 128-bit gathers of the force kernels are conflict-free; 0 = scan order (a
                               cheaper build, more bank conflicts per force evaluation).  Invalidates the lists.      */
    MD_OPT_FUSE_STEPS = 5,  /* multi-step graphs of md_integrate, staged LJ / FENE VERTEX in fp32: 1 (default) = the force kernel of
                               an inner step applies the kicks and the drift of the next step itself (no kick+drift kernel, no
                               force store; positions alternate between the caller's array and a scratch plane inside the
                               graph and end in the caller's array); 0 = separate kernels.  Same arithmetic, same results. */
    MD_OPT_BUILD_DIRECT = 4 /* staged Verlet build, dense cells: 1 (default) = the scheduled rows are emitted straight from the
                               hit words of the transposed scan (candidates enumerated by bank column); 0 = through the
                               column buckets in scratch memory (the form before it).  Same rows bit for bit.
                               Invalidates the lists.                                                                */
} md_option;

/* md_probe kinds: machine ceilings other than HBM bandwidth that bound the force kernels (S:8(d)). */
typedef enum {
    MD_PROBE_FFMA = 0,              /* fp32 FFMA issue rate          -> TFLOP/s                                    */
    MD_PROBE_FFMA2 = 1,             /* packed f32x2 FFMA2 issue rate -> TFLOP/s                                    */
    MD_PROBE_MUFU = 2,              /* MUFU.EX2 rate                 -> Tops/s                                     */
    MD_PROBE_RED_V4_SCATTER = 3,    /* red.global.add.v4.f32 to hashed particles     -> G lane-operations/s       */
    MD_PROBE_RED_F32_SCATTER = 4,   /* red.global.add.f32 to hashed components       -> G lane-operations/s       */
    MD_PROBE_RED_V4_COALESCED = 5,  /* red.global.add.v4.f32, consecutive lanes -> consecutive particles           */
    MD_PROBE_RED_F32_COALESCED = 6
} md_probe_kind;

/* Extended counters of md_stats_ex (host struct, filled up to `bytes`). */
typedef struct {
    int64_t n_edges;            /* E = 1/2 sum |L_i| at the last build                                         */
    int64_t n_full_entries;     /* sum |L_i|                                                                          */
    int64_t n_rebuilds;         /* skin-triggered device-side rebuilds inside md_integrate so far                      */
    int64_t n_in_cutoff;        /* E_in: pairs of the current list with d2 < rcut^2 at the current positions (S:Q16),
                                   counted by a kernel of its own with the fp64 predicate of S:Q5                      */
    int32_t max_neigh_seen;     /* max |L_i| at the last build                                                         */
    int32_t max_stage;          /* largest staged neighbourhood (particles) of a 256-particle block at the last build  */
    int32_t stage_launch;       /* staged-particle capacity the staged VERTEX kernels are launched with               */
    int32_t threads_per_particle; /* 1, 2 or 4: which instantiation of the staged LJ VERTEX kernel that capacity selects
                                   (0: the staged path is not in use)                                                  */
    int32_t cluster_size;       /* owners per cluster of MD_SCATTER_CLUSTER (0 until that list is built)              */
    int32_t pad0;
    int64_t n_cluster_units;    /* (cluster, j) units of MD_SCATTER_CLUSTER = L2 reductions of its j side at most      */
} md_stats_ex_t;

/* Bytes of device workspace md_create needs for these parameters.  host pointers. */
md_status md_workspace_bytes(int64_t N, const double box[3], double rcut, double skin,
                             const md_potential* pot, int32_t max_neigh, size_t* bytes);

/* Create a system of N particles in the periodic orthorhombic box[3] (cells of width >= r_v =
 * rcut + skin, Verlet lists of radius r_v).  box, pot: host.  workspace: DEVICE pointer, 256-byte
 * aligned, workspace_bytes >= md_workspace_bytes(...), owned by the caller and borrowed until
 * md_destroy.  cuda_stream: a cudaStream_t (may be NULL for the legacy default stream).
 * max_neigh: capacity of every L_i (rounded up to a multiple of 4), at most 480.
 * MD_ERR_INVALID if N <= 0, max_neigh > 480, N*max_neigh >= 2^31, box[k] < 2 (rcut + 2 skin), box[k] not exactly
 * representable in fp32, bad potential. */
md_status md_create(md_system** out, int64_t N, const double box[3], double rcut, double skin,
                    const md_potential* pot, int32_t max_neigh, void* workspace, size_t workspace_bytes,
                    void* cuda_stream);

/* Bind the state arrays (DEVICE pointers to float4[N]; quat/angmom/torque may be NULL unless
 * kind == MD_POT_PATCHY), taken to be in ORIGINAL id order: binding resets the slot map to the identity and
 * invalidates cells, lists and forces.  Positions may lie anywhere; md_build_cells wraps them into [0, box_k). */
md_status md_bind_state(md_system*, void* pos, void* vel, void* force, void* quat, void* angmom, void* torque);

/* Storage order applied at every list build ("sorted along a Hilbert curve"). Default NONE. */
md_status md_set_order(md_system*, int32_t order);

/* precision of md_integrate's state (default MD_PREC_F32).  In MD_PREC_MIXED the library keeps fp64 copies of
 * the integrated arrays in its workspace: they are taken from the bound fp32 arrays by the first md_build_cells /
 * md_integrate / md_step_host after md_bind_state or md_set_precision, advanced by md_integrate, wrapped and
 * reordered with the fp32 arrays, and the fp32 arrays are rewritten from them (round to nearest) at every step, so
 * every other call sees the same interface.  State written into the fp32 arrays behind the library's back is not
 * seen until the next md_bind_state.  MD_ERR_INVALID for an unknown value. */
md_status md_set_precision(md_system*, int32_t precision);

/* P:53 "Brownian dynamics simulations in the NVT ensemble, with the thermostat described in Ref. 27" -- Ref. 27 is not
 * in the container; reading DESIGN.md QT: an Andersen-type velocity refresh.  One application: each particle,
 * independently and with probability p_trans, gets a velocity drawn from the Maxwell-Boltzmann distribution at
 * temperature T (components Gaussian, variance T / mass); with kind == MD_POT_PATCHY each body, with probability
 * p_rot, likewise an angular momentum of variance T * inertia.  Draws come from Philox4x32-10 keyed by `seed`, counter
 * (ORIGINAL particle id, `call`, stream, block): the result depends on neither the storage order nor the launch
 * shape.  Positions and forces are untouched (forces stay valid); in MD_PREC_MIXED the fp64 copies are refreshed too.
 * md_thermostat applies it once (asynchronous, on the stream).  md_set_thermostat makes md_integrate (and
 * md_step_host) apply it after every n_newt-th step counted from this call, with call = steps / n_newt;
 * n_newt = 0 switches it off (the default: NVE, B:5).  MD_ERR_INVALID for T <= 0, a probability outside [0, 1] or
 * n_newt < 0; MD_ERR_STATE without a bound state. */
md_status md_set_thermostat(md_system*, double T, int64_t n_newt, double p_trans, double p_rot, uint64_t seed);
md_status md_thermostat(md_system*, double T, double p_trans, double p_rot, uint64_t seed, uint32_t call);

/* The fp64 state of MD_PREC_MIXED in ORIGINAL id order: pos_host, vel_host = HOST double[3 N] (x, y, z per particle),
 * either may be NULL.  Synchronises.  MD_ERR_STATE unless the precision is MD_PREC_MIXED and the copies exist. */
md_status md_get_state_double(md_system*, double* pos_host, double* vel_host);

/* S:A2/A3 ("cell filling ... one-particle-per-thread"): wrap positions into [0, box), bin into
 * cells, counting sort; with an order set, permute all bound state arrays into cell / Hilbert order. */
md_status md_build_cells(md_system*);

/* S:A4: L_i = { j != i : |r_ij|^2 < r_v^2 }, predicate evaluated in fp64 on the fp32 positions in
 * the fixed order of S:O0 (bit-exact pair set).  Emits the full list (VERTEX) and the half list i<j
 * sorted by i (EDGE, "number of threads = sum_i |L_i| / 2"), and records the reference
 * positions of the skin criterion.  Requires md_build_cells since the last position change. */
md_status md_build_verlet(md_system*);

/* S:A6/A7: forces, per-particle energies (force.w) and torques for the current positions.
 * Lists must be valid (no particle moved more than skin/2 since md_build_verlet). */
md_status md_forces(md_system*, int32_t strategy, int32_t scatter);

/* S:A10 (B:5): nsteps of NVE velocity-Verlet (S:O6; rigid bodies S:O7) in fp32 state.  Each step:
 * half kick, drift, skin check max_i |x_i - x_i^ref|^2 > (skin/2)^2 -> rebuild cells + lists on the
 * device without host synchronisation, forces, half kick.  Requires valid forces on entry. */
md_status md_integrate(md_system*, double dt, int64_t nsteps, int32_t strategy, int32_t scatter);
/* Note on capacity: the shared-memory staged VERTEX variant is launched with room for the largest block neighbourhood
 * seen at the last synchronising call plus 15-30 %.  A block whose neighbourhood outgrows that room in a device-side
 * rebuild (a lattice melting) is still computed, from global memory through its segment table (slower, same pairs and
 * decisions); calling md_stats every ~100 steps while the structure changes lets the capacity follow.  Only a
 * neighbourhood beyond the BUILD capacity (a quarter of a million staged bytes per block) is an error, MD_ERR_CAPACITY. */

/* S:A9: U = sum_i pe_i, K_t = 1/2 m sum |v|^2, K_r = sum |L|^2 / (2 I), accumulated in fp64.
 * Host output pointers.  Synchronises; reports latched device errors. */
md_status md_energy(md_system*, double* e_pot, double* e_kin_trans, double* e_kin_rot);

/* Counters (host pointers, any may be NULL).  n_edges = E = 1/2 sum |L_i|. Synchronises. */
md_status md_stats(md_system*, int64_t* n_edges, int64_t* n_full_entries, int32_t* max_neigh_seen,
                   int64_t* n_rebuilds);

/* md_stats plus the counters above; `bytes` = sizeof(md_stats_ex_t) of the caller.  Needs built lists for n_in_cutoff
 * (else that field is -1).  Synchronises. */
md_status md_stats_ex(md_system*, md_stats_ex_t* out, size_t bytes);

/* Set a behaviour switch (md_option).  MD_ERR_INVALID for an unknown option or a negative value. */
md_status md_set_option(md_system*, int32_t option, int64_t value);

/* Measure one machine ceiling (md_probe_kind) on the handle's device and stream; *value (host) in the unit listed with
 * the kind.  Uses the permutation scratch of the workspace: lists, cells and forces stay valid, a state reordering in
 * flight does not exist (the call synchronises before and after).  ~10 ms. */
md_status md_probe(md_system*, int32_t kind, double* value);

/* Copy the half list to the HOST as pairs of ORIGINAL ids (lo, hi), unsorted. pairs_host has room for
 * `capacity` pairs (2 int32 each); *n receives the pair count (even if > capacity). Synchronises. */
md_status md_get_pairs(md_system*, int32_t* pairs_host, int64_t capacity, int64_t* n);

/* ids_host[s] = original id of the particle stored in slot s (identity for MD_ORDER_NONE). Synchronises. */
md_status md_get_ids(md_system*, int32_t* ids_host);

/* End-to-end entry with HOST buffers (float4[N] each; quat/angmom/torque NULL unless patchy):
 * copies pos, vel (quat, angmom) host->device into the bound arrays, builds cells and lists,
 * evaluates forces, runs nsteps of md_integrate, and copies pos, vel, force (quat, angmom, torque)
 * back to the host in ORIGINAL id order.  Synchronises. */
md_status md_step_host(md_system*, void* pos_host, void* vel_host, void* force_host, void* quat_host,
                       void* angmom_host, void* torque_host, double dt, int64_t nsteps, int32_t strategy,
                       int32_t scatter);

/* ---------------------------------------------------------------------------------------------------------------------
 * Space decomposition ("space-decomposition: the domain ... partitioned into smaller subsets"; S:8(e), S:8(f4)).
 * One handle per rank holds the particles the rank OWNS (original ids 0 .. n_active-1) followed by GHOST copies of the
 * neighbouring ranks' particles within the halo width of its sub-domain (ids n_active .. N-1), all in GLOBAL coordinates
 * and the GLOBAL periodic box, so cells, Verlet lists and both force strategies run unchanged; every pair that involves
 * an owned particle is evaluated by the owner's rank (pairs across a face by both ranks: redundant arithmetic instead of
 * a reverse force exchange), forces on ghosts are discarded.  Protocol of one step (paper_1401_4350_b200/dd.py):
 *   md_half_step(KICK_DRIFT) -> halo refresh: md_gather_ids(send list) / send / recv / md_scatter_ids(ghost ids)
 *   -> md_rebuild_flag on every rank, all-reduce(max) -> [migration + new halo + md_resize + md_bind_state + builds]
 *   -> md_forces -> md_half_step(KICK).
 * ------------------------------------------------------------------------------------------------------------------- */
typedef enum { MD_ARRAY_POS = 0, MD_ARRAY_VEL = 1, MD_ARRAY_FORCE = 2, MD_ARRAY_QUAT = 3, MD_ARRAY_ANGMOM = 4, MD_ARRAY_TORQUE = 5 } md_array;
typedef enum { MD_STEP_KICK_DRIFT = 0, MD_STEP_KICK = 1 } md_step_part;

/* Change the particle count of the handle to n_new in [1, N at creation] (the workspace was carved for the creation N;
 * cells and capacities keep the creation geometry).  Unbinds the state: md_bind_state arrays of the new length next.
 * Resets n_active to n_new. */
md_status md_resize(md_system*, int64_t n_new);

/* Particles with ORIGINAL id >= n_active are ghosts: md_integrate / md_half_step neither kick nor drift them (the halo
 * refresh moves them), md_energy leaves them out; forces and lists treat them like any particle.  Default: N (none).
 * fp32 precision only (MD_ERR_STATE in MD_PREC_MIXED). */
md_status md_set_active(md_system*, int64_t n_active);

/* One half of a velocity-Verlet step (S:O6 / S:O7) on the owned particles, asynchronous:
 *   MD_STEP_KICK_DRIFT  v += dt/2 F/m, x += dt v (rigid bodies: L, q likewise) and the skin check of S:Q4 on ALL particles,
 *                       which latches the device-side rebuild flag; the forces are stale afterwards (call md_forces)
 *   MD_STEP_KICK        v += dt/2 F/m with the forces of the new positions.
 * MD_ERR_STATE without valid forces. */
md_status md_half_step(md_system*, double dt, int32_t part);

/* *flag (host) = 1 if the skin criterion has tripped since the last list build.  Synchronises. */
md_status md_rebuild_flag(md_system*, int32_t* flag);

/* dst_dev[k] = array[particle with original id ids_dev[k]] (ids_dev == NULL: id first_id + k), k < n; float4 each, DEVICE
 * pointers; array = md_array.  Asynchronous.  md_scatter_ids is the inverse for the id range [first_id, first_id + n):
 * array[particle first_id + k] = src_dev[k] (writing positions or quaternions invalidates the forces). */
md_status md_gather_ids(md_system*, int32_t array, const int32_t* ids_dev, int64_t first_id, int64_t n, void* dst_dev);
md_status md_scatter_ids(md_system*, int32_t array, int64_t first_id, int64_t n, const void* src_dev);

/* Stable compaction (ascending index) of { i < n : lo <= pos_dev[i][axis] < hi } into idx_out_dev[capacity] (may be NULL to
 * count only); *count_host receives the count (even if > capacity).  pos_dev: DEVICE float4[n]; the bounds are compared
 * in fp32.  scratch_dev: DEVICE, >= 4 * (n / 1024 + 3) bytes, 4-byte aligned.  Independent of any handle.  Synchronises
 * cuda_stream. */
md_status md_dd_select(const void* pos_dev, int64_t n, int32_t axis, double lo, double hi, int32_t* idx_out_dev, int64_t capacity,
                       int64_t* count_host, void* scratch_dev, size_t scratch_bytes, void* cuda_stream);

/* -------------------------------------------------------------------------------------------------------------------
 * No-allocation entry point (md_static.cu).  For callers that cannot call cudaMalloc (code under CUDA graph capture,
 * serving loops, harnesses that forbid it): the energy sums of md_energy (S:A9: U = sum_i pe_i, K_t = 1/2 m sum |v|^2,
 * K_r = sum |L|^2 / (2 I), fp32 terms accumulated in fp64, two deterministic stages) with NO handle and NO workspace.
 * The block partials live in a file-scope device array of 48 KiB that every GPU loading the library holds until exit;
 * the call performs no cudaMalloc / cudaFree and no allocating library routine.
 *   vel_dev, force_dev   DEVICE float4[n] (16-byte aligned), force.w = pe_i as left by md_forces
 *   angmom_dev           DEVICE float4[n] or NULL (then e_out[2] = 0)
 *   n                    1 .. MD_ENERGY_STATIC_MAX_N; beyond it MD_ERR_CAPACITY (nothing is launched)
 *   e_out_dev            DEVICE double[3] = (U, K_t, K_r), written on cuda_stream; the caller owns it
 *   err, err_len         optional HOST buffer for a message on failure (may be NULL / 0)
 * All n particles are summed (no ghost exclusion: that needs a handle's id table).  Runs on the CURRENT device, on
 * cuda_stream, asynchronously.  The first call on each device looks up the array's device address
 * (cudaGetSymbolAddress): make that call outside a graph capture.  All calls on a device share the array: calls that
 * overlap on the GPU (two streams, two host threads) race on it and must be serialised by the caller; it keeps the last
 * call's contents, and every call overwrites all partials it reads (nothing has to be cleared). */
#define MD_ENERGY_STATIC_MAX_N 16777216
md_status md_energy_static(const void* vel_dev, const void* force_dev, const void* angmom_dev, int64_t n, double mass,
                           double inv_inertia, double* e_out_dev, void* cuda_stream, char* err, size_t err_len);

/* Number of kernels this library has launched on behalf of the handle (for bench.py's gpu_launches). */
int64_t md_launch_count(const md_system*);

const char* md_last_error(const md_system*);
void md_destroy(md_system*);

#ifdef __cplusplus
}
#endif
#endif /* MD_B200_H */
