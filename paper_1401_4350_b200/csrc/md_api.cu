// md_api.cu -- the C ABI of include/md_b200.h: argument checks, workspace carving, call order, error latching.
// Host logic only; every step of the path runs in the kernels of md_build.cu / md_forces.cu / md_integrate.cu.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <vector>
#include "md_internal.cuh"

namespace {

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Geometry {
    int nc[3];
    int64_t ncell;
    int cap, ntiles;
    size_t ecap, ucap;
    int rcap, nblk, stage_cap, mask_words;   // staged path
};

// S:Q8: n_k = max(1, floor(L_k / (r_v (1 + 1e-5)))) cells per axis, width >= r_v
bool make_geometry(int64_t N, const double box[3], double rcut, double skin, int max_neigh, Geometry* g) {
    if (N <= 0 || N > (1ll << 30) || !(rcut > 0) || !(skin >= 0) || max_neigh <= 0) return false;
    double rv = rcut + skin;
    g->ncell = 1;
    for (int k = 0; k < 3; ++k) {
        if (!(box[k] > 0) || box[k] < 2.0 * (rcut + 2.0 * skin)) return false;
        if ((double)(float)box[k] != box[k]) return false;   // S:Q7: fp32 minimum image and fp64 predicates share one box
        int n = (int)floor(box[k] / (rv * (1.0 + 1e-5)));
        g->nc[k] = n < 1 ? 1 : n;
        g->ncell *= g->nc[k];
    }
    if (g->ncell > (1ll << 30)) return false;
    if (max_neigh > 480) return false;            // the staged build keeps column populations in 8-bit fields (md_staged.cu pass B)
    g->cap = (max_neigh + 3) / 4 * 4;
    g->ntiles = (int)((N + MD_TILE - 1) / MD_TILE);
    if ((int64_t)g->ntiles * MD_TILE * g->cap >= (1ll << 31)) return false;
    g->ecap = (size_t)N * g->cap / 2 + 64;
    g->ucap = g->ecap + 2 * (size_t)N + 64;      // cluster units: at most one per pair, plus the padding of every last round
    if (g->ucap >= (1ull << 31)) g->ucap = (1ull << 31) - 64;
    // staged path: rows of 16-bit local indices in chunks of 4 entries; smem capacity of the build kernel
    g->rcap = (g->cap + 31) / 32 * 32;
    g->nblk = (int)((N + MD_TB - 1) / MD_TB);
    // largest neighbourhood (entries) a force kernel can stage: 16 B (+16 B quaternion) each in <= 224 KB of shared memory
    g->stage_cap = 0;   // set by the caller (depends on the potential)
    {   // candidate masks of the staged build: room for twice the mean cell population plus 24
        const double ppc = (double)N / (double)g->ncell;
        g->mask_words = (int)((2.0 * ppc + 24.0 + 31.0) / 32.0);
        if (g->mask_words < 1) g->mask_words = 1;
    }
    return true;
}

// carve the workspace; with base == nullptr only the size is computed
size_t carve(char* base, int64_t N, const Geometry& g, bool rigid, DevBuffers* B) {
    size_t off = 0;
    auto take = [&](size_t bytes) -> char* {
        char* p = base ? base + off : nullptr;
        off = align_up(off + bytes, 256);
        return p;
    };
    DevBuffers b;
    memset(&b, 0, sizeof(b));
    const size_t Npad = (size_t)g.ntiles * MD_TILE;
    b.ctrl = (DevCtrl*)take(sizeof(DevCtrl));
    b.cell_of = (int*)take(4 * Npad);
    b.cell_count = (int*)take(4 * (size_t)(g.ncell + 1));
    b.cell_start = (int*)take(4 * (size_t)(g.ncell + 1));
    b.cell_rank = (int*)take(4 * (size_t)g.ncell);
    b.items_tmp = (int*)take(4 * Npad);
    b.items = (int*)take(4 * Npad);
    b.ids = (int*)take(4 * Npad);
    b.ids_tmp = (int*)take(4 * Npad);
    b.slot_of_id = (int*)take(4 * Npad);
    b.tmp4 = (float4*)take(16 * Npad * (rigid ? 14 : 7));   // permutation scratch, one plane per state array and fp64 half
    for (int k = 0; k < (rigid ? 8 : 4); ++k) b.shadow[k] = (float4*)take(16 * Npad);
    b.pos_ref = (float4*)take(16 * Npad);
    b.nl_count = (int*)take(4 * Npad);
    b.nl_full = (int*)take(4 * Npad * g.cap);
    b.tile_info = (int2*)take(8 * (size_t)g.ntiles);
    b.half_count = (int*)take(4 * Npad);
    b.edge_off = (unsigned int*)take(4 * (Npad + 1));
    b.edges = (int2*)take(8 * g.ecap);
    b.in_off = (unsigned int*)take(4 * (Npad + 1));
    b.in_edge = (unsigned int*)take(4 * g.ecap);
    b.edge_f = (float4*)take(16 * g.ecap);
    if (rigid) {
        b.edge_ti = (float4*)take(16 * g.ecap);
        b.edge_tj = (float4*)take(16 * g.ecap);
    }
    size_t nscan = (std::max<size_t>(Npad, (size_t)g.ncell + 1) + 4095) / 4096 + 8;
    b.scan_blk = (unsigned int*)take(4 * nscan);
    b.e_part = (double*)take(8 * 3 * 2048);
    b.e_out = (double*)take(8 * 4);
    b.cell_lin = (int*)take(4 * (size_t)g.ncell);
    b.rows = (unsigned short*)take(2 * (size_t)g.nblk * MD_TB * (size_t)g.rcap);
    b.rows_tmp = (unsigned short*)take(2 * (size_t)g.nblk * MD_TB * (size_t)(8 * ((g.rcap + 2) / 2) + g.rcap + 2));   // 8 column buckets + list form
    b.cmask = (unsigned int*)take(4 * (size_t)g.nblk * 27 * (size_t)g.mask_words * MD_TB);   // scan order + sorted by column
    b.row_count = (int*)take(4 * Npad);
    b.lo_count = (int*)take(4 * Npad);
    b.cl_units = (uint2*)take(8 * g.ucap);
    b.cl_info = (int2*)take(8 * (((size_t)N + MD_CLUSTER - 1) / MD_CLUSTER));
    b.blk = (BlkInfo*)take(sizeof(BlkInfo) * (size_t)g.nblk);
    b.seg = (int2*)take(8 * (size_t)g.nblk * MD_SEGMAX);
    if (B) *B = b;
    return off;
}

bool check_pot(const md_potential* p, double rcut) {
    if (!p) return false;
    if (p->kind < MD_POT_LJ || p->kind > MD_POT_PATCHY_PP) return false;
    if (!(p->epsilon > 0) || !(p->sigma > 0) || !(p->mass > 0)) return false;
    if (p->kind == MD_POT_FENE_WCA && (p->chain_len < 1 || !(p->fene_K > 0) || !(p->fene_R0 > 0))) return false;
    if (p->kind == MD_POT_PATCHY_PP) {
        const double ne = p->patch_exponent, ce = p->core_exponent;
        if (!(p->patch_radius > 0) || !(p->rcut_patch > 0)) return false;
        if (!(ne >= 2 && ne <= 400 && ne == 2 * floor(ne / 2)) || !(ce >= 2 && ce <= 400 && ce == 2 * floor(ce / 2))) return false;
        if (rcut < (2.0 * p->patch_radius + p->rcut_patch) * (1.0 - 1e-6)) return false;   // a patch pair in range would be missed
    }
    if (p->kind == MD_POT_PATCHY || p->kind == MD_POT_PATCHY_PP) {
        if (p->n_patches < 1 || p->n_patches > MD_MAX_PATCH) return false;
        if (!(p->inertia > 0) || !(p->patch_sigma_r > 0) || !(p->patch_sigma_ang > 0) || !(p->rcut_core > 0)) return false;
        if (p->rcut_core > rcut) return false;
        for (int a = 0; a < p->n_patches; ++a) {
            double n2 = 0;
            for (int k = 0; k < 3; ++k) n2 += (double)p->patch_dir[a][k] * p->patch_dir[a][k];
            if (fabs(n2 - 1.0) > 1e-4) return false;   // S:8(b): non-unit patch vectors are invalid
        }
    }
    return true;
}

// 3-D Hilbert index of cell (x,y,z) on a 2^bits grid ("8-vertex Hilbert curve" = 2x2x2 recursion).
// Skilling's transpose construction ("Programming the Hilbert curve", AIP Conf. Proc. 707, 2004), restated.
uint64_t hilbert3(uint32_t x, uint32_t y, uint32_t z, int bits) {
    uint32_t X[3] = { x, y, z };
    const uint32_t M = 1u << (bits - 1);
    for (uint32_t Q = M; Q > 1; Q >>= 1) {          // inverse undo excess work
        uint32_t Pm = Q - 1;
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) X[0] ^= Pm;
            else { uint32_t t = (X[0] ^ X[i]) & Pm; X[0] ^= t; X[i] ^= t; }
        }
    }
    for (int i = 1; i < 3; ++i) X[i] ^= X[i - 1];   // Gray encode
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1; Q >>= 1) if (X[2] & Q) t ^= Q - 1;
    for (int i = 0; i < 3; ++i) X[i] ^= t;
    uint64_t h = 0;                                  // interleave the transposed bits, X[0] most significant
    for (int b = bits - 1; b >= 0; --b)
        for (int i = 0; i < 3; ++i) h = (h << 1) | ((X[i] >> b) & 1u);
    return h;
}

void make_cell_rank(const int nc[3], int order, std::vector<int>& rank) {
    const int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    rank.resize((size_t)ncell);
    if (order != MD_ORDER_HILBERT) {
        for (int64_t c = 0; c < ncell; ++c) rank[(size_t)c] = (int)c;
        return;
    }
    int bits = 1;
    while ((1 << bits) < std::max(nc[0], std::max(nc[1], nc[2]))) ++bits;
    std::vector<std::pair<uint64_t, int>> keys((size_t)ncell);
    for (int x = 0; x < nc[0]; ++x)
        for (int y = 0; y < nc[1]; ++y)
            for (int z = 0; z < nc[2]; ++z) {
                int lin = (x * nc[1] + y) * nc[2] + z;
                keys[(size_t)lin] = { hilbert3((uint32_t)x, (uint32_t)y, (uint32_t)z, bits), lin };
            }
    std::sort(keys.begin(), keys.end());
    for (int64_t r = 0; r < ncell; ++r) rank[(size_t)keys[(size_t)r].second] = (int)r;
}

void drop_step_graph(md_system* s) {
    if (s->step_exec) { cudaGraphExecDestroy(s->step_exec); s->step_exec = nullptr; }
    if (s->multi_exec) { cudaGraphExecDestroy(s->multi_exec); s->multi_exec = nullptr; }
    if (s->oct_exec) { cudaGraphExecDestroy(s->oct_exec); s->oct_exec = nullptr; }
    if (s->quad_exec) { cudaGraphExecDestroy(s->quad_exec); s->quad_exec = nullptr; }
    if (s->pair_exec) { cudaGraphExecDestroy(s->pair_exec); s->pair_exec = nullptr; }
}

md_status fail(md_system* s, md_status code, const char* msg) {
    if (s) snprintf(s->errmsg, sizeof(s->errmsg), "%s", msg);
    return code;
}

md_status check_cuda(md_system* s, const char* where) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(s->errmsg, sizeof(s->errmsg), "CUDA error at %s: %s", where, cudaGetErrorString(e));
        s->sticky = MD_ERR_CUDA;
        return MD_ERR_CUDA;
    }
    return MD_OK;
}

// cell_rank[linear cell] = storage rank and its inverse cell_lin[rank] = linear cell
void upload_cell_rank(md_system* s, const std::vector<int>& rank) {
    std::vector<int> inv(rank.size());
    for (size_t c = 0; c < rank.size(); ++c) inv[(size_t)rank[c]] = (int)c;
    cudaMemcpyAsync(s->B.cell_rank, rank.data(), 4 * rank.size(), cudaMemcpyHostToDevice, s->stream);
    cudaMemcpyAsync(s->B.cell_lin, inv.data(), 4 * inv.size(), cudaMemcpyHostToDevice, s->stream);
    cudaStreamSynchronize(s->stream);   // host temporaries
}

// slot s holds original id s (state arrays given in original id order): a kernel, no host temporaries, no synchronisation
void reset_ids(md_system* s) { md_launch_iota_ids(s); }

// synchronise and surface latched device errors
md_status sync_and_check(md_system* s, const char* where) {
    DevCtrl c;
    cudaError_t e = cudaMemcpyAsync(&c, s->B.ctrl, sizeof(c), cudaMemcpyDeviceToHost, s->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
    if (e != cudaSuccess) {
        snprintf(s->errmsg, sizeof(s->errmsg), "CUDA error at %s: %s", where, cudaGetErrorString(e));
        s->sticky = MD_ERR_CUDA;
        return MD_ERR_CUDA;
    }
    if (c.err) {
        // latched device conditions are reported once and cleared (the header documents only MD_ERR_CUDA as sticky):
        // after md_bind_state / a rebuild with valid data the handle works again
        cudaMemsetAsync(&s->B.ctrl->err, 0, sizeof(int), s->stream);
    }
    if (c.err & MD_DEVERR_CAPACITY) {
        snprintf(s->errmsg, sizeof(s->errmsg), "neighbour capacity exceeded: a particle has %d Verlet neighbours, max_neigh = %d", c.max_seen, s->P.cap);
        s->lists_valid = s->staged_valid = s->legacy_valid = s->cluster_valid = false;
        s->forces_valid = false;
        return MD_ERR_CAPACITY;
    }
    if (c.err & MD_DEVERR_STAGE) {
        snprintf(s->errmsg, sizeof(s->errmsg), "staged build capacity exceeded: a block needs %d staged particles / %d segments "
                 "(build capacity %d, segment capacity %d)", c.max_stage, c.max_seg, s->P.stage_cap, MD_SEGMAX);
        s->lists_valid = s->staged_valid = false;
        s->forces_valid = false;
        return MD_ERR_CAPACITY;
    }
    s->n_edges_host = (long long)c.n_edges;
    if (s->order != MD_ORDER_NONE && c.max_stage > 0) {
        // size the staged force launches from the largest neighbourhood seen, with 15 % head room for the
        // device-side rebuilds that happen before the next synchronising call; if that head room alone costs a
        // resident block per SM, keep only as much of it as still fits the block count of a tight (4 %) fit
        // (30 % for systems of fewer blocks than SMs: their maximum fluctuates more and occupancy does not matter there)
        const int sms = s->sm_count;
        int want = (int)(c.max_stage * (s->P.nblk >= sms ? 1.15 : 1.30)) + 64;
        want = (want + 63) / 64 * 64;
        want = std::min(want, ((int)s->N + 1 + 63) / 64 * 64);   // a neighbourhood never holds more than the whole system
        const size_t per_entry = s->rigid ? 32 : 16, sm_bytes = s->smem_per_sm, xch = s->rigid ? 0 : 24 * MD_TB;
        auto per_block = [&](int se) {
            size_t b = 16 + per_entry * (size_t)se;
            if (b > 75 * 1024) b += xch;
            return b + 1024;
        };
        const int tight = ((int)(c.max_stage * 1.04) + 32 + 63) / 64 * 64;
        const int nb_t = (int)std::min<size_t>(4, sm_bytes / per_block(tight)), nb_w = (int)std::min<size_t>(4, sm_bytes / per_block(want));
        // only where it matters and where the maximum over blocks is statistically stable: at least one block per SM
        if (nb_t == nb_w && nb_w >= 1 && nb_w <= 4 && s->P.nblk >= sms) {
            // head room that costs nothing: up to 30 % if the same number of blocks stays resident
            size_t budget = sm_bytes / nb_w - 1024 - 16;
            if (budget > 75 * 1024 + xch) budget -= xch;
            const int fit = (int)(budget / per_entry) / 64 * 64;
            const int roomy = ((int)(c.max_stage * 1.30) + 64 + 63) / 64 * 64;
            if (fit > want && per_block(std::min(fit, roomy)) * nb_w <= sm_bytes) want = std::min(fit, roomy);
        } else if (nb_t > nb_w && s->P.nblk >= sms) {
            size_t budget = sm_bytes / nb_t - 1024 - 16;
            if (budget > 75 * 1024 + xch) budget -= xch;
            const int fit = (int)(budget / per_entry) / 64 * 64;
            if (fit >= tight && fit < want) want = fit;
        }
        s->stage_launch = want;
    }
    if (c.err & MD_DEVERR_FENE) {
        snprintf(s->errmsg, sizeof(s->errmsg), "FENE bond length reached R0");
        s->forces_valid = false;
        return MD_ERR_NUMERIC;
    }
    return MD_OK;
}

}  // namespace

void md_drop_graphs(md_system* s) { drop_step_graph(s); }

extern "C" {

md_status md_workspace_bytes(int64_t N, const double box[3], double rcut, double skin, const md_potential* pot,
                             int32_t max_neigh, size_t* bytes) {
    Geometry g;
    if (!bytes || !box || !check_pot(pot, rcut) || !make_geometry(N, box, rcut, skin, max_neigh, &g)) return MD_ERR_INVALID;
    *bytes = carve(nullptr, N, g, pot->kind == MD_POT_PATCHY || pot->kind == MD_POT_PATCHY_PP, nullptr);
    return MD_OK;
}

md_status md_create(md_system** out, int64_t N, const double box[3], double rcut, double skin, const md_potential* pot,
                    int32_t max_neigh, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!out) return MD_ERR_INVALID;
    *out = nullptr;
    Geometry g;
    if (!box || !check_pot(pot, rcut) || !make_geometry(N, box, rcut, skin, max_neigh, &g)) return MD_ERR_INVALID;
    const bool rigid = pot->kind == MD_POT_PATCHY || pot->kind == MD_POT_PATCHY_PP;
    size_t need = carve(nullptr, N, g, rigid, nullptr);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < need) return MD_ERR_INVALID;

    md_system* s = (md_system*)calloc(1, sizeof(md_system));
    if (!s) return MD_ERR_INVALID;
    s->N = N;
    s->N_capacity = N;
    s->stream = (cudaStream_t)cuda_stream;
    s->rcut = rcut; s->skin = skin;
    s->pot = *pot;
    s->rigid = rigid;
    s->order = MD_ORDER_NONE;
    s->workspace = workspace; s->workspace_bytes = workspace_bytes;
    s->ecap = g.ecap;
    s->ucap = g.ucap;
    carve((char*)workspace, N, g, rigid, &s->B);

    DevParams& P = s->P;
    P.N = (int)N; P.n_active = (int)N; P.ntiles = g.ntiles; P.cap = g.cap; P.capg = g.cap / 4;
    P.dLx = box[0]; P.dLy = box[1]; P.dLz = box[2];
    P.Lx = (float)box[0]; P.Ly = (float)box[1]; P.Lz = (float)box[2];
    P.hLx = 0.5f * P.Lx; P.hLy = 0.5f * P.Ly; P.hLz = 0.5f * P.Lz;
    const double rv = rcut + skin;
    P.rv2d = rv * rv;
    P.rc2d = rcut * rcut;
    P.ncx = g.nc[0]; P.ncy = g.nc[1]; P.ncz = g.nc[2]; P.ncell = (int)g.ncell;
    P.cscale_x = g.nc[0] / box[0]; P.cscale_y = g.nc[1] / box[1]; P.cscale_z = g.nc[2] / box[2];
    P.rc2 = (float)P.rc2d;
    P.band_abs = (float)(P.rc2d * 1e-6);   // S:H10 band; the fp32 d2 is accurate to ~3e-7 relative
    P.half_skin2 = (float)(0.25 * skin * skin);
    P.rv2 = (float)P.rv2d;
    P.band_rv = (float)(P.rv2d * 1e-6);    // S:Q6 band of the list predicate
    P.nblk = g.nblk; P.rcap = g.rcap; P.mask_words = g.mask_words;
    P.use_masks = ((double)N / (double)g.ncell >= 8.0) ? 1 : 0;
    P.row_schedule = 1;   // measured: masks win at 17.7 particles per cell, lists at 2.5-3
    P.build_direct = 1;
    s->fuse_steps = true;
    P.stage_cap = (int)((224 * 1024 - 16) / (rigid ? 32 : 16)) - 1;
    P.skinf = (float)skin;
    P.shift_margin = (float)(rv + skin);
    s->stage_launch = P.stage_cap;
    s->stage_limit = 0;
    {   // the device the handle lives on: SM count and shared-memory sizes come from its properties, not from literals
        cudaDeviceProp prop;
        if (cudaGetDevice(&s->device) != cudaSuccess || cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) { cudaGetLastError(); free(s); return MD_ERR_CUDA; }
        s->sm_count = prop.multiProcessorCount;
        s->smem_per_sm = prop.sharedMemPerMultiprocessor;
        s->smem_optin = std::min<size_t>(prop.sharedMemPerBlockOptin, 224 * 1024);   // the workspace was sized for <= 224 KB per block
        if (s->smem_optin < 96 * 1024) { free(s); return MD_ERR_INVALID; }            // not a device this library was written for
        P.stage_cap = (int)((s->smem_optin - 16) / (rigid ? 32 : 16)) - 1;
        s->stage_launch = P.stage_cap;
        md_staged_configure(s);
        md_cluster_configure(s);
    }
    P.kind = rigid ? MD_POT_PATCHY : pot->kind;   // both rigid-body models run on the same kernels (P.pp_model tells them apart)
    P.eps = pot->epsilon; P.sig2 = pot->sigma * pot->sigma; P.mass = pot->mass; P.inv_mass = 1.0f / pot->mass;
    P.sigma = pot->sigma;
    P.c48 = 48.0f * pot->epsilon; P.c24 = 24.0f * pot->epsilon; P.c4 = 4.0f * pot->epsilon;
    {
        const double s6 = pow((double)pot->sigma, 6.0), e = pot->epsilon;
        P.lj_a = (float)(48.0 * e * s6 * s6); P.lj_b = (float)(24.0 * e * s6);
        P.lj_c = (float)(4.0 * e * s6 * s6);  P.lj_d = (float)(4.0 * e * s6);
    }
    {
        double s2 = (double)pot->sigma * pot->sigma / (rcut * rcut), s6 = s2 * s2 * s2;
        double vc = 4.0 * pot->epsilon * s6 * (s6 - 1.0);
        bool shift = pot->shift_energy != 0 || pot->kind == MD_POT_FENE_WCA;   // WCA is always shifted (B:9)
        P.vshift = (rigid || !shift) ? 0.0f : (float)vc;
    }
    P.k_nrc2 = make_float2(-P.rc2, -P.rc2); P.k_na = make_float2(-P.lj_a, -P.lj_a); P.k_b = make_float2(P.lj_b, P.lj_b);
    P.k_c = make_float2(P.lj_c, P.lj_c); P.k_nd = make_float2(-P.lj_d, -P.lj_d); P.k_nvs = make_float2(-P.vshift, -P.vshift);
    if (rigid) {
        double rc = pot->rcut_core;
        double s2 = (double)pot->sigma * pot->sigma / (rc * rc), s6 = s2 * s2 * s2;
        P.core_rc2 = (float)(rc * rc);
        P.core_vshift = (float)(4.0 * pot->epsilon * s6 * (s6 - 1.0));
        P.n_patches = pot->n_patches;
        for (int a = 0; a < MD_MAX_PATCH; ++a)
            for (int k = 0; k < 3; ++k) P.pdir[a][k] = a < pot->n_patches ? pot->patch_dir[a][k] : 0.0f;
        {   // config 4's patch set (S:O4): b_1..b_4 = (1,1,1), (1,-1,-1), (-1,1,-1), (-1,-1,1) / sqrt(3), in this order
            static const float tet[4][3] = { { 1, 1, 1 }, { 1, -1, -1 }, { -1, 1, -1 }, { -1, -1, 1 } };
            P.tetra = pot->n_patches == 4 ? 1 : 0;
            for (int a = 0; a < 4 && P.tetra; ++a)
                for (int k = 0; k < 3; ++k)
                    if (fabsf(pot->patch_dir[a][k] - tet[a][k] * 0.57735026918962576f) > 1e-6f) P.tetra = 0;
        }
        P.eps_patch = pot->eps_patch;
        P.inv_sr2 = 1.0f / (pot->patch_sigma_r * pot->patch_sigma_r);
        P.inv_2sr2 = 0.5f * P.inv_sr2;
        P.inv_w2 = 1.0f / (pot->patch_sigma_ang * pot->patch_sigma_ang);
        P.inv_inertia = 1.0f / pot->inertia;
        P.pp_model = pot->kind == MD_POT_PATCHY_PP ? 1 : 0;
        if (P.pp_model) {
            P.pp_core_half = (int)(pot->core_exponent / 2); P.pp_half_n = (int)(pot->patch_exponent / 2);
            P.pp_core_n = pot->core_exponent; P.pp_n = pot->patch_exponent;
            P.pp_radius = pot->patch_radius;
            P.pp_inv_w2 = 1.0f / (pot->patch_sigma_r * pot->patch_sigma_r);
            P.pp_rc2 = pot->rcut_patch * pot->rcut_patch;
        }
    }
    if (pot->kind == MD_POT_FENE_WCA) {
        P.fene_K = pot->fene_K;
        P.fene_R02 = pot->fene_R0 * pot->fene_R0;
        P.fene_invR02 = 1.0f / P.fene_R02;
        P.chain_len = pot->chain_len;
    } else {
        P.chain_len = 1;
    }

    // device-side initial state: control block zero, ids = identity, cell rank table
    cudaMemsetAsync(s->B.ctrl, 0, sizeof(DevCtrl), s->stream);
    {
        reset_ids(s);
        std::vector<int> rank;
        make_cell_rank(g.nc, MD_ORDER_NONE, rank);
        upload_cell_rank(s, rank);
    }
    if (check_cuda(s, "md_create") != MD_OK) { free(s); return MD_ERR_CUDA; }
    *out = s;
    return MD_OK;
}

md_status md_bind_state(md_system* s, void* pos, void* vel, void* force, void* quat, void* angmom, void* torque) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!pos || !vel || !force) return fail(s, MD_ERR_INVALID, "md_bind_state: pos, vel and force are required");
    if (s->rigid && (!quat || !angmom || !torque)) return fail(s, MD_ERR_INVALID, "md_bind_state: rigid bodies need quat, angmom and torque");
    void* all[6] = { pos, vel, force, quat, angmom, torque };
    for (int k = 0; k < 6; ++k)
        if (all[k] && ((uintptr_t)all[k] & 15)) return fail(s, MD_ERR_INVALID, "md_bind_state: pointers must be 16-byte aligned");
    s->pos = (float4*)pos; s->vel = (float4*)vel; s->force = (float4*)force;
    s->quat = s->rigid ? (float4*)quat : nullptr;
    s->angmom = s->rigid ? (float4*)angmom : nullptr;
    s->torque = s->rigid ? (float4*)torque : nullptr;
    s->bound = true;
    s->shadow_valid = false;
    s->cells_valid = s->lists_valid = s->forces_valid = s->seg_valid = s->staged_valid = s->legacy_valid = s->cluster_valid = false;
    drop_step_graph(s);   // the step graph bakes the state pointers in
    reset_ids(s);   // the arrays are taken to be in original id order
    return check_cuda(s, "md_bind_state");
}

md_status md_set_order(md_system* s, int32_t order) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (order < MD_ORDER_NONE || order > MD_ORDER_HILBERT) return fail(s, MD_ERR_INVALID, "md_set_order: unknown order");
    s->order = order;
    drop_step_graph(s);
    std::vector<int> rank;
    int nc[3] = { s->P.ncx, s->P.ncy, s->P.ncz };
    make_cell_rank(nc, order, rank);
    upload_cell_rank(s, rank);
    s->cells_valid = s->lists_valid = s->seg_valid = s->staged_valid = s->legacy_valid = s->cluster_valid = false;
    return check_cuda(s, "md_set_order");
}

// mixed precision: the fp64 copies are taken from the bound fp32 arrays the first time they are needed after a bind
static void ensure_shadows(md_system* s) {
    if (s->precision != MD_PREC_MIXED || s->shadow_valid) return;
    md_launch_shadow_init(s);
    s->shadow_valid = true;
}

md_status md_set_precision(md_system* s, int32_t precision) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (precision != MD_PREC_F32 && precision != MD_PREC_MIXED) return fail(s, MD_ERR_INVALID, "md_set_precision: unknown precision");
    if (precision == MD_PREC_MIXED && s->P.n_active < s->P.N) return fail(s, MD_ERR_STATE, "md_set_precision: ghosts (md_set_active) need MD_PREC_F32");
    if (precision != s->precision) {
        s->precision = precision;
        s->shadow_valid = false;
        drop_step_graph(s);   // the step graph bakes the integration kernels in
    }
    return MD_OK;
}

md_status md_get_state_double(md_system* s, double* pos_host, double* vel_host) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (s->precision != MD_PREC_MIXED || !s->bound || !s->shadow_valid)
        return fail(s, MD_ERR_STATE, "md_get_state_double: needs MD_PREC_MIXED and a bound state that md_build_cells or md_integrate has seen");
    const size_t n = (size_t)s->N;
    std::vector<double> plane(2 * n);
    std::vector<int> ids(n);
    cudaMemcpyAsync(ids.data(), s->B.ids, 4 * n, cudaMemcpyDeviceToHost, s->stream);
    md_status st = sync_and_check(s, "md_get_state_double");
    if (st != MD_OK) return st;
    double* outs[2] = { pos_host, vel_host };
    for (int a = 0; a < 2; ++a) {
        if (!outs[a]) continue;
        for (int h = 0; h < 2; ++h) {   // plane 2a: (x, y), plane 2a+1: (z, -)
            cudaMemcpyAsync(plane.data(), s->B.shadow[2 * a + h], 16 * n, cudaMemcpyDeviceToHost, s->stream);
            if ((st = sync_and_check(s, "md_get_state_double")) != MD_OK) return st;
            for (size_t i = 0; i < n; ++i) {
                double* o = outs[a] + 3 * (size_t)ids[i];
                if (h == 0) { o[0] = plane[2 * i]; o[1] = plane[2 * i + 1]; }
                else o[2] = plane[2 * i];
            }
        }
    }
    return MD_OK;
}

md_status md_build_cells(md_system* s) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->bound) return fail(s, MD_ERR_STATE, "md_build_cells: no state bound");
    ensure_shadows(s);
    md_launch_build_cells(s, false);
    s->cells_valid = true;
    s->lists_valid = s->seg_valid = s->staged_valid = s->legacy_valid = s->cluster_valid = false;
    return check_cuda(s, "md_build_cells");
}

md_status md_build_verlet(md_system* s) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->bound || !s->cells_valid) return fail(s, MD_ERR_STATE, "md_build_verlet: call md_build_cells first");
    s->staged_valid = s->legacy_valid = s->seg_valid = s->cluster_valid = false;
    if (s->order != MD_ORDER_NONE) {
        // cell-sorted storage: rows of block-local indices (md_staged.cu); the explicit global-slot lists of the
        // L2-gather variants are derived lazily from the same cells and the build-time positions (ensure_explicit)
        md_launch_build_staged(s, false);
        md_launch_build_end(s, false);
        s->lists_valid = true;
        md_status st = sync_and_check(s, "md_build_verlet");   // reads the largest staged neighbourhood: sizes the launches
        if (st != MD_OK) { s->lists_valid = false; return st; }
        s->staged_valid = true;
    } else {
        md_launch_build_verlet(s, false, s->pos);
        md_launch_build_end(s, false);
        s->lists_valid = true;
        s->legacy_valid = true;
    }
    s->cells_valid = false;   // cells describe the positions at build time only
    return check_cuda(s, "md_build_verlet");
}

// The explicit lists (tile-transposed full list + (i, j) edge list) for the current build.  The cell arrays still
// describe the build-time positions kept in pos_ref (no md_build_cells since), so the lists can be made on demand.
static void ensure_explicit(md_system* s) {
    if (s->legacy_valid) return;
    md_launch_build_verlet(s, false, s->B.pos_ref);
    s->legacy_valid = true;
    s->seg_valid = false;
}

// The (cluster, j) unit list of MD_SCATTER_CLUSTER for the current build, made on demand like the explicit lists.
static md_status ensure_cluster(md_system* s) {
    if (s->cluster_valid) return MD_OK;
    // (the build recounts E from its own units and rewrites the list counters: they must come out the same)
    if (!md_launch_build_cluster(s, false, s->B.pos_ref)) return fail(s, MD_ERR_CAPACITY, "MD_SCATTER_CLUSTER: max_neigh too large for the cluster build's shared memory");
    s->cluster_valid = true;
    return MD_OK;
}

static bool wants_cluster(int32_t strategy, int32_t variant) { return strategy == MD_EDGE && variant == MD_SCATTER_CLUSTER; }

// which list representation a (strategy, variant) pair runs on
static bool wants_staged(const md_system* s, int32_t strategy, int32_t variant) {
    if (s->order == MD_ORDER_NONE) return false;
    return strategy == MD_VERTEX && variant != MD_GATHER_L2;
}

static md_status check_strategy(md_system* s, int32_t strategy, int32_t scatter) {
    if (strategy != MD_VERTEX && strategy != MD_EDGE && strategy != MD_VERTEX_N3) return fail(s, MD_ERR_INVALID, "unknown strategy");
    if (strategy == MD_VERTEX_N3) {
        const int64_t m = scatter == 0 ? 12 : scatter;
        if (scatter < 0 || m > 64) return fail(s, MD_ERR_INVALID, "MD_VERTEX_N3: the number of force copies m must be 1..64 (0 = 12)");
        if ((size_t)(m * s->N) > s->ecap) return fail(s, MD_ERR_INVALID, "MD_VERTEX_N3: m * N exceeds the edge capacity N * max_neigh / 2");
        return MD_OK;
    }
    if (strategy == MD_EDGE && (scatter < MD_SCATTER_RED || scatter > MD_SCATTER_CLUSTER)) return fail(s, MD_ERR_INVALID, "unknown scatter variant");
    if (strategy == MD_VERTEX && (scatter < MD_GATHER_AUTO || scatter > MD_GATHER_SMEM)) return fail(s, MD_ERR_INVALID, "unknown gather variant");
    if (s->order == MD_ORDER_NONE && strategy == MD_VERTEX && scatter == MD_GATHER_SMEM)
        return fail(s, MD_ERR_STATE, "the shared-memory staged variant needs cell-sorted storage: md_set_order(MD_ORDER_CELL or MD_ORDER_HILBERT)");
    return MD_OK;
}

// energy = false: nobody can observe force.w of this evaluation (an inner step of a multi-step graph)
static md_status launch_forces_any(md_system* s, int32_t strategy, int32_t scatter, bool energy = true) {
    if (wants_staged(s, strategy, scatter)) {
        if (!md_launch_forces_staged(s, energy)) return fail(s, MD_ERR_CAPACITY, "staged neighbourhood does not fit in shared memory");
    } else {
        md_launch_forces(s, strategy, scatter);
    }
    return MD_OK;
}

// One step of md_integrate captured as a graph.  The rebuild chain (cells, reordering, Verlet rows, bookkeeping) sits
// in the body of a conditional IF node: when the skin flag is clear it costs nothing, where the plain-launch path pays
// a dozen gated no-op kernels per step.  Returns false (and leaves no graph) if any graph call fails.
#define GCHK(call) do { if (ok) { cudaError_t e_ = (call); if (e_ != cudaSuccess) { ok = false; \
    snprintf(s->errmsg, sizeof(s->errmsg), "step graph: %s -> %s", #call, cudaGetErrorString(e_)); \
    if (s->debug) fprintf(stderr, "%s\n", s->errmsg); } } } while (0)
static bool build_step_graph(md_system* s, float fdt, int32_t strategy, int32_t scatter, bool staged, bool seg, int reps,
                             cudaGraphExec_t* exec_out, int* nodes_out) {
    // capture happens on two internal streams (the caller's stream may be the legacy default stream, which cannot be
    // captured); the instantiated graph is launched on the caller's stream
    if (!s->aux_stream && cudaStreamCreateWithFlags(&s->aux_stream, cudaStreamNonBlocking) != cudaSuccess) return false;
    if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return false;
    const int64_t launches0 = s->launches;
    cudaStream_t user_stream = s->stream;
    cudaStream_t main_stream = s->cap_stream;
    s->stream = main_stream;
    cudaGraph_t graph = nullptr;
    bool ok = true;
    GCHK(cudaStreamBeginCapture(main_stream, cudaStreamCaptureModeRelaxed));
    if (!ok) { cudaGetLastError(); s->stream = user_stream; return false; }
    cudaStreamCaptureStatus st;
    cudaGraph_t cg = nullptr;
    const cudaGraphNode_t* deps = nullptr;
    size_t ndeps = 0;
    int tail_nodes = 0, main_nodes = 0;
    bool aux_open = false;
    // Fused step tails (multi-step graphs, staged LJ / FENE VERTEX, fp32, no ghosts): the force kernel of an inner step applies
    // the kicks and the drift of the next step itself (FuseArgs), so steps 2..reps have no kick+drift kernel and no force
    // store.  The new positions go to the other of two position arrays (the caller's and plane 6 of the permutation
    // scratch); with the opening kick+drift of step 1 also written across there are `reps` (even) switches per graph and
    // the state ends in the caller's array.  The rebuild chain of a step is captured on the array that is current there.
    float4* const pos_user = s->pos;
    float4* const pos_alt = s->B.tmp4 + (size_t)6 * s->P.ntiles * MD_TILE;
    const bool fuse = s->fuse_steps && reps > 1 && reps % 2 == 0 && staged && !s->rigid && s->precision != MD_PREC_MIXED &&
                      s->P.n_active >= s->P.N;
    float4* cur = pos_user;
    for (int rep_i = 0; rep_i < reps && ok; ++rep_i) {   // `reps` consecutive steps in one graph, one IF node each
    cudaGraphConditionalHandle handle = 0;
    GCHK(cudaStreamGetCaptureInfo(main_stream, &st, nullptr, &cg, &deps, &ndeps));
    GCHK(cudaGraphConditionalHandleCreate(&handle, cg, 0, cudaGraphCondAssignDefault));
    if (ok) {
        if (!fuse) md_launch_kick_drift(s, fdt, rep_i > 0);   // sets the device rebuild flag (S:A5); carries the previous step's closing kick
        else if (rep_i == 0) { float4* other = cur == pos_user ? pos_alt : pos_user; md_launch_kick_drift_to(s, fdt, other); cur = other; }
        s->pos = cur;                              // everything below reads (and the rebuild permutes) the current array
        md_launch_set_cond(s, handle);
        GCHK(cudaStreamGetCaptureInfo(main_stream, &st, nullptr, &cg, &deps, &ndeps));
    }
    cudaGraphNode_t cond_node = nullptr;
    if (ok) {
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = handle;
        np.conditional.type = cudaGraphCondTypeIf;
        np.conditional.size = 1;
        GCHK(cudaGraphAddNode(&cond_node, cg, deps, ndeps, &np));
        if (ok) {
            cudaGraph_t body = np.conditional.phGraph_out[0];
            GCHK(cudaStreamBeginCaptureToGraph(s->aux_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
            if (ok) {
                aux_open = true;
                s->stream = s->aux_stream;
                md_launch_build_cells(s, true);
                if (staged) md_launch_build_staged(s, true);
                else if (wants_cluster(strategy, scatter)) md_launch_build_cluster(s, true, s->pos);
                else md_launch_build_verlet(s, true, s->pos);
                if (seg) md_launch_seg_index(s, true);
                md_launch_build_end(s, true);
                s->stream = main_stream;
                cudaGraph_t tmp = nullptr;
                aux_open = false;       // ended here whatever the outcome
                { cudaError_t e_ = cudaStreamEndCapture(s->aux_stream, &tmp); if (e_ != cudaSuccess && ok) { ok = false;
                    snprintf(s->errmsg, sizeof(s->errmsg), "step graph: end of body capture -> %s", cudaGetErrorString(e_)); } }
            }
        }
        GCHK(cudaStreamUpdateCaptureDependencies(main_stream, &cond_node, 1, cudaStreamSetCaptureDependencies));
    }
    const int64_t before_tail = s->launches;
    if (ok) {
        if (fuse && rep_i < reps - 1) {
            float4* other = cur == pos_user ? pos_alt : pos_user;
            ok = md_launch_forces_staged(s, false, FuseArgs{ s->vel, other, fdt });
            cur = other;
        } else {
            ok = launch_forces_any(s, strategy, scatter, rep_i == reps - 1) == MD_OK;   // md_energy sees the last step only
        }
        if (rep_i == reps - 1) md_launch_kick(s, fdt);   // inner steps: fused into the next kick+drift
    }
    tail_nodes = (int)(s->launches - before_tail);
    main_nodes += ((fuse && rep_i > 0) ? 1 : 2) + tail_nodes;   // kernels outside the conditional body
    }
    s->pos = pos_user;
    if (fuse && cur != pos_user) ok = false;       // (cannot happen: reps is even)
    if (aux_open) {   // a failure while the body capture was open: close it, or aux_stream stays in capture mode for good
        cudaGraph_t tmp = nullptr;
        cudaStreamEndCapture(s->aux_stream, &tmp);
        aux_open = false;
    }
    { cudaError_t e_ = cudaStreamEndCapture(main_stream, &graph); if (e_ != cudaSuccess) { if (ok && s->debug) fprintf(stderr, "step graph: end capture -> %s\n", cudaGetErrorString(e_)); ok = false; } }
    s->launches = launches0;
    s->stream = user_stream;
    GCHK(cudaGraphInstantiate(exec_out, graph, 0));
    if (graph) cudaGraphDestroy(graph);
    if (!ok) { cudaGetLastError(); drop_step_graph(s); return false; }
    s->step_strategy = strategy; s->step_variant = scatter; s->step_dt = fdt; s->step_dt_d = s->dt_d; s->step_stage = s->stage_launch;
    *nodes_out = main_nodes;
    return true;
}

md_status md_forces(md_system* s, int32_t strategy, int32_t scatter) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->bound || !s->lists_valid) return fail(s, MD_ERR_STATE, "md_forces: lists are not built (md_build_cells, md_build_verlet)");
    md_status st = check_strategy(s, strategy, scatter);
    if (st != MD_OK) return st;
    if (wants_staged(s, strategy, scatter)) {
        if (!s->staged_valid) return fail(s, MD_ERR_STATE, "md_forces: staged lists are not valid, call md_build_cells + md_build_verlet");
    } else if (wants_cluster(strategy, scatter)) {
        if ((st = ensure_cluster(s)) != MD_OK) return st;
    } else {
        ensure_explicit(s);
        if (strategy == MD_EDGE && scatter == MD_SCATTER_SEGMENTED && !s->seg_valid) {
            md_launch_seg_index(s, false);
            s->seg_valid = true;
        }
    }
    if ((st = launch_forces_any(s, strategy, scatter)) != MD_OK) return st;
    s->forces_valid = true;
    return check_cuda(s, "md_forces");
}

md_status md_set_thermostat(md_system* s, double T, int64_t n_newt, double p_trans, double p_rot, uint64_t seed) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (n_newt < 0 || (n_newt > 0 && (!(T > 0) || !(p_trans >= 0 && p_trans <= 1) || !(p_rot >= 0 && p_rot <= 1))))
        return fail(s, MD_ERR_INVALID, "md_set_thermostat: n_newt >= 0, T > 0 and probabilities in [0, 1] required");
    s->thermo_n = n_newt; s->thermo_steps = 0;
    s->thermo_T = T; s->thermo_pt = p_trans; s->thermo_pr = p_rot; s->thermo_seed = seed;
    return MD_OK;
}

md_status md_thermostat(md_system* s, double T, double p_trans, double p_rot, uint64_t seed, uint32_t call) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->bound) return fail(s, MD_ERR_STATE, "md_thermostat: no state bound");
    if (!(T > 0) || !(p_trans >= 0 && p_trans <= 1) || !(p_rot >= 0 && p_rot <= 1))
        return fail(s, MD_ERR_INVALID, "md_thermostat: T > 0 and probabilities in [0, 1] required");
    ensure_shadows(s);
    md_launch_thermostat(s, T, p_trans, p_rot, seed, call);
    return check_cuda(s, "md_thermostat");
}

static md_status integrate_nve(md_system* s, double dt, int64_t nsteps, int32_t strategy, int32_t scatter);

// NVE velocity-Verlet (B:5), with the thermostat of reading QT after every thermo_n-th step when it is set
md_status md_integrate(md_system* s, double dt, int64_t nsteps, int32_t strategy, int32_t scatter) {
    if (!s) return MD_ERR_INVALID;
    if (s->thermo_n <= 0 || nsteps <= 0) return integrate_nve(s, dt, nsteps, strategy, scatter);
    int64_t done = 0;
    while (done < nsteps) {
        const int64_t to_next = s->thermo_n - s->thermo_steps % s->thermo_n;
        const int64_t chunk = to_next < nsteps - done ? to_next : nsteps - done;
        md_status st = integrate_nve(s, dt, chunk, strategy, scatter);
        if (st != MD_OK) return st;
        s->thermo_steps += chunk; done += chunk;
        if (s->thermo_steps % s->thermo_n == 0)
            md_launch_thermostat(s, s->thermo_T, s->thermo_pt, s->thermo_pr, s->thermo_seed, (unsigned int)(s->thermo_steps / s->thermo_n));
    }
    return check_cuda(s, "md_integrate");
}

static md_status integrate_nve(md_system* s, double dt, int64_t nsteps, int32_t strategy, int32_t scatter) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->bound || !s->lists_valid || !s->forces_valid) return fail(s, MD_ERR_STATE, "md_integrate: needs built lists and valid forces on entry");
    if (!(dt > 0) || nsteps < 0) return fail(s, MD_ERR_INVALID, "md_integrate: dt > 0 and nsteps >= 0 required");
    md_status st = check_strategy(s, strategy, scatter);
    if (st != MD_OK) return st;
    const bool staged = wants_staged(s, strategy, scatter);
    const bool seg = strategy == MD_EDGE && scatter == MD_SCATTER_SEGMENTED;
    if (staged && !s->staged_valid) return fail(s, MD_ERR_STATE, "md_integrate: staged lists are not valid, call md_build_cells + md_build_verlet");
    const bool cluster = wants_cluster(strategy, scatter);
    if (cluster) { if ((st = ensure_cluster(s)) != MD_OK) return st; }
    else if (!staged) ensure_explicit(s);
    if (seg && !s->seg_valid) { md_launch_seg_index(s, false); s->seg_valid = true; }
    const float fdt = (float)dt;
    s->dt_d = dt;
    ensure_shadows(s);
    int64_t k0 = 0;
    if (!s->graphs_off && !s->no_graph && nsteps > 0) {   // MD_OPT_NO_GRAPH: plain launches (profilers list every kernel)
        if (!s->step_exec || s->step_strategy != strategy || s->step_variant != scatter || s->step_dt != fdt ||
            s->step_dt_d != dt || s->step_stage != s->stage_launch) {
            drop_step_graph(s);
            if (!build_step_graph(s, fdt, strategy, scatter, staged, seg, 1, &s->step_exec, &s->step_nodes) ||
                !build_step_graph(s, fdt, strategy, scatter, staged, seg, 2, &s->pair_exec, &s->pair_nodes) ||
                !build_step_graph(s, fdt, strategy, scatter, staged, seg, 4, &s->quad_exec, &s->quad_nodes) ||
                !build_step_graph(s, fdt, strategy, scatter, staged, seg, 8, &s->oct_exec, &s->oct_nodes) ||
                !build_step_graph(s, fdt, strategy, scatter, staged, seg, MD_GRAPH_STEPS, &s->multi_exec, &s->multi_nodes)) s->graphs_off = true;
        }
        if (s->step_exec && s->pair_exec && s->quad_exec && s->oct_exec && s->multi_exec) {
            while (k0 < nsteps) {      // MD_GRAPH_STEPS steps per launch while they fit, then 8, 4, 2, 1 for the rest
                const int64_t left = nsteps - k0;
                const int reps = left >= MD_GRAPH_STEPS ? MD_GRAPH_STEPS : left >= 8 ? 8 : left >= 4 ? 4 : left >= 2 ? 2 : 1;
                cudaGraphExec_t ex = reps == MD_GRAPH_STEPS ? s->multi_exec : reps == 8 ? s->oct_exec : reps == 4 ? s->quad_exec : reps == 2 ? s->pair_exec : s->step_exec;
                if (cudaGraphLaunch(ex, s->stream) != cudaSuccess) break;
                k0 += reps;
                s->launches += reps == MD_GRAPH_STEPS ? s->multi_nodes : reps == 8 ? s->oct_nodes : reps == 4 ? s->quad_nodes : reps == 2 ? s->pair_nodes : s->step_nodes;
            }
        }
    }
    for (int64_t k = k0; k < nsteps; ++k) {
        md_launch_kick_drift(s, fdt, false);     // sets the device rebuild flag (S:A5)
        md_launch_build_cells(s, true);          // gated on the flag: no host synchronisation (S:H6)
        if (staged) md_launch_build_staged(s, true);
        else if (cluster) md_launch_build_cluster(s, true, s->pos);
        else md_launch_build_verlet(s, true, s->pos);
        if (seg) md_launch_seg_index(s, true);
        md_launch_build_end(s, true);
        if ((st = launch_forces_any(s, strategy, scatter)) != MD_OK) return st;
        md_launch_kick(s, fdt);
    }
    if (nsteps > 0) {
        // a device-side rebuild may have replaced the lists of the representation in use; the other one is stale
        if (staged) { s->legacy_valid = false; s->seg_valid = false; s->cluster_valid = false; }
        else if (cluster) { s->legacy_valid = false; s->seg_valid = false; s->staged_valid = false; }
        else { s->staged_valid = false; s->cluster_valid = false; if (!seg) s->seg_valid = false; }
        s->cells_valid = false;
    }
    return check_cuda(s, "md_integrate");
}

md_status md_energy(md_system* s, double* e_pot, double* e_kin_trans, double* e_kin_rot) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->bound || !s->forces_valid) return fail(s, MD_ERR_STATE, "md_energy: needs valid forces (md_forces)");
    md_launch_energy(s);
    double e[3];
    cudaMemcpyAsync(e, s->B.e_out, sizeof(e), cudaMemcpyDeviceToHost, s->stream);
    md_status st = sync_and_check(s, "md_energy");
    if (st != MD_OK) return st;
    if (e_pot) *e_pot = e[0];
    if (e_kin_trans) *e_kin_trans = e[1];
    if (e_kin_rot) *e_kin_rot = s->rigid ? e[2] : 0.0;
    return MD_OK;
}

md_status md_stats(md_system* s, int64_t* n_edges, int64_t* n_full_entries, int32_t* max_neigh_seen, int64_t* n_rebuilds) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    DevCtrl c;
    cudaMemcpyAsync(&c, s->B.ctrl, sizeof(c), cudaMemcpyDeviceToHost, s->stream);
    md_status st = sync_and_check(s, "md_stats");
    if (n_edges) *n_edges = c.n_edges;
    if (n_full_entries) *n_full_entries = (int64_t)c.n_full;
    if (max_neigh_seen) *max_neigh_seen = c.max_seen;
    if (n_rebuilds) *n_rebuilds = c.n_rebuilds;
    return st;
}

md_status md_stats_ex(md_system* s, md_stats_ex_t* out, size_t bytes) {
    if (!s || !out || bytes == 0) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    const bool have_lists = s->bound && s->lists_valid;
    if (have_lists) {
        ensure_explicit(s);
        md_launch_count_in_cutoff(s);
    }
    DevCtrl c;
    cudaMemcpyAsync(&c, s->B.ctrl, sizeof(c), cudaMemcpyDeviceToHost, s->stream);
    md_status st = sync_and_check(s, "md_stats_ex");
    md_stats_ex_t r;
    memset(&r, 0, sizeof(r));
    r.n_edges = c.n_edges; r.n_full_entries = (int64_t)c.n_full; r.n_rebuilds = c.n_rebuilds;
    r.n_in_cutoff = have_lists ? (int64_t)c.n_in : -1;
    r.max_neigh_seen = c.max_seen; r.max_stage = c.max_stage; r.stage_launch = s->stage_launch;
    r.threads_per_particle = s->staged_valid ? md_staged_threads_per_particle(s) : 0;
    r.cluster_size = s->cluster_valid ? MD_CLUSTER : 0;
    r.n_cluster_units = s->cluster_valid ? (int64_t)c.n_units : 0;
    memcpy(out, &r, bytes < sizeof(r) ? bytes : sizeof(r));
    return st;
}

md_status md_set_option(md_system* s, int32_t option, int64_t value) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (value < 0) return fail(s, MD_ERR_INVALID, "md_set_option: negative value");
    switch (option) {
    case MD_OPT_STAGE_LIMIT:
        s->stage_limit = (int)std::min<int64_t>(value, 1 << 30);
        drop_step_graph(s);            // the step graph bakes the launch capacity in
        return MD_OK;
    case MD_OPT_NO_GRAPH: s->no_graph = value != 0; return MD_OK;
    case MD_OPT_ROW_SCHEDULE:
        s->P.row_schedule = value != 0 ? 1 : 0;
        drop_step_graph(s);            // the graph bakes the parameter block in
        s->lists_valid = s->staged_valid = s->legacy_valid = s->seg_valid = s->cluster_valid = false;
        return MD_OK;
    case MD_OPT_FUSE_STEPS:
        s->fuse_steps = value != 0;
        drop_step_graph(s);
        return MD_OK;
    case MD_OPT_BUILD_DIRECT:
        s->P.build_direct = value != 0 ? 1 : 0;
        drop_step_graph(s);
        s->lists_valid = s->staged_valid = s->legacy_valid = s->seg_valid = s->cluster_valid = false;
        return MD_OK;
    case MD_OPT_DEBUG: s->debug = value != 0; return MD_OK;
    default: return fail(s, MD_ERR_INVALID, "md_set_option: unknown option");
    }
}

md_status md_probe(md_system* s, int32_t kind, double* value) {
    if (!s || !value) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (kind < MD_PROBE_FFMA || kind > MD_PROBE_RED_F32_COALESCED) return fail(s, MD_ERR_INVALID, "md_probe: unknown kind");
    cudaStreamSynchronize(s->stream);
    if (!md_run_probe(s, kind, value)) {
        md_status st = check_cuda(s, "md_probe");
        return st != MD_OK ? st : fail(s, MD_ERR_INVALID, "md_probe: the system is too small to hold the probe's scratch");
    }
    s->launches += 4;
    return check_cuda(s, "md_probe");
}

md_status md_rebuild_flag(md_system* s, int32_t* flag) {
    if (!s || !flag) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    DevCtrl c;
    cudaMemcpyAsync(&c, s->B.ctrl, sizeof(c), cudaMemcpyDeviceToHost, s->stream);
    md_status st = sync_and_check(s, "md_rebuild_flag");
    *flag = c.rebuild != 0 ? 1 : 0;
    return st;
}

md_status md_get_ids(md_system* s, int32_t* ids_host) {
    if (!s || !ids_host) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    cudaMemcpyAsync(ids_host, s->B.ids, 4 * (size_t)s->N, cudaMemcpyDeviceToHost, s->stream);
    cudaStreamSynchronize(s->stream);
    return check_cuda(s, "md_get_ids");
}

md_status md_get_pairs(md_system* s, int32_t* pairs_host, int64_t capacity, int64_t* n) {
    if (!s || !n) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->lists_valid) return fail(s, MD_ERR_STATE, "md_get_pairs: lists are not built");
    if (s->staged_valid && !s->legacy_valid) {   // export what the staged kernels use: rows -> explicit (i, j) pairs
        md_launch_edge_offsets(s, false);
        md_launch_edges_from_rows(s);
        s->seg_valid = false;                     // the edge array now follows the row order, not the explicit build
    }
    DevCtrl c;
    cudaMemcpyAsync(&c, s->B.ctrl, sizeof(c), cudaMemcpyDeviceToHost, s->stream);
    md_status st = sync_and_check(s, "md_get_pairs");
    if (st != MD_OK) return st;
    *n = c.n_edges;
    int64_t m = std::min<int64_t>(capacity, c.n_edges);
    if (m <= 0 || !pairs_host) return MD_OK;
    std::vector<int> ids((size_t)s->N);
    cudaMemcpyAsync(ids.data(), s->B.ids, 4 * (size_t)s->N, cudaMemcpyDeviceToHost, s->stream);
    cudaMemcpyAsync(pairs_host, s->B.edges, 8 * (size_t)m, cudaMemcpyDeviceToHost, s->stream);
    cudaStreamSynchronize(s->stream);
    for (int64_t e = 0; e < m; ++e) {   // slots -> original ids, (lo, hi); drop the image flag
        int a = ids[(size_t)pairs_host[2 * e]];
        int b = ids[(size_t)(pairs_host[2 * e + 1] & 0x7fffffff)];
        pairs_host[2 * e] = a < b ? a : b;
        pairs_host[2 * e + 1] = a < b ? b : a;
    }
    return check_cuda(s, "md_get_pairs");
}

md_status md_step_host(md_system* s, void* pos_host, void* vel_host, void* force_host, void* quat_host, void* angmom_host,
                       void* torque_host, double dt, int64_t nsteps, int32_t strategy, int32_t scatter) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->bound) return fail(s, MD_ERR_STATE, "md_step_host: no state bound");
    if (!pos_host || !vel_host || !force_host) return fail(s, MD_ERR_INVALID, "md_step_host: pos, vel, force host buffers required");
    if (s->rigid && (!quat_host || !angmom_host || !torque_host)) return fail(s, MD_ERR_INVALID, "md_step_host: rigid bodies need quat, angmom, torque");
    md_status st = check_strategy(s, strategy, scatter);
    if (st != MD_OK) return st;
    const size_t bytes = 16 * (size_t)s->N;
    reset_ids(s);   // host buffers are in ORIGINAL id order
    s->shadow_valid = false;
    // Cells and lists need the positions only: velocities (and angular momenta) are uploaded on a second stream, into free
    // planes of the permutation scratch, while the lists are built, and enter the slot order afterwards through ids[].
    const size_t plane_in = (size_t)s->P.ntiles * MD_TILE;
    float4* const vel_in = s->B.tmp4 + (size_t)(s->rigid ? 12 : 6) * plane_in;
    float4* const ang_in = s->B.tmp4 + (size_t)13 * plane_in;     // rigid bodies only (14 planes)
    bool split = s->order != MD_ORDER_NONE;
    if (split && !s->aux_stream && cudaStreamCreateWithFlags(&s->aux_stream, cudaStreamNonBlocking) != cudaSuccess) split = false;
    if (split && !s->ev_in && (cudaEventCreateWithFlags(&s->ev_in, cudaEventDisableTiming) != cudaSuccess ||
                               cudaEventCreateWithFlags(&s->ev_vel, cudaEventDisableTiming) != cudaSuccess)) split = false;
    if (!split) cudaGetLastError();
    cudaMemcpyAsync(s->pos, pos_host, bytes, cudaMemcpyHostToDevice, s->stream);
    if (split) {
        cudaEventRecord(s->ev_in, s->stream);                       // the scratch planes are free once earlier work has drained
        cudaStreamWaitEvent(s->aux_stream, s->ev_in, 0);
        cudaMemcpyAsync(vel_in, vel_host, bytes, cudaMemcpyHostToDevice, s->aux_stream);
        if (s->rigid) cudaMemcpyAsync(ang_in, angmom_host, bytes, cudaMemcpyHostToDevice, s->aux_stream);
        cudaEventRecord(s->ev_vel, s->aux_stream);
    } else {
        cudaMemcpyAsync(s->vel, vel_host, bytes, cudaMemcpyHostToDevice, s->stream);
        if (s->rigid) cudaMemcpyAsync(s->angmom, angmom_host, bytes, cudaMemcpyHostToDevice, s->stream);
    }
    if (s->rigid) cudaMemcpyAsync(s->quat, quat_host, bytes, cudaMemcpyHostToDevice, s->stream);
    if ((st = md_build_cells(s)) != MD_OK) return st;
    if ((st = md_build_verlet(s)) != MD_OK) return st;
    if (split) {
        cudaStreamWaitEvent(s->stream, s->ev_vel, 0);
        md_launch_permute_in(s, vel_in, s->vel);
        if (s->rigid) md_launch_permute_in(s, ang_in, s->angmom);
    }
    if ((st = md_forces(s, strategy, scatter)) != MD_OK) return st;
    if (nsteps > 0 && (st = md_integrate(s, dt, nsteps, strategy, scatter)) != MD_OK) return st;
    struct { float4* dev; void* host; } outs[6] = { { s->pos, pos_host }, { s->vel, vel_host }, { s->force, force_host },
                                                    { s->quat, quat_host }, { s->angmom, angmom_host }, { s->torque, torque_host } };
    // back to ORIGINAL id order: every array goes through its own plane of the permutation scratch, so the un-permute
    // kernels and the device->host copies queue back to back with no dependency between arrays
    const size_t plane = (size_t)s->P.ntiles * MD_TILE;
    for (int k = 0; k < 6; ++k) {
        if (!outs[k].dev || !outs[k].host) continue;
        if (s->order == MD_ORDER_NONE) {
            cudaMemcpyAsync(outs[k].host, outs[k].dev, bytes, cudaMemcpyDeviceToHost, s->stream);
        } else {
            md_launch_unpermute(s, outs[k].dev, s->B.tmp4 + (size_t)k * plane);
            cudaMemcpyAsync(outs[k].host, s->B.tmp4 + (size_t)k * plane, bytes, cudaMemcpyDeviceToHost, s->stream);
        }
    }
    return sync_and_check(s, "md_step_host");
}

int64_t md_launch_count(const md_system* s) { return s ? s->launches : 0; }

const char* md_last_error(const md_system* s) { return s ? s->errmsg : "null handle"; }

void md_destroy(md_system* s) {
    if (!s) return;
    drop_step_graph(s);
    if (s->ev_in) cudaEventDestroy(s->ev_in);
    if (s->ev_vel) cudaEventDestroy(s->ev_vel);
    if (s->aux_stream) cudaStreamDestroy(s->aux_stream);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    free(s);
}

}  // extern "C"
