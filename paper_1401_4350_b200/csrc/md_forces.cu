// md_forces.cu -- the two thread mappings of arXiv 1401.4350 for the short-range force/torque evaluation.
//   VERTEX: one thread per particle i loops over its Verlet list L_i, accumulates F_i (tau_i, pe_i)
//                  in registers, one 128-bit store per output array; every pair evaluated twice; no atomics.
//   EDGE: one thread per unordered pair of the list, the pair function evaluated once,
//                  F_ij = -F_ji scattered to both particles only when the pair is inside the cutoff
//                  ("only if the force is actually non-zero").  Four scatter paths (B:5, S:A7).
// fp32 arithmetic; the in-cutoff decision is the fp64 predicate of S:O0/S:Q5, taken in fp32 with an fp64
// recheck inside a relative band of 1e-6 around r_c^2 (S:H10), so it always equals the oracle's decision.
#include <stdio.h>
#include "md_internal.cuh"

static inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

#include "md_pair.cuh"

// FENE partners of slot i (ids id-1 and id+1 inside its chain) -> accumulates into (f, pe)
__device__ __forceinline__ void fene_vertex(const DevParams& P, const DevBuffers& B, const float4* __restrict__ pos,
                                            int i, float4 xi, float& fx, float& fy, float& fz, float& pe) {
    int id = B.ids[i];
    int m = id % P.chain_len;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        int pid = s == 0 ? id - 1 : id + 1;
        bool ok = s == 0 ? (m != 0) : (m != P.chain_len - 1 && pid < P.N);
        if (!ok) continue;
        float4 xj = pos[B.slot_of_id[pid]];
        float dx = min_image(xj.x, xi.x, P.Lx, P.hLx);
        float dy = min_image(xj.y, xi.y, P.Ly, P.hLy);
        float dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
        float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        float g, V;
        if (!fene_pair(P, d2, g, V)) atomicOr(&B.ctrl->err, MD_DEVERR_FENE);
        fx -= g * dx; fy -= g * dy; fz -= g * dz;   // force on i = -(force on j)
        pe += V;
    }
}

// ------------------------------------------------------------------------------------------------
// VERTEX kernels (S:A6).  List layout: tile of 32 particles, int4 groups: entry k of lane l at
// ((tile*capg + k/4)*32 + l)*4 + k%4  -> one coalesced 128-bit load per 4 visits.
// ------------------------------------------------------------------------------------------------
// Per-thread accumulators of the LJ VERTEX loop.  `band` tracks min |d2 - rc^2|: if any visit came within the
// fp64-recheck band (S:H10) the particle is recomputed by vertex_lj_careful after the loop, which keeps the
// hot loop free of calls and branches.
struct LJAcc { float fx, fy, fz, pe, band; int nin; };

template <bool IMG, bool TAIL>
__device__ __forceinline__ void vertex_lj_visit(const DevParams& P, float4 xi, float4 xj, bool valid, LJAcc& a) {
    float dx, dy, dz;
    if (IMG) {
        dx = min_image(xj.x, xi.x, P.Lx, P.hLx);
        dy = min_image(xj.y, xi.y, P.Ly, P.hLy);
        dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
    } else {
        dx = xj.x - xi.x; dy = xj.y - xi.y; dz = xj.z - xi.z;
    }
    float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (TAIL) d2 = fmaxf(d2, 1e-12f);           // padding entries point at the particle itself
    const float t = d2 - P.rc2;
    bool in = t < 0.0f;
    if (TAIL) in = in && valid;
    a.band = fminf(a.band, fabsf(t));
    const float inv = rcp_approx(d2);
    float inv3 = inv * inv * inv;
    inv3 = in ? inv3 : 0.0f;
    const float g = inv * inv3 * fmaf(P.lj_a, inv3, -P.lj_b);     // 24 eps s6 (2 s6 - 1) / d2
    a.fx = fmaf(-g, dx, a.fx); a.fy = fmaf(-g, dy, a.fy); a.fz = fmaf(-g, dz, a.fz);
    a.pe = fmaf(inv3, fmaf(P.lj_c, inv3, -P.lj_d), a.pe);        // 4 eps s6 (s6 - 1); the shift is nin * V_c
    a.nin += in ? 1 : 0;
}

template <bool IMG>
__device__ __forceinline__ void vertex_lj_loop(const DevParams& P, const float4* __restrict__ pos, const int4* __restrict__ row,
                                               float4 xi, int cnt, int gmin, int gmax, LJAcc& a) {
    int g = 0;
#pragma unroll 2
    for (; g < gmin; ++g) {                        // every lane of the warp has 4 real neighbours here
        const int4 jj = row[g * MD_TILE];
        const float4 x0 = ldg4(pos + jj.x), x1 = ldg4(pos + jj.y), x2 = ldg4(pos + jj.z), x3 = ldg4(pos + jj.w);
        vertex_lj_visit<IMG, false>(P, xi, x0, true, a);
        vertex_lj_visit<IMG, false>(P, xi, x1, true, a);
        vertex_lj_visit<IMG, false>(P, xi, x2, true, a);
        vertex_lj_visit<IMG, false>(P, xi, x3, true, a);
    }
    for (; g < gmax; ++g) {                        // ragged tail: entries k >= cnt are padding
        const int4 jj = row[g * MD_TILE];
        const int k = g * 4;
        const float4 x0 = ldg4(pos + jj.x), x1 = ldg4(pos + jj.y), x2 = ldg4(pos + jj.z), x3 = ldg4(pos + jj.w);
        vertex_lj_visit<IMG, true>(P, xi, x0, k < cnt, a);
        vertex_lj_visit<IMG, true>(P, xi, x1, k + 1 < cnt, a);
        vertex_lj_visit<IMG, true>(P, xi, x2, k + 2 < cnt, a);
        vertex_lj_visit<IMG, true>(P, xi, x3, k + 3 < cnt, a);
    }
}

// Rare path: some visit of this particle fell inside the recheck band -> redo the particle with the fp64
// decision of S:O0 / S:Q5 for every banded pair (same accumulation order as the fast loop).  Scalar arguments
// only (a by-value parameter block would live on the stack); the result goes through `out` (global memory).
__device__ __noinline__ void vertex_lj_careful(const float4* __restrict__ pos, const int* __restrict__ row_i, int cnt, float4 xi,
                                              float Lx, float Ly, float Lz, float rc2, float band_abs,
                                              float lj_a, float lj_b, float lj_c, float lj_d, float vshift,
                                              double dLx, double dLy, double dLz, double rc2d, float4* out) {
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f;
    int nin = 0;
    for (int k = 0; k < cnt; ++k) {
        const int j = row_i[(k >> 2) * (MD_TILE * 4) + (k & 3)];
        const float4 xj = pos[j];
        const float dx = min_image(xj.x, xi.x, Lx, 0.5f * Lx);
        const float dy = min_image(xj.y, xi.y, Ly, 0.5f * Ly);
        const float dz = min_image(xj.z, xi.z, Lz, 0.5f * Lz);
        const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        const float t = d2 - rc2;
        bool in = t < 0.0f;
        if (fabsf(t) < band_abs) in = inside_fp64(xi, xj, dLx, dLy, dLz, rc2d);
        const float inv = rcp_approx(d2);
        float inv3 = inv * inv * inv;
        inv3 = in ? inv3 : 0.0f;
        const float g = inv * inv3 * fmaf(lj_a, inv3, -lj_b);
        fx = fmaf(-g, dx, fx); fy = fmaf(-g, dy, fy); fz = fmaf(-g, dz, fz);
        pe = fmaf(inv3, fmaf(lj_c, inv3, -lj_d), pe);
        nin += in ? 1 : 0;
    }
    *out = make_float4(fx, fy, fz, fmaf(-(float)nin, vshift, pe));
}

template <bool BONDS>
__global__ void __launch_bounds__(128, 8) k_vertex_lj(DevParams P, DevBuffers B, const float4* __restrict__ pos, float4* __restrict__ force) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31, tile = i >> 5;
    if (tile >= P.ntiles) return;
    const bool live = i < P.N;
    const int cnt = live ? B.nl_count[i] : 0;
    const int2 info = B.tile_info[tile];                 // (kmax | img << 30, kmin)
    const int kmax = info.x & 0x3fffffff;
    const float4 xi = pos[live ? i : 0];
    const int4* __restrict__ row = reinterpret_cast<const int4*>(B.nl_full) + (size_t)tile * P.capg * MD_TILE + lane;
    LJAcc a = { 0.f, 0.f, 0.f, 0.f, 3.0e38f, 0 };
    if (info.x >> 30) vertex_lj_loop<true>(P, pos, row, xi, cnt, info.y >> 2, (kmax + 3) >> 2, a);
    else vertex_lj_loop<false>(P, pos, row, xi, cnt, info.y >> 2, (kmax + 3) >> 2, a);
    if (!live) return;
    if (a.band < P.band_abs) {
        vertex_lj_careful(pos, reinterpret_cast<const int*>(row), cnt, xi, P.Lx, P.Ly, P.Lz, P.rc2, P.band_abs,
                          P.lj_a, P.lj_b, P.lj_c, P.lj_d, P.vshift, P.dLx, P.dLy, P.dLz, P.rc2d, force + i);
        const float4 r = force[i];
        a.fx = r.x; a.fy = r.y; a.fz = r.z; a.pe = r.w; a.nin = 0;
    }
    float pe = 0.5f * fmaf(-(float)a.nin, P.vshift, a.pe);
    if (BONDS) {
        float bpe = 0.f;
        fene_vertex(P, B, pos, i, xi, a.fx, a.fy, a.fz, bpe);
        pe += 0.5f * bpe;
    }
    force[i] = make_float4(a.fx, a.fy, a.fz, pe);
}

template <bool IMG, bool PP>
__device__ __forceinline__ void vertex_patchy_visit(const DevParams& P, const float4* __restrict__ pos, const float4* __restrict__ quat,
                                                    float4 xi, const Rot& Ri, int j, float& fx, float& fy, float& fz, float& pe,
                                                    float& tx, float& ty, float& tz) {
    float4 xj = ldg4(pos + j);
    float dx, dy, dz;
    if (IMG) {
        dx = min_image(xj.x, xi.x, P.Lx, P.hLx);
        dy = min_image(xj.y, xi.y, P.Ly, P.hLy);
        dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
    } else {
        dx = xj.x - xi.x; dy = xj.y - xi.y; dz = xj.z - xi.z;
    }
    float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (in_cutoff(P, d2, xi, xj)) {
        float4 qj = ldg4(quat + j);
        float gx, gy, gz, V, a, b, c, u, v, w;
        rigid_pair<false, PP>(P, dx, dy, dz, d2, Ri, qj, gx, gy, gz, V, a, b, c, u, v, w);
        fx -= gx; fy -= gy; fz -= gz;
        tx += a; ty += b; tz += c;
        pe += V;
    }
}

template <bool PP>
__global__ void __launch_bounds__(128) k_vertex_patchy(DevParams P, DevBuffers B, const float4* __restrict__ pos,
                                                       const float4* __restrict__ quat, float4* __restrict__ force,
                                                       float4* __restrict__ torque) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31, tile = i >> 5;
    if (i >= P.N) return;
    const int cnt = B.nl_count[i];
    const int2 info = B.tile_info[tile];
    const float4 xi = pos[i], qi = quat[i];
    const int* __restrict__ row = B.nl_full + ((size_t)tile * P.capg * MD_TILE + lane) * 4;
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f, tx = 0.f, ty = 0.f, tz = 0.f;
    const Rot Ri = quat_to_rot(qi);     // once per particle
    for (int k = 0; k < cnt; ++k) {
        int j = row[(k >> 2) * (MD_TILE * 4) + (k & 3)];
        if (info.x >> 30) vertex_patchy_visit<true, PP>(P, pos, quat, xi, Ri, j, fx, fy, fz, pe, tx, ty, tz);
        else vertex_patchy_visit<false, PP>(P, pos, quat, xi, Ri, j, fx, fy, fz, pe, tx, ty, tz);
    }
    force[i] = make_float4(fx, fy, fz, 0.5f * pe);
    torque[i] = make_float4(tx, ty, tz, 0.f);
}

// ------------------------------------------------------------------------------------------------
// EDGE kernels (S:A7)
// ------------------------------------------------------------------------------------------------
__global__ void k_zero4(DevParams P, float4* a, float4* b) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < P.N) {
        a[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (b) b[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// evaluate one edge: returns true if inside the cutoff; F_j = (fx,fy,fz), V full pair energy
// first half of an edge: separation and the cutoff decision (cheap: two position loads, ~25 instructions)
__device__ __forceinline__ bool edge_test(const DevParams& P, const float4* __restrict__ pos, int i, int jw,
                                          float& dx, float& dy, float& dz, float& d2) {
    const int j = jw & 0x7fffffff;
    float4 xi = ldg4(pos + i), xj = ldg4(pos + j);
    dx = xj.x - xi.x; dy = xj.y - xi.y; dz = xj.z - xi.z;
    if (jw < 0) {   // the pair crosses a periodic face (flag set at build time)
        dx = min_image(xj.x, xi.x, P.Lx, P.hLx);
        dy = min_image(xj.y, xi.y, P.Ly, P.hLy);
        dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
    }
    d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    return in_cutoff(P, d2, xi, xj);
}

// second half: the pair function of an edge inside the cutoff.  F_j = (fx,fy,fz), V full pair energy
template <int KIND>
__device__ __forceinline__ void edge_force(const DevParams& P, const float4* __restrict__ quat, int i, int jw,
                                           float dx, float dy, float dz, float d2, float& fx, float& fy, float& fz, float& V,
                                           float& tix, float& tiy, float& tiz, float& tjx, float& tjy, float& tjz) {
    if (md_is_rigid(KIND)) {
        const int j = jw & 0x7fffffff;
        float4 qi = ldg4(quat + i), qj = ldg4(quat + j);
        const Rot Ri = quat_to_rot(qi);
        rigid_pair<true, KIND == MD_POT_PATCHY_PP>(P, dx, dy, dz, d2, Ri, qj, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz);
    } else {
        float g;
        lj_pair(P, d2, g, V);
        fx = g * dx; fy = g * dy; fz = g * dz;
    }
}

// evaluate one edge: returns true if inside the cutoff
template <int KIND>
__device__ __forceinline__ bool edge_eval(const DevParams& P, const float4* __restrict__ pos, const float4* __restrict__ quat,
                                          int i, int jw, float& fx, float& fy, float& fz, float& V,
                                          float& tix, float& tiy, float& tiz, float& tjx, float& tjy, float& tjz) {
    float dx, dy, dz, d2;
    if (!edge_test(P, pos, i, jw, dx, dy, dz, d2)) return false;
    edge_force<KIND>(P, quat, i, jw, dx, dy, dz, d2, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz);
    return true;
}

// (a) red.global.add.f32 per component / (b) red.global.add.v4.f32 per particle and array
template <int KIND, bool V4>
__global__ void __launch_bounds__(256) k_edge_red(DevParams P, DevBuffers B, const float4* __restrict__ pos,
                                                  const float4* __restrict__ quat, float4* force, float4* torque) {
    const unsigned int E = B.ctrl->n_edges;
    const unsigned int stride = gridDim.x * blockDim.x;
    unsigned int e = blockIdx.x * blockDim.x + threadIdx.x;
    for (;;) {
        // every lane scans forward to its next edge inside the cutoff (the others cost a distance test and nothing
        // else), so that the lanes of a warp enter the pair function together: for the rigid bodies, where that function is
        // ~250 instructions and half of the listed pairs are outside r_c, this is what the time goes into
        int2 ij;
        float dx, dy, dz, d2;
        bool have = false;
        while (e < E) {
            ij = B.edges[e];
            e += stride;
            if (edge_test(P, pos, ij.x, ij.y, dx, dy, dz, d2)) { have = true; break; }
        }
        if (!have) break;
        float fx, fy, fz, V, tix = 0.f, tiy = 0.f, tiz = 0.f, tjx = 0.f, tjy = 0.f, tjz = 0.f;
        edge_force<KIND>(P, quat, ij.x, ij.y, dx, dy, dz, d2, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz);
        const int j = ij.y & 0x7fffffff;
        const float hV = 0.5f * V;
        if (V4) {
            red_add_v4(force + ij.x, -fx, -fy, -fz, hV);
            red_add_v4(force + j, fx, fy, fz, hV);
            if (md_is_rigid(KIND)) {
                red_add_v4(torque + ij.x, tix, tiy, tiz, 0.f);
                red_add_v4(torque + j, tjx, tjy, tjz, 0.f);
            }
        } else {
            float* fi = reinterpret_cast<float*>(force + ij.x);
            float* fj = reinterpret_cast<float*>(force + j);
            red_add_f32(fi + 0, -fx); red_add_f32(fi + 1, -fy); red_add_f32(fi + 2, -fz); red_add_f32(fi + 3, hV);
            red_add_f32(fj + 0, fx);  red_add_f32(fj + 1, fy);  red_add_f32(fj + 2, fz);  red_add_f32(fj + 3, hV);
            if (md_is_rigid(KIND)) {
                float* ti = reinterpret_cast<float*>(torque + ij.x);
                float* tj = reinterpret_cast<float*>(torque + j);
                red_add_f32(ti + 0, tix); red_add_f32(ti + 1, tiy); red_add_f32(ti + 2, tiz);
                red_add_f32(tj + 0, tjx); red_add_f32(tj + 1, tjy); red_add_f32(tj + 2, tjz);
            }
        }
    }
}

// (c) warp-aggregated by the owning particle: SLICE lanes walk the half row of particle i (edges sorted by
// i), keep the i-side sum in registers, combine it with __shfl_xor and issue ONE red per particle and array;
// the j side is scattered with red.v4.
// EDGE_SLICE lanes per owner: 8 for long half rows (LJ at r_c >= 2.5), 4 or 2 for the short rows of the polymer and patchy
// configs (an 8-lane slice on a 6-entry half row leaves most lanes idle)
template <int KIND, int EDGE_SLICE>
__global__ void __launch_bounds__(256) k_edge_warp(DevParams P, DevBuffers B, const float4* __restrict__ pos,
                                                   const float4* __restrict__ quat, float4* force, float4* torque) {
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    const int sl = threadIdx.x & (EDGE_SLICE - 1);
    const int per_warp = 32 / EDGE_SLICE;
    const int nslices = (gridDim.x * blockDim.x) / EDGE_SLICE;
    // warp-uniform outer loop (the shuffles below need all 32 lanes); each aligned group of EDGE_SLICE lanes owns one i
    for (int i0 = (gtid >> 5) * per_warp; i0 < P.N; i0 += nslices) {
        const int i = i0 + ((threadIdx.x & 31) / EDGE_SLICE);
        const bool act = i < P.N;
        const unsigned int e0 = act ? B.edge_off[i] : 0u, e1 = act ? B.edge_off[i + 1] : 0u;
        float ax = 0.f, ay = 0.f, az = 0.f, ape = 0.f, atx = 0.f, aty = 0.f, atz = 0.f;
        for (unsigned int e = e0 + sl; e < e1; e += EDGE_SLICE) {
            int2 ij = B.edges[e];
            float fx, fy, fz, V, tix = 0.f, tiy = 0.f, tiz = 0.f, tjx = 0.f, tjy = 0.f, tjz = 0.f;
            if (!edge_eval<KIND>(P, pos, quat, i, ij.y, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz)) continue;
            const int j = ij.y & 0x7fffffff;
            const float hV = 0.5f * V;
            ax -= fx; ay -= fy; az -= fz; ape += hV;
            red_add_v4(force + j, fx, fy, fz, hV);
            if (md_is_rigid(KIND)) {
                atx += tix; aty += tiy; atz += tiz;
                red_add_v4(torque + j, tjx, tjy, tjz, 0.f);
            }
        }
        // slices of a warp may own different particles: reduce inside aligned groups of EDGE_SLICE lanes
#pragma unroll
        for (int o = EDGE_SLICE / 2; o > 0; o >>= 1) {
            ax += __shfl_xor_sync(0xffffffffu, ax, o);
            ay += __shfl_xor_sync(0xffffffffu, ay, o);
            az += __shfl_xor_sync(0xffffffffu, az, o);
            ape += __shfl_xor_sync(0xffffffffu, ape, o);
            if (md_is_rigid(KIND)) {
                atx += __shfl_xor_sync(0xffffffffu, atx, o);
                aty += __shfl_xor_sync(0xffffffffu, aty, o);
                atz += __shfl_xor_sync(0xffffffffu, atz, o);
            }
        }
        if (sl == 0 && e1 > e0) {   // one reduction per owning particle
            red_add_v4(force + i, ax, ay, az, ape);
            if (md_is_rigid(KIND)) red_add_v4(torque + i, atx, aty, atz, 0.f);
        }
    }
}

// (c') the same aggregation for short half rows (polymer, rigid bodies: 4..8 listed pairs per particle, half of them
// outside r_c): a slice per owner leaves most lanes idle, so here a warp walks a CONTIGUOUS range of the edge list,
// compacts the pairs inside the cutoff into a 64-entry ring in shared memory and evaluates them 32 at a time.  The ring
// keeps the edge order, edges are sorted by owner, so equal owners sit in adjacent lanes: a segmented shuffle reduction
// leaves one red.v4 per owner and array at the head lane of each run.  The j side is scattered with red.v4 as before.
template <int KIND>
__global__ void __launch_bounds__(256) k_edge_warp_queue(DevParams P, DevBuffers B, const float4* __restrict__ pos,
                                                         const float4* __restrict__ quat, float4* force, float4* torque) {
    __shared__ int2 q_ij[8][64];
    __shared__ float4 q_d[8][64];
    const unsigned int full = 0xffffffffu;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const unsigned int E = B.ctrl->n_edges;
    const unsigned int nw = gridDim.x * 8u;
    const unsigned int chunk = ((E + nw - 1) / nw + 31u) & ~31u;
    const uint64_t b0 = (uint64_t)(blockIdx.x * 8u + w) * chunk;
    unsigned int e = b0 < E ? (unsigned int)b0 : E;
    const unsigned int e_end = (uint64_t)e + chunk < E ? e + chunk : E;
    unsigned int head = 0, count = 0;
    for (;;) {
        while (count < 32u && e < e_end) {       // warp-uniform
            const unsigned int my = e + lane;
            bool hit = false;
            int2 ij = make_int2(0, 0);
            float dx = 0.f, dy = 0.f, dz = 0.f, d2 = 0.f;
            if (my < e_end) {
                ij = B.edges[my];
                hit = edge_test(P, pos, ij.x, ij.y, dx, dy, dz, d2);
            }
            const unsigned int m = __ballot_sync(full, hit);
            if (hit) {
                const unsigned int p = (head + count + __popc(m & ((1u << lane) - 1u))) & 63u;
                q_ij[w][p] = ij;
                q_d[w][p] = make_float4(dx, dy, dz, d2);
            }
            count += __popc(m);
            e += 32u;
        }
        if (count == 0u) break;
        __syncwarp();
        const unsigned int n = count < 32u ? count : 32u;
        const bool act = (unsigned int)lane < n;
        int key = -1;
        float ax = 0.f, ay = 0.f, az = 0.f, ape = 0.f, atx = 0.f, aty = 0.f, atz = 0.f;
        int2 ij = make_int2(0, 0);
        float4 d = make_float4(0.f, 0.f, 0.f, 0.f);
        if (act) { ij = q_ij[w][(head + lane) & 63u]; d = q_d[w][(head + lane) & 63u]; }
        __syncwarp();                            // the ring slots just read may be refilled below
        head = (head + n) & 63u;
        count -= n;
        if (act) {
            float fx, fy, fz, V, tix = 0.f, tiy = 0.f, tiz = 0.f, tjx = 0.f, tjy = 0.f, tjz = 0.f;
            edge_force<KIND>(P, quat, ij.x, ij.y, d.x, d.y, d.z, d.w, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz);
            const int j = ij.y & 0x7fffffff;
            const float hV = 0.5f * V;
            key = ij.x;
            ax = -fx; ay = -fy; az = -fz; ape = hV;
            red_add_v4(force + j, fx, fy, fz, hV);
            if (md_is_rigid(KIND)) {
                atx = tix; aty = tiy; atz = tiz;
                red_add_v4(torque + j, tjx, tjy, tjz, 0.f);
            }
        }
        // runs of equal owners are contiguous (edge order): after the step of distance o a lane holds the sum over
        // [lane, lane + 2o) cut at the end of its run
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int ko = __shfl_down_sync(full, key, o);
            const bool same = lane + o < 32 && ko == key;
            float t;
            t = __shfl_down_sync(full, ax, o); if (same) ax += t;
            t = __shfl_down_sync(full, ay, o); if (same) ay += t;
            t = __shfl_down_sync(full, az, o); if (same) az += t;
            t = __shfl_down_sync(full, ape, o); if (same) ape += t;
            if (md_is_rigid(KIND)) {
                t = __shfl_down_sync(full, atx, o); if (same) atx += t;
                t = __shfl_down_sync(full, aty, o); if (same) aty += t;
                t = __shfl_down_sync(full, atz, o); if (same) atz += t;
            }
        }
        const int kprev = __shfl_up_sync(full, key, 1);
        if (act && (lane == 0 || kprev != key)) {
            red_add_v4(force + key, ax, ay, az, ape);
            if (md_is_rigid(KIND)) red_add_v4(torque + key, atx, aty, atz, 0.f);
        }
    }
}

// (d) per-edge store, then an atomic-free per-particle sum over own edges (+) and incoming edges (-)
template <int KIND>
__global__ void __launch_bounds__(256) k_edge_store(DevParams P, DevBuffers B, const float4* __restrict__ pos,
                                                    const float4* __restrict__ quat) {
    const unsigned int E = B.ctrl->n_edges;
    const unsigned int stride = gridDim.x * blockDim.x;
    for (unsigned int e = blockIdx.x * blockDim.x + threadIdx.x; e < E; e += stride) {
        int2 ij = B.edges[e];
        float fx = 0.f, fy = 0.f, fz = 0.f, V = 0.f, tix = 0.f, tiy = 0.f, tiz = 0.f, tjx = 0.f, tjy = 0.f, tjz = 0.f;
        if (!edge_eval<KIND>(P, pos, quat, ij.x, ij.y, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz)) {
            fx = fy = fz = V = 0.f; tix = tiy = tiz = tjx = tjy = tjz = 0.f;
        }
        B.edge_f[e] = make_float4(fx, fy, fz, V);
        if (md_is_rigid(KIND)) {
            B.edge_ti[e] = make_float4(tix, tiy, tiz, 0.f);
            B.edge_tj[e] = make_float4(tjx, tjy, tjz, 0.f);
        }
    }
}

template <int KIND>
__global__ void __launch_bounds__(128) k_edge_segsum(DevParams P, DevBuffers B, float4* __restrict__ force, float4* __restrict__ torque) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P.N) return;
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f, tx = 0.f, ty = 0.f, tz = 0.f;
    for (unsigned int e = B.edge_off[p]; e < B.edge_off[p + 1]; ++e) {   // p is the first member: F_i = -F_j
        float4 f = B.edge_f[e];
        fx -= f.x; fy -= f.y; fz -= f.z; pe += f.w;
        if (md_is_rigid(KIND)) { float4 t = B.edge_ti[e]; tx += t.x; ty += t.y; tz += t.z; }
    }
    for (unsigned int t = B.in_off[p]; t < B.in_off[p + 1]; ++t) {       // p is the second member
        unsigned int e = B.in_edge[t];
        float4 f = B.edge_f[e];
        fx += f.x; fy += f.y; fz += f.z; pe += f.w;
        if (md_is_rigid(KIND)) { float4 q = B.edge_tj[e]; tx += q.x; ty += q.y; tz += q.z; }
    }
    force[p] = make_float4(fx, fy, fz, 0.5f * pe);
    if (md_is_rigid(KIND)) torque[p] = make_float4(tx, ty, tz, 0.f);
}

// S:A8 bonded pass for EDGE (C3): one thread per static bond (id, id+1), FENE only, scatter with red.v4
__global__ void k_edge_bonds(DevParams P, DevBuffers B, const float4* __restrict__ pos, float4* force) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= P.N - 1 || (id % P.chain_len) == P.chain_len - 1) return;
    const int i = B.slot_of_id[id], j = B.slot_of_id[id + 1];
    float4 xi = pos[i], xj = pos[j];
    float dx = min_image(xj.x, xi.x, P.Lx, P.hLx);
    float dy = min_image(xj.y, xi.y, P.Ly, P.hLy);
    float dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
    float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    float g, V;
    if (!fene_pair(P, d2, g, V)) atomicOr(&B.ctrl->err, MD_DEVERR_FENE);
    red_add_v4(force + i, -g * dx, -g * dy, -g * dz, 0.5f * V);
    red_add_v4(force + j, g * dx, g * dy, g * dz, 0.5f * V);
}

// ------------------------------------------------------------------------------------------------
// VERTEX with Newton's third law and m private force copies per particle (S:8(f1))
// ------------------------------------------------------------------------------------------------
// One thread per particle i over its half row (the edges (i, j) sorted by i): own side in registers and one plain
// store, -f (and the j-side torque) added with red.v4 into copy (i mod m) of particle j (DESIGN Q20: the paper does
// not say how a writer picks its copy).  Pairs outside the cutoff issue no atomics.
template <int KIND>
__global__ void __launch_bounds__(128) k_vertex_n3(DevParams P, DevBuffers B, const float4* __restrict__ pos,
                                                   const float4* __restrict__ quat, float4* __restrict__ force,
                                                   float4* __restrict__ torque, float4* fcopy, float4* tcopy, int m) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const size_t plane = (size_t)(i % m) * (size_t)P.N;
    float4* fc = fcopy + plane;
    float4* tc = md_is_rigid(KIND) ? tcopy + plane : nullptr;
    const unsigned int e0 = B.edge_off[i], e1 = B.edge_off[i + 1];
    float ax = 0.f, ay = 0.f, az = 0.f, ape = 0.f, atx = 0.f, aty = 0.f, atz = 0.f;
    for (unsigned int e = e0; e < e1; ++e) {
        const int jw = B.edges[e].y;
        float fx, fy, fz, V, tix = 0.f, tiy = 0.f, tiz = 0.f, tjx = 0.f, tjy = 0.f, tjz = 0.f;
        if (!edge_eval<KIND>(P, pos, quat, i, jw, fx, fy, fz, V, tix, tiy, tiz, tjx, tjy, tjz)) continue;
        const int j = jw & 0x7fffffff;
        const float hV = 0.5f * V;
        ax -= fx; ay -= fy; az -= fz; ape += hV;
        red_add_v4(fc + j, fx, fy, fz, hV);
        if (md_is_rigid(KIND)) {
            atx += tix; aty += tiy; atz += tiz;
            red_add_v4(tc + j, tjx, tjy, tjz, 0.f);
        }
    }
    force[i] = make_float4(ax, ay, az, ape);
    if (md_is_rigid(KIND)) torque[i] = make_float4(atx, aty, atz, 0.f);
}

// "then the vectors are combined to obtain the total force acting on each particle": copies added in index order
__global__ void __launch_bounds__(256) k_n3_combine(DevParams P, float4* __restrict__ force, float4* __restrict__ torque,
                                                    const float4* __restrict__ fcopy, const float4* __restrict__ tcopy, int m) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    float4 f = force[i];
    for (int c = 0; c < m; ++c) {
        const float4 g = fcopy[(size_t)c * P.N + i];
        f.x += g.x; f.y += g.y; f.z += g.z; f.w += g.w;
    }
    force[i] = f;
    if (torque) {
        float4 t = torque[i];
        for (int c = 0; c < m; ++c) {
            const float4 g = tcopy[(size_t)c * P.N + i];
            t.x += g.x; t.y += g.y; t.z += g.z;
        }
        torque[i] = t;
    }
}

template <int KIND>
static void launch_vertex_n3(md_system* s, int m) {
    const DevParams& P = s->P;
    float4* tq = md_is_rigid(KIND) ? s->torque : nullptr;
    float4* fcopy = s->B.edge_f;                                   // the per-edge scratch of the segmented variant
    float4* tcopy = md_is_rigid(KIND) ? s->B.edge_tj : nullptr;
    cudaMemsetAsync(fcopy, 0, 16 * (size_t)m * P.N, s->stream);
    if (tcopy) cudaMemsetAsync(tcopy, 0, 16 * (size_t)m * P.N, s->stream);
    k_vertex_n3<KIND><<<cdiv(P.N, 128), 128, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, tq, fcopy, tcopy, m);
    k_n3_combine<<<cdiv(P.N, 256), 256, 0, s->stream>>>(P, s->force, tq, fcopy, tcopy, m);
    s->launches += 2;
    if (P.kind == MD_POT_FENE_WCA) {
        k_edge_bonds<<<cdiv(P.N, 256), 256, 0, s->stream>>>(P, s->B, s->pos, s->force);
        s->launches += 1;
    }
}

// E_in (S:Q16): pairs of the explicit edge list inside the cutoff at the current positions, by the decision every force
// kernel takes (fp32 away from the threshold, the fp64 predicate of S:Q5 inside the band) -> ctrl->n_in
__global__ void __launch_bounds__(256) k_count_in_cutoff(DevParams P, DevBuffers B, const float4* __restrict__ pos) {
    const unsigned int E = B.ctrl->n_edges;
    const unsigned int stride = gridDim.x * blockDim.x;
    unsigned int n = 0;
    for (unsigned int e = blockIdx.x * blockDim.x + threadIdx.x; e < E; e += stride) {
        const int2 ij = B.edges[e];
        float dx, dy, dz, d2;
        n += edge_test(P, pos, ij.x, ij.y, dx, dy, dz, d2) ? 1u : 0u;
    }
    n = __reduce_add_sync(0xffffffffu, n);
    if ((threadIdx.x & 31) == 0 && n) atomicAdd(&B.ctrl->n_in, (unsigned long long)n);
}

void md_launch_count_in_cutoff(md_system* s) {
    cudaMemsetAsync(&s->B.ctrl->n_in, 0, sizeof(unsigned long long), s->stream);
    k_count_in_cutoff<<<s->sm_count * 8, 256, 0, s->stream>>>(s->P, s->B, s->pos);
    s->launches += 1;
}

// ------------------------------------------------------------------------------------------------
// host-side dispatch
// ------------------------------------------------------------------------------------------------
template <int KIND>
static void launch_edge(md_system* s, int scatter) {
    const DevParams& P = s->P;
    const int nbN = cdiv(P.N, 256);
    const int persistent = s->sm_count * 8;   // 8 CTAs of 256 threads per SM, grid-stride over the device-resident edge count
    float4* tq = md_is_rigid(KIND) ? s->torque : nullptr;
    if (scatter == MD_SCATTER_SEGMENTED) {
        k_edge_store<KIND><<<persistent, 256, 0, s->stream>>>(P, s->B, s->pos, s->quat);
        k_edge_segsum<KIND><<<cdiv(P.N, 128), 128, 0, s->stream>>>(P, s->B, s->force, tq);
        s->launches += 2;
    } else {
        k_zero4<<<nbN, 256, 0, s->stream>>>(P, s->force, tq);
        s->launches += 1;
        if (scatter == MD_SCATTER_CLUSTER) { md_launch_edge_cluster(s); s->launches -= 1; }
        else if (scatter == MD_SCATTER_RED) k_edge_red<KIND, false><<<persistent, 256, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, tq);
        else if (scatter == MD_SCATTER_RED_V4) k_edge_red<KIND, true><<<persistent, 256, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, tq);
        else {
            const double half_row = (double)s->n_edges_host / (double)P.N;   // E / N at the last synchronised build (0 if unknown)
            // rigid bodies with short rows: the compacting walk (measured: patchy N = 2^20 melted 134 -> 98 us, C4 37.7 -> 35.4;
            // the polymer and LJ configs are faster with slices: 23.2 vs 25.2 us at C3, 196 vs 312 us at C2a)
            if (md_is_rigid(KIND) && half_row > 0 && half_row < 14.0) k_edge_warp_queue<KIND><<<persistent, 256, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, tq);
            else
            if (half_row > 0 && half_row < 8.0) k_edge_warp<KIND, 2><<<persistent, 256, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, tq);
            else if (half_row > 0 && half_row < 14.0) k_edge_warp<KIND, 4><<<persistent, 256, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, tq);
            else k_edge_warp<KIND, 8><<<persistent, 256, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, tq);
        }
        s->launches += 1;
    }
    if (P.kind == MD_POT_FENE_WCA) {
        k_edge_bonds<<<nbN, 256, 0, s->stream>>>(P, s->B, s->pos, s->force);
        s->launches += 1;
    }
}

void md_launch_forces(md_system* s, int strategy, int scatter) {
    const DevParams& P = s->P;
    if (strategy == MD_VERTEX) {
        int nb = cdiv((int64_t)P.ntiles * MD_TILE, 128);
        if (P.kind == MD_POT_PATCHY && P.pp_model) k_vertex_patchy<true><<<nb, 128, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, s->torque);
        else if (P.kind == MD_POT_PATCHY) k_vertex_patchy<false><<<nb, 128, 0, s->stream>>>(P, s->B, s->pos, s->quat, s->force, s->torque);
        else if (P.kind == MD_POT_FENE_WCA) k_vertex_lj<true><<<nb, 128, 0, s->stream>>>(P, s->B, s->pos, s->force);
        else k_vertex_lj<false><<<nb, 128, 0, s->stream>>>(P, s->B, s->pos, s->force);
        s->launches += 1;
    } else if (strategy == MD_VERTEX_N3) {
        const int m = scatter == 0 ? 12 : scatter;
        if (P.kind == MD_POT_PATCHY && P.pp_model) launch_vertex_n3<MD_POT_PATCHY_PP>(s, m);
        else if (P.kind == MD_POT_PATCHY) launch_vertex_n3<MD_POT_PATCHY>(s, m);
        else launch_vertex_n3<MD_POT_LJ>(s, m);
    } else {
        if (P.kind == MD_POT_PATCHY && P.pp_model) launch_edge<MD_POT_PATCHY_PP>(s, scatter);
        else if (P.kind == MD_POT_PATCHY) launch_edge<MD_POT_PATCHY>(s, scatter);
        else launch_edge<MD_POT_LJ>(s, scatter);
    }
}
