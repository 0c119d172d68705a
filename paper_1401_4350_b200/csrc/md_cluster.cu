// md_cluster.cu -- EDGE with cluster-aggregated scatter (MD_SCATTER_CLUSTER, S:A7).
//
// The ceiling of every red.global-based EDGE variant on B200 is the NUMBER of L2 reductions (~170 G lane-operations/s
// whatever their width, md_probe), and the warp-aggregated variant still issues one per in-cutoff pair for the j side
// (27.6 M at config C2a).  Here the j side is aggregated before it reaches L2:
//   * MD_CLUSTER = 16 consecutive slots (neighbours in space when the storage is cell / Hilbert ordered) form a
//     cluster of OWNERS.  The half list (i < j) of the cluster is stored as UNITS (j, mask): bit k of mask = pair
//     (owner k, j) is in the Verlet list.  One unit stands for popcount(mask) pairs (~4.2 at C2a).
//   * force kernel: one warp per cluster, one LANE per unit at a time.  The lane walks the set bits of its unit --
//     one lane-iteration per listed pair ("one thread per interacting pair"), the pair function evaluated once,
//     +f / -f applied to both members -- keeping the j side in REGISTERS (one red.v4 per unit, none if no pair of the
//     unit is inside the cutoff: "only if the force is actually non-zero") and adding the owner side to a
//     lane-private row of a shared-memory accumulator [16 owners][32 lanes] (no atomics, no bank conflicts), which is
//     summed once per cluster: 16 red.v4 per cluster for the owner side.
//   * units are sorted by popcount and dealt to the lanes in a snake over rounds of 32, so that every lane of the
//     warp has about the same number of pairs; the lanes run a flattened loop (next unit as soon as the mask is empty).
// Reductions per evaluation at C2a: ~6.9 M (j side) + 1 M (owner side) instead of 28.6 M.
#include <stdio.h>
#include "md_pair.cuh"

#define GATE(B, gated) if ((gated) && (B).ctrl->rebuild == 0) return

static inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

#define CLB_WARPS 4                 // clusters (warps) per block of the build kernel
#define CL_CELLCAP (27 * MD_CLUSTER)

__global__ void k_cluster_begin(DevBuffers B, int gated) {
    GATE(B, gated);
    B.ctrl->cl_cursor = 0u;
    B.ctrl->n_units = 0ull;
    B.ctrl->n_cl_pairs = 0ull;
}

// the bookkeeping the other list builds leave behind: E = sum of popcounts, sum |L_i| = 2 E
__global__ void k_cluster_end(DevBuffers B, int gated) {
    GATE(B, gated);
    B.ctrl->n_edges = (unsigned int)B.ctrl->n_cl_pairs;
    B.ctrl->n_full = 2ull * B.ctrl->n_cl_pairs;
}

// ------------------------------------------------------------------------------------------------
// S:A4 for the cluster list: one warp per cluster.  Candidates = the particles of the distinct cells in the union of
// the 27-cell stencils (S:Q8) of the owners' cells; lane = candidate j, tested against the 16 owners with the list
// predicate of S:O0 (fp32 filter with the robust minimum image, fp64 decision inside the band, S:Q6).
// IDENT: storage is cell-sorted (slot == position in the cell-sorted item list).
// ------------------------------------------------------------------------------------------------
template <bool IDENT>
__global__ void __launch_bounds__(32 * CLB_WARPS) k_build_cluster(DevParams P, DevBuffers B, int gated, const float4* __restrict__ pos,
                                                                  int ucap_w, unsigned int ucap_total, int write_ref) {
    GATE(B, gated);
    extern __shared__ __align__(16) unsigned char smraw[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const size_t per_warp = 32 * (size_t)MD_CLUSTER + 4 * (size_t)(CL_CELLCAP + MD_CLUSTER + 40) + 8 * (size_t)ucap_w;
    unsigned char* base = smraw + (size_t)w * ((per_warp + 15) / 16 * 16);
    float4* pi = reinterpret_cast<float4*>(base);                       // [16] owner positions
    int* cells = reinterpret_cast<int*>(pi + 2 * MD_CLUSTER);           // [CL_CELLCAP] distinct candidate cells (ranks); pi[16..31] = raw owner positions
    int* own = cells + CL_CELLCAP;                                      // [16] distinct own cells
    int* hist = own + MD_CLUSTER;                                       // [17] popcount histogram, [17..33] cursors
    uint2* ubuf = reinterpret_cast<uint2*>(hist + 40);                  // [ucap_w] units in scan order
    const int ncl = (P.N + MD_CLUSTER - 1) / MD_CLUSTER;
    const int c = blockIdx.x * CLB_WARPS + w;
    if (c >= ncl) return;
    const int i0 = c * MD_CLUSTER;
    const int nown = min(MD_CLUSTER, P.N - i0);

    // 1. owners
    int oc = -1 - lane;                                                 // distinct dummies for dead lanes
    if (lane < MD_CLUSTER) {
        float4 xi = make_float4(1.0e15f, 1.0e15f, 1.0e15f, 0.f);
        if (lane < nown) {
            xi = pos[i0 + lane];
            oc = B.cell_of[i0 + lane];
            if (write_ref) B.pos_ref[i0 + lane] = xi;
        }
        pi[lane] = xi;
    }
    if (lane < 34) hist[lane] = 0;
    // 2. distinct own cells
    const unsigned int grp = __match_any_sync(0xffffffffu, oc);
    const bool head = lane < nown && (__ffs(grp) - 1) == lane;
    const unsigned int heads = __ballot_sync(0xffffffffu, head);
    if (head) own[__popc(heads & ((1u << lane) - 1u))] = oc;
    const int n_own = __popc(heads);
    __syncwarp();
    // 3. distinct non-empty candidate cells
    int L = 0;
    for (int m = 0; m < n_own; ++m) {
        const int lin = B.cell_lin[own[m]];
        const int cz = lin % P.ncz, cy = (lin / P.ncz) % P.ncy, cx = lin / (P.ncz * P.ncy);
        int r = -1 - lane;
        if (lane < 27) {
            int ax = cx + lane / 9 - 1, ay = cy + (lane / 3) % 3 - 1, az = cz + lane % 3 - 1;
            if (ax < 0) ax += P.ncx; else if (ax >= P.ncx) ax -= P.ncx;
            if (ay < 0) ay += P.ncy; else if (ay >= P.ncy) ay -= P.ncy;
            if (az < 0) az += P.ncz; else if (az >= P.ncz) az -= P.ncz;
            // an axis with one cell: cx - 1 wraps to ncx - 1 = 0 and cx + 1 to 0 as well; with two cells -1 and +1 coincide
            ax = min(max(ax, 0), P.ncx - 1); ay = min(max(ay, 0), P.ncy - 1); az = min(max(az, 0), P.ncz - 1);
            r = B.cell_rank[(ax * P.ncy + ay) * P.ncz + az];
        }
        const unsigned int same = __match_any_sync(0xffffffffu, r);
        bool keep = lane < 27 && (__ffs(same) - 1) == lane && B.cell_start[r + 1] > B.cell_start[r];
        if (keep) for (int t = 0; t < L; ++t) if (cells[t] == r) { keep = false; break; }
        const unsigned int kb = __ballot_sync(0xffffffffu, keep);
        if (keep) cells[L + __popc(kb & ((1u << lane) - 1u))] = r;
        L += __popc(kb);
        __syncwarp();
    }
    // 3b. Can plain differences stand in for the minimum image?  Per axis: yes if the owners (+ r_v) stay clear of the
    //     periodic face (mode 0), or, with the upper half of the box shifted down by L (exact in fp32: Sterbenz), clear of
    //     the seam at +-L/2 (mode 1); else the cluster takes the robust minimum image for every pair (small boxes, storage
    //     order NONE).  Shifted coordinates give bit-identical differences to min_image() for every pair within r_v.
    float4 xo = lane < MD_CLUSTER ? pi[lane] : make_float4(0.f, 0.f, 0.f, 0.f);
    const bool live_o = lane < nown;
    int mode[3];
    {
        const float Ls[3] = { P.Lx, P.Ly, P.Lz };
        const float xs[3] = { xo.x, xo.y, xo.z };
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float L = Ls[a], hL = 0.5f * L, rv = P.shift_margin;           // r_v + skin: a safe margin
            const float v = xs[a], tv = v > hL ? v - L : v;
            float lo = live_o ? v : 3.0e38f, hi = live_o ? v : -3.0e38f, tlo = live_o ? tv : 3.0e38f, thi = live_o ? tv : -3.0e38f;
            for (int o = 16; o > 0; o >>= 1) {
                lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
                tlo = fminf(tlo, __shfl_xor_sync(0xffffffffu, tlo, o)); thi = fmaxf(thi, __shfl_xor_sync(0xffffffffu, thi, o));
            }
            mode[a] = (lo - rv >= 0.0f && hi + rv < L) ? 0 : ((tlo - rv > -hL && thi + rv < hL) ? 1 : 2);
        }
    }
    const bool fast = mode[0] < 2 && mode[1] < 2 && mode[2] < 2;
    const float sLx = mode[0] == 1 ? P.Lx : 0.0f, sLy = mode[1] == 1 ? P.Ly : 0.0f, sLz = mode[2] == 1 ? P.Lz : 0.0f;
    float4* pr = pi + MD_CLUSTER;                                         // raw owner positions (fp64 band decisions)
    if (lane < MD_CLUSTER) {
        pr[lane] = xo;
        if (fast) {
            int fl = 0;
            if (xo.x > P.hLx && mode[0] == 1) { xo.x -= sLx; fl |= 1; }
            if (xo.y > P.hLy && mode[1] == 1) { xo.y -= sLy; fl |= 2; }
            if (xo.z > P.hLz && mode[2] == 1) { xo.z -= sLz; fl |= 4; }
            xo.w = __int_as_float(fl);
            pi[lane] = xo;
        }
    }
    __syncwarp();
    // 4. candidates -> units
    int nunits = 0;
    unsigned long long npairs = 0ull;
    bool overflow = false;
    for (int ci = 0; ci < L; ++ci) {
        const int r = cells[ci];
        const int s0 = B.cell_start[r], n = B.cell_start[r + 1] - s0;
        if (IDENT && s0 + n <= i0 + 1) continue;                         // half list: only j above the lowest owner can pair
        for (int t0 = 0; t0 < n; t0 += 32) {
            const int t = t0 + lane;
            unsigned int mask = 0u, img = 0u;
            int j = 0;
            if (t < n) {
                j = IDENT ? s0 + t : B.items[s0 + t];
                const float4 xr = pos[j];
                if (fast) {
                    float4 xj = xr;
                    int fj = 0;
                    if (xj.x > P.hLx && mode[0] == 1) { xj.x -= sLx; fj |= 1; }
                    if (xj.y > P.hLy && mode[1] == 1) { xj.y -= sLy; fj |= 2; }
                    if (xj.z > P.hLz && mode[2] == 1) { xj.z -= sLz; fj |= 4; }
#pragma unroll 4
                    for (int k = 0; k < MD_CLUSTER; ++k) {
                        const float4 xi = pi[k];
                        const float dx = xj.x - xi.x, dy = xj.y - xi.y, dz = xj.z - xi.z;
                        const float tt = fmaf(dz, dz, fmaf(dy, dy, dx * dx)) - P.rv2;
                        bool in = tt < 0.0f;
                        if (fabsf(tt) < P.band_rv) in = inside_fp64(pr[k], xr, P.dLx, P.dLy, P.dLz, P.rv2d);
                        in = in && j > i0 + k && k < nown;              // half list: slot of the owner < slot of j
                        if (in) {
                            mask |= 1u << k;
                            img |= (fj != __float_as_int(xi.w)) ? 1u : 0u;   // exactly one member was shifted on some axis: the pair crosses a face
                        }
                    }
                } else {
#pragma unroll 4
                    for (int k = 0; k < MD_CLUSTER; ++k) {
                        const float4 xi = pr[k];
                        const float dx = min_image(xr.x, xi.x, P.Lx, P.hLx), dy = min_image(xr.y, xi.y, P.Ly, P.hLy),
                                    dz = min_image(xr.z, xi.z, P.Lz, P.hLz);
                        const float tt = fmaf(dz, dz, fmaf(dy, dy, dx * dx)) - P.rv2;
                        bool in = tt < 0.0f;
                        if (fabsf(tt) < P.band_rv) in = inside_fp64(xi, xr, P.dLx, P.dLy, P.dLz, P.rv2d);
                        in = in && j > i0 + k && k < nown;
                        if (in) {
                            mask |= 1u << k;
                            img |= (fabsf(xr.x - xi.x) > P.hLx) | (fabsf(xr.y - xi.y) > P.hLy) | (fabsf(xr.z - xi.z) > P.hLz);
                        }
                    }
                }
            }
            const unsigned int ub = __ballot_sync(0xffffffffu, mask != 0u);
            if (mask) {
                const int p = nunits + __popc(ub & ((1u << lane) - 1u));
                if (p < ucap_w) ubuf[p] = make_uint2((unsigned int)j | (img << 31), mask); else overflow = true;
                npairs += __popc(mask);
                atomicAdd(&hist[__popc(mask)], 1);
            }
            nunits += __popc(ub);
        }
    }
    overflow = __any_sync(0xffffffffu, overflow);
    __syncwarp();
    // 5. sort by popcount (descending) and deal the units to the lanes in a snake over rounds of 32
    if (lane == 0) {
        int acc = 0;
        for (int pc = MD_CLUSTER; pc >= 1; --pc) { hist[17 + pc] = acc; acc += hist[pc]; }
    }
    const int R = overflow ? 0 : (nunits + 31) >> 5;
    unsigned int gbase = 0u;
    if (lane == 0) {
        gbase = atomicAdd(&B.ctrl->cl_cursor, (unsigned int)R * 32u);
        if (overflow || gbase + (unsigned int)R * 32u > ucap_total) { atomicOr(&B.ctrl->err, MD_DEVERR_CAPACITY); gbase = 0xffffffffu; }
    }
    gbase = __shfl_sync(0xffffffffu, gbase, 0);
    __syncwarp();
    if (gbase == 0xffffffffu) {
        if (lane == 0) B.cl_info[c] = make_int2(0, 0);
        return;
    }
    for (int p = lane; p < R * 32; p += 32) {
        uint2 u = make_uint2(0u, 0u);
        int sp = p;                                                     // padding fills the tail of the last round
        if (p < nunits) {
            u = ubuf[p];
            sp = atomicAdd(&hist[17 + __popc(u.y)], 1);
        }
        // (the padding slots are exactly the sorted positions >= nunits: nobody else writes them)
        const int rr = sp >> 5, ix = sp & 31;
        B.cl_units[gbase + rr * 32 + ((rr & 1) ? 31 - ix : ix)] = u;
    }
    // 6. bookkeeping
    for (int o = 16; o > 0; o >>= 1) npairs += __shfl_xor_sync(0xffffffffu, npairs, o);
    if (lane == 0) {
        B.cl_info[c] = make_int2((int)gbase, R);
        atomicAdd(&B.ctrl->n_units, (unsigned long long)nunits);
        atomicAdd(&B.ctrl->n_cl_pairs, npairs);
    }
}

// ------------------------------------------------------------------------------------------------
// S:A7 force kernel.  One warp per cluster (grid-stride), 4 warps per block.  Shared memory per warp:
//   px/py/pz[16] owner positions (+ qi[16] quaternions for rigid bodies), acc[16][32] float4 owner-side accumulators
//   (+ tacc[16][32] torques): row k = owner, column = lane -> every lane reads and writes its own column only.
// ------------------------------------------------------------------------------------------------
#define CLF_WARPS 4

template <int KIND>
struct ClusterSmem {
    float px[MD_CLUSTER + 4], py[MD_CLUSTER + 4], pz[MD_CLUSTER + 4], pw[MD_CLUSTER + 4];   // [MD_CLUSTER] = the dummy owner at 1e15   // owner positions, one 64-byte row per coordinate:
                                                                            // a lookup by a lane-varying owner index is three
                                                                            // conflict-free broadcast loads (one wavefront each)
    float4 qi[md_is_rigid(KIND) ? MD_CLUSTER : 1];
    float4 acc[(MD_CLUSTER + 1) * 32];      // row MD_CLUSTER: the dummy owner (collects exact zeros)
    float4 tacc[md_is_rigid(KIND) ? MD_CLUSTER * 32 : 1];
};

template <int KIND>
__global__ void __launch_bounds__(32 * CLF_WARPS) k_edge_cluster(DevParams P, DevBuffers B, const float4* __restrict__ pos,
                                                                 const float4* __restrict__ quat, float4* force, float4* torque) {
    extern __shared__ __align__(16) unsigned char smraw[];
    constexpr bool RIGID = md_is_rigid(KIND);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    ClusterSmem<KIND>& S = reinterpret_cast<ClusterSmem<KIND>*>(smraw)[w];
    const int ncl = (P.N + MD_CLUSTER - 1) / MD_CLUSTER;
    const int nwarps = gridDim.x * CLF_WARPS;
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int k = 0; k <= MD_CLUSTER; ++k) S.acc[k * 32 + lane] = zero4;
    if (RIGID) for (int k = 0; k < MD_CLUSTER; ++k) S.tacc[k * 32 + lane] = zero4;
    if (lane < 4) { S.px[MD_CLUSTER + lane] = 1.0e15f; S.py[MD_CLUSTER + lane] = 1.0e15f; S.pz[MD_CLUSTER + lane] = 1.0e15f; }
    const uint2* __restrict__ units = B.cl_units;
    // potential constants of the LJ pair function pinned in registers (otherwise reloaded from the constant bank per pair)
    const float c_band = P.band_abs;
    const float2 c2_nrc2 = make_float2(-P.rc2, -P.rc2), c2_a = make_float2(P.lj_a, P.lj_a), c2_nb = make_float2(-P.lj_b, -P.lj_b),
                 c2_hc = make_float2(0.5f * P.lj_c, 0.5f * P.lj_c), c2_nhd = make_float2(-0.5f * P.lj_d, -0.5f * P.lj_d),
                 c2_nhvs = make_float2(-0.5f * P.vshift, -0.5f * P.vshift);
    for (int c = blockIdx.x * CLF_WARPS + w; c < ncl; c += nwarps) {
        const int i0 = c * MD_CLUSTER;
        const int2 info = B.cl_info[c];
        const int R = info.y;
        const uint2* __restrict__ ul = units + (unsigned int)info.x + lane;
        __syncwarp();                    // the previous cluster's owner rows have been read back (and zeroed)
        if (lane < MD_CLUSTER) {
            const bool ok = i0 + lane < P.N;
            const float4 xo = ok ? pos[i0 + lane] : make_float4(1.0e15f, 1.0e15f, 1.0e15f, 0.f);
            S.px[lane] = xo.x; S.py[lane] = xo.y; S.pz[lane] = xo.z; S.pw[lane] = xo.w;
            if (RIGID) S.qi[lane] = ok ? quat[i0 + lane] : make_float4(1.f, 0.f, 0.f, 0.f);
        }
        // Rounds of 32 units, one per lane; the unit and the gathered position of the NEXT round are in flight while this
        // round's pairs are evaluated.  Units are sorted by popcount, so the lanes of a round hold about the same number of
        // pairs; the warp leaves the inner loop when its longest unit is done.
        uint2 un = R > 0 ? ul[0] : make_uint2(0u, 0u);
        float4 xn = ldg4(pos + (un.x & 0x7fffffffu));
        float4 qn = zero4;
        if (RIGID) qn = ldg4(quat + (un.x & 0x7fffffffu));
        __syncwarp();
        for (int r = 0; r < R; ++r) {
            unsigned int mask = un.y;
            const int j = (int)(un.x & 0x7fffffffu);
            const bool img = (un.x >> 31) != 0u;
            const float4 xj = xn, qj = qn;
            if (r + 1 < R) {
                un = ul[(r + 1) * 32];
                xn = ldg4(pos + (un.x & 0x7fffffffu));
                if (RIGID) qn = ldg4(quat + (un.x & 0x7fffffffu));
            }
            float fjx = 0.f, fjy = 0.f, fjz = 0.f, pej = 0.f, tjx = 0.f, tjy = 0.f, tjz = 0.f;
            if (RIGID) {
                while (mask) {           // one lane-iteration per listed pair
                    const int k = 31 - __clz(mask);
                    mask ^= 1u << k;
                    const float4 xi = make_float4(S.px[k], S.py[k], S.pz[k], 0.f);
                    float dx = xj.x - xi.x, dy = xj.y - xi.y, dz = xj.z - xi.z;
                    if (img) {
                        dx = min_image(xj.x, xi.x, P.Lx, P.hLx); dy = min_image(xj.y, xi.y, P.Ly, P.hLy); dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
                    }
                    const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    if (in_cutoff(P, d2, xi, xj)) {
                        const Rot Ri = quat_to_rot(S.qi[k]);
                        float fx, fy, fz, V, tix, tiy, tiz, ax, ay, az;
                        rigid_pair<true, KIND == MD_POT_PATCHY_PP>(P, dx, dy, dz, d2, Ri, qj, fx, fy, fz, V, tix, tiy, tiz, ax, ay, az);
                        const float hV = 0.5f * V;
                        fjx += fx; fjy += fy; fjz += fz; pej += hV;
                        tjx += ax; tjy += ay; tjz += az;
                        float4 a = S.acc[k * 32 + lane], tq = S.tacc[k * 32 + lane];
                        a.x -= fx; a.y -= fy; a.z -= fz; a.w += hV;
                        tq.x += tix; tq.y += tiy; tq.z += tiz;
                        S.acc[k * 32 + lane] = a; S.tacc[k * 32 + lane] = tq;
                    }
                }
            } else {
                // LJ / WCA: TWO listed pairs of the unit per lane-iteration (owners ka, kb; kb = the dummy owner MD_CLUSTER, parked
                // at 1e15, when the unit has an odd pair left): two independent dependency chains per lane, and the cutoff
                // factor, 1/d2, s6 and the force / energy polynomials of both pairs in packed f32x2 instructions.  The
                // cutoff enters as a 0/1 factor m (s = m / d2): force and energy of an outside pair are exactly zero.
                while (mask) {
                    const int ka = 31 - __clz(mask);
                    mask ^= 1u << ka;
                    int kb = 31 - __clz(mask);                       // -1 when the mask is empty now
                    kb = kb < 0 ? MD_CLUSTER : kb;
                    mask &= ~(1u << kb);
                    const float4 xa = make_float4(S.px[ka], S.py[ka], S.pz[ka], 0.f), xb = make_float4(S.px[kb], S.py[kb], S.pz[kb], 0.f);
                    float dxa = xj.x - xa.x, dya = xj.y - xa.y, dza = xj.z - xa.z;
                    float dxb = xj.x - xb.x, dyb = xj.y - xb.y, dzb = xj.z - xb.z;
                    if (img) {
                        dxa = min_image(xj.x, xa.x, P.Lx, P.hLx); dya = min_image(xj.y, xa.y, P.Ly, P.hLy); dza = min_image(xj.z, xa.z, P.Lz, P.hLz);
                        dxb = min_image(xj.x, xb.x, P.Lx, P.hLx); dyb = min_image(xj.y, xb.y, P.Ly, P.hLy); dzb = min_image(xj.z, xb.z, P.Lz, P.hLz);
                    }
                    const float2 d2 = make_float2(fmaf(dza, dza, fmaf(dya, dya, dxa * dxa)), fmaf(dzb, dzb, fmaf(dyb, dyb, dxb * dxb)));
                    const float2 tt = __fadd2_rn(d2, c2_nrc2);
                    float2 m = make_float2(tt.x < 0.0f ? 1.0f : 0.0f, tt.y < 0.0f ? 1.0f : 0.0f);
                    if (fminf(fabsf(tt.x), fabsf(tt.y)) < c_band) {          // S:Q5 / S:H10: fp64 decision inside the band (rare)
                        if (fabsf(tt.x) < c_band) m.x = inside_fp64(xa, xj, P.dLx, P.dLy, P.dLz, P.rc2d) ? 1.0f : 0.0f;
                        if (fabsf(tt.y) < c_band) m.y = inside_fp64(xb, xj, P.dLx, P.dLy, P.dLz, P.rc2d) ? 1.0f : 0.0f;
                    }
                    const float2 s = __fmul2_rn(make_float2(rcp_approx(d2.x), rcp_approx(d2.y)), m);
                    const float2 z3 = __fmul2_rn(__fmul2_rn(s, s), s);
                    const float2 g = __fmul2_rn(__fmul2_rn(s, z3), __ffma2_rn(c2_a, z3, c2_nb));     // 24 eps s6 (2 s6 - 1) / d2
                    const float2 hV = __ffma2_rn(m, c2_nhvs, __fmul2_rn(z3, __ffma2_rn(c2_hc, z3, c2_nhd)));   // (4 eps s6 (s6 - 1) - V_c) / 2
                    fjx = fmaf(g.x, dxa, fjx); fjy = fmaf(g.x, dya, fjy); fjz = fmaf(g.x, dza, fjz);
                    fjx = fmaf(g.y, dxb, fjx); fjy = fmaf(g.y, dyb, fjy); fjz = fmaf(g.y, dzb, fjz);
                    pej += hV.x + hV.y;
                    float4 a = S.acc[ka * 32 + lane], b = S.acc[kb * 32 + lane];
                    a.x = fmaf(-g.x, dxa, a.x); a.y = fmaf(-g.x, dya, a.y); a.z = fmaf(-g.x, dza, a.z); a.w += hV.x;
                    b.x = fmaf(-g.y, dxb, b.x); b.y = fmaf(-g.y, dyb, b.y); b.z = fmaf(-g.y, dzb, b.z); b.w += hV.y;
                    S.acc[ka * 32 + lane] = a; S.acc[kb * 32 + lane] = b;
                }
            }
            // a unit none of whose pairs is inside the cutoff contributes exact zeros and issues no reduction
            if (fjx != 0.f || fjy != 0.f || fjz != 0.f || pej != 0.f) {
                red_add_v4(force + j, fjx, fjy, fjz, pej);
                if (RIGID) red_add_v4(torque + j, tjx, tjy, tjz, 0.f);
            }
        }
        __syncwarp();
        // owner side: lane l sums half a row (owner l >> 1, columns (l & 1) * 16 ...), entries rotated by the lane so that
        // the 8 lanes of a quarter-warp read 8 different 16-byte columns; rows are zeroed as they are read
        {
            const int k = lane >> 1, h = lane & 1;
            float sx = 0.f, sy = 0.f, sz = 0.f, sw = 0.f, tx = 0.f, ty = 0.f, tz = 0.f;
#pragma unroll
            for (int t = 0; t < 16; ++t) {
                const int col = h * 16 + ((t + lane) & 15);
                const float4 a = S.acc[k * 32 + col];
                S.acc[k * 32 + col] = zero4;
                sx += a.x; sy += a.y; sz += a.z; sw += a.w;
                if (RIGID) {
                    const float4 b = S.tacc[k * 32 + col];
                    S.tacc[k * 32 + col] = zero4;
                    tx += b.x; ty += b.y; tz += b.z;
                }
            }
            sx += __shfl_xor_sync(0xffffffffu, sx, 1); sy += __shfl_xor_sync(0xffffffffu, sy, 1);
            sz += __shfl_xor_sync(0xffffffffu, sz, 1); sw += __shfl_xor_sync(0xffffffffu, sw, 1);
            if (RIGID) {
                tx += __shfl_xor_sync(0xffffffffu, tx, 1); ty += __shfl_xor_sync(0xffffffffu, ty, 1);
                tz += __shfl_xor_sync(0xffffffffu, tz, 1);
            }
            if (h == 0 && i0 + k < P.N && R > 0) {
                red_add_v4(force + i0 + k, sx, sy, sz, sw);
                if (RIGID) red_add_v4(torque + i0 + k, tx, ty, tz, 0.f);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
static int cluster_ucap_w(const md_system* s) { return (8 * s->P.cap + 31) / 32 * 32; }   // units one cluster may hold

static size_t cluster_build_smem(const md_system* s) {
    const size_t per_warp = 32 * (size_t)MD_CLUSTER + 4 * (size_t)(CL_CELLCAP + MD_CLUSTER + 40) + 8 * (size_t)cluster_ucap_w(s);
    return CLB_WARPS * ((per_warp + 15) / 16 * 16);
}

void md_cluster_configure(md_system* s) {
    const int optin = (int)s->smem_optin;
    cudaFuncSetAttribute(k_build_cluster<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_build_cluster<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_edge_cluster<MD_POT_LJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_edge_cluster<MD_POT_PATCHY>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_edge_cluster<MD_POT_PATCHY_PP>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_edge_cluster<MD_POT_LJ>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_edge_cluster<MD_POT_PATCHY>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_edge_cluster<MD_POT_PATCHY_PP>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
}

// the unit list from the cells of the last md_build_cells and the positions `pos_src` (the live positions inside a
// rebuild, the build-time positions pos_ref when the list is made on demand).  false: the build does not fit in shared memory.
bool md_launch_build_cluster(md_system* s, bool gated, const float4* pos_src) {
    const DevParams& P = s->P;
    const int g = gated ? 1 : 0;
    const size_t smem = cluster_build_smem(s);
    if (smem > s->smem_optin) return false;
    const int ncl = (P.N + MD_CLUSTER - 1) / MD_CLUSTER;
    const int write_ref = pos_src != s->B.pos_ref ? 1 : 0;
    k_cluster_begin<<<1, 1, 0, s->stream>>>(s->B, g);
    if (s->order != MD_ORDER_NONE)
        k_build_cluster<true><<<cdiv(ncl, CLB_WARPS), 32 * CLB_WARPS, smem, s->stream>>>(P, s->B, g, pos_src, cluster_ucap_w(s), (unsigned int)s->ucap, write_ref);
    else
        k_build_cluster<false><<<cdiv(ncl, CLB_WARPS), 32 * CLB_WARPS, smem, s->stream>>>(P, s->B, g, pos_src, cluster_ucap_w(s), (unsigned int)s->ucap, write_ref);
    k_cluster_end<<<1, 1, 0, s->stream>>>(s->B, g);
    s->launches += 3;
    return true;
}

template <int KIND>
static void launch_cluster_kind(md_system* s) {
    const size_t smem = CLF_WARPS * sizeof(ClusterSmem<KIND>);
    int per_sm = (int)((s->smem_per_sm - 1024) / (smem + 1024));
    if (per_sm > 8) per_sm = 8;
    if (per_sm < 1) per_sm = 1;
    const int ncl = (s->P.N + MD_CLUSTER - 1) / MD_CLUSTER;
    int grid = s->sm_count * per_sm;
    if (grid > cdiv(ncl, CLF_WARPS)) grid = cdiv(ncl, CLF_WARPS);
    k_edge_cluster<KIND><<<grid, 32 * CLF_WARPS, smem, s->stream>>>(s->P, s->B, s->pos, s->quat, s->force, md_is_rigid(KIND) ? s->torque : nullptr);
    s->launches += 1;
}

// force and torque must have been zeroed by the caller (md_forces.cu launch_edge)
void md_launch_edge_cluster(md_system* s) {
    if (s->P.kind == MD_POT_PATCHY && s->P.pp_model) launch_cluster_kind<MD_POT_PATCHY_PP>(s);
    else if (s->P.kind == MD_POT_PATCHY) launch_cluster_kind<MD_POT_PATCHY>(s);
    else launch_cluster_kind<MD_POT_LJ>(s);
}
