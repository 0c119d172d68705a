// md_staged.cu -- the shared-memory staged path.
//
// Storage is cell-sorted (MD_ORDER_CELL / MD_ORDER_HILBERT), so the particles of a cell are one
// contiguous slot range.  A block owns MD_TB consecutive slots; the union of the 27-cell stencils (P:53
// "standard cell algorithm") of its cells is a short list of contiguous slot SEGMENTS.  Both the Verlet-list
// build and the force kernels first copy those segments into shared memory -- the force kernels with 1-D bulk
// TMA copies (cp.async.bulk + mbarrier) -- and then address neighbours by a 16-bit block-LOCAL index:
//   * the Verlet row of particle i (S:A4) holds |L_i| local indices sorted by slot; entries with slot < i come
//     first, so the EDGE half list (i < j) is the suffix of the same row;
//   * VERTEX and EDGE run one SLICE of 4 or 8 lanes per particle: consecutive lanes read
//     consecutive sorted neighbours, i.e. mostly consecutive float4 in shared memory (few bank conflicts),
//     instead of one 128-byte L1 line per lane from global memory (profiles/r01a_first_path.md).
// The pair arithmetic, the fp64 recheck band (S:H10) and all tolerances are those of md_forces.cu.
#include <stdio.h>
#include <stdlib.h>
#include <algorithm>
#include "md_pair.cuh"

#define GATE(B, gated) if ((gated) && (B).ctrl->rebuild == 0) return

static inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// ------------------------------------------------------------------------------------------------
// PTX wrappers: mbarrier + 1-D bulk TMA copy global -> shared
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, void* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

#define DUMMY_COORD 1.0e15f   // the padding entry of every staged neighbourhood: d2 ~ 3e30, never inside a cutoff

// ------------------------------------------------------------------------------------------------
// block scan over TB threads (exclusive), total in *tot
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int blk_excl_scan(int v, int* tot, int* sh /* >= 33 ints */) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) sh[w] = x;
    __syncthreads();
    if (w == 0) {
        int s = lane < nw ? sh[lane] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += y;
        }
        if (lane < nw) sh[lane] = s;
    }
    __syncthreads();
    const int base = w ? sh[w - 1] : 0;
    *tot = sh[nw - 1];
    __syncthreads();
    return base + x - v;
}

__device__ __forceinline__ int pack_coord(int cx, int cy, int cz) { return cx | (cy << 10) | (cz << 20); }

// Candidate scan of one stencil cell for interior / shift-transformed blocks: all lanes of a warp walk the same cell, so
// the loop is branch-free.  The result is a BITMASK per 32 candidates (bit k = candidate k of the cell is inside r_v,
// from the sign bit of d2 - r_v^2), written with one coalesced 32-bit store per word -- a list of indices would be ~70
// scattered 16-bit stores per thread.  mrow = word 0 of this cell for this thread (words are MD_TB apart).
// self = index of the particle itself in this cell, or -1.  Returns the number of neighbours found.
template <bool SHIFT>
__device__ __forceinline__ int scan_cell_mask(const float4* __restrict__ cellpos, int n, int self, float4 xi, float rv2,
                                              float hLx, float hLy, float hLz, float tLx, float tLy, float tLz,
                                              unsigned int* mrow, float& bandmin) {
    int found = 0;
    for (int k0 = 0; k0 < n; k0 += 32) {
        const int kn = min(32, n - k0);
        unsigned int mask = 0u, bit = 1u;
#pragma unroll 8
        for (int k = 0; k < kn; ++k) {
            float4 xj = __ldg(cellpos + k0 + k);
            if (SHIFT) {
                if (xj.x > hLx) xj.x -= tLx;
                if (xj.y > hLy) xj.y -= tLy;
                if (xj.z > hLz) xj.z -= tLz;
            }
            const float ddx = xj.x - xi.x, ddy = xj.y - xi.y, ddz = xj.z - xi.z;
            const float tt = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx)) - rv2;
            bandmin = fminf(bandmin, fabsf(tt));
            mask |= (unsigned int)(__float_as_int(tt) >> 31) & bit;      // sign bit: inside r_v
            bit <<= 1;
        }
        if ((unsigned int)(self - k0) < 32u) mask &= ~(1u << (self - k0));
        mrow[(size_t)(k0 >> 5) * MD_TB] = mask;
        found += __popc(mask);
    }
    return found;
}

// Candidate scan of one stencil cell FUSED with the column bucketing of pass B (dense cells).  All lanes of a warp walk the
// same cell, candidate by candidate, so the bank column of the candidate (local index & 7) is warp-uniform: the walk is
// aligned to groups of eight local indices and unrolled by eight, which makes the column a compile-time constant of every
// unrolled slot -- the eight column populations pc[] stay in registers with static indexing and a neighbour goes to its
// bucket with one predicated 16-bit store.  No candidate masks are written or decoded (they were 226 MB of scratch traffic
// and a decode loop that ran at 9 of 32 lanes, profiles/r01d_ncu.md).  tb = bucket 0, entry 0 of this thread (entries are
// MD_TB apart, buckets cap8 entries apart); a bucket that outgrows cap8 keeps overwriting its last slot and is reported
// by the caller (pc[u] > cap8).
template <bool SHIFT, bool SELF>
__device__ __forceinline__ void scan_cell_bucket(const float4* __restrict__ cellpos, int n, int t0, int me, float4 xi, float rv2,
                                                 float hLx, float hLy, float hLz, float tLx, float tLy, float tLz,
                                                 unsigned short* __restrict__ tb, int cap8, int (&pc)[8], float& bandmin) {
    const int a = t0 & 7;
    const float4* __restrict__ cp = cellpos - a;     // index kk = candidate + a: local index tb0 + kk has column kk & 7
    const int tb0 = t0 - a, kend = n + a;
    auto one = [&](int u, int kk) {
        float4 xj = __ldg(cp + kk);
        if (SHIFT) {
            if (xj.x > hLx) xj.x -= tLx;
            if (xj.y > hLy) xj.y -= tLy;
            if (xj.z > hLz) xj.z -= tLz;
        }
        const float ddx = xj.x - xi.x, ddy = xj.y - xi.y, ddz = xj.z - xi.z;
        const float tt = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx)) - rv2;
        bandmin = fminf(bandmin, fabsf(tt));
        int m = __float_as_int(tt) >> 31;                    // -1 inside r_v, 0 outside
        const int t = tb0 + kk;
        if (SELF) m = (t == me) ? 0 : m;
        const int p = min(pc[u], cap8 - 1);
        if (m) tb[(size_t)(u * cap8 + p) * MD_TB] = (unsigned short)t;
        pc[u] -= m;
    };
    for (int g = 0; g < kend; g += 8) {
        if (g >= a && g + 8 <= kend) {                       // a full aligned group: no bounds checks
#pragma unroll
            for (int u = 0; u < 8; ++u) one(u, g + u);
        } else {
#pragma unroll
            for (int u = 0; u < 8; ++u)
                if (g + u >= a && g + u < kend) one(u, g + u);
        }
    }
}

// LIST form of the candidate scan, used when cells hold few particles (mask_words == 0: at 2-3 particles per cell 27
// mostly empty mask words per thread cost more than ~10 index stores).  All lanes of a warp walk the same cell, so
// the loop is kept branch-free: a predicated store at the thread's write offset, which advances (by one scratch row)
// when the candidate is inside r_v (sign bit of d2 - r_v^2), clamped at the overflow row cap + 1.
template <bool SHIFT, bool SELF>
__device__ __forceinline__ void scan_cell_fast(const float4* __restrict__ cellpos, int n, int t0, int me, float4 xi, float rv2,
                                               float hLx, float hLy, float hLz, float tLx, float tLy, float tLz,
                                               unsigned short* tmp_blk, unsigned int& off, unsigned int offmax, float& bandmin,
                                               float near_gap) {
    // near_gap = r_v^2 - r_c^2 for the rigid bodies (else a negative number: never near): bit 15 of the stored index marks a
    // neighbour inside the CUTOFF at build time, so that the row can start with the pairs that will be evaluated
#pragma unroll 8
    for (int k = 0; k < n; ++k) {
        float4 xj = __ldg(cellpos + k);
        if (SHIFT) {
            if (xj.x > hLx) xj.x -= tLx;
            if (xj.y > hLy) xj.y -= tLy;
            if (xj.z > hLz) xj.z -= tLz;
        }
        const float ddx = xj.x - xi.x, ddy = xj.y - xi.y, ddz = xj.z - xi.z;
        const float tt = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx)) - rv2;
        bandmin = fminf(bandmin, fabsf(tt));
        int m = __float_as_int(tt) >> 31;                  // -1 inside r_v, 0 outside
        if (SELF) m = (t0 + k == me) ? 0 : m;
        const unsigned int nearbit = (tt + near_gap < 0.0f) ? 0x8000u : 0u;   // d2 < r_c^2
        if (m) *reinterpret_cast<unsigned short*>(reinterpret_cast<char*>(tmp_blk) + off) = (unsigned short)((unsigned int)(t0 + k) | nearbit);
        off = min(off + ((unsigned int)m & (2u * MD_TB)), offmax);
    }
}

// The same scan with every decision taken carefully: minimum image (blocks whose neighbourhood crosses a periodic face
// without a valid shift transform) and the fp64 predicate inside the band (S:Q6).  Rare path.
__device__ __noinline__ int scan_cell_slow(const float4* __restrict__ cellpos, int n, int self, float4 xi,
                                           float Lx, float Ly, float Lz, float rv2, float bandv, double dLx, double dLy,
                                           double dLz, double rv2d, unsigned int* mrow) {
    int found = 0;
    for (int k0 = 0; k0 < n; k0 += 32) {
        const int kn = min(32, n - k0);
        unsigned int mask = 0u;
        for (int k = 0; k < kn; ++k) {
            if (k0 + k == self) continue;
            const float4 xj = __ldg(cellpos + k0 + k);
            // raw (untransformed) coordinates of both particles: the robust minimum image is right for every pair
            const float ddx = min_image(xj.x, xi.x, Lx, 0.5f * Lx), ddy = min_image(xj.y, xi.y, Ly, 0.5f * Ly),
                        ddz = min_image(xj.z, xi.z, Lz, 0.5f * Lz);
            const float tt = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx)) - rv2;
            bool in = tt < 0.0f;
            if (fabsf(tt) < bandv) in = inside_fp64(xi, xj, dLx, dLy, dLz, rv2d);
            if (in) mask |= 1u << k;
        }
        mrow[(size_t)(k0 >> 5) * MD_TB] = mask;
        found += __popc(mask);
    }
    return found;
}

// ------------------------------------------------------------------------------------------------
// S:A4 staged Verlet build.  One block per MD_TB slots, one thread per particle.
// ------------------------------------------------------------------------------------------------
#define TS_CB 24     // transposed scan: hit words (32 candidates each) per owner and pass
#define TS_OC 32     // transposed scan: own cells per block it is sized for (more -> the per-thread scan)
#define TS_ROW (MD_TB + 2 * TS_OC)   // hit words of one chunk: the owners of every own cell start at an even index
#define TS_OFF_HITW (16 * MD_TB)     // after three planes of MD_TB + 2 floats
#define TS_OFF_OWNF (TS_OFF_HITW + 4 * TS_CB * TS_ROW)
#define TS_OFF_PCS (TS_OFF_OWNF + 2 * (5 * (TS_OC + 2) + 28 * TS_OC) + 12)    // 16-byte aligned
#define TS_OFF_CTAB (TS_OFF_PCS + 16 * MD_TB)                                  // direct form: per warp, 28 x 8 column prefixes (bytes)
#define TS_OFF_PRE13 (TS_OFF_CTAB + (MD_TB / 32) * 28 * 8)
#define TS_SMEM_BYTES (TS_OFF_PRE13 + 8 * TS_OC)
static_assert(TS_OFF_PCS % 16 == 0 && TS_OFF_PRE13 % 8 == 0, "shared-memory layout of the transposed scan");

// per-column populations (t & 7 == c, one byte each) of the local-index range [t0, t1)
__device__ __forceinline__ unsigned long long col_counts8(int t0, int t1) {
    unsigned long long r = 0ull;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const int f = t0 + ((c - t0) & 7);
        const int n = f < t1 ? (t1 - f + 7) >> 3 : 0;
        r |= (unsigned long long)n << (8 * c);
    }
    return r;
}
template <bool MASKS>
__global__ void __launch_bounds__(MD_TB, 4) k_build_staged(DevParams P, DevBuffers B, int gated, const float4* __restrict__ pos,
                                                        int ncand_cap, int umax, int tbl_cap) {
    GATE(B, gated);
    extern __shared__ __align__(16) unsigned char smraw[];
    // The build reads candidate positions straight from global memory (all lanes of a warp read the same candidate: one
    // sector, L1-resident), so its shared memory holds only the cell tables and four blocks fit on an SM.
    int* cand = reinterpret_cast<int*>(smraw);                       // [ncand_cap]
    int* urank = cand + (tbl_cap >> 1);                              // [umax]  (cand[]: max(hash set, stencil table) = tbl_cap / 2 ints)
    int* ubase = urank + umax;                                       // [umax + 1]
    int* ustart = ubase + umax + 1;                                  // [umax] first slot of the cell
    int* own_rank = ustart + umax;                                   // [MD_TB]
    int* own_xyz = own_rank + MD_TB;                                 // [MD_TB] packed cell coordinates of the own cells (pack_coord)
    // transposed scan (MASKS variant): owners' positions, hit words, per-own-cell candidate prefixes
    const int ts_off = (4 * ((tbl_cap >> 1) + 3 * umax + 1 + 2 * MD_TB) + 15) & ~15;     // byte offset from smraw: keeps the shared address space
    float* xown = reinterpret_cast<float*>(smraw + ts_off);                           // [3][MD_TB + 2] owners' x, y, z planes (pairs of owners load as f32x2)
    unsigned int* hitw = reinterpret_cast<unsigned int*>(smraw + ts_off + TS_OFF_HITW);   // [TS_CB][TS_ROW]
    unsigned short* own_first = reinterpret_cast<unsigned short*>(smraw + ts_off + TS_OFF_OWNF);   // [TS_OC + 1] first thread of own cell oc
    unsigned short* task_base = own_first + TS_OC + 2;               // [TS_OC + 1] chunks of 32 candidates before own cell oc
    unsigned short* pbase = task_base + TS_OC + 2;                   // [TS_OC + 1] first hit-word index of own cell oc (even)
    unsigned short* nchs = pbase + TS_OC + 2;                        // [TS_OC] direct form: chunks of own cell oc (column-sorted enumeration)
    unsigned short* cbase = nchs + TS_OC + 2;                        // [TS_OC + 1] direct form: chunks before own cell oc
    unsigned short* pref = cbase + TS_OC + 2;                        // [TS_OC][28] candidates before stencil cell sc of own cell oc
    unsigned char* ctab = smraw + ts_off + TS_OFF_CTAB;              // [warps][28][8] direct form: candidates of column c before stencil cell a
    unsigned long long* pre13 = reinterpret_cast<unsigned long long*>(smraw + ts_off + TS_OFF_PRE13);   // [TS_OC] per-column candidates before the own cell
    unsigned short* pcs = reinterpret_cast<unsigned short*>(smraw + ts_off + TS_OFF_PCS);   // [8][MD_TB] column populations of pass B
    __shared__ int sh_scan[33];
    __shared__ int s_tsok, s_direct;
    __shared__ int s_flags, s_err, s_own_base, s_U;

    const int b = blockIdx.x, tid = threadIdx.x;
    const int i0 = b * MD_TB, i1 = min(P.N, i0 + MD_TB);
    const int i = i0 + tid;
    const bool live = i < i1;
    if (tid == 0) { s_flags = 0; s_err = 0; s_own_base = 0; s_U = 0; }

    // cell coordinates of the own cells: three 10-bit fields when every axis has at most 1024 cells, else the linear index
    const bool xyz_packed = P.ncx <= 1024 && P.ncy <= 1024 && P.ncz <= 1024;
    auto cell_xyz = [&](int v, int& cx, int& cy, int& cz) {
        if (xyz_packed) { cx = v & 1023; cy = (v >> 10) & 1023; cz = v >> 20; }
        else { cz = v % P.ncz; cy = (v / P.ncz) % P.ncy; cx = v / (P.ncz * P.ncy); }
    };
    // 1. the block's non-empty cells (storage ranks, ascending), compacted
    const int myrank = live ? B.cell_of[i] : -1;
    const int head = live && (tid == 0 || B.cell_of[i - 1] != myrank) ? 1 : 0;
    int nownc;
    const int oc_ex = blk_excl_scan(head, &nownc, sh_scan);
    if (head) {
        own_rank[oc_ex] = myrank;
        const int lin = B.cell_lin[myrank];      // the divisions by the cell counts happen once per own cell, not per stencil entry
        own_xyz[oc_ex] = xyz_packed ? pack_coord(lin / (P.ncz * P.ncy), (lin / P.ncz) % P.ncy, lin % P.ncz) : lin;
    }
    const int myoc = oc_ex + head - 1;       // ordinal of this thread's cell among the block's own cells
    __syncthreads();

    // 2. candidate cells: the 27-cell stencil of every own cell (S:Q8)
    const int n = 27 * nownc;
    if (n > tbl_cap) {      // the stencil table (27 16-bit entries per own cell, in the storage of the hash set) was sized smaller
        if (tid == 0) { atomicOr(&B.ctrl->err, MD_DEVERR_STAGE); B.blk[b] = BlkInfo{ 0, 0, 0, 0 }; }
        if (live) { B.row_count[i] = 0; B.lo_count[i] = 0; B.half_count[i] = 0; B.pos_ref[i] = pos[i]; }
        return;
    }
    // the candidates go through a shared-memory hash set (cand[], open addressing, native 32-bit CAS): neighbouring own
    // cells share most of their stencils, so only the DISTINCT cells (a few hundred) are compacted and sorted, not the
    // 27 x own-cells candidates (thousands at 2-3 particles per cell)
    const int hmask = ncand_cap - 1;                  // ncand_cap is a power of two >= 2 umax (or > 27 x own cells)
    for (int t = tid; t < ncand_cap; t += MD_TB) cand[t] = 0x7fffffff;
    __syncthreads();
    for (int t = tid; t < n; t += MD_TB) {
        const int s = t % 27;
        int cx, cy, cz;
        cell_xyz(own_xyz[t / 27], cx, cy, cz);
        int ax = cx + s / 9 - 1, ay = cy + (s / 3) % 3 - 1, az = cz + s % 3 - 1;
        int wrapped = 0;   // bit a: the stencil crosses the periodic face of axis a
        if (ax < 0) { ax += P.ncx; wrapped |= 1; } else if (ax >= P.ncx) { ax -= P.ncx; wrapped |= 1; }
        if (ay < 0) { ay += P.ncy; wrapped |= 2; } else if (ay >= P.ncy) { ay -= P.ncy; wrapped |= 2; }
        if (az < 0) { az += P.ncz; wrapped |= 4; } else if (az >= P.ncz) { az -= P.ncz; wrapped |= 4; }
        // fewer than 3 cells on an axis: the wrap lands on a cell of the axis again; the set removes the duplicates
        if (wrapped) atomicOr(&s_flags, wrapped);
        const int r = B.cell_rank[(ax * P.ncy + ay) * P.ncz + az];
        if (B.cell_start[r + 1] > B.cell_start[r]) {      // empty cells contribute nothing
            unsigned int h = ((unsigned int)r * 2654435761u) >> 7;
            for (int probes = 0;; ++probes) {
                if (probes > hmask) { atomicAdd(&s_U, umax + 1); break; }   // set full: more distinct cells than it was sized for
                h &= hmask;
                const int old = atomicCAS(&cand[h], 0x7fffffff, r);
                if (old == 0x7fffffff) {                  // first sighting of this cell: append it to the distinct list
                    const int idx = atomicAdd(&s_U, 1);
                    if (idx < umax) urank[idx] = r;
                    break;
                }
                if (old == r) break;
                ++h;
            }
        }
    }
    __syncthreads();

    // 3. the distinct ranks were appended to urank[0..U) as they entered the set (arbitrary order, sorted next)
    const int U = s_U;
    if (U > umax) {
        if (tid == 0) { atomicOr(&B.ctrl->err, MD_DEVERR_STAGE); B.blk[b] = BlkInfo{ 0, 0, 0, 0 }; }
        if (live) { B.row_count[i] = 0; B.lo_count[i] = 0; B.half_count[i] = 0; B.pos_ref[i] = pos[i]; }
        return;
    }
    // 4. bitonic sort of the distinct ranks (ascending rank = ascending slot)
    int U2 = 32;
    while (U2 < U) U2 <<= 1;                          // U2 <= umax (a power of two)
    if (U <= MD_TB) {
        // few distinct cells (dense cells: ~100): rank sort, one element per thread, two barriers instead of the ~30 of the
        // bitonic network (the values are distinct: position = number of smaller ones)
        int r = 0, p = 0;
        if (tid < U) {
            r = urank[tid];
            for (int x = 0; x < U; ++x) p += urank[x] < r ? 1 : 0;
        }
        __syncthreads();
        if (tid < U) urank[p] = r;
        __syncthreads();
        U2 = 0;                                        // skip the network below
    } else {
        for (int t = U + tid; t < U2; t += MD_TB) urank[t] = 0x7fffffff;
        __syncthreads();
    }
    for (int k = 2; k <= U2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = tid; t < U2; t += MD_TB) {
                const int x = t ^ j;
                if (x > t) {
                    const int a = urank[t], c = urank[x];
                    const bool asc = (t & k) == 0;
                    if ((a > c) == asc) { urank[t] = c; urank[x] = a; }
                }
            }
            __syncthreads();
        }
    }

    // 5. local base of every distinct cell (exclusive scan of the cell populations), packed cell coordinates
    int M = 0;
    for (int base = 0; base < U; base += MD_TB) {
        const int u = base + tid;
        int c = 0;
        if (u < U) {
            const int r = urank[u];
            const int s0 = B.cell_start[r];
            c = B.cell_start[r + 1] - s0;
            ustart[u] = s0;
        }
        int tot;
        const int p = blk_excl_scan(c, &tot, sh_scan);
        if (u < U) ubase[u] = M + p;
        M += tot;
    }
    if (tid == 0) ubase[U] = M;
    if (M + 1 > P.stage_cap) {
        if (tid == 0) { atomicOr(&B.ctrl->err, MD_DEVERR_STAGE); atomicMax(&B.ctrl->max_stage, M + 1); B.blk[b] = BlkInfo{ 0, 0, 0, 0 }; }
        if (live) { B.row_count[i] = 0; B.lo_count[i] = 0; B.half_count[i] = 0; B.pos_ref[i] = pos[i]; }
        return;
    }
    __syncthreads();

    // 6. contiguous slot segments -> global segment table (first slot, first local index)
    int nseg = 0;
    for (int base = 0; base < U; base += MD_TB) {
        const int u = base + tid;
        int f = 0;
        if (u < U) f = (u == 0 || B.cell_start[urank[u - 1] + 1] != B.cell_start[urank[u]]) ? 1 : 0;
        int tot;
        const int p = blk_excl_scan(f, &tot, sh_scan);
        if (f && nseg + p < MD_SEGMAX) B.seg[(size_t)b * MD_SEGMAX + nseg + p] = make_int2(B.cell_start[urank[u]], ubase[u]);
        nseg += tot;
    }
    if (nseg > MD_SEGMAX) {
        if (tid == 0) { atomicOr(&B.ctrl->err, MD_DEVERR_STAGE); B.blk[b] = BlkInfo{ 0, 0, 0, 0 }; }
        if (live) { B.row_count[i] = 0; B.lo_count[i] = 0; B.half_count[i] = 0; B.pos_ref[i] = pos[i]; }
        return;
    }

    // 6b. pack the segment length beside its first local index: seg.y = local << 16 | len (both < 65536), so the force
    //     kernels can issue a segment's bulk copy from its own table entry alone
    {
        __syncthreads();
        int2* sgt = B.seg + (size_t)b * MD_SEGMAX;
        int ys[MD_SEGMAX / MD_TB], ln[MD_SEGMAX / MD_TB];
#pragma unroll
        for (int q = 0; q < MD_SEGMAX / MD_TB; ++q) {
            const int sg = q * MD_TB + tid;
            ys[q] = 0; ln[q] = 0;
            if (sg < nseg) { ys[q] = sgt[sg].y; ln[q] = (sg + 1 < nseg ? sgt[sg + 1].y : M) - ys[q]; }
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < MD_SEGMAX / MD_TB; ++q) {
            const int sg = q * MD_TB + tid;
            if (sg < nseg) sgt[sg].y = (ys[q] << 16) | ln[q];
        }
    }

    // 7. locate the block's own particles in the local index space
    if (tid == 0) {
        const int r0 = own_rank[0];
        int lo = 0, hi = U - 1;
        while (lo < hi) { const int mid = (lo + hi) >> 1; if (urank[mid] < r0) lo = mid + 1; else hi = mid; }
        s_own_base = ubase[lo] + (i0 - B.cell_start[r0]);
    }
    // 7b. stencil table (reuses cand[]): cand[oc * 27 + s] = index into urank of stencil cell s of own cell oc, or -1 for
    //     an empty cell / a cell already listed for this own cell (axes with fewer than 3 cells, S:Q8)
    {
        const bool small_axis = P.ncx < 3 || P.ncy < 3 || P.ncz < 3;
        auto stencil_rank = [&](int xyz, int st) {
            int cx, cy, cz;
            cell_xyz(xyz, cx, cy, cz);
            int ax = cx + st / 9 - 1, ay = cy + (st / 3) % 3 - 1, az = cz + st % 3 - 1;
            if (ax < 0) ax += P.ncx; else if (ax >= P.ncx) ax -= P.ncx;
            if (ay < 0) ay += P.ncy; else if (ay >= P.ncy) ay -= P.ncy;
            if (az < 0) az += P.ncz; else if (az >= P.ncz) az -= P.ncz;
            return B.cell_rank[(ax * P.ncy + ay) * P.ncz + az];
        };
        __syncthreads();   // cand[] is no longer read by the unique pass
        for (int t = tid; t < n; t += MD_TB) {
            const int lin = own_xyz[t / 27];
            const int st = t % 27;
            const int r = stencil_rank(lin, st);
            int lo = 0, hi = U - 1;
            while (lo < hi) { const int mid = (lo + hi) >> 1; if (urank[mid] < r) lo = mid + 1; else hi = mid; }
            int u = (U > 0 && urank[lo] == r) ? lo : -1;
            if (small_axis && u >= 0)
                for (int s2 = 0; s2 < st; ++s2) if (stencil_rank(lin, s2) == r) { u = -1; break; }
            reinterpret_cast<short*>(cand)[t] = (short)u;   // u < umax <= 4096
        }
    }
    __syncthreads();
    const int own_base = s_own_base;
    // 7c. periodic blocks.  wrap_axes = axes on which the neighbourhood crosses a periodic face.  The shift-down transform
    //     T(x) = x > L/2 ? x - L : x (exact in fp32, Sterbenz) turns every minimum image of a listed pair into a plain
    //     difference provided no pair straddles L/2 unwrapped, now or before the next rebuild: guaranteed when no staged
    //     coordinate of a wrapped axis lies within r_v + skin of L/2 (always true unless the box is a few cells wide).
    //     Then the staged copy is transformed and the scan below needs no minimum image; else the block is flagged for
    //     the minimum-image variants of the scan and of the force kernels.
    const int wrap_axes = s_flags & 7;
    __syncthreads();
    if (tid == 0) s_flags = 0;   // from here on: bit a = axis a violates the margin criterion
    __syncthreads();
    if (wrap_axes) {
        // tested per staged CELL (its coordinate interval, widened by 1 % of a cell for the rounding of the binning)
        // instead of per staged position: a superset of the positions, 25x fewer tests
        int bad = 0;
        for (int u = tid; u < U; u += MD_TB) {
            const int lin = B.cell_lin[urank[u]];
            const int cz = lin % P.ncz, cy = (lin / P.ncz) % P.ncy, cx = lin / (P.ncz * P.ncy);
            auto near_half = [&](int c, double cscale, float hL) {
                const float lo = (float)(((double)c - 0.01) / cscale), hi = (float)(((double)c + 1.01) / cscale);
                return lo <= hL + P.shift_margin && hi >= hL - P.shift_margin;
            };
            if ((wrap_axes & 1) && near_half(cx, P.cscale_x, P.hLx)) bad |= 1;
            if ((wrap_axes & 2) && near_half(cy, P.cscale_y, P.hLy)) bad |= 2;
            if ((wrap_axes & 4) && near_half(cz, P.cscale_z, P.hLz)) bad |= 4;
        }
        if (bad) atomicOr(&s_flags, bad);
    }
    __syncthreads();
    const bool small_box = P.ncx < 3 || P.ncy < 3 || P.ncz < 3;
    const bool shift_ok = wrap_axes != 0 && (s_flags & 7) == 0 && !small_box;
    const bool maywrap = (wrap_axes != 0 && !shift_ok) || small_box;
    // the transform is applied on the fly to the coordinates this kernel reads (and to the staged copy in the force kernels)
    const float tLx = (shift_ok && (wrap_axes & 1)) ? P.Lx : 0.0f, tLy = (shift_ok && (wrap_axes & 2)) ? P.Ly : 0.0f,
                tLz = (shift_ok && (wrap_axes & 4)) ? P.Lz : 0.0f;
    auto load_pos = [&](int slot) {
        float4 x = __ldg(pos + slot);
        if (shift_ok) {
            if (x.x > P.hLx) x.x -= tLx;
            if (x.y > P.hLy) x.y -= tLy;
            if (x.z > P.hLz) x.z -= tLz;
        }
        return x;
    };

    // 8. L_i = { j != i : d2 < r_v^2 }, fp32 filter + fp64 decision inside the band (S:Q6).  Pass A leaves, per
    //    stencil cell, a bitmask of the candidates inside r_v (scan_cell_mask); pass B turns the masks into the row.
    int cnt = 0, lo_cnt = 0;
    bool bucketed = false, bucket_over = false;                   // dense cells: the scan already filled the column buckets
    // Rigid bodies (few, expensive pairs; half of the listed pairs outside r_c): rows start with the neighbours that were
    // inside the CUTOFF at build time, in scan order, instead of being scheduled by bank column (their 12-entry rows put no
    // load on the shared-memory pipe).  The lanes of a warp then meet the pairs they evaluate at the same row positions
    // and the in-cutoff branch of the force kernel diverges only where a pair has crossed r_c since the build.
    const bool near_first = !MASKS && P.kind == MD_POT_PATCHY && P.row_schedule && P.stage_cap < 32768;
    unsigned long long pops_pre = 0ull;
    const int W = P.mask_words;                                   // 32-bit mask words per stencil cell
    constexpr bool use_masks = MASKS;                             // else: list form (few particles per cell)
    unsigned int* cm = B.cmask + (size_t)b * 27 * W * MD_TB + tid;   // word (cell sc, w) at cm[(sc * W + w) * MD_TB]
    const int cap8 = (P.rcap + 2) >> 1;                             // capacity of one column bucket of pass B
    unsigned short* tmp_blk = B.rows_tmp + ((size_t)P.nblk * 8 * cap8 + (size_t)b * (P.rcap + 2)) * MD_TB;   // list form: neighbours in scan order
    unsigned short* tmp = tmp_blk + tid;
    const short* __restrict__ mycells = reinterpret_cast<const short*>(cand) + max(myoc, 0) * 27;
    const int me = own_base + tid;
    // 8a. TRANSPOSED scan (dense cells, no minimum image needed).  The per-thread scan below spends 58 issue slots per
    //     candidate (lanes in different own cells diverge, ragged cell heads and tails, bucket bookkeeping on every
    //     candidate).  Here a warp takes one own cell and 32 of the candidates of its stencil (enumerated across the 27
    //     cells, so every lane holds one): the lane keeps ITS candidate in registers and the warp walks the owners of the
    //     cell, whose position is one broadcast shared-memory load -- ~15 instructions per 32 tests, one ballot word per
    //     (owner, 32 candidates).  Each owner thread then turns its hit words into the column buckets of pass B.  The band
    //     decision (S:Q6) is taken in place, in fp64 on the raw coordinates, by the lanes that meet it.
    bool tdone = false;
    bool tdirect = false;                   // direct form: rows emitted from the hit words (8b), no buckets
    int d_myhw = 0, d_nch = 0;              // this thread's hit words: hitw[j * TS_ROW + d_myhw], j < d_nch
    unsigned long long d_rem = 0ull;        // neighbours per column, one byte each
    const unsigned short* d_cl = nullptr;   // candidate list of the thread's own cell: local index of (chunk j, lane l) at [j * 32 + l]
    if (MASKS && !maywrap && nownc <= TS_OC) {
        const int lane = tid & 31, wid = tid >> 5;
        if (tid == 0) s_tsok = 1;
        if (head) own_first[myoc] = (unsigned short)tid;
        if (tid == 0) own_first[nownc] = (unsigned short)(i1 - i0);
        { const float4 xo = live ? load_pos(i) : make_float4(DUMMY_COORD, DUMMY_COORD, DUMMY_COORD, 0.f);
          xown[tid] = xo.x; xown[MD_TB + 2 + tid] = xo.y; xown[2 * (MD_TB + 2) + tid] = xo.z; }
        // per own cell: candidates before every stencil cell (pref), per-column totals -> chunks of the direct form (nchs),
        // per-column candidates before the own cell itself (pre13).  One warp per own cell, lane a = stencil cell a.
        for (int oc = wid; oc < nownc; oc += MD_TB / 32) {
            int n = 0;
            unsigned long long cc8 = 0ull;                      // per-column candidate counts of the lane's cell, one byte each
            if (lane < 27) {
                const int u = reinterpret_cast<const short*>(cand)[oc * 27 + lane];
                if (u >= 0) { const int t0 = ubase[u], t1 = ubase[u + 1]; n = t1 - t0; cc8 = col_counts8(t0, t1); }
            }
            int ninc = n;
            unsigned long long cinc = cc8;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, ninc, d);
                const unsigned long long z = __shfl_up_sync(0xffffffffu, cinc, d);
                if (lane >= d) { ninc += y; cinc += z; }
            }
            if (lane < 28) pref[oc * 28 + lane] = (unsigned short)min(ninc - n, 65535);
            if (lane == 13) pre13[oc] = cinc - cc8;
            if (lane == 27) {
                int mx = 0;
#pragma unroll
                for (int c = 0; c < 8; ++c) mx = max(mx, (int)((cinc >> (8 * c)) & 255ull));
                // a column holds at most total / 8 + 27 candidates: no byte overflows while total <= 32 TS_CB
                nchs[oc] = (unsigned short)(ninc <= 32 * TS_CB ? (mx + 3) >> 2 : 0xffff);
            }
        }
        __syncthreads();
        if (wid == 0) {
            // exclusive prefixes over the own cells (nownc <= 32: lane = own cell): chunks of the bucket form (task_base), owner
            // pairs from an even thread (pbase), chunks of the direct form (cbase)
            const bool in = lane < nownc;
            const int ch = in ? ((int)pref[lane * 28 + 27] + 31) >> 5 : 0;
            const int pw2 = in ? (((int)own_first[lane + 1] + 1) & ~1) - ((int)own_first[lane] & ~1) : 0;
            const int nd = in ? (int)nchs[lane] : 0;
            const bool dok = nd <= TS_CB;
            int a1 = ch, a2 = pw2, a3 = dok ? nd : 0;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int y1 = __shfl_up_sync(0xffffffffu, a1, d), y2 = __shfl_up_sync(0xffffffffu, a2, d), y3 = __shfl_up_sync(0xffffffffu, a3, d);
                if (lane >= d) { a1 += y1; a2 += y2; a3 += y3; }
            }
            if (in) {
                task_base[lane] = (unsigned short)min(a1 - ch, 65535);
                pbase[lane] = (unsigned short)(a2 - pw2);
                cbase[lane] = (unsigned short)(a3 - (dok ? nd : 0));
            }
            const int tb = __shfl_sync(0xffffffffu, a1, 31), cb = __shfl_sync(0xffffffffu, a3, 31);
            const int mx = __reduce_max_sync(0xffffffffu, ch);
            const bool alld = __all_sync(0xffffffffu, dok);
            if (lane == 0) {
                task_base[nownc] = (unsigned short)min(tb, 65535);
                // the candidate lists (local index of candidate k of own cell oc) live in this block's part of the mask scratch
                const size_t capu16 = (size_t)2 * 27 * P.mask_words * MD_TB;
                if ((size_t)tb * 32 > capu16 || tb > 65535) s_tsok = 0;
                s_U = mx;       // most chunks of any own cell (s_U is free after step 3)
                // direct form: every own cell fits one pass of hit words in its column-sorted enumeration
                s_direct = (P.build_direct && alld && (size_t)cb * 32 <= capu16) ? 1 : 0;
            }
        }
        __syncthreads();
        if (s_tsok && s_direct) {
            // DIRECT form.  The candidates of an own cell's stencil are enumerated BY BANK COLUMN: lane l of chunk j holds
            // candidate 4 j + (l & 3) of column l >> 2 (column = local index & 7), in stencil order within the column.  A hit
            // word then holds one nibble per column; transposed per owner (below) the nibbles of a column form a bit string
            // whose bit r is "candidate r of the column is a neighbour", and the scheduled emission of 8b takes "the next
            // neighbour of column c" with one find-first-set: no buckets in scratch memory, no decode pass.  One warp takes a
            // whole own cell, chunk after chunk.
            tdone = true;
            tdirect = true;
            unsigned short* __restrict__ clist = reinterpret_cast<unsigned short*>(B.cmask + (size_t)b * 27 * P.mask_words * MD_TB);
            const short* __restrict__ cand_s = reinterpret_cast<const short*>(cand);
            const float rv2 = P.rv2, bandv = P.band_rv;
            const float* __restrict__ xox = xown, * __restrict__ xoy = xown + MD_TB + 2, * __restrict__ xoz = xown + 2 * (MD_TB + 2);
            unsigned char* __restrict__ tab = ctab + wid * (28 * 8);       // tab[a * 8 + c]
            for (int oc = wid; oc < nownc; oc += MD_TB / 32) {
                const int nch = nchs[oc];
                const int o0 = own_first[oc], o1 = own_first[oc + 1];
                const int c = lane >> 2, q = lane & 3;
                // per-column prefix table of the 27 stencil cells: lane a takes cell a, an exclusive warp scan of the packed
                // byte counts (no byte overflows: see nchs), one 64-bit store per cell
                int ct0 = 0, cus = 0;
                unsigned long long cc8 = 0ull;
                if (lane < 27) {
                    const int u = cand_s[oc * 27 + lane];
                    if (u >= 0) { ct0 = ubase[u]; cc8 = col_counts8(ct0, ubase[u + 1]); cus = ustart[u] - ct0; }
                }
                unsigned long long inc = cc8;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const unsigned long long y = __shfl_up_sync(0xffffffffu, inc, d);
                    if (lane >= d) inc += y;
                }
                __syncwarp();                                       // the table of the previous own cell is no longer read
                if (lane < 28) *reinterpret_cast<unsigned long long*>(tab + lane * 8) = inc - cc8;
                __syncwarp();
                unsigned int* __restrict__ hw0 = hitw + (int)pbase[oc] - (o0 & ~1);
                unsigned short* __restrict__ clo = clist + (size_t)cbase[oc] * 32;
                const int ncol = tab[27 * 8 + c];                   // candidates of the lane's column
                // the lane's rank grows by 4 per chunk: it walks the cells of its column forwards (a = last cell whose
                // prefix pa is <= r, pn = prefix of the next cell)
                int a = 0, pa = 0, pn = tab[8 + c];
                for (int j = 0; j < nch; ++j) {
                    const int r = 4 * j + q;
                    const bool valid = r < ncol;
                    while (a < 26 && pn <= r) { ++a; pa = pn; pn = tab[(a + 1) * 8 + c]; }
                    // the cell's first local index and slot offset come from the lane that holds cell a
                    const int t0 = __shfl_sync(0xffffffffu, ct0, a), usl = __shfl_sync(0xffffffffu, cus, a);
                    const int t = t0 + ((c - t0) & 7) + 8 * (r - pa);
                    const int slot = valid ? usl + t : 0;
                    float4 xj = make_float4(DUMMY_COORD, DUMMY_COORD, DUMMY_COORD, 0.f);
                    if (valid) {
                        xj = load_pos(slot);
                        clo[j * 32 + lane] = (unsigned short)t;
                    }
                    unsigned int* __restrict__ hw = hw0 + j * TS_ROW;      // hw[o]: word of owner thread o
                    unsigned int hp = smem_u32(hw + (o0 & ~1));             // running shared-memory address of the pair's two words
                    float bmin = 3.0e38f;
                    const float2 nxjx = make_float2(-xj.x, -xj.x), nxjy = make_float2(-xj.y, -xj.y), nxjz = make_float2(-xj.z, -xj.z);
                    const float2 nrv2 = make_float2(-rv2, -rv2);
#pragma unroll 2
                    for (int o = o0 & ~1; o < o1; o += 2) {
                        const float2 ox = *reinterpret_cast<const float2*>(xox + o), oy = *reinterpret_cast<const float2*>(xoy + o),
                                     oz = *reinterpret_cast<const float2*>(xoz + o);
                        const float2 ddx = __fadd2_rn(ox, nxjx), ddy = __fadd2_rn(oy, nxjy), ddz = __fadd2_rn(oz, nxjz);
                        const float2 d2 = __ffma2_rn(ddz, ddz, __ffma2_rn(ddy, ddy, __fmul2_rn(ddx, ddx)));
                        const float2 tt = __fadd2_rn(d2, nrv2);
                        bmin = fminf(fminf(bmin, fabsf(tt.x)), fabsf(tt.y));
                        const unsigned int wa = __ballot_sync(0xffffffffu, tt.x < 0.0f);
                        const unsigned int wb = __ballot_sync(0xffffffffu, tt.y < 0.0f);
                        if (lane == 0) asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(hp), "r"(wa), "r"(wb) : "memory");   // padded layout: always in range
                        hp += 8u;
                    }
                    if (__any_sync(0xffffffffu, bmin < bandv)) {    // rare: a pair inside the band -> fp64 on the raw coordinates (S:Q6)
                        for (int o = o0; o < o1; ++o) {
                            const float ddx = xj.x - xox[o], ddy = xj.y - xoy[o], ddz = xj.z - xoz[o];
                            const float tt = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx)) - rv2;
                            bool in = tt < 0.0f;
                            if (fabsf(tt) < bandv) in = inside_fp64(__ldg(pos + i0 + o), __ldg(pos + slot), P.dLx, P.dLy, P.dLz, P.rv2d);
                            const unsigned int word = __ballot_sync(0xffffffffu, in);
                            if (lane == 0) hw[o] = word;
                        }
                    }
                }
            }
            __syncthreads();
            if (live) {
                d_nch = nchs[myoc];
                d_myhw = (int)pbase[myoc] + tid - ((int)own_first[myoc] & ~1);
                d_cl = clist + (size_t)cbase[myoc] * 32;
                unsigned int* myw = hitw + d_myhw;
                {   // the particle itself is a hit of its own column: clear it
                    const int cme = me & 7;
                    const int t0 = ubase[cand_s[myoc * 27 + 13]];
                    const int f = t0 + ((cme - t0) & 7);
                    const int rs = (int)((pre13[myoc] >> (8 * cme)) & 255ull) + ((me - f) >> 3);
                    myw[(rs >> 2) * TS_ROW] &= ~(1u << (cme * 4 + (rs & 3)));
                }
                // transpose, in place, eight words at a time: word (8 g + c) becomes the bit string of column c over the chunks
                // 8 g .. 8 g + 7 (bit 4 jj + q = candidate 4 (8 g + jj) + q of the column)
                unsigned long long rem = 0ull;
                for (int g = 0; 8 * g < d_nch; ++g) {
                    unsigned int x[8];
#pragma unroll
                    for (int jj = 0; jj < 8; ++jj) x[jj] = 8 * g + jj < d_nch ? myw[(8 * g + jj) * TS_ROW] : 0u;
                    // 8 x 8 nibble transpose: three butterfly stages (16-, 8-, 4-bit blocks)
#pragma unroll
                    for (int i = 0; i < 4; ++i) { const unsigned int t = ((x[i] >> 16) ^ x[i + 4]) & 0x0000ffffu; x[i + 4] ^= t; x[i] ^= t << 16; }
#pragma unroll
                    for (int i = 0; i < 8; ++i) if (!(i & 2)) { const unsigned int t = ((x[i] >> 8) ^ x[i + 2]) & 0x00ff00ffu; x[i + 2] ^= t; x[i] ^= t << 8; }
#pragma unroll
                    for (int i = 0; i < 8; i += 2) { const unsigned int t = ((x[i] >> 4) ^ x[i + 1]) & 0x0f0f0f0fu; x[i + 1] ^= t; x[i] ^= t << 4; }
#pragma unroll
                    for (int cc = 0; cc < 8; ++cc) {
                        myw[(8 * g + cc) * TS_ROW] = x[cc];
                        rem += (unsigned long long)__popc(x[cc]) << (8 * cc);
                    }
                }
                d_rem = rem;
#pragma unroll
                for (int cc = 0; cc < 8; ++cc) cnt += (int)((rem >> (8 * cc)) & 255ull);
            }
        } else if (s_tsok) {
            tdone = true;
            const int ntask = task_base[nownc], maxch = s_U;
            unsigned short* __restrict__ clist = reinterpret_cast<unsigned short*>(B.cmask + (size_t)b * 27 * P.mask_words * MD_TB);
            const short* __restrict__ cand_s = reinterpret_cast<const short*>(cand);
            const float rv2 = P.rv2, bandv = P.band_rv;
            unsigned short* __restrict__ tmp2 = B.rows_tmp + (size_t)b * 8 * cap8 * MD_TB + tid;
            const int plim = min(cap8, 255);
            bool over = false;
#pragma unroll
            for (int c = 0; c < 8; ++c) pcs[c * MD_TB + tid] = 0;
            for (int cb0 = 0; cb0 < maxch; cb0 += TS_CB) {
                if (cb0) __syncthreads();       // the hit words of the previous pass have been consumed
                int oc = 0;
                for (int tk = wid; tk < ntask; tk += MD_TB / 32) {
                    while ((int)task_base[oc + 1] <= tk) ++oc;      // own cell of the task (tasks ascend)
                    const int chunk = tk - (int)task_base[oc];
                    if (chunk < cb0 || chunk >= cb0 + TS_CB) continue;
                    // candidate k of the own cell's stencil -> (stencil cell, rank in it): binary search over the 27 prefixes,
                    // held one per lane
                    const int prl = pref[oc * 28 + min(lane, 27)];
                    const int ktot = __shfl_sync(0xffffffffu, prl, 27);
                    const int k = chunk * 32 + lane;
                    const bool valid = k < ktot;
                    int a = 0;
#pragma unroll
                    for (int st = 16; st > 0; st >>= 1) {
                        const int pm = __shfl_sync(0xffffffffu, prl, min(a + st, 26));
                        if (a + st <= 26 && pm <= k) a += st;
                    }
                    float4 xj = make_float4(DUMMY_COORD, DUMMY_COORD, DUMMY_COORD, 0.f);
                    int slot = 0;
                    const int pa = __shfl_sync(0xffffffffu, prl, a);
                    if (valid) {
                        const int u = cand_s[oc * 27 + a];          // pr[a] <= k < pr[a + 1]: cell a is not empty, so u >= 0
                        const int r = k - pa;
                        slot = ustart[u] + r;
                        xj = load_pos(slot);
                        clist[(size_t)tk * 32 + lane] = (unsigned short)(ubase[u] + r);
                    }
                    const int o0 = own_first[oc], o1 = own_first[oc + 1];
                    unsigned int* __restrict__ hw = hitw + (chunk - cb0) * TS_ROW + (int)pbase[oc] - (o0 & ~1);   // hw[o]: words of owner thread o
                    unsigned int* __restrict__ hwc = hw;
                    // two owners per step in packed f32x2 (FADD2 / FMUL2 / FFMA2): pairs start at even threads, the owner
                    // before o0 / after o1 - 1 of a ragged end is computed and not stored
                    float bmin = 3.0e38f;
                    const float2 nxjx = make_float2(-xj.x, -xj.x), nxjy = make_float2(-xj.y, -xj.y), nxjz = make_float2(-xj.z, -xj.z);   // (a - b)^2 == (b - a)^2 exactly
                    const float2 nrv2 = make_float2(-rv2, -rv2);
                    const float* __restrict__ xox = xown, * __restrict__ xoy = xown + MD_TB + 2, * __restrict__ xoz = xown + 2 * (MD_TB + 2);
#pragma unroll 2
                    for (int o = o0 & ~1; o < o1; o += 2) {
                        const float2 ox = *reinterpret_cast<const float2*>(xox + o), oy = *reinterpret_cast<const float2*>(xoy + o),
                                     oz = *reinterpret_cast<const float2*>(xoz + o);
                        const float2 ddx = __fadd2_rn(ox, nxjx), ddy = __fadd2_rn(oy, nxjy), ddz = __fadd2_rn(oz, nxjz);
                        const float2 d2 = __ffma2_rn(ddz, ddz, __ffma2_rn(ddy, ddy, __fmul2_rn(ddx, ddx)));
                        const float2 tt = __fadd2_rn(d2, nrv2);
                        bmin = fminf(fminf(bmin, fabsf(tt.x)), fabsf(tt.y));
                        const unsigned int wa = __ballot_sync(0xffffffffu, tt.x < 0.0f);
                        const unsigned int wb = __ballot_sync(0xffffffffu, tt.y < 0.0f);
                        if (lane == 0) *reinterpret_cast<uint2*>(hwc + o) = make_uint2(wa, wb);   // padded layout: always in range
                    }
                    const bool banded = bmin < bandv;
                    if (__any_sync(0xffffffffu, banded)) {          // rare: a pair inside the band -> fp64 on the raw coordinates (S:Q6)
                        for (int o = o0; o < o1; ++o) {
                            const float ddx = xj.x - xox[o], ddy = xj.y - xoy[o], ddz = xj.z - xoz[o];
                            const float tt = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx)) - rv2;
                            bool in = tt < 0.0f;
                            if (fabsf(tt) < bandv) in = inside_fp64(__ldg(pos + i0 + o), __ldg(pos + slot), P.dLx, P.dLy, P.dLz, P.rv2d);
                            const unsigned int word = __ballot_sync(0xffffffffu, in);
                            if (lane == 0) hw[o] = word;
                        }
                    }
                }
                __syncthreads();
                if (live) {
                    const int nw = min(TS_CB, (((int)pref[myoc * 28 + 27] + 31) >> 5) - cb0);
                    const int myhw = (int)pbase[myoc] + tid - ((int)own_first[myoc] & ~1);
                    const unsigned short* cl = clist + ((size_t)task_base[myoc] + cb0) * 32;
                    // one flat loop over the set bits of all hit words (a loop per word would run at the pace of the lane with
                    // the most hits in that word); the candidate-list entry of the NEXT hit is requested before the current one
                    // is filed, so the two memory latencies overlap
                    int w = -1;
                    unsigned int bits = 0u;
                    auto next_hit = [&]() {
                        while (bits == 0u) {
                            if (++w >= nw) return -1;
                            bits = hitw[w * TS_ROW + myhw];
                        }
                        const int bit = __ffs(bits) - 1;
                        bits &= bits - 1u;
                        return w * 32 + bit;
                    };
                    int idx = next_hit();
                    int tn = idx >= 0 ? (int)cl[idx] : me;
                    while (idx >= 0) {
                        const int t = tn;
                        idx = next_hit();
                        if (idx >= 0) tn = cl[idx];
                        if (t != me) {
                            const int c = t & 7;
                            const int pp = (int)pcs[c * MD_TB + tid];
                            if (pp < plim) { tmp2[(size_t)(c * cap8 + pp) * MD_TB] = (unsigned short)t; pcs[c * MD_TB + tid] = (unsigned short)(pp + 1); } else over = true;
                        }
                    }
                }
            }
            if (live) {
                unsigned long long pops = 0ull;
#pragma unroll
                for (int c = 0; c < 8; ++c) { const int pc1 = (int)pcs[c * MD_TB + tid]; cnt += pc1; pops |= (unsigned long long)pc1 << (8 * c); }
                pops_pre = pops;
                bucketed = true;
                bucket_over = over;
            }
        }
    }
    if (live) {
        const float4 xi_raw = __ldg(pos + i);
        const float4 xi = load_pos(i);
        const float hLx = P.hLx, hLy = P.hLy, hLz = P.hLz;
        float bandmin = maywrap ? 0.0f : 3.0e38f;                 // maywrap blocks go straight to the careful scan
        if (tdone) {
            // the transposed scan above has filled the buckets
        } else if (!maywrap && !use_masks) {
            const float rv2 = P.rv2;
            const float near_gap = near_first ? P.rv2 - P.rc2 : -1.0f;
            unsigned int off = 2u * tid;
            const unsigned int offmax = (unsigned int)(P.cap + 1) * (2u * MD_TB) + 2u * tid;
            for (int sc = 0; sc < 27; ++sc) {
                const int u = mycells[sc];
                if (u < 0) continue;
                const int t0 = ubase[u], n = ubase[u + 1] - t0;
                const float4* cellpos = pos + ustart[u];
                if (sc == 13) {                           // stencil entry 13 is the own cell: exclude the particle itself
                    if (shift_ok) scan_cell_fast<true, true>(cellpos, n, t0, me, xi, rv2, hLx, hLy, hLz, tLx, tLy, tLz, tmp_blk, off, offmax, bandmin, near_gap);
                    else scan_cell_fast<false, true>(cellpos, n, t0, me, xi, rv2, hLx, hLy, hLz, tLx, tLy, tLz, tmp_blk, off, offmax, bandmin, near_gap);
                } else {
                    if (shift_ok) scan_cell_fast<true, false>(cellpos, n, t0, me, xi, rv2, hLx, hLy, hLz, tLx, tLy, tLz, tmp_blk, off, offmax, bandmin, near_gap);
                    else scan_cell_fast<false, false>(cellpos, n, t0, me, xi, rv2, hLx, hLy, hLz, tLx, tLy, tLz, tmp_blk, off, offmax, bandmin, near_gap);
                }
            }
            cnt = (int)((off - 2u * tid) / (2u * MD_TB));   // cap + 1 = overflow
        } else if (!maywrap) {
            const float rv2 = P.rv2;
            unsigned short* __restrict__ tb = B.rows_tmp + (size_t)b * 8 * cap8 * MD_TB + tid;
            int pc[8] = { 0, 0, 0, 0, 0, 0, 0, 0 };
            for (int sc = 0; sc < 27; ++sc) {
                const int u = mycells[sc];
                if (u < 0) continue;
                const int t0 = ubase[u];
                int n = ubase[u + 1] - t0;
                if (n > 32 * W) { n = 32 * W; atomicOr(&B.ctrl->err, MD_DEVERR_STAGE); }   // cell fuller than the mask capacity of the careful path
                const float4* cellpos = pos + ustart[u];
                if (sc == 13) {                           // stencil entry 13 is the own cell: exclude the particle itself
                    if (shift_ok) scan_cell_bucket<true, true>(cellpos, n, t0, me, xi, rv2, hLx, hLy, hLz, tLx, tLy, tLz, tb, cap8, pc, bandmin);
                    else scan_cell_bucket<false, true>(cellpos, n, t0, me, xi, rv2, hLx, hLy, hLz, tLx, tLy, tLz, tb, cap8, pc, bandmin);
                } else {
                    if (shift_ok) scan_cell_bucket<true, false>(cellpos, n, t0, me, xi, rv2, hLx, hLy, hLz, tLx, tLy, tLz, tb, cap8, pc, bandmin);
                    else scan_cell_bucket<false, false>(cellpos, n, t0, me, xi, rv2, hLx, hLy, hLz, tLx, tLy, tLz, tb, cap8, pc, bandmin);
                }
            }
            bucketed = true;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                cnt += pc[c];
                if (pc[c] > cap8 || pc[c] > 255) bucket_over = true;
                pops_pre |= (unsigned long long)(pc[c] & 255) << (8 * c);
            }
        }
        if (bandmin < P.band_rv) {      // rare: a banded candidate (or a block that needs the minimum image)
            cnt = 0;
            bucketed = false;           // the careful scan leaves masks: pass B decodes them (and overwrites the buckets)
            for (int sc = 0; sc < 27; ++sc) {
                const int u = mycells[sc];
                if (u < 0) continue;
                const int t0 = ubase[u];
                int n = ubase[u + 1] - t0;
                if (n > 32 * W) { n = 32 * W; atomicOr(&B.ctrl->err, MD_DEVERR_STAGE); }
                const int self = (me >= t0 && me < t0 + n) ? me - t0 : -1;   // (small boxes: the own cell may sit elsewhere in the stencil)
                cnt += scan_cell_slow(pos + ustart[u], n, self, xi_raw, P.Lx, P.Ly, P.Lz, P.rv2, P.band_rv, P.dLx, P.dLy, P.dLz,
                                      P.rv2d, cm + (size_t)sc * W * MD_TB);
            }
            if (!use_masks) {           // list form: expand the careful masks into the scan-order list
                int k = 0;
                for (int sc = 0; sc < 27; ++sc) {
                    const int u = mycells[sc];
                    if (u < 0) continue;
                    const int t0 = ubase[u];
                    const int nw = min(W, (ubase[u + 1] - t0 + 31) >> 5);
                    for (int w = 0; w < nw; ++w) {
                        unsigned int m = cm[(size_t)(sc * W + w) * MD_TB];
                        while (m) {
                            const int bit = __ffs(m) - 1;
                            m &= m - 1;
                            if (k < P.cap) tmp[(size_t)k * MD_TB] = (unsigned short)(t0 + 32 * w + bit);
                            ++k;
                        }
                    }
                }
            }
        }
        if (cnt > P.cap) atomicOr(&B.ctrl->err, MD_DEVERR_CAPACITY);
    }
    // every set bit of the thread's masks = one neighbour (local index t), visited cell by cell in ascending t
    auto for_each_neighbour = [&](auto&& f) {
        if (!use_masks) {
            const int c2l = min(cnt, P.cap);
            for (int k = 0; k < c2l; ++k) f((int)(tmp[(size_t)k * MD_TB] & 0x7fffu));
            return;
        }
        for (int sc = 0; sc < 27; ++sc) {
            const int u = mycells[sc];
            if (u < 0) continue;
            const int t0 = ubase[u];
            const int nw = min(W, (ubase[u + 1] - t0 + 31) >> 5);
            for (int w = 0; w < nw; ++w) {
                unsigned int m = cm[(size_t)(sc * W + w) * MD_TB];
                const int tb = t0 + 32 * w;
                while (m) { const int bit = __ffs(m) - 1; m &= m - 1; f(tb + bit); }
            }
        }
    };
    // 8b. Pass B: emit the row in the order the force kernels read it.  Thread tid (lane p of its quarter-warp) reads
    //     entry k at the same time as the 7 other lanes of the quarter read theirs; a 128-bit shared-memory gather is
    //     conflict-free when the 8 lanes hit 8 different columns, so lane p takes, at step k, a neighbour of column
    //     (k + p) mod 8 while it has one (else of its fullest column).  Row layout: block-transposed chunks of four
    //     16-bit local indices, rows[((b * nchunk) + k/4) * MD_TB + tid] -> one coalesced 64-bit load per 4 visits.
    {
        const int c2 = (live && cnt <= P.cap) ? cnt : 0;
        const int nchunk = P.rcap >> 2;
        uint2* __restrict__ rowb = reinterpret_cast<uint2*>(B.rows) + (size_t)b * nchunk * MD_TB + tid;
        unsigned int w[4] = { 0u, 0u, 0u, 0u };
        const int rsh = (M + 1 <= 4096) ? 4 : 0;   // MD_BLK_SH4: entries are byte offsets into the staged float4 array
        const unsigned int dummy = (unsigned int)M << rsh;
        // one decoding sweep drops every neighbour into the bucket of its column (8 buckets of cap8 entries: a column with
        // more than half a row's capacity is reported as a capacity error)
        unsigned short* __restrict__ tmp2 = B.rows_tmp + (size_t)b * 8 * cap8 * MD_TB + tid;
        // the eight column populations live in one 64-bit register, 8 bits each (a column holds <= cap8 <= 255 entries)
        unsigned long long pops = 0ull, rem8 = 0ull;
        int c2e = c2;                                      // entries to emit (0 after a bucket overflow)
        int lo_e = 0;                                      // neighbours with a lower slot, counted while emitting
        if (c2 > 0 && tdirect) {
            // direct form: the schedule (column (k + p) mod 8 while it has one, else the fullest) takes "the next neighbour of
            // column c" = the lowest set bit of the column's bit string (three 32-bit words per column, transposed above)
            unsigned int* myw = hitw + d_myhw;
            unsigned int rlo = (unsigned int)d_rem, rhi = (unsigned int)(d_rem >> 32);   // neighbours left per column, one byte each
            const int ng = (d_nch + 7) >> 3;
            // one scheduled pick: returns the position of the neighbour in the candidate list
            auto pick = [&](int k) {
                int c = (k + tid) & 7;
                if ((__byte_perm(rlo, rhi, c) & 0xffu) == 0u) {            // preferred column exhausted: the fullest one (first of equals)
                    // key = count * 8 + (7 - column): the largest key is the fullest column, the lowest column among equals
                    unsigned int best = 0u;
#pragma unroll
                    for (int cc = 0; cc < 8; ++cc) {
                        const unsigned int bc = __byte_perm(cc < 4 ? rlo : rhi, 0u, 0x4440u | (unsigned int)(cc & 3));
                        best = max(best, bc * 8u + (unsigned int)(7 - cc));
                    }
                    c = 7 - (int)(best & 7u);
                }
                const unsigned int dec = 1u << (8 * (c & 3));
                if (c < 4) rlo -= dec; else rhi -= dec;
                unsigned int* pw = myw + c * TS_ROW;
                unsigned int bits = pw[0];
                int g = 0;
                if (bits == 0u && ng > 1) { pw += 8 * TS_ROW; bits = pw[0]; g = 1; }
                if (bits == 0u && ng > 2) { pw += 8 * TS_ROW; bits = pw[0]; g = 2; }
                const int bit = __ffs(bits) - 1;                            // (bits != 0: the column has neighbours left)
                pw[0] = bits & (bits - 1u);
                const int rr = 32 * g + bit;                                // rank of the candidate in its column
                return (rr >> 2) * 32 + c * 4 + (rr & 3);
            };
            int k0 = 0;
            for (; k0 + 4 <= c2; k0 += 4) {
                int src[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) src[q] = pick(k0 + q);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const unsigned int tq = d_cl[src[q]];
                    lo_e += (int)tq < me ? 1 : 0;
                    w[q] = tq << rsh;
                }
                rowb[(size_t)(k0 >> 2) * MD_TB] = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
            }
            if (k0 < c2) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    w[q] = dummy;
                    if (k0 + q < c2) {
                        const unsigned int tq = d_cl[pick(k0 + q)];
                        lo_e += (int)tq < me ? 1 : 0;
                        w[q] = tq << rsh;
                    }
                }
                rowb[(size_t)(k0 >> 2) * MD_TB] = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
            }
            lo_cnt = lo_e;
            c2e = 0;                                       // nothing left for the scheduled emission below
        } else if (c2 > 0 && near_first) {
            // two sweeps over the scan-order list: near neighbours first, then the rest (careful-path lists carry no flags: all "rest")
            int kout = 0;
            for (int pass = 0; pass < 2; ++pass) {
                for (int k = 0; k < c2; ++k) {
                    const unsigned int raw = tmp[(size_t)k * MD_TB];
                    if (((raw >> 15) & 1u) == (unsigned int)pass) continue;      // pass 0 takes the flagged entries
                    const unsigned int tq = raw & 0x7fffu;
                    lo_e += (int)tq < me ? 1 : 0;
                    w[kout & 3] = tq << rsh;
                    if ((kout & 3) == 3) rowb[(size_t)(kout >> 2) * MD_TB] = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
                    ++kout;
                }
            }
            if (kout & 3) {
                for (int q = kout & 3; q < 4; ++q) w[q] = dummy;
                rowb[(size_t)(kout >> 2) * MD_TB] = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
            }
            lo_cnt = lo_e;
            c2e = 0;                                       // nothing left for the scheduled emission below
        } else if (c2 > 0 && !P.row_schedule && !use_masks) {
            // scan order, no column scheduling: the list the candidate scan left in scratch goes straight into the row
            for (int k0 = 0; k0 < c2; k0 += 4) {
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int k = k0 + q;
                    const unsigned int tq = k < c2 ? (unsigned int)(tmp[(size_t)k * MD_TB] & 0x7fffu) : 0x7fffffffu;
                    lo_e += (int)tq < me ? 1 : 0;
                    w[q] = k < c2 ? (tq << rsh) : dummy;
                }
                rowb[(size_t)(k0 >> 2) * MD_TB] = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
            }
            lo_cnt = lo_e;
            c2e = 0;                                       // nothing left for the scheduled emission below
        } else if (c2 > 0 && bucketed) {
            pops = pops_pre;                               // buckets filled by scan_cell_bucket; lo_cnt is counted below
            if (bucket_over) { atomicOr(&B.ctrl->err, MD_DEVERR_CAPACITY); c2e = 0; }
            rem8 = pops;
        } else if (c2 > 0) {
            int lo_b = 0;
            bool over = false;
            for_each_neighbour([&](int t) {
                const int c = t & 7, sh8 = c * 8;
                const int p = (int)((pops >> sh8) & 255ull);
                if (p < cap8) { tmp2[(size_t)(c * cap8 + p) * MD_TB] = (unsigned short)t; pops += 1ull << sh8; } else over = true;
                lo_b += t < me;
            });
            lo_cnt = lo_b;
            if (over) { atomicOr(&B.ctrl->err, MD_DEVERR_CAPACITY); c2e = 0; }
            rem8 = pops;
        }
        for (int k0 = 0; k0 < c2e; k0 += 4) {
            int src[4];                                   // scratch positions of the four entries (-1 = padding)
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int k = k0 + q;
                src[q] = -1;
                if (k < c2e) {
                    int c = (k + tid) & 7;
                    int r = (int)((rem8 >> (8 * c)) & 255ull);
                    if (r == 0) {                          // preferred column exhausted: take the fullest one
#pragma unroll
                        for (int cc = 0; cc < 8; ++cc) { const int v = (int)((rem8 >> (8 * cc)) & 255ull); if (v > r) { r = v; c = cc; } }
                    }
                    src[q] = c * cap8 + (int)((pops >> (8 * c)) & 255ull) - r;    // next unused entry of column c
                    rem8 -= 1ull << (8 * c);
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const unsigned int tq = src[q] >= 0 ? (unsigned int)tmp2[(size_t)src[q] * MD_TB] : 0x7fffffffu;
                lo_e += (int)tq < me ? 1 : 0;              // local indices ascend with the slot: t < me <=> slot < i  (padding never counts)
                w[q] = src[q] >= 0 ? (tq << rsh) : dummy;
            }
            rowb[(size_t)(k0 >> 2) * MD_TB] = make_uint2(w[0] | (w[1] << 16), w[2] | (w[3] << 16));
        }
        if (bucketed && P.row_schedule) lo_cnt = lo_e;
        if (live) {
            B.row_count[i] = c2;
            B.lo_count[i] = cnt > P.cap ? 0 : lo_cnt;
            B.half_count[i] = cnt > P.cap ? 0 : cnt - lo_cnt;
            B.pos_ref[i] = pos[i];      // the skin reference is the untransformed position
        }
    }
    // 9. block totals
    int tot_full, tot_half;
    blk_excl_scan(min(cnt, P.cap), &tot_full, sh_scan);
    blk_excl_scan(cnt > P.cap ? 0 : cnt - lo_cnt, &tot_half, sh_scan);
    const int seen = __reduce_max_sync(0xffffffffu, cnt);
    if ((tid & 31) == 0) atomicMax(&B.ctrl->max_seen, seen);
    __syncthreads();
    if (tid == 0) {
        int out = 0;
        if (wrap_axes || small_box) {
            out = MD_BLK_WRAP | (wrap_axes * MD_BLK_AXIS_SHIFT);
            if (shift_ok) out |= MD_BLK_SHIFT_OK;
        }
        if (M + 1 <= 4096) out |= MD_BLK_SH4;
        B.blk[b] = BlkInfo{ nseg, M, own_base, out };
        atomicAdd(&B.ctrl->n_full, (unsigned long long)tot_full);
        atomicAdd(&B.ctrl->n_edges, (unsigned int)tot_half);
        atomicMax(&B.ctrl->max_stage, M + 1);
        atomicMax(&B.ctrl->max_seg, nseg);
    }
}

__global__ void k_staged_begin(DevBuffers B, int gated) {
    GATE(B, gated);
    B.ctrl->max_seen = 0;
    B.ctrl->n_full = 0ull;
    B.ctrl->n_edges = 0u;
    B.ctrl->max_stage = 0;
    B.ctrl->max_seg = 0;
}

static void staged_build_sizes(const md_system* s, int* ncand_cap, int* umax, int* tbl_cap, size_t* smem) {
    const DevParams& P = s->P;
    const double ppc = (double)P.N / (double)P.ncell;
    double own = (double)MD_TB / (ppc > 1e-9 ? ppc : 1e-9);
    if (own > MD_TB) own = MD_TB;
    int nc = 64;
    while (nc < 27 * (2 * own + 4) && nc < MD_NCAND) nc <<= 1;
    if (nc > MD_NCAND) nc = MD_NCAND;
    int um = nc < MD_UMAX ? nc : MD_UMAX;
    int region = nc;                                  // ints shared by the hash set and, after it, the stencil table
    if (4 * ((size_t)nc + 3 * (size_t)um + 1 + MD_TB) > 40 * 1024) {
        // sparse cells (2-3 particles per cell): ~100 own cells per block.  The set holds DISTINCT cells only, about
        // (own^(1/3) + 2)^3 of them for a compact block: size it (4x that, load <= 1/2) instead of 27 x own cells, and
        // keep the table at its hard bound of 27 x MD_TB 16-bit entries -- 42 KB instead of 83 KB per block at 2.5
        // particles per cell, five resident blocks instead of one.
        const double side = cbrt(own) + 2.0;
        int want = 256;
        while (want < 4.0 * side * side * side && want < MD_UMAX) want <<= 1;
        um = want < um ? want : um;
        nc = 2 * um;
        region = nc > (27 * MD_TB + 1) / 2 ? nc : (27 * MD_TB + 1) / 2;
    }
    else {
        // dense cells: the distinct-cell tables need no more than the sparse sizing gives (4x the cells of a compact block);
        // the transposed scan wants the shared memory (four resident blocks)
        const double side = cbrt(own) + 2.0;
        int want = 256;
        while (want < 4.0 * side * side * side && want < MD_UMAX) want <<= 1;
        um = want < um ? want : um;
    }
    *ncand_cap = nc;
    *umax = um;
    *tbl_cap = 2 * region;
    *smem = 4 * ((size_t)region + 3 * (size_t)um + 1 + 2 * MD_TB) + 16;
}

void md_launch_build_staged(md_system* s, bool gated) {
    const DevParams& P = s->P;
    const int g = gated ? 1 : 0;
    int nc, um, tc;
    size_t smem;
    staged_build_sizes(s, &nc, &um, &tc, &smem);
    // candidates are read through L1: with the small tables of dense cells leave it as large as the resident blocks allow
    // (measured at C2a: carveout 25 -> 1.96 ms, 50 -> 1.65, 75 -> 1.82, 100 -> 2.02); the 42 KB tables of sparse cells need
    // the shared memory itself (five resident blocks instead of two)
    const bool tscan = P.use_masks && P.row_schedule;           // k_build_staged<true>: + the arrays of the transposed scan
    if (tscan) smem += TS_SMEM_BYTES + 16;
    const int carve = smem > 30 * 1024 ? (int)cudaSharedmemCarveoutMaxShared : 50;
    if (carve != s->build_carve) {      // per handle = per device (function attributes are per device)
        cudaFuncSetAttribute(k_build_staged<true>, cudaFuncAttributePreferredSharedMemoryCarveout, carve);
        cudaFuncSetAttribute(k_build_staged<false>, cudaFuncAttributePreferredSharedMemoryCarveout, carve);
        s->build_carve = carve;
    }
    k_staged_begin<<<1, 1, 0, s->stream>>>(s->B, g);
    if (tscan) k_build_staged<true><<<P.nblk, MD_TB, smem, s->stream>>>(P, s->B, g, s->pos, nc, um, tc);
    else k_build_staged<false><<<P.nblk, MD_TB, smem, s->stream>>>(P, s->B, g, s->pos, nc, um, tc);
    s->launches += 2;
}

// ------------------------------------------------------------------------------------------------
// explicit (i, j) edge list from the staged rows: i < j slots, sorted by i, bit 31 of j = periodic image flag.
// Used by md_get_pairs (list parity export).  Needs edge_off = exclusive scan of half_count.  Local indices
// ascend with the slot, so the half list (i < j) of particle i is { t in row : t > own local index }.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned int row_entry(const uint2* __restrict__ rowb, int k, int shift) {
    const uint2 pk = rowb[(size_t)(k >> 2) * MD_TB];
    const unsigned int w = (k & 2) ? pk.y : pk.x;
    return ((k & 1) ? (w >> 16) : (w & 0xffffu)) >> shift;   // local index
}

__global__ void __launch_bounds__(MD_TB) k_edges_from_rows(DevParams P, DevBuffers B, const float4* __restrict__ pos) {
    extern __shared__ __align__(16) unsigned char smraw[];
    int* sslot = reinterpret_cast<int*>(smraw);   // [M]
    const int b = blockIdx.x, tid = threadIdx.x;
    const BlkInfo bi = B.blk[b];
    const int2* __restrict__ seg = B.seg + (size_t)b * MD_SEGMAX;
    for (int sg = tid >> 5; sg < bi.nseg; sg += MD_TB / 32) {
        const int2 s0 = seg[sg];
        const int l0 = (int)((unsigned)s0.y >> 16), len = s0.y & 0xffff;
        for (int k = tid & 31; k < len; k += 32) sslot[l0 + k] = s0.x + k;
    }
    __syncthreads();
    const int i = b * MD_TB + tid;
    if (i >= P.N) return;
    const int cnt = B.row_count[i], me = bi.own_base + tid;
    const uint2* __restrict__ rowb = reinterpret_cast<const uint2*>(B.rows) + (size_t)b * (P.rcap >> 2) * MD_TB + tid;
    const float4 xi = pos[i];
    unsigned int o = B.edge_off[i];
    for (int k = 0; k < cnt; ++k) {
        const int t = (int)row_entry(rowb, k, (bi.flags & MD_BLK_SH4) ? 4 : 0);
        if (t <= me) continue;
        const int j = sslot[t];
        const float4 xj = pos[j];
        const int w = (fabsf(xj.x - xi.x) > P.hLx) | (fabsf(xj.y - xi.y) > P.hLy) | (fabsf(xj.z - xi.z) > P.hLz);
        B.edges[o++] = make_int2(i, j | (w << 31));
    }
}

void md_launch_edges_from_rows(md_system* s) {
    const DevParams& P = s->P;
    k_edges_from_rows<<<P.nblk, MD_TB, 4 * (size_t)P.stage_cap, s->stream>>>(P, s->B, s->pos);
    s->launches += 1;
}

// ------------------------------------------------------------------------------------------------
// staging prologue of the force kernels: bulk TMA copies of the block's segments into shared memory
// ------------------------------------------------------------------------------------------------
struct Stage {
    float4* spos;    // [M + 1]  (entry M = dummy)
    float4* squat;   // [M + 1]  rigid bodies only
};

// Segment copies are issued by ALL warps: a bulk copy takes uniform operands, so the lanes of a warp issue theirs one
// after the other; spreading the ~100 segments of a block over its 8 warps (segment l*8+w to lane l of warp w) cuts
// the issue chain from ~100 to ~13 copies.  Each thread's first table entry is loaded at kernel entry together with
// the block header, so the staging copies wait for ONE memory latency.
struct SegPre { int2 e; int sg; };
__device__ __forceinline__ SegPre seg_preload(const DevBuffers& B, int b) {
    SegPre sp;
    const int nw = blockDim.x >> 5;
    sp.sg = (threadIdx.x & 31) * nw + (threadIdx.x >> 5);
    sp.e = B.seg[(size_t)b * MD_SEGMAX + sp.sg];   // always inside the table; entries >= nseg are ignored
    return sp;
}

template <bool QUAT>
__device__ __forceinline__ Stage stage_issue(const DevParams& P, const DevBuffers& B, const BlkInfo bi, int b, int stage_entries,
                                             const SegPre& pre, const float4* __restrict__ pos, const float4* __restrict__ quat,
                                             unsigned char* smraw) {
    Stage st;
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smraw);
    st.spos = reinterpret_cast<float4*>(smraw + 16);
    st.squat = QUAT ? st.spos + stage_entries : nullptr;
    const int2* __restrict__ seg = B.seg + (size_t)b * MD_SEGMAX;
    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_expect_tx(bar, (unsigned)bi.M * 16u * (QUAT ? 2u : 1u));
    }
    if (tid == 32) {
        st.spos[bi.M] = make_float4(DUMMY_COORD, DUMMY_COORD, DUMMY_COORD, 0.f);
        if (QUAT) st.squat[bi.M] = make_float4(1.f, 0.f, 0.f, 0.f);
    }
    __syncthreads();          // barrier initialised and armed before any copy is issued; dummy entry written
    if (pre.sg < bi.nseg) {
        const int l0 = (int)((unsigned)pre.e.y >> 16), len = pre.e.y & 0xffff;
        bulk_g2s(st.spos + l0, pos + pre.e.x, (unsigned)len * 16u, bar);
        if (QUAT) bulk_g2s(st.squat + l0, quat + pre.e.x, (unsigned)len * 16u, bar);
    }
    for (int sg = pre.sg + (int)blockDim.x; sg < bi.nseg; sg += blockDim.x) {
        const int2 s0 = seg[sg];
        const int l0 = (int)((unsigned)s0.y >> 16), len = s0.y & 0xffff;
        bulk_g2s(st.spos + l0, pos + s0.x, (unsigned)len * 16u, bar);
        if (QUAT) bulk_g2s(st.squat + l0, quat + s0.x, (unsigned)len * 16u, bar);
    }
    return st;
}

// second half of the prologue: wait for the bulk copies, then the periodic shift transform
__device__ __forceinline__ void stage_wait(const DevParams& P, const BlkInfo bi, const Stage& st, unsigned char* smraw) {
    const int tid = threadIdx.x;
    mbar_wait(smraw, 0);      // all segments have landed
    // periodic blocks: shift the upper half of the box down by L on the wrapped axes (exact in fp32: Sterbenz),
    // after which plain differences ARE the minimum images (verified pair by pair at build time)
    if ((bi.flags & MD_BLK_WRAP) && (bi.flags & MD_BLK_SHIFT_OK)) {
        const bool sx = bi.flags & (MD_BLK_AXIS_SHIFT << 0), sy = bi.flags & (MD_BLK_AXIS_SHIFT << 1), sz = bi.flags & (MD_BLK_AXIS_SHIFT << 2);
        for (int t = tid; t < bi.M; t += blockDim.x) {
            float4 x = st.spos[t];
            if (sx && x.x > P.hLx) x.x -= P.Lx;
            if (sy && x.y > P.hLy) x.y -= P.Ly;
            if (sz && x.z > P.hLz) x.z -= P.Lz;
            st.spos[t] = x;
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// VERTEX, LJ / WCA (+ FENE bonds), staged (S:A6): one thread per particle loops over its row; neighbour
// positions come from the block's shared-memory neighbourhood by 128-bit gathers whose bank columns were
// de-conflicted at build time (k_build_staged pass B).  No atomics, every pair computed twice.
// ------------------------------------------------------------------------------------------------
struct LJAccS { float fx, fy, fz, band; float2 pe, nin; };

// streamed row chunk: read once per evaluation, so it bypasses L1 allocation (the L1 left beside the staged
// neighbourhoods is small) (no_allocate)
__device__ __forceinline__ uint2 ld_row(const uint2* p) {
    uint2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}

// staged position of a row entry: entries hold (local index << SH); SH == 4 makes the entry the byte offset
// sp32 = 32-bit shared-window address of the staged array, computed once per thread
template <int SH>
__device__ __forceinline__ float4 staged_pos(unsigned int sp32, unsigned int e) {
    float4 v;
    const unsigned int a = sp32 + (SH == 4 ? e : (e << 4));
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}

// Two visits (a, b) at once.  Distances and the force accumulation are scalar fp32; the chain in between --
// cutoff mask, 1/d2, s6, force and energy polynomials -- runs on both visits with packed f32x2 instructions
// (FADD2 / FMUL2 / FFMA2: half the issue slots).  The cutoff enters as a 0/1 mask m (no branch, no select):
// s = m / d2, so force and energy of an outside pair are exactly zero; the energy shift is -m V_c.
// `band` tracks min |d2 - rc^2| for the fp64 recheck (S:H10).
template <bool IMG>
__device__ __forceinline__ void lj_visit2_s(const DevParams& P, float4 xi, float4 xa, float4 xb, LJAccS& a) {
    float dxa, dya, dza, dxb, dyb, dzb;
    if (IMG) {
        dxa = min_image(xa.x, xi.x, P.Lx, P.hLx); dya = min_image(xa.y, xi.y, P.Ly, P.hLy); dza = min_image(xa.z, xi.z, P.Lz, P.hLz);
        dxb = min_image(xb.x, xi.x, P.Lx, P.hLx); dyb = min_image(xb.y, xi.y, P.Ly, P.hLy); dzb = min_image(xb.z, xi.z, P.Lz, P.hLz);
    } else {
        dxa = xa.x - xi.x; dya = xa.y - xi.y; dza = xa.z - xi.z;
        dxb = xb.x - xi.x; dyb = xb.y - xi.y; dzb = xb.z - xi.z;
    }
    const float2 d2 = make_float2(fmaf(dza, dza, fmaf(dya, dya, dxa * dxa)), fmaf(dzb, dzb, fmaf(dyb, dyb, dxb * dxb)));
    const float2 t = __fadd2_rn(d2, P.k_nrc2);
    const float2 m = make_float2(t.x < 0.0f ? 1.0f : 0.0f, t.y < 0.0f ? 1.0f : 0.0f);
    a.band = fminf(fminf(a.band, fabsf(t.x)), fabsf(t.y));
    const float2 inv = make_float2(rcp_approx(d2.x), rcp_approx(d2.y));
    const float2 s = __fmul2_rn(inv, m);                       // m / d2
    const float2 s2 = __fmul2_rn(s, s);
    const float2 u = __fmul2_rn(s2, s);                        // m / d2^3  (sigma^-6 s6)
    const float2 w = __fmul2_rn(s2, s2);                       // m / d2^4
    const float2 ng = __fmul2_rn(w, __ffma2_rn(P.k_na, u, P.k_b));   // -24 eps s6 (2 s6 - 1) / d2
    a.fx = fmaf(ng.x, dxa, a.fx); a.fy = fmaf(ng.x, dya, a.fy); a.fz = fmaf(ng.x, dza, a.fz);
    a.fx = fmaf(ng.y, dxb, a.fx); a.fy = fmaf(ng.y, dyb, a.fy); a.fz = fmaf(ng.y, dzb, a.fz);
    a.pe = __ffma2_rn(u, __ffma2_rn(P.k_c, u, P.k_nd), a.pe);  // 4 eps s6 (s6 - 1)
    a.pe = __ffma2_rn(m, P.k_nvs, a.pe);                       // - V_c
}

// rare path (~1.6e-4 of the particles at rc = 2.5): a visit of this particle fell inside the fp64-recheck band.
// Re-scan the row for the banded pairs only and, where the S:O0 / S:Q5 fp64 decision differs from the fp32 one the
// fast loop took, add or remove that pair's contribution.  acc = (fx, fy, fz, pe) of the fast loop, corrected in place.
template <bool IMG>
__device__ __noinline__ void lj_fix_band_s(const float4* spos, const uint2* __restrict__ rowb, int cnt, int shift, float4 xi,
                                           float Lx, float Ly, float Lz, float rc2, float band_abs, float lj_a, float lj_b,
                                           float lj_c, float lj_d, float vshift, double dLx, double dLy, double dLz, double rc2d,
                                           float4* acc) {
    float4 a = *acc;
    for (int k = 0; k < cnt; ++k) {
        const float4 xj = spos[row_entry(rowb, k, shift)];
        float dx, dy, dz;
        if (IMG) {
            dx = min_image(xj.x, xi.x, Lx, 0.5f * Lx); dy = min_image(xj.y, xi.y, Ly, 0.5f * Ly); dz = min_image(xj.z, xi.z, Lz, 0.5f * Lz);
        } else {
            dx = xj.x - xi.x; dy = xj.y - xi.y; dz = xj.z - xi.z;
        }
        const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        const float t = d2 - rc2;
        if (!(fabsf(t) < band_abs)) continue;
        const bool in32 = t < 0.0f;
        const bool in64 = inside_fp64(xi, xj, dLx, dLy, dLz, rc2d);
        if (in32 == in64) continue;
        const float sgn = in64 ? 1.0f : -1.0f;
        const float inv = rcp_approx(d2);
        const float u = inv * inv * inv;
        const float ng = sgn * (inv * u) * fmaf(-lj_a, u, lj_b);
        a.x = fmaf(ng, dx, a.x); a.y = fmaf(ng, dy, a.y); a.z = fmaf(ng, dz, a.z);
        a.w += sgn * (fmaf(u, fmaf(lj_c, u, -lj_d), -vshift));
    }
    *acc = a;
}

// FENE partners of slot i (ids id-1 and id+1 inside its chain), global gathers through slot_of_id
__device__ __forceinline__ void fene_vertex_s(const DevParams& P, const DevBuffers& B, const float4* __restrict__ pos, int i,
                                              float& fx, float& fy, float& fz, float& pe) {
    const float4 xi = pos[i];
    const int id = B.ids[i];
    const int m = id % P.chain_len;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
        const int pid = s == 0 ? id - 1 : id + 1;
        const bool ok = s == 0 ? (m != 0) : (m != P.chain_len - 1 && pid < P.N);
        if (!ok) continue;
        const float4 xj = pos[B.slot_of_id[pid]];
        const float dx = min_image(xj.x, xi.x, P.Lx, P.hLx);
        const float dy = min_image(xj.y, xi.y, P.Ly, P.hLy);
        const float dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
        const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        float g, V;
        if (!fene_pair(P, d2, g, V)) atomicOr(&B.ctrl->err, MD_DEVERR_FENE);
        fx -= g * dx; fy -= g * dy; fz -= g * dz;
        pe += V;
    }
}

// The same two visits in reduced units for sigma == 1 (every BASELINE config): with s = m / d2 the sums
//   A = sum (s^4 - 2 s^7) d,  pe = sum (s^6 - s^3),  nin = sum m
// need no potential constants inside the loop (F_i = 24 eps A, V = 4 eps pe - V_c nin are applied once per particle),
// which removes the per-chunk constant reloads and eight registers.  a.pe holds sum (s^6 - s^3), a.nin the count.
// ENERGY = false: the per-particle energy is not needed (inner steps of a multi-step md_integrate graph: md_energy can only
// observe the forces of the LAST step) -- the pe and nin sums are dropped, ~7 % of the loop's issue slots.
template <bool IMG, bool ENERGY>
__device__ __forceinline__ void lj_visit2_unit_s(const DevParams& P, float4 xi, float4 xa, float4 xb, LJAccS& a) {
    float dxa, dya, dza, dxb, dyb, dzb;
    if (IMG) {
        dxa = min_image(xa.x, xi.x, P.Lx, P.hLx); dya = min_image(xa.y, xi.y, P.Ly, P.hLy); dza = min_image(xa.z, xi.z, P.Lz, P.hLz);
        dxb = min_image(xb.x, xi.x, P.Lx, P.hLx); dyb = min_image(xb.y, xi.y, P.Ly, P.hLy); dzb = min_image(xb.z, xi.z, P.Lz, P.hLz);
    } else {
        dxa = xa.x - xi.x; dya = xa.y - xi.y; dza = xa.z - xi.z;
        dxb = xb.x - xi.x; dyb = xb.y - xi.y; dzb = xb.z - xi.z;
    }
    const float2 d2 = make_float2(fmaf(dza, dza, fmaf(dya, dya, dxa * dxa)), fmaf(dzb, dzb, fmaf(dyb, dyb, dxb * dxb)));
    const float2 t = __fadd2_rn(d2, P.k_nrc2);
    const float2 m = make_float2(t.x < 0.0f ? 1.0f : 0.0f, t.y < 0.0f ? 1.0f : 0.0f);
    a.band = fminf(fminf(a.band, fabsf(t.x)), fabsf(t.y));
    const float2 inv = make_float2(rcp_approx(d2.x), rcp_approx(d2.y));
    const float2 s = __fmul2_rn(inv, m);
    const float2 s2 = __fmul2_rn(s, s);
    const float2 z3 = __fmul2_rn(s2, s);
    const float2 z4 = __fmul2_rn(s2, s2);
    const float2 z7 = __fmul2_rn(z4, z3);
    const float2 ng = __ffma2_rn(z7, make_float2(-2.0f, -2.0f), z4);
    a.fx = fmaf(ng.x, dxa, a.fx); a.fy = fmaf(ng.x, dya, a.fy); a.fz = fmaf(ng.x, dza, a.fz);
    a.fx = fmaf(ng.y, dxb, a.fx); a.fy = fmaf(ng.y, dyb, a.fy); a.fz = fmaf(ng.y, dzb, a.fz);
    if (ENERGY) {
        a.pe = __fadd2_rn(a.pe, __ffma2_rn(z3, z3, make_float2(-z3.x, -z3.y)));
        a.nin = __fadd2_rn(a.nin, m);
    }
}

template <bool IMG, int SH, bool UNIT, bool ENERGY>
__device__ __forceinline__ void lj_chunk_s(const DevParams& P, unsigned int sp32, float4 xi, uint2 cur, LJAccS& a) {
    const float4 x0 = staged_pos<SH>(sp32, cur.x & 0xffffu), x1 = staged_pos<SH>(sp32, cur.x >> 16);
    const float4 x2 = staged_pos<SH>(sp32, cur.y & 0xffffu), x3 = staged_pos<SH>(sp32, cur.y >> 16);
    if (UNIT) {
        lj_visit2_unit_s<IMG, ENERGY>(P, xi, x0, x1, a);
        lj_visit2_unit_s<IMG, ENERGY>(P, xi, x2, x3, a);
    } else {
        lj_visit2_s<IMG>(P, xi, x0, x1, a);
        lj_visit2_s<IMG>(P, xi, x2, x3, a);
    }
}

// cnt, pk[0..3]: |L_i| and the first four row chunks, loaded by the caller while the staging copies were in flight.
// The row streams from HBM (~1300 cycles under load); chunks are consumed four per iteration through four separate
// load instructions, each re-issued four chunks (~350 instructions of arithmetic) ahead of its use.
// NS = threads per particle (1; 2 or 4 when the staged neighbourhood is so large that only one or two 256-particle blocks
// fit on an SM: the block then runs 512 threads, thread h * 256 + p takes the row chunks c = h mod 2 of particle p and the
// two partial sums meet in shared memory -- twice the warps for the same shared memory).  xch = exchange buffer (NS == 2).
// fused step tail (FuseArgs, md_internal.cuh): v += hk f twice (closing kick of this step, opening kick of the next: two
// roundings, as k_kick followed by k_kick_drift), x' = x + dt v into the other position array, skin check (S:Q4).
// Not inlined: its registers must not compete with the row loop of the caller.
__device__ __noinline__ void fuse_kick_drift(float hk, float dt, float half_skin2, float4* __restrict__ vel, const float4* __restrict__ pos,
                                             float4* __restrict__ pos_next, const float4* __restrict__ pos_ref, int* __restrict__ rebuild,
                                             int i, float fx, float fy, float fz) {
    float4 v = vel[i];
    float4 x = pos[i];                                      // raw position (the staged copy may be shift-transformed)
    const float4 r = pos_ref[i];
    v.x = fmaf(hk, fx, v.x); v.y = fmaf(hk, fy, v.y); v.z = fmaf(hk, fz, v.z);
    v.x = fmaf(hk, fx, v.x); v.y = fmaf(hk, fy, v.y); v.z = fmaf(hk, fz, v.z);
    x.x = fmaf(dt, v.x, x.x); x.y = fmaf(dt, v.y, x.y); x.z = fmaf(dt, v.z, x.z);
    vel[i] = v;
    pos_next[i] = x;
    const float dx = x.x - r.x, dy = x.y - r.y, dz = x.z - r.z;
    if ((dx * dx + dy * dy + dz * dz) > half_skin2) *rebuild = 1;     // S:Q4 strict '>'
}

template <bool IMG, int SH, bool UNIT, int NS, bool ENERGY>
__device__ __forceinline__ void vertex_lj_rows(const DevParams& P, const DevBuffers& B, const BlkInfo bi, const Stage& st, int i,
                                               bool live, int cnt, const uint2* __restrict__ rowb, uint2 pkA, uint2 pkB, uint2 pkC,
                                               uint2 pkD, float* xch, const float4* __restrict__ pos, float4* __restrict__ force,
                                               bool bonds, const FuseArgs& fuse) {
    const int tp = threadIdx.x % MD_TB, h = threadIdx.x / MD_TB;
    const float4 xi = st.spos[bi.own_base + (live ? tp : 0)];
    const unsigned int sp = smem_u32(st.spos);
    const int nall = (cnt + 3) >> 2;                       // the last chunk is padded with the dummy entry
    const int nch = (nall - h + NS - 1) / NS;              // chunks h, h + NS, ... of the row
    const uint2* __restrict__ rowh = rowb + (size_t)h * MD_TB;
    const size_t cs = (size_t)NS * MD_TB;                  // stride between this thread's chunks
    LJAccS a = { 0.f, 0.f, 0.f, 3.0e38f, make_float2(0.f, 0.f), make_float2(0.f, 0.f) };
    for (int c = 0; c < nch; c += 4) {
        const uint2 curA = pkA;
        if (c + 4 < nch) pkA = ld_row(rowh + (size_t)(c + 4) * cs);
        lj_chunk_s<IMG, SH, UNIT, ENERGY>(P, sp, xi, curA, a);
        if (c + 1 >= nch) break;
        const uint2 curB = pkB;
        if (c + 5 < nch) pkB = ld_row(rowh + (size_t)(c + 5) * cs);
        lj_chunk_s<IMG, SH, UNIT, ENERGY>(P, sp, xi, curB, a);
        if (c + 2 >= nch) break;
        const uint2 curC = pkC;
        if (c + 6 < nch) pkC = ld_row(rowh + (size_t)(c + 6) * cs);
        lj_chunk_s<IMG, SH, UNIT, ENERGY>(P, sp, xi, curC, a);
        if (c + 3 >= nch) break;
        const uint2 curD = pkD;
        if (c + 7 < nch) pkD = ld_row(rowh + (size_t)(c + 7) * cs);
        lj_chunk_s<IMG, SH, UNIT, ENERGY>(P, sp, xi, curD, a);
    }
    float pe2 = a.pe.x + a.pe.y;
    float nin = a.nin.x + a.nin.y;
    if (NS > 1) {                                          // threads h > 0 hand their partial sums to thread h == 0
        if (h > 0) {
            float* x = xch + (size_t)(h - 1) * 6 * MD_TB;
            x[tp] = a.fx; x[MD_TB + tp] = a.fy; x[2 * MD_TB + tp] = a.fz; x[3 * MD_TB + tp] = pe2;
            x[4 * MD_TB + tp] = nin; x[5 * MD_TB + tp] = a.band;
        }
        __syncthreads();
        if (h > 0) return;
#pragma unroll
        for (int k = 0; k < NS - 1; ++k) {                 // fixed order: run-to-run reproducible
            const float* x = xch + (size_t)k * 6 * MD_TB;
            a.fx += x[tp]; a.fy += x[MD_TB + tp]; a.fz += x[2 * MD_TB + tp]; pe2 += x[3 * MD_TB + tp];
            nin += x[4 * MD_TB + tp]; a.band = fminf(a.band, x[5 * MD_TB + tp]);
        }
    }
    if (!live) return;
    if (UNIT) {   // back from reduced units: F = 24 eps A, V = 4 eps sum (s^6 - s^3) - V_c nin
        a.fx *= P.c24; a.fy *= P.c24; a.fz *= P.c24;
        pe2 = fmaf(P.c4, pe2, -P.vshift * nin);
    }
    if (a.band < P.band_abs) {
        float4* scratch = force + i;           // own output slot as scratch (rewritten below)
        *scratch = make_float4(a.fx, a.fy, a.fz, pe2);
        lj_fix_band_s<IMG>(st.spos, rowb, cnt, SH, xi, P.Lx, P.Ly, P.Lz, P.rc2, P.band_abs, P.lj_a, P.lj_b,
                           P.lj_c, P.lj_d, P.vshift, P.dLx, P.dLy, P.dLz, P.rc2d, scratch);
        const float4 r = *scratch;
        a.fx = r.x; a.fy = r.y; a.fz = r.z; pe2 = r.w;
    }
    float pe = 0.5f * pe2;
    if (bonds) {
        float bpe = 0.f;
        fene_vertex_s(P, B, pos, i, a.fx, a.fy, a.fz, bpe);
        pe += 0.5f * bpe;
    }
    if (fuse.vel) fuse_kick_drift(0.5f * fuse.dt * P.inv_mass, fuse.dt, P.half_skin2, fuse.vel, pos, fuse.pos_next, B.pos_ref, &B.ctrl->rebuild, i, a.fx, a.fy, a.fz);
    else force[i] = make_float4(a.fx, a.fy, a.fz, pe);
}

// Blocks whose neighbourhood does not fit the launch (it grew past the head room since the last synchronising call)
// are not failed: they take this slow path, which reads the same rows but fetches each neighbour from global memory --
// local index -> slot through the block's segment table (sorted by local base: binary search), raw positions, minimum
// image.  Same pair set, same decisions (fp64 band), so the result stays within the parity tolerance.
__device__ __forceinline__ int staged_slot_of_local(const int2* __restrict__ seg, int nseg, int t) {
    int lo = 0, hi = nseg - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if ((int)((unsigned)seg[mid].y >> 16) <= t) lo = mid; else hi = mid - 1;
    }
    const int2 sg = seg[lo];
    return sg.x + (t - (int)((unsigned)sg.y >> 16));
}

template <bool RIGID, bool PP>
__device__ __forceinline__ void vertex_rows_unstaged(const DevParams& P, const DevBuffers& B, const BlkInfo bi, int b,
                                                  const float4* __restrict__ pos, const float4* __restrict__ quat,
                                                  float4* __restrict__ force, float4* __restrict__ torque,
                                                  const FuseArgs& fuse = FuseArgs{ nullptr, nullptr, 0.0f }) {
    if (threadIdx.x >= MD_TB) return;
    const int i = b * MD_TB + threadIdx.x;
    if (i >= P.N) return;
    const int cnt = B.row_count[i];
    const int sh = (bi.flags & MD_BLK_SH4) ? 4 : 0;
    const int2* __restrict__ seg = B.seg + (size_t)b * MD_SEGMAX;
    const unsigned short* __restrict__ row = B.rows + ((size_t)b * (P.rcap >> 2) * MD_TB + threadIdx.x) * 4;
    const float4 xi = pos[i];
    Rot Ri;
    if (RIGID) Ri = quat_to_rot(quat[i]);
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f, tx = 0.f, ty = 0.f, tz = 0.f;
    for (int k = 0; k < cnt; ++k) {
        const int t = (int)row[(size_t)(k >> 2) * MD_TB * 4 + (k & 3)] >> sh;
        const int j = staged_slot_of_local(seg, bi.nseg, t);
        const float4 xj = pos[j];
        const float dx = min_image(xj.x, xi.x, P.Lx, P.hLx), dy = min_image(xj.y, xi.y, P.Ly, P.hLy), dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
        const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        if (!in_cutoff(P, d2, xi, xj)) continue;
        if (RIGID) {
            float gx, gy, gz, V, a, bb, c, u, v, w;
            rigid_pair<false, PP>(P, dx, dy, dz, d2, Ri, quat[j], gx, gy, gz, V, a, bb, c, u, v, w);
            fx -= gx; fy -= gy; fz -= gz; pe += V;
            tx += a; ty += bb; tz += c;
        } else {
            float g, V;
            lj_pair(P, d2, g, V);
            fx = fmaf(-g, dx, fx); fy = fmaf(-g, dy, fy); fz = fmaf(-g, dz, fz); pe += V;
        }
    }
    pe *= 0.5f;
    if (!RIGID && P.kind == MD_POT_FENE_WCA) {
        float bpe = 0.f;
        fene_vertex_s(P, B, pos, i, fx, fy, fz, bpe);
        pe += 0.5f * bpe;
    }
    if (!RIGID && fuse.vel) { fuse_kick_drift(0.5f * fuse.dt * P.inv_mass, fuse.dt, P.half_skin2, fuse.vel, pos, fuse.pos_next, B.pos_ref, &B.ctrl->rebuild, i, fx, fy, fz); return; }
    force[i] = make_float4(fx, fy, fz, pe);
    if (RIGID) torque[i] = make_float4(tx, ty, tz, 0.f);
}

template <int NS, bool ENERGY>
__global__ void __launch_bounds__(MD_TB * NS, NS == 1 ? 4 : (NS == 2 ? 2 : 1)) k_vertex_lj_staged(DevParams P, DevBuffers B, int stage_entries,
                                                                                  const float4* __restrict__ pos,
                                                                                  float4* __restrict__ force, FuseArgs fuse) {
    extern __shared__ __align__(16) unsigned char smraw[];
    const int b = blockIdx.x;
    const int tp = threadIdx.x % MD_TB, h = threadIdx.x / MD_TB;
    // everything the block needs from global memory before it can compute is requested at once: the block header, the
    // head of its segment table, |L_i| and the first four row chunks of this thread (rows hold >= 8 chunks; chunks past
    // |L_i| are loaded but never consumed)
    const SegPre pre = seg_preload(B, b);
    const int i = b * MD_TB + tp;
    const bool live = i < P.N;
    const uint2* __restrict__ rowb = reinterpret_cast<const uint2*>(B.rows) + (size_t)b * (P.rcap >> 2) * MD_TB + tp;
    const uint2* __restrict__ rowh = rowb + (size_t)h * MD_TB;
    const uint2 pkA = ld_row(rowh), pkB = ld_row(rowh + NS * MD_TB), pkC = ld_row(rowh + 2 * NS * MD_TB), pkD = ld_row(rowh + 3 * NS * MD_TB);
    const int cnt = live ? B.row_count[i] : 0;
    const BlkInfo bi = B.blk[b];
    if (bi.M <= 0) return;                         // the build failed for this block and latched the error: never guess
    if (bi.M + 1 > stage_entries) {                // launch sized too small for this block: slow path from global memory
        vertex_rows_unstaged<false, false>(P, B, bi, b, pos, nullptr, force, nullptr, fuse);
        return;
    }
    const Stage st = stage_issue<false>(P, B, bi, b, stage_entries, pre, pos, nullptr, smraw);
    float* xch = reinterpret_cast<float*>(st.spos + stage_entries);     // [NS - 1][6][MD_TB] floats, NS > 1 only
    stage_wait(P, bi, st, smraw);
    if (NS == 1 && !live) return;
    const bool bonds = P.kind == MD_POT_FENE_WCA;
    const bool img = (bi.flags & MD_BLK_WRAP) && !(bi.flags & MD_BLK_SHIFT_OK);
    const bool unit = P.sig2 == 1.0f;
#define LJ_ROWS(IMG_, SH_, UNIT_, EN_) vertex_lj_rows<IMG_, SH_, UNIT_, NS, EN_>(P, B, bi, st, i, live, cnt, rowb, pkA, pkB, pkC, pkD, xch, pos, force, bonds, fuse)
    // (the energy-free form exists for the reduced-unit loop only: sigma == 1 in every config)
    if (bi.flags & MD_BLK_SH4) {
        if (unit) { if (img) LJ_ROWS(true, 4, true, ENERGY); else LJ_ROWS(false, 4, true, ENERGY); }
        else { if (img) LJ_ROWS(true, 4, false, true); else LJ_ROWS(false, 4, false, true); }
    } else {
        if (unit) { if (img) LJ_ROWS(true, 0, true, ENERGY); else LJ_ROWS(false, 0, true, ENERGY); }
        else { if (img) LJ_ROWS(true, 0, false, true); else LJ_ROWS(false, 0, false, true); }
    }
#undef LJ_ROWS
}

// ------------------------------------------------------------------------------------------------
// VERTEX, patchy rigid bodies, staged: positions and quaternions of the neighbourhood in shared memory
// ------------------------------------------------------------------------------------------------
template <bool IMG, bool PP>
__device__ __forceinline__ void patchy_visit_s(const DevParams& P, const Stage& st, float4 xi, const Rot& Ri, unsigned int t,
                                               float& fx, float& fy, float& fz, float& pe, float& tx, float& ty, float& tz) {
    const float4 xj = st.spos[t];
    float dx, dy, dz;
    if (IMG) {
        dx = min_image(xj.x, xi.x, P.Lx, P.hLx); dy = min_image(xj.y, xi.y, P.Ly, P.hLy); dz = min_image(xj.z, xi.z, P.Lz, P.hLz);
    } else {
        dx = xj.x - xi.x; dy = xj.y - xi.y; dz = xj.z - xi.z;
    }
    const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (in_cutoff(P, d2, xi, xj)) {
        const float4 qj = st.squat[t];
        float gx, gy, gz, V, a, bb, c, u, v, w;
        rigid_pair<false, PP>(P, dx, dy, dz, d2, Ri, qj, gx, gy, gz, V, a, bb, c, u, v, w);
        fx -= gx; fy -= gy; fz -= gz;
        tx += a; ty += bb; tz += c;
        pe += V;
    }
}

template <bool IMG, bool PP>
__device__ __forceinline__ void vertex_patchy_rows(const DevParams& P, const DevBuffers& B, const BlkInfo bi, const Stage& st, int b,
                                                   float4* __restrict__ force, float4* __restrict__ torque) {
    const int tid = threadIdx.x;
    const int i = b * MD_TB + tid;
    if (i >= P.N) return;
    const int cnt = B.row_count[i];
    const int me = bi.own_base + tid;
    const float4 xi = st.spos[me], qi = st.squat[me];
    const uint2* __restrict__ rowb = reinterpret_cast<const uint2*>(B.rows) + (size_t)b * (P.rcap >> 2) * MD_TB + tid;
    const int nch = (cnt + 3) >> 2;
    float fx = 0.f, fy = 0.f, fz = 0.f, pe = 0.f, tx = 0.f, ty = 0.f, tz = 0.f;
    const int sh = (bi.flags & MD_BLK_SH4) ? 4 : 0;
    const Rot Ri = quat_to_rot(qi);     // once per particle
    for (int c = 0; c < nch; ++c) {
        const uint2 cur = __ldg(rowb + (size_t)c * MD_TB);     // padding entries = dummy (far away -> outside the cutoff)
        patchy_visit_s<IMG, PP>(P, st, xi, Ri, (cur.x & 0xffffu) >> sh, fx, fy, fz, pe, tx, ty, tz);
        patchy_visit_s<IMG, PP>(P, st, xi, Ri, (cur.x >> 16) >> sh, fx, fy, fz, pe, tx, ty, tz);
        patchy_visit_s<IMG, PP>(P, st, xi, Ri, (cur.y & 0xffffu) >> sh, fx, fy, fz, pe, tx, ty, tz);
        patchy_visit_s<IMG, PP>(P, st, xi, Ri, (cur.y >> 16) >> sh, fx, fy, fz, pe, tx, ty, tz);
    }
    force[i] = make_float4(fx, fy, fz, 0.5f * pe);
    torque[i] = make_float4(tx, ty, tz, 0.f);
}

template <bool PP>
__global__ void __launch_bounds__(MD_TB, 4) k_vertex_patchy_staged(DevParams P, DevBuffers B, int stage_entries, const float4* __restrict__ pos,
                                                                const float4* __restrict__ quat, float4* __restrict__ force,
                                                                float4* __restrict__ torque) {
    extern __shared__ __align__(16) unsigned char smraw[];
    const int b = blockIdx.x;
    const BlkInfo bi = B.blk[b];
    if (bi.M <= 0) return;
    if (bi.M + 1 > stage_entries) {                // as in k_vertex_lj_staged
        vertex_rows_unstaged<true, PP>(P, B, bi, b, pos, quat, force, torque);
        return;
    }
    const SegPre pre = seg_preload(B, b);
    const Stage st = stage_issue<true>(P, B, bi, b, stage_entries, pre, pos, quat, smraw);
    stage_wait(P, bi, st, smraw);
    if ((bi.flags & MD_BLK_WRAP) && !(bi.flags & MD_BLK_SHIFT_OK)) vertex_patchy_rows<true, PP>(P, B, bi, st, b, force, torque);
    else vertex_patchy_rows<false, PP>(P, B, bi, st, b, force, torque);
}

// ------------------------------------------------------------------------------------------------
// host-side dispatch
// ------------------------------------------------------------------------------------------------
size_t md_staged_smem_bytes(const md_system* s, int stage_entries) {
    return 16 + 16 * (size_t)stage_entries * (s->rigid ? 2 : 1);
}

// Function attributes are per DEVICE: set for the handle's device at md_create (a second handle on another GPU of the
// same process gets its own opt-in), never behind a process-wide flag.
void md_staged_configure(md_system* s) {
    const int optin = (int)s->smem_optin;
    cudaFuncSetAttribute(k_build_staged<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_build_staged<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_edges_from_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_vertex_lj_staged<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_vertex_lj_staged<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_vertex_lj_staged<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_vertex_lj_staged<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_vertex_lj_staged<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_vertex_lj_staged<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    // the neighbourhoods live in shared memory and the rows bypass L1: ask for the largest shared-memory carveout so that
    // as many blocks as the sizing in sync_and_check counted on are resident
    cudaFuncSetAttribute(k_vertex_lj_staged<1, true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_vertex_lj_staged<1, false>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_vertex_lj_staged<2, true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_vertex_lj_staged<2, false>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_vertex_lj_staged<4, true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_vertex_lj_staged<4, false>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_vertex_patchy_staged<false>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_vertex_patchy_staged<true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaFuncSetAttribute(k_vertex_patchy_staged<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    cudaFuncSetAttribute(k_vertex_patchy_staged<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
    s->build_carve = -1;
}

// which instantiation of k_vertex_lj_staged a launch capacity of `smem` bytes selects: threads per particle
static int staged_lj_ns(const md_system* s, size_t smem) {
    const size_t optin = s->smem_optin, per_sm = s->smem_per_sm;
    if (2 * (smem + 24 * MD_TB + 1024) > per_sm - 1024 && smem + 72 * MD_TB <= optin && s->P.rcap >= 64) return 4;   // one block per SM
    if (smem > 75 * 1024 && smem + 24 * MD_TB <= optin) return 2;                                                      // <= 2 blocks per SM
    return 1;
}

static int staged_launch_entries(const md_system* s) {
    int se = s->stage_launch;
    if (s->stage_limit > 0) se = std::min(se, s->stage_limit);   // MD_OPT_STAGE_LIMIT (tests): force blocks onto the unstaged path
    return se;
}

int md_staged_threads_per_particle(const md_system* s) {
    if (s->rigid || s->order == MD_ORDER_NONE) return 0;
    return staged_lj_ns(s, md_staged_smem_bytes(s, staged_launch_entries(s)));
}

// VERTEX on the staged rows.  Returns false if the neighbourhood does not fit in shared memory.
bool md_launch_forces_staged(md_system* s, bool energy, FuseArgs fuse) {
    const DevParams& P = s->P;
    const int se = staged_launch_entries(s);
    const size_t smem = md_staged_smem_bytes(s, se);
    if (smem > s->smem_optin) return false;
    if (P.kind == MD_POT_PATCHY && P.pp_model) k_vertex_patchy_staged<true><<<P.nblk, MD_TB, smem, s->stream>>>(P, s->B, se, s->pos, s->quat, s->force, s->torque);
    else if (P.kind == MD_POT_PATCHY) k_vertex_patchy_staged<false><<<P.nblk, MD_TB, smem, s->stream>>>(P, s->B, se, s->pos, s->quat, s->force, s->torque);
    else {
        const int ns = staged_lj_ns(s, smem);
        if (ns == 4)        // one block per SM: four threads per particle (1024-thread blocks, 32 warps on the SM)
            { if (energy) k_vertex_lj_staged<4, true><<<P.nblk, 4 * MD_TB, smem + 72 * MD_TB, s->stream>>>(P, s->B, se, s->pos, s->force, fuse);
              else k_vertex_lj_staged<4, false><<<P.nblk, 4 * MD_TB, smem + 72 * MD_TB, s->stream>>>(P, s->B, se, s->pos, s->force, fuse); }
        else if (ns == 2)   // <= 2 blocks per SM: two threads per particle
            { if (energy) k_vertex_lj_staged<2, true><<<P.nblk, 2 * MD_TB, smem + 24 * MD_TB, s->stream>>>(P, s->B, se, s->pos, s->force, fuse);
              else k_vertex_lj_staged<2, false><<<P.nblk, 2 * MD_TB, smem + 24 * MD_TB, s->stream>>>(P, s->B, se, s->pos, s->force, fuse); }
        else if (energy) k_vertex_lj_staged<1, true><<<P.nblk, MD_TB, smem, s->stream>>>(P, s->B, se, s->pos, s->force, fuse);
        else k_vertex_lj_staged<1, false><<<P.nblk, MD_TB, smem, s->stream>>>(P, s->B, se, s->pos, s->force, fuse);
    }
    s->launches += 1;
    return true;
}
