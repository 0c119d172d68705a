// md_build.cu -- cell binning + counting sort (S:A2), optional cell/Hilbert reordering (S:A3),
// Verlet-list build (S:A4), edge list and the incoming-edge index of the segmented scatter.
// Every kernel takes its data-dependent sizes from device memory and can be "gated" on the device-side
// rebuild flag (S:H6), so md_integrate never synchronises with the host.
#include <stdio.h>
#include "md_internal.cuh"

#define GATE(B, gated) if ((gated) && (B).ctrl->rebuild == 0) return

static inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// ------------------------------------------------------------------------------------------------
// generic exclusive scan of unsigned int (three kernels, deterministic)
// ------------------------------------------------------------------------------------------------
#define SCAN_THREADS 256
#define SCAN_ITEMS 16
#define SCAN_CHUNK (SCAN_THREADS * SCAN_ITEMS)

__device__ __forceinline__ unsigned int block_excl_scan(unsigned int v, unsigned int* total, unsigned int* sh) {
    // exclusive scan of one value per thread across the block (blockDim.x <= 1024, multiple of 32)
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    unsigned int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) sh[w] = x;
    __syncthreads();
    if (w == 0) {
        unsigned int s = lane < nw ? sh[lane] : 0u;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned int y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += y;
        }
        if (lane < nw) sh[lane] = s;   // inclusive over warps
    }
    __syncthreads();
    unsigned int base = w ? sh[w - 1] : 0u;
    *total = sh[nw - 1];
    __syncthreads();
    return base + x - v;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(DevBuffers B, int gated, const unsigned int* in, int n) {
    GATE(B, gated);
    __shared__ unsigned int sh[32];
    int base = blockIdx.x * SCAN_CHUNK;
    unsigned int s = 0;
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        int idx = base + k * SCAN_THREADS + threadIdx.x;
        if (idx < n) s += in[idx];
    }
    unsigned int tot;
    block_excl_scan(s, &tot, sh);
    if (threadIdx.x == 0) B.scan_blk[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) k_scan_top(DevBuffers B, int gated, int nb, unsigned int* total_out) {
    GATE(B, gated);
    __shared__ unsigned int sh[32];
    __shared__ unsigned int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        int idx = base + threadIdx.x;
        unsigned int v = idx < nb ? B.scan_blk[idx] : 0u;
        unsigned int tot;
        unsigned int ex = block_excl_scan(v, &tot, sh);
        unsigned int c = carry;
        if (idx < nb) B.scan_blk[idx] = c + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry = c + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0 && total_out) *total_out = carry;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(DevBuffers B, int gated, const unsigned int* in, unsigned int* out, int n) {
    GATE(B, gated);
    __shared__ unsigned int sh[32];
    int base = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;   // thread owns SCAN_ITEMS consecutive items
    unsigned int v[SCAN_ITEMS];
    unsigned int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        int idx = base + k;
        v[k] = idx < n ? in[idx] : 0u;
        s += v[k];
    }
    unsigned int tot;
    unsigned int ex = block_excl_scan(s, &tot, sh) + B.scan_blk[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        int idx = base + k;
        if (idx < n) out[idx] = ex;
        ex += v[k];
        if (idx == n - 1) out[n] = ex;   // out has n+1 entries
    }
}

// out[0..n] = exclusive scan of in[0..n-1]; *total_out (device) = sum.  in and out may alias.
static void launch_scan(md_system* s, bool gated, const unsigned int* in, unsigned int* out, int n, unsigned int* total_out) {
    int nb = cdiv(n, SCAN_CHUNK);
    k_scan_reduce<<<nb, SCAN_THREADS, 0, s->stream>>>(s->B, gated, in, n);
    k_scan_top<<<1, 1024, 0, s->stream>>>(s->B, gated, nb, total_out);
    k_scan_apply<<<nb, SCAN_THREADS, 0, s->stream>>>(s->B, gated, in, out, n);
    s->launches += 3;
}

// ------------------------------------------------------------------------------------------------
// S:A2 cell binning ("cell filling ... one-particle-per-thread")
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float wrap1(float x, float L) {
    // S:Q7: x - L*floor(x/L); the fp32 result may equal L -> clamp to 0
    if (x >= 0.0f && x < L) return x;
    float w = x - L * floorf(x / L);
    if (!(w >= 0.0f) || w >= L) w = 0.0f;
    return w;
}

__device__ __forceinline__ int cell_coord(float x, double scale, int n) {
    int c = (int)floor((double)x * scale);   // binning in double: exact classification of the stored fp32 value (S:H2)
    return c < 0 ? 0 : (c >= n ? n - 1 : c);
}

__global__ void k_zero_counts(DevParams P, DevBuffers B, int gated) {
    GATE(B, gated);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i <= P.ncell) B.cell_count[i] = 0;
}

__global__ void k_wrap_bin(DevParams P, DevBuffers B, int gated, float4* pos) {
    GATE(B, gated);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    float4 x = pos[i];
    x.x = wrap1(x.x, P.Lx); x.y = wrap1(x.y, P.Ly); x.z = wrap1(x.z, P.Lz);
    pos[i] = x;
    int cx = cell_coord(x.x, P.cscale_x, P.ncx);
    int cy = cell_coord(x.y, P.cscale_y, P.ncy);
    int cz = cell_coord(x.z, P.cscale_z, P.ncz);
    int c = B.cell_rank[(cx * P.ncy + cy) * P.ncz + cz];
    B.cell_of[i] = c;
    B.ids_tmp[i] = atomicAdd(&B.cell_count[c], 1);   // arrival index inside the cell (order fixed below)
}

// mixed precision: the fp64 position is wrapped, the fp32 position is its rounding, kept inside [0, L)
__device__ __forceinline__ double wrap1d(double x, double L) {
    if (x >= 0.0 && x < L) return x;
    double w = x - L * floor(x / L);
    if (!(w >= 0.0) || w >= L) w = 0.0;
    return w;
}
__device__ __forceinline__ float round_inside(double x, float L) {
    float f = (float)x;
    return f < L ? f : nextafterf(L, 0.0f);   // a double just below L may round up to L
}
__global__ void k_wrap_bin_mixed(DevParams P, DevBuffers B, int gated, float4* pos) {
    GATE(B, gated);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    double2* pxy = reinterpret_cast<double2*>(B.shadow[0]);
    double2* pz = reinterpret_cast<double2*>(B.shadow[1]);
    double2 xy = pxy[i], z_ = pz[i];
    xy.x = wrap1d(xy.x, P.dLx); xy.y = wrap1d(xy.y, P.dLy); z_.x = wrap1d(z_.x, P.dLz);
    pxy[i] = xy; pz[i] = z_;
    float4 x = pos[i];
    x.x = round_inside(xy.x, P.Lx); x.y = round_inside(xy.y, P.Ly); x.z = round_inside(z_.x, P.Lz);
    pos[i] = x;
    int cx = cell_coord(x.x, P.cscale_x, P.ncx);
    int cy = cell_coord(x.y, P.cscale_y, P.ncy);
    int cz = cell_coord(x.z, P.cscale_z, P.ncz);
    int c = B.cell_rank[(cx * P.ncy + cy) * P.ncz + cz];
    B.cell_of[i] = c;
    B.ids_tmp[i] = atomicAdd(&B.cell_count[c], 1);
}

__global__ void k_cell_scatter(DevParams P, DevBuffers B, int gated) {
    GATE(B, gated);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    B.items_tmp[B.cell_start[B.cell_of[i]] + B.ids_tmp[i]] = i;
}

// deterministic order inside a cell: ascending slot (rank by counting; cells hold tens of particles)
__global__ void k_cell_rank_sort(DevParams P, DevBuffers B, int gated) {
    GATE(B, gated);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    int c = B.cell_of[i];
    int s = B.cell_start[c], e = B.cell_start[c + 1];
    int r = 0;
    for (int t = s; t < e; ++t) r += (B.items_tmp[t] < i);
    B.items[s + r] = i;
}

// ------------------------------------------------------------------------------------------------
// S:A3 physical reordering: new slot s takes the particle of old slot items[s]
// ------------------------------------------------------------------------------------------------
struct StateArrays { float4* a[14]; int n; };   // six fp32 arrays + up to eight fp64 half planes (mixed precision)

// all bound state arrays, ids and cell indices in one pass: plane k of tmp4 takes array k in the new order
__global__ void k_gather_state(DevParams P, DevBuffers B, int gated, StateArrays S, size_t plane) {
    GATE(B, gated);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int o = B.items[i];
    const int id = B.ids[o], cell = B.cell_of[o];
    for (int k0 = 0; k0 < S.n; k0 += 4) {        // four loads in flight before the first store (the arrays may alias for the compiler)
        float4 v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) if (k0 + q < S.n) v[q] = S.a[k0 + q][o];
#pragma unroll
        for (int q = 0; q < 4; ++q) if (k0 + q < S.n) B.tmp4[(k0 + q) * plane + i] = v[q];
    }
    B.ids_tmp[i] = id;
    B.items_tmp[i] = cell;
}
__global__ void k_commit_state(DevParams P, DevBuffers B, int gated, StateArrays S, size_t plane) {
    GATE(B, gated);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int id = B.ids_tmp[i], cell = B.items_tmp[i];
    for (int k0 = 0; k0 < S.n; k0 += 4) {
        float4 v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) if (k0 + q < S.n) v[q] = B.tmp4[(k0 + q) * plane + i];
#pragma unroll
        for (int q = 0; q < 4; ++q) if (k0 + q < S.n) S.a[k0 + q][i] = v[q];
    }
    B.ids[i] = id;
    B.slot_of_id[id] = i;
    B.cell_of[i] = cell;
    B.items[i] = i;   // storage order == cell order from now on
}

void md_launch_build_cells(md_system* s, bool gated) {
    const DevParams& P = s->P;
    int g = gated ? 1 : 0;
    int nbN = cdiv(P.N, 256);
    k_zero_counts<<<cdiv(P.ncell + 1, 256), 256, 0, s->stream>>>(P, s->B, g);
    const bool mixed = s->precision == MD_PREC_MIXED && s->shadow_valid;
    if (mixed) k_wrap_bin_mixed<<<nbN, 256, 0, s->stream>>>(P, s->B, g, s->pos);
    else k_wrap_bin<<<nbN, 256, 0, s->stream>>>(P, s->B, g, s->pos);
    s->launches += 2;
    launch_scan(s, gated, (const unsigned int*)s->B.cell_count, (unsigned int*)s->B.cell_start, P.ncell, nullptr);
    k_cell_scatter<<<nbN, 256, 0, s->stream>>>(P, s->B, g);
    k_cell_rank_sort<<<nbN, 256, 0, s->stream>>>(P, s->B, g);
    s->launches += 2;
    if (s->order != MD_ORDER_NONE) {
        // inside md_integrate (gated) the rebuild sits between the drift and the force evaluation: forces and torques are
        // dead there and are recomputed in the new order right after, so they are not carried through the permutation
        float4* arrs[6] = { s->pos, s->vel, gated ? nullptr : s->force, s->quat, s->angmom, gated ? nullptr : s->torque };
        StateArrays S;
        S.n = 0;
        for (int a = 0; a < 6; ++a) if (arrs[a]) S.a[S.n++] = arrs[a];
        if (mixed) for (int k = 0; k < (s->rigid ? 8 : 4); ++k) S.a[S.n++] = s->B.shadow[k];
        const size_t plane = (size_t)P.ntiles * MD_TILE;
        k_gather_state<<<nbN, 256, 0, s->stream>>>(P, s->B, g, S, plane);
        k_commit_state<<<nbN, 256, 0, s->stream>>>(P, s->B, g, S, plane);
        s->launches += 2;
    }
}

// ------------------------------------------------------------------------------------------------
// S:A4 Verlet list ("Verlet lists updating ... one-particle-per-thread").
// Predicate S:O0 in fp64 on the fp32 positions, fixed operation order, no FMA contraction.
// ------------------------------------------------------------------------------------------------
__global__ void k_build_begin(DevBuffers B, int gated) {
    GATE(B, gated);
    B.ctrl->max_seen = 0;
    B.ctrl->n_full = 0ull;
}

__device__ __forceinline__ int full_index(int tile, int lane, int k, int capg) {
    return ((tile * capg + (k >> 2)) * MD_TILE + lane) * 4 + (k & 3);
}

template <bool IDENT>
__global__ void __launch_bounds__(128) k_build_verlet(DevParams P, DevBuffers B, int gated, const float4* __restrict__ pos) {
    GATE(B, gated);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31, tile = i >> 5;
    int cnt = 0, half = 0, img = 0;
    if (i < P.N) {
        const float4 xi4 = pos[i];
        const double xi = xi4.x, yi = xi4.y, zi = xi4.z;
        const int cx = cell_coord(xi4.x, P.cscale_x, P.ncx);
        const int cy = cell_coord(xi4.y, P.cscale_y, P.ncy);
        const int cz = cell_coord(xi4.z, P.cscale_z, P.ncz);
        // S:Q8: 27-cell stencil, each distinct cell once when an axis has fewer than 3 cells
        const int x0 = P.ncx >= 3 ? -1 : 0, x1 = P.ncx >= 3 ? 1 : P.ncx - 1;
        const int y0 = P.ncy >= 3 ? -1 : 0, y1 = P.ncy >= 3 ? 1 : P.ncy - 1;
        const int z0 = P.ncz >= 3 ? -1 : 0, z1 = P.ncz >= 3 ? 1 : P.ncz - 1;
        const double hx = 0.5 * P.dLx, hy = 0.5 * P.dLy, hz = 0.5 * P.dLz;
        for (int ox = x0; ox <= x1; ++ox) {
            int ax = P.ncx >= 3 ? (cx + ox + P.ncx) % P.ncx : ox;
            for (int oy = y0; oy <= y1; ++oy) {
                int ay = P.ncy >= 3 ? (cy + oy + P.ncy) % P.ncy : oy;
                for (int oz = z0; oz <= z1; ++oz) {
                    int az = P.ncz >= 3 ? (cz + oz + P.ncz) % P.ncz : oz;
                    const int c = B.cell_rank[(ax * P.ncy + ay) * P.ncz + az];
                    const int s = B.cell_start[c], e = B.cell_start[c + 1];
                    for (int t = s; t < e; ++t) {
                        const int j = IDENT ? t : B.items[t];
                        if (j == i) continue;
                        const float4 xj = pos[j];
                        int w = 0;
                        double dx = (double)xj.x - xi;
                        if (dx > hx) { dx -= P.dLx; w = 1; } else if (dx < -hx) { dx += P.dLx; w = 1; }
                        double dy = (double)xj.y - yi;
                        if (dy > hy) { dy -= P.dLy; w = 1; } else if (dy < -hy) { dy += P.dLy; w = 1; }
                        double dz = (double)xj.z - zi;
                        if (dz > hz) { dz -= P.dLz; w = 1; } else if (dz < -hz) { dz += P.dLz; w = 1; }
                        const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
                        if (d2 < P.rv2d) {
                            if (cnt < P.cap) B.nl_full[full_index(tile, lane, cnt, P.capg)] = j;
                            ++cnt;
                            half += (j > i);
                            img |= w;
                        }
                    }
                }
            }
        }
        if (cnt > P.cap) { atomicOr(&B.ctrl->err, MD_DEVERR_CAPACITY); }
        B.nl_count[i] = cnt < P.cap ? cnt : P.cap;
        B.half_count[i] = cnt > P.cap ? 0 : half;
        B.pos_ref[i] = xi4;
    }
    int c2 = cnt < P.cap ? cnt : P.cap;
    int kmax = __reduce_max_sync(0xffffffffu, c2);
    int kmin = __reduce_min_sync(0xffffffffu, i < P.N ? c2 : 0);   // a tile with dead lanes takes the checked loop
    int tot = __reduce_add_sync(0xffffffffu, c2);
    int seen = __reduce_max_sync(0xffffffffu, cnt);
    int anyimg = __any_sync(0xffffffffu, img);
    // pad every row of the tile up to the tile's rounded-up length with the particle's own slot (masked by the
    // force kernels' validity test; keeps the gathers of the ragged tail in bounds)
    if (tile < P.ntiles) {
        const int self = i < P.N ? i : 0;
        for (int k = c2; k < ((kmax + 3) & ~3); ++k) B.nl_full[full_index(tile, lane, k, P.capg)] = self;
    }
    if (lane == 0 && tile < P.ntiles) {
        B.tile_info[tile] = make_int2(kmax | (anyimg << 30), kmin);
        atomicMax(&B.ctrl->max_seen, seen);
        atomicAdd(&B.ctrl->n_full, (unsigned long long)tot);
    }
}

// one EDGE thread per unordered pair -> explicit (i, j) list, i < j (slots), sorted by i.
// Bit 31 of j marks a pair whose minimum image crosses a periodic face.
__global__ void __launch_bounds__(128) k_fill_edges(DevParams P, DevBuffers B, int gated, const float4* __restrict__ pos) {
    GATE(B, gated);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= P.N) return;
    const int lane = i & 31, tile = i >> 5;
    const int cnt = B.nl_count[i];
    const float4 xi = pos[i];
    unsigned int o = B.edge_off[i];
    for (int k = 0; k < cnt; ++k) {
        int j = B.nl_full[full_index(tile, lane, k, P.capg)];
        if (j > i) {
            // a listed pair is either closer than r_v in raw coordinates or more than L - r_v apart: the fp32 test is safe
            const float4 xj = pos[j];
            int w = (fabsf(xj.x - xi.x) > P.hLx) | (fabsf(xj.y - xi.y) > P.hLy) | (fabsf(xj.z - xi.z) > P.hLz);
            B.edges[o++] = make_int2(i, j | (w << 31));
        }
    }
}

__global__ void k_build_end(DevBuffers B, int gated) {
    GATE(B, gated);
    if (gated) B.ctrl->n_rebuilds += 1;
    B.ctrl->rebuild = 0;
}

void md_launch_build_verlet(md_system* s, bool gated, const float4* pos_src) {
    const DevParams& P = s->P;
    int g = gated ? 1 : 0;
    k_build_begin<<<1, 1, 0, s->stream>>>(s->B, g);
    int nb = cdiv((int64_t)P.ntiles * MD_TILE, 128);
    if (s->order != MD_ORDER_NONE) k_build_verlet<true><<<nb, 128, 0, s->stream>>>(P, s->B, g, pos_src);
    else k_build_verlet<false><<<nb, 128, 0, s->stream>>>(P, s->B, g, pos_src);
    s->launches += 2;
    launch_scan(s, gated, (const unsigned int*)s->B.half_count, s->B.edge_off, P.N, &s->B.ctrl->n_edges);
    k_fill_edges<<<cdiv(P.N, 128), 128, 0, s->stream>>>(P, s->B, g, pos_src);
    s->launches += 1;
}

void md_launch_edge_offsets(md_system* s, bool gated) {
    launch_scan(s, gated, (const unsigned int*)s->B.half_count, s->B.edge_off, s->P.N, nullptr);
}

void md_launch_build_end(md_system* s, bool gated) {
    k_build_end<<<1, 1, 0, s->stream>>>(s->B, gated ? 1 : 0);
    s->launches += 1;
}

// ------------------------------------------------------------------------------------------------
// incoming-edge index for MD_SCATTER_SEGMENTED ("parallel segmented reduction"): for particle p the
// ids of the edges (q, p), q < p, in the order of p's own list -> a deterministic, atomic-free sum.
// ------------------------------------------------------------------------------------------------
__global__ void k_in_count(DevParams P, DevBuffers B, int gated) {
    GATE(B, gated);
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < P.N) B.items_tmp[i] = B.nl_count[i] - B.half_count[i];
}

__global__ void __launch_bounds__(128) k_in_fill(DevParams P, DevBuffers B, int gated) {
    GATE(B, gated);
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P.N) return;
    const int lane = p & 31, tile = p >> 5;
    const int cnt = B.nl_count[p];
    unsigned int o = B.in_off[p];
    for (int k = 0; k < cnt; ++k) {
        int q = B.nl_full[full_index(tile, lane, k, P.capg)];
        if (q < p) {
            unsigned int e0 = B.edge_off[q], e1 = B.edge_off[q + 1];
            for (unsigned int e = e0; e < e1; ++e)
                if ((B.edges[e].y & 0x7fffffff) == p) { B.in_edge[o++] = e; break; }
        }
    }
}

// gated = part of a device-side rebuild inside md_integrate (runs only when the rebuild flag is set)
void md_launch_seg_index(md_system* s, bool gated) {
    const DevParams& P = s->P;
    int g = gated ? 1 : 0;
    k_in_count<<<cdiv(P.N, 256), 256, 0, s->stream>>>(P, s->B, g);
    s->launches += 1;
    launch_scan(s, gated, (const unsigned int*)s->B.items_tmp, s->B.in_off, P.N, nullptr);
    k_in_fill<<<cdiv(P.N, 128), 128, 0, s->stream>>>(P, s->B, g);
    s->launches += 1;
}

// slot s holds original id s
__global__ void k_iota_ids(DevParams P, DevBuffers B) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < P.N) { B.ids[i] = i; B.slot_of_id[i] = i; }
}
void md_launch_iota_ids(md_system* s) {
    k_iota_ids<<<cdiv(s->P.N, 256), 256, 0, s->stream>>>(s->P, s->B);
    s->launches += 1;
}

// dst[ids[s]] = src[s]  (slot order -> original id order)
__global__ void k_unpermute(DevParams P, DevBuffers B, const float4* src, float4* dst) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < P.N) dst[B.ids[i]] = src[i];
}
// dst[s] = src[ids[s]]  (original id order -> slot order)
__global__ void k_permute_in(DevParams P, DevBuffers B, const float4* __restrict__ src, float4* __restrict__ dst) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < P.N) dst[i] = src[B.ids[i]];
}
void md_launch_permute_in(md_system* s, const float4* src, float4* dst) {
    k_permute_in<<<cdiv(s->P.N, 256), 256, 0, s->stream>>>(s->P, s->B, src, dst);
    s->launches += 1;
}
void md_launch_unpermute(md_system* s, const float4* src, float4* dst) {
    k_unpermute<<<cdiv(s->P.N, 256), 256, 0, s->stream>>>(s->P, s->B, src, dst);
    s->launches += 1;
}
