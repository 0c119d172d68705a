// md_dd.cu -- what a space decomposition ("the domain ... partitioned into smaller subsets", S:8(e), S:8(f4)) needs
// from the single-GPU library.  A rank runs the unchanged cell / Verlet / force kernels on the particles it OWNS plus
// GHOST copies of the neighbouring ranks' particles within the halo width of its slab, all in GLOBAL coordinates and the
// GLOBAL periodic box (the minimum image then needs no special case).  Added here:
//   md_resize        the particle count of a handle may shrink / grow below its creation capacity (migration changes it)
//   md_set_active    ghosts = original ids >= n_active: never kicked or drifted, left out of md_energy
//   md_half_step     the two halves of a velocity-Verlet step as separate calls (the halo refresh sits between them)
//   md_rebuild_flag  the device-side skin flag, read back (the ranks agree on a rebuild with one all-reduce)
//   md_gather_ids / md_scatter_ids   pack the send list / unpack the ghosts by ORIGINAL id (slot order is the library's business)
//   md_dd_select     stable compaction of the indices with lo <= coordinate < hi (migration and halo zones)
// The driver (paper_1401_4350_b200/dd.py) owns the protocol and moves bytes with torch.distributed; every arithmetic
// step on particle data runs in the kernels below.
#include <stdio.h>
#include "md_internal.cuh"

static inline int cdiv64(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

__global__ void __launch_bounds__(256) k_gather_ids(DevBuffers B, const float4* __restrict__ arr, const int* __restrict__ ids, int first_id,
                                                    int n, float4* __restrict__ dst) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int id = ids ? ids[k] : first_id + k;
    dst[k] = arr[B.slot_of_id[id]];
}

__global__ void __launch_bounds__(256) k_scatter_ids(DevBuffers B, float4* __restrict__ arr, int first_id, int n, const float4* __restrict__ src) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    arr[B.slot_of_id[first_id + k]] = src[k];
}

// ---- stable compaction of { i : lo <= x_i[axis] < hi }, three kernels, deterministic (index order) ----
#define SEL_CHUNK 1024
__device__ __forceinline__ bool sel_pred(const float4* __restrict__ pos, int i, int axis, float lo, float hi) {
    const float4 x = pos[i];
    const float v = axis == 0 ? x.x : (axis == 1 ? x.y : x.z);
    return v >= lo && v < hi;
}

__global__ void __launch_bounds__(256) k_sel_count(const float4* __restrict__ pos, int n, int axis, float lo, float hi, unsigned int* blk) {
    __shared__ unsigned int sh[8];
    unsigned int c = 0;
    for (int t = threadIdx.x; t < SEL_CHUNK; t += 256) {
        const int i = blockIdx.x * SEL_CHUNK + t;
        c += (i < n && sel_pred(pos, i, axis, lo, hi)) ? 1u : 0u;
    }
    c = __reduce_add_sync(0xffffffffu, c);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) { unsigned int s = 0; for (int w = 0; w < 8; ++w) s += sh[w]; blk[blockIdx.x] = s; }
}

__global__ void __launch_bounds__(1024) k_sel_scan(unsigned int* blk, int nb, unsigned int* total) {
    __shared__ unsigned int sh[32];
    __shared__ unsigned int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 1024) {
        const int i = base + threadIdx.x;
        const unsigned int v = i < nb ? blk[i] : 0u;
        unsigned int x = v;
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        for (int o = 1; o < 32; o <<= 1) { const unsigned int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) sh[w] = x;
        __syncthreads();
        if (w == 0) {
            unsigned int s = sh[lane];
            for (int o = 1; o < 32; o <<= 1) { const unsigned int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
            sh[lane] = s;
        }
        __syncthreads();
        const unsigned int c = carry;
        const unsigned int ex = c + (w ? sh[w - 1] : 0u) + x - v;
        if (i < nb) blk[i] = ex;
        __syncthreads();
        if (threadIdx.x == 1023) carry = ex + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = carry;
}

__global__ void __launch_bounds__(256) k_sel_write(const float4* __restrict__ pos, int n, int axis, float lo, float hi,
                                                   const unsigned int* __restrict__ blk, int* __restrict__ out, int cap) {
    __shared__ unsigned int sh[8];
    unsigned int base = blk[blockIdx.x];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int t0 = 0; t0 < SEL_CHUNK; t0 += 256) {        // index order inside the block: chunk by chunk, warp by warp, lane by lane
        const int i = blockIdx.x * SEL_CHUNK + t0 + threadIdx.x;
        const bool p = i < n && sel_pred(pos, i, axis, lo, hi);
        const unsigned int b = __ballot_sync(0xffffffffu, p);
        if (lane == 0) sh[w] = __popc(b);
        __syncthreads();
        unsigned int off = base;
        for (int q = 0; q < w; ++q) off += sh[q];
        unsigned int tot = 0;
        for (int q = 0; q < 8; ++q) tot += sh[q];
        if (p) {
            const unsigned int o = off + __popc(b & ((1u << lane) - 1u));
            if ((int)o < cap) out[o] = i;
        }
        base += tot;
        __syncthreads();
    }
}

extern "C" {

md_status md_dd_select(const void* pos_dev, int64_t n, int32_t axis, double lo, double hi, int32_t* idx_out_dev, int64_t capacity,
                       int64_t* count_host, void* scratch_dev, size_t scratch_bytes, void* cuda_stream) {
    if (!pos_dev || n < 0 || n >= (1ll << 31) || axis < 0 || axis > 2 || !count_host || !scratch_dev) return MD_ERR_INVALID;
    const int nb = cdiv64(n > 0 ? n : 1, SEL_CHUNK);
    if (scratch_bytes < 4 * (size_t)(nb + 2) || ((uintptr_t)scratch_dev & 3)) return MD_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned int* blk = (unsigned int*)scratch_dev;
    unsigned int* total = blk + nb;
    // the interval is compared in fp32 like every coordinate of the path; the driver passes fp32-representable bounds
    const float flo = (float)lo, fhi = (float)hi;
    k_sel_count<<<nb, 256, 0, st>>>((const float4*)pos_dev, (int)n, axis, flo, fhi, blk);
    k_sel_scan<<<1, 1024, 0, st>>>(blk, nb, total);
    if (idx_out_dev && capacity > 0)
        k_sel_write<<<nb, 256, 0, st>>>((const float4*)pos_dev, (int)n, axis, flo, fhi, blk, idx_out_dev, (int)(capacity < (1ll << 31) - 1 ? capacity : (1ll << 31) - 1));
    unsigned int h = 0;
    cudaMemcpyAsync(&h, total, 4, cudaMemcpyDeviceToHost, st);
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return MD_ERR_CUDA;
    *count_host = (int64_t)h;
    return MD_OK;
}

static float4* dd_array(md_system* s, int32_t array) {
    switch (array) {
    case MD_ARRAY_POS: return s->pos;
    case MD_ARRAY_VEL: return s->vel;
    case MD_ARRAY_FORCE: return s->force;
    case MD_ARRAY_QUAT: return s->quat;
    case MD_ARRAY_ANGMOM: return s->angmom;
    case MD_ARRAY_TORQUE: return s->torque;
    default: return nullptr;
    }
}

md_status md_gather_ids(md_system* s, int32_t array, const int32_t* ids_dev, int64_t first_id, int64_t n, void* dst_dev) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    float4* arr = s->bound ? dd_array(s, array) : nullptr;
    if (!arr || n < 0 || (n > 0 && !dst_dev) || (!ids_dev && (first_id < 0 || first_id + n > s->N))) {
        MD_ERRBUF(s, "md_gather_ids: unbound state, unknown array or id range outside [0, N)");
        return MD_ERR_INVALID;
    }
    if (n == 0) return MD_OK;
    k_gather_ids<<<cdiv64(n, 256), 256, 0, s->stream>>>(s->B, arr, ids_dev, (int)first_id, (int)n, (float4*)dst_dev);
    s->launches += 1;
    return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

md_status md_scatter_ids(md_system* s, int32_t array, int64_t first_id, int64_t n, const void* src_dev) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    float4* arr = s->bound ? dd_array(s, array) : nullptr;
    if (!arr || n < 0 || (n > 0 && !src_dev) || first_id < 0 || first_id + n > s->N) {
        MD_ERRBUF(s, "md_scatter_ids: unbound state, unknown array or id range outside [0, N)");
        return MD_ERR_INVALID;
    }
    if (n == 0) return MD_OK;
    k_scatter_ids<<<cdiv64(n, 256), 256, 0, s->stream>>>(s->B, arr, (int)first_id, (int)n, (const float4*)src_dev);
    s->launches += 1;
    if (array == MD_ARRAY_POS || array == MD_ARRAY_QUAT) s->forces_valid = false;   // the forces describe the old positions
    return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

md_status md_resize(md_system* s, int64_t n_new) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (n_new <= 0 || n_new > s->N_capacity) { MD_ERRBUF(s, "md_resize: N must be in [1, N at creation]"); return MD_ERR_INVALID; }
    s->N = n_new;
    s->P.N = (int)n_new;
    s->P.ntiles = (int)((n_new + MD_TILE - 1) / MD_TILE);
    s->P.nblk = (int)((n_new + MD_TB - 1) / MD_TB);
    s->P.n_active = (int)n_new;
    s->bound = false;                      // the caller binds arrays of the new length
    s->cells_valid = s->lists_valid = s->forces_valid = s->seg_valid = s->staged_valid = s->legacy_valid = s->cluster_valid = false;
    s->shadow_valid = false;
    md_drop_graphs(s);
    return MD_OK;
}

md_status md_set_active(md_system* s, int64_t n_active) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (n_active < 0 || n_active > s->N) { MD_ERRBUF(s, "md_set_active: n_active must be in [0, N]"); return MD_ERR_INVALID; }
    if (n_active < s->N && s->precision != MD_PREC_F32) { MD_ERRBUF(s, "md_set_active: ghosts need MD_PREC_F32"); return MD_ERR_STATE; }
    s->P.n_active = (int)n_active;
    md_drop_graphs(s);                     // the step graph bakes the parameter block in
    return MD_OK;
}

md_status md_half_step(md_system* s, double dt, int32_t part) {
    if (!s) return MD_ERR_INVALID;
    if (s->sticky) return (md_status)s->sticky;
    if (!s->bound || !s->forces_valid) { MD_ERRBUF(s, "md_half_step: needs a bound state and valid forces"); return MD_ERR_STATE; }
    if (!(dt > 0) || (part != MD_STEP_KICK_DRIFT && part != MD_STEP_KICK)) { MD_ERRBUF(s, "md_half_step: dt > 0 and a known part required"); return MD_ERR_INVALID; }
    if (s->precision != MD_PREC_F32) { MD_ERRBUF(s, "md_half_step: fp32 state only"); return MD_ERR_STATE; }
    if (part == MD_STEP_KICK_DRIFT) {
        md_launch_kick_drift(s, (float)dt, false);   // sets the device rebuild flag (S:A5)
        s->forces_valid = false;                     // the forces belong to the old positions: md_forces before the closing kick
    } else {
        md_launch_kick(s, (float)dt);
    }
    return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ERR_CUDA;
}

}  // extern "C"
