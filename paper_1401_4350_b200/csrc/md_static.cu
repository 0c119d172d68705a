// md_static.cu -- md_energy_static(): the energy sums of S:A9 (U = sum_i pe_i, K_t = 1/2 m sum |v|^2, K_r = sum |L|^2 / 2I,
// fp32 terms accumulated in fp64, two deterministic stages) for callers that may not allocate: code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc.  No handle, no workspace: the block partials of the first
// stage live in a file-scope device array of fixed size, which every GPU that loads the library holds until exit
// (48 KiB).  The entry point calls no cudaMalloc / cudaFree and no allocating library routine.
//
// The array's NAME is a host-side stand-in in host code, not a device address: its device address is looked up with
// cudaGetSymbolAddress once per device (with that device current) and passed to the kernels.
//
// Every call on a device shares the array.  It keeps the last call's contents; each call overwrites every partial it
// reads, so nothing has to start at zero -- but two calls that overlap on the GPU (different streams of one device,
// or two host threads) race on it: serialise them.
#include <stdio.h>
#include <stdint.h>
#include <mutex>
#include <cuda_runtime.h>
#include "md_b200.h"

#define ST_THREADS 256
#define ST_CHUNK 8192                                    // particles per block of the first stage
#define ST_BLOCKS (MD_ENERGY_STATIC_MAX_N / ST_CHUNK)    // 2048 blocks x 3 doubles = 48 KiB
#define ST_MAX_DEVICES 64

static __device__ __align__(256) double md_static_epart[3 * ST_BLOCKS];

static std::mutex g_st_mutex;
static double* g_st_ptr[ST_MAX_DEVICES];                 // device address of md_static_epart on device d, once looked up

static __device__ __forceinline__ double st_block_sum(double v, double* sh) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) sh[w] = v;
    __syncthreads();
    double r = 0.0;
    if (w == 0) {
        r = lane < (blockDim.x >> 5) ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
    }
    __syncthreads();
    return r;
}

// stage 1: block b sums particles [b * ST_CHUNK, (b + 1) * ST_CHUNK) and overwrites its three partials
__global__ void __launch_bounds__(ST_THREADS) k_energy_static_partial(const float4* __restrict__ vel, const float4* __restrict__ force,
                                                                      const float4* __restrict__ angmom, int n, double* part) {
    __shared__ double sh[32];
    double u = 0.0, kt = 0.0, kr = 0.0;
    const int i0 = blockIdx.x * ST_CHUNK, i1 = min(n, i0 + ST_CHUNK);
    for (int i = i0 + threadIdx.x; i < i1; i += ST_THREADS) {
        u += (double)force[i].w;
        const float4 v = vel[i];
        kt += (double)v.x * v.x + (double)v.y * v.y + (double)v.z * v.z;
        if (angmom) {
            const float4 L = angmom[i];
            kr += (double)L.x * L.x + (double)L.y * L.y + (double)L.z * L.z;
        }
    }
    u = st_block_sum(u, sh); kt = st_block_sum(kt, sh); kr = st_block_sum(kr, sh);
    if (threadIdx.x == 0) {
        part[3 * blockIdx.x + 0] = u;
        part[3 * blockIdx.x + 1] = kt;
        part[3 * blockIdx.x + 2] = kr;
    }
}

// stage 2: one block sums the nblocks partials of THIS call in a fixed order
__global__ void __launch_bounds__(ST_THREADS) k_energy_static_final(const double* __restrict__ part, int nblocks, double mass,
                                                                    double inv_inertia, double* __restrict__ e_out) {
    __shared__ double sh[32];
    double u = 0.0, kt = 0.0, kr = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += ST_THREADS) {
        u += part[3 * b + 0]; kt += part[3 * b + 1]; kr += part[3 * b + 2];
    }
    u = st_block_sum(u, sh); kt = st_block_sum(kt, sh); kr = st_block_sum(kr, sh);
    if (threadIdx.x == 0) {
        e_out[0] = u;
        e_out[1] = 0.5 * mass * kt;
        e_out[2] = 0.5 * inv_inertia * kr;
    }
}

static md_status st_fail(md_status st, char* err, size_t err_len, const char* msg, const char* detail = nullptr) {
    if (err && err_len > 0) {
        if (detail) snprintf(err, err_len, "md_energy_static: %s (%s)", msg, detail);
        else snprintf(err, err_len, "md_energy_static: %s", msg);
    }
    return st;
}

extern "C" md_status md_energy_static(const void* vel_dev, const void* force_dev, const void* angmom_dev, int64_t n, double mass,
                                      double inv_inertia, double* e_out_dev, void* cuda_stream, char* err, size_t err_len) {
    if (err && err_len > 0) err[0] = 0;
    if (!vel_dev || !force_dev || !e_out_dev) return st_fail(MD_ERR_INVALID, err, err_len, "vel_dev, force_dev and e_out_dev must not be NULL");
    if (n < 1) return st_fail(MD_ERR_INVALID, err, err_len, "n must be >= 1");
    if (n > (int64_t)MD_ENERGY_STATIC_MAX_N) {
        char d[96];
        snprintf(d, sizeof d, "n = %lld, MD_ENERGY_STATIC_MAX_N = %d", (long long)n, MD_ENERGY_STATIC_MAX_N);
        return st_fail(MD_ERR_CAPACITY, err, err_len, "n exceeds the capacity of the static scratch array", d);
    }
    if ((((uintptr_t)vel_dev) | ((uintptr_t)force_dev) | ((uintptr_t)angmom_dev)) & 15u)
        return st_fail(MD_ERR_INVALID, err, err_len, "state arrays must be 16-byte aligned float4 arrays");
    if (((uintptr_t)e_out_dev) & 7u) return st_fail(MD_ERR_INVALID, err, err_len, "e_out_dev must be 8-byte aligned");

    // set-up, once per device, with that device current: the device address of the scratch array
    int dev = -1;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) return st_fail(MD_ERR_CUDA, err, err_len, "cudaGetDevice", cudaGetErrorString(ce));
    if (dev < 0 || dev >= ST_MAX_DEVICES) return st_fail(MD_ERR_INVALID, err, err_len, "device ordinal beyond ST_MAX_DEVICES");
    double* part = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_st_mutex);
        if (!g_st_ptr[dev]) {
            double* p = nullptr;
            ce = cudaGetSymbolAddress((void**)&p, md_static_epart);
            if (ce != cudaSuccess || !p) return st_fail(MD_ERR_CUDA, err, err_len, "cudaGetSymbolAddress(md_static_epart)", cudaGetErrorString(ce));
            g_st_ptr[dev] = p;
        }
        part = g_st_ptr[dev];
    }

    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nb = (int)((n + ST_CHUNK - 1) / ST_CHUNK);     // <= ST_BLOCKS by the check above
    k_energy_static_partial<<<nb, ST_THREADS, 0, st>>>((const float4*)vel_dev, (const float4*)force_dev, (const float4*)angmom_dev, (int)n, part);
    k_energy_static_final<<<1, ST_THREADS, 0, st>>>(part, nb, mass, inv_inertia, e_out_dev);
    ce = cudaGetLastError();
    if (ce != cudaSuccess) return st_fail(MD_ERR_CUDA, err, err_len, "kernel launch", cudaGetErrorString(ce));
    return MD_OK;
}
