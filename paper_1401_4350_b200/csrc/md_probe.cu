// md_probe.cu -- md_probe(): the machine ceilings other than HBM that bound the force kernels, measured on the device
// the handle lives on (S:8(d): "the builder must measure an FFMA-chain and a MUFU-chain micro-benchmark on the box";
// "micro-benchmark red.global.add.f32 and .v4.f32 at random and at clustered addresses before interpreting EDGE
// numbers").  bench.py calls it in the same run as the timed kernels, so `roofline` quotes a peak measured under
// the same clocks.  Scratch comes from the caller's workspace (the permutation planes): nothing is allocated here.
#include <stdio.h>
#include "md_internal.cuh"

#define PROBE_NIT 4096
#define PROBE_CHAINS 8

// issue rates: 8 independent chains per thread, 8 blocks of 256 threads per SM
template <int MODE>
__global__ void __launch_bounds__(256) k_probe_alu(float* out, float s) {
    float a[PROBE_CHAINS], b[PROBE_CHAINS];
    float2 p[PROBE_CHAINS], q[PROBE_CHAINS];
    for (int k = 0; k < PROBE_CHAINS; ++k) {
        a[k] = threadIdx.x * 0.001f + k + 1.0f; b[k] = s + k;
        p[k] = make_float2(a[k], b[k]); q[k] = make_float2(b[k], a[k]);
    }
    const float2 c2 = make_float2(s, s * 0.5f);
    for (int it = 0; it < PROBE_NIT; ++it) {
#pragma unroll
        for (int k = 0; k < PROBE_CHAINS; ++k) {
            if (MODE == MD_PROBE_FFMA) a[k] = fmaf(a[k], b[k], s);
            if (MODE == MD_PROBE_FFMA2) p[k] = __ffma2_rn(p[k], q[k], c2);
            if (MODE == MD_PROBE_MUFU) { float r; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a[k])); a[k] = r * s; }
        }
    }
    float r = 0;
    for (int k = 0; k < PROBE_CHAINS; ++k) r += a[k] + b[k] + p[k].x + p[k].y + q[k].x;
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

// L2 reductions into n float4 accumulators (L2-resident, like force[]): every lane issues nred operations.
// PATTERN 0: addresses hashed over the whole array (a scatter to random particles); 1: consecutive lanes hit consecutive
// float4 (the flush of a contiguous accumulator range); V4: red.global.add.v4.f32, else red.global.add.f32.
template <int V4, int PATTERN>
__global__ void __launch_bounds__(256) k_probe_red(float4* acc, unsigned int n, int nred) {
    const unsigned int g = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int h = g * 2654435761u + 12345u;
    for (int r = 0; r < nred; ++r) {
        unsigned int j;
        if (PATTERN == 0) { h = h * 1664525u + 1013904223u; j = (h >> 8) % n; }
        else j = (g + (unsigned int)r * gridDim.x * blockDim.x) % n;
        if (V4) asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(acc + j), "f"(1.f), "f"(2.f), "f"(3.f), "f"(4.f) : "memory");
        else asm volatile("red.global.add.f32 [%0], %1;" ::"l"(reinterpret_cast<float*>(acc + j) + (r & 3)), "f"(1.f) : "memory");
    }
}

template <typename F>
static bool probe_time(cudaStream_t st, F launch, float* ms) {
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return false;
    launch();                                   // warm-up
    cudaStreamSynchronize(st);
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(a, st);
        launch();
        cudaEventRecord(b, st);
        if (cudaEventSynchronize(b) != cudaSuccess) { cudaEventDestroy(a); cudaEventDestroy(b); return false; }
        float t;
        cudaEventElapsedTime(&t, a, b);
        best = t < best ? t : best;
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    *ms = best;
    return cudaGetLastError() == cudaSuccess;
}

// value: TFLOP/s (FFMA, FFMA2), Tops/s (MUFU), G lane-operations/s (the reductions).  false on a CUDA error.
bool md_run_probe(md_system* s, int kind, double* value) {
    int nb = s->sm_count * 8;
    float* out = reinterpret_cast<float*>(s->B.tmp4);                 // nb * 256 floats of the permutation scratch
    const size_t plane_bytes = 16 * (size_t)s->P.ntiles * MD_TILE * 7;
    if ((size_t)nb * 256 * 4 > plane_bytes) nb = (int)(plane_bytes / 1024);   // a small system: fewer blocks (the rates then read low)
    if (nb < 1) return false;
    float ms = 0.f;
    const double winstr = (double)nb * 8 * PROBE_NIT * PROBE_CHAINS;   // warp instructions of the measured kind
    cudaStream_t st = s->stream;
    switch (kind) {
    case MD_PROBE_FFMA:
        if (!probe_time(st, [&] { k_probe_alu<MD_PROBE_FFMA><<<nb, 256, 0, st>>>(out, 1.0001f); }, &ms)) return false;
        *value = winstr * 64.0 / (ms * 1e-3) * 1e-12;
        return true;
    case MD_PROBE_FFMA2:
        if (!probe_time(st, [&] { k_probe_alu<MD_PROBE_FFMA2><<<nb, 256, 0, st>>>(out, 1.0001f); }, &ms)) return false;
        *value = winstr * 128.0 / (ms * 1e-3) * 1e-12;
        return true;
    case MD_PROBE_MUFU:
        if (!probe_time(st, [&] { k_probe_alu<MD_PROBE_MUFU><<<nb, 256, 0, st>>>(out, 1.0001f); }, &ms)) return false;
        *value = winstr * 32.0 / (ms * 1e-3) * 1e-12;
        return true;
    default: break;
    }
    // reductions: the accumulators are the first N float4 of the permutation scratch (left dirty: scratch)
    const unsigned int n = (unsigned int)s->P.N;
    const int nred = 32;
    const double ops = (double)nb * 256 * nred;
    bool ok = false;
    if (kind == MD_PROBE_RED_V4_SCATTER) ok = probe_time(st, [&] { k_probe_red<1, 0><<<nb, 256, 0, st>>>(s->B.tmp4, n, nred); }, &ms);
    else if (kind == MD_PROBE_RED_F32_SCATTER) ok = probe_time(st, [&] { k_probe_red<0, 0><<<nb, 256, 0, st>>>(s->B.tmp4, n, nred); }, &ms);
    else if (kind == MD_PROBE_RED_V4_COALESCED) ok = probe_time(st, [&] { k_probe_red<1, 1><<<nb, 256, 0, st>>>(s->B.tmp4, n, nred); }, &ms);
    else if (kind == MD_PROBE_RED_F32_COALESCED) ok = probe_time(st, [&] { k_probe_red<0, 1><<<nb, 256, 0, st>>>(s->B.tmp4, n, nred); }, &ms);
    if (!ok) return false;
    *value = ops / (ms * 1e-3) * 1e-9;
    return true;
}
