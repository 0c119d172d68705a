// microbench.cu -- the machine numbers DESIGN.md quotes for the non-HBM ceilings of the force kernels (SURVEY 8(d):
// "the builder must measure an FFMA-chain and a MUFU-chain micro-benchmark on the box"; "micro-benchmark
// red.global.add.f32 and .v4.f32 at random and at clustered addresses before interpreting EDGE numbers").
// Stand-alone, not part of libmd_b200.so:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o microbench paper_1401_4350_b200/csrc/microbench.cu && ./microbench
#include <cstdio>
#include <vector>
#include <cuda_runtime.h>

#define NIT 4096
// ---- issue rates: 8 independent chains per thread, 8 blocks of 256 threads per SM ----
template <int MODE>
__global__ void __launch_bounds__(256) k_alu(float* out, float s) {
    float a[8], b[8];
    float2 p[8], q[8];
    for (int k = 0; k < 8; ++k) { a[k] = threadIdx.x * 0.001f + k + 1.0f; b[k] = s + k; p[k] = make_float2(a[k], b[k]); q[k] = make_float2(b[k], a[k]); }
    const float2 c2 = make_float2(s, s * 0.5f);
    for (int it = 0; it < NIT; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (MODE == 0) a[k] = fmaf(a[k], b[k], s);                 // FFMA
            if (MODE == 1) p[k] = __ffma2_rn(p[k], q[k], c2);          // FFMA2 (packed f32x2)
            if (MODE == 2) a[k] = a[k] + b[k];                         // FADD
            if (MODE == 3) { float r; asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a[k])); a[k] = r + s; }   // MUFU.RCP (+FADD)
            if (MODE == 4) { float r; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a[k])); a[k] = r * s; }   // MUFU.EX2 (+FMUL)
            if (MODE == 5) { a[k] = fmaf(a[k], b[k], s); b[k] = fminf(b[k], a[k]); }   // FFMA + FMNMX (fma pipe + alu pipe)
        }
    }
    float r = 0;
    for (int k = 0; k < 8; ++k) r += a[k] + b[k] + p[k].x + p[k].y + q[k].x;
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

// ---- L2 reductions: every lane issues NRED red operations; MODE 0 scalar f32, 1 v4.f32;
//      addresses: idx[] (random over the array, or clustered = neighbours in a 2 KB window, like an MD neighbourhood) ----
template <int V4>
__global__ void __launch_bounds__(256) k_red(float4* acc, const int* __restrict__ idx, int n_idx, int nred) {
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    for (int r = 0; r < nred; ++r) {
        const int j = idx[(size_t)(g + (size_t)r * gridDim.x * blockDim.x) % n_idx];
        if (V4) asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(acc + j), "f"(1.f), "f"(2.f), "f"(3.f), "f"(4.f) : "memory");
        else asm volatile("red.global.add.f32 [%0], %1;" ::"l"(reinterpret_cast<float*>(acc + j) + (r & 3)), "f"(1.f) : "memory");
    }
}

template <typename F>
static float timeit(F f) {
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    f(); cudaDeviceSynchronize();
    cudaEventRecord(a); f(); cudaEventRecord(b); cudaEventSynchronize(b);
    float ms; cudaEventElapsedTime(&ms, a, b);
    return ms;
}

int main() {
    cudaDeviceProp pr; cudaGetDeviceProperties(&pr, 0);
    const int sms = pr.multiProcessorCount;
    int khz = 0; cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    const double ghz = khz * 1e-6;
    printf("%s, %d SMs, %.3f GHz (max SM clock)\n", pr.name, sms, ghz);
    float* out; cudaMalloc(&out, (size_t)sms * 8 * 256 * 4);
    const int nb = sms * 8;
    const char* names[] = { "FFMA", "FFMA2 (f32x2)", "FADD", "MUFU.RCP + FADD", "MUFU.EX2 + FMUL", "FFMA + FMNMX" };
    const double per[] = { 1, 1, 1, 2, 2, 2 };
    float ms[6];
    ms[0] = timeit([&] { k_alu<0><<<nb, 256>>>(out, 1.0001f); });
    ms[1] = timeit([&] { k_alu<1><<<nb, 256>>>(out, 1.0001f); });
    ms[2] = timeit([&] { k_alu<2><<<nb, 256>>>(out, 1.0001f); });
    ms[3] = timeit([&] { k_alu<3><<<nb, 256>>>(out, 1.0001f); });
    ms[4] = timeit([&] { k_alu<4><<<nb, 256>>>(out, 1.0001f); });
    ms[5] = timeit([&] { k_alu<5><<<nb, 256>>>(out, 1.0001f); });
    for (int m = 0; m < 6; ++m) {
        const double winstr = (double)nb * 8 * NIT * 8 * per[m];
        const double per_cyc = winstr / (ms[m] * 1e6) / sms / ghz;
        printf("%-18s %7.3f ms  %5.2f warp-instr / cycle / SM", names[m], ms[m], per_cyc);
        if (m == 0) printf("  -> %.1f TFLOP/s fp32 (FFMA = 2 flop x 32 lanes)", per_cyc * 64 * sms * ghz * 1e-3);
        if (m == 1) printf("  -> %.1f TFLOP/s fp32 (FFMA2 = 4 flop x 32 lanes)", per_cyc * 128 * sms * ghz * 1e-3);
        if (m == 3 || m == 4) printf("  -> MUFU %.2f / cycle / SM = %.2f Tops/s", per_cyc / 2, per_cyc / 2 * 32 * sms * ghz * 1e-3);
        printf("\n");
    }
    // reductions
    const int N = 1 << 20;                      // 16 MiB of float4 accumulators (L2-resident), like force[] at N = 2^20
    float4* acc; cudaMalloc(&acc, (size_t)N * 16); cudaMemset(acc, 0, (size_t)N * 16);
    const int n_idx = 1 << 24;
    std::vector<int> h(n_idx);
    int* d; cudaMalloc(&d, (size_t)n_idx * 4);
    const int threads = sms * 8 * 256, nred = 32;
    for (int pat = 0; pat < 2; ++pat) {
        unsigned s = 12345u;
        for (int t = 0; t < n_idx; ++t) {
            s = s * 1664525u + 1013904223u;
            if (pat == 0) h[t] = (int)((s >> 8) % N);                                  // random over the whole array
            else h[t] = (int)(((unsigned)(t % threads) * (unsigned)(N / threads + 1) + ((s >> 8) % 128)) % N);   // within a 2 KB window of "its own" slot
        }
        cudaMemcpy(d, h.data(), (size_t)n_idx * 4, cudaMemcpyHostToDevice);
        for (int v4 = 0; v4 < 2; ++v4) {
            const float t = v4 ? timeit([&] { k_red<1><<<sms * 8, 256>>>(acc, d, n_idx, nred); })
                               : timeit([&] { k_red<0><<<sms * 8, 256>>>(acc, d, n_idx, nred); });
            const double ops = (double)threads * nred;
            printf("red.global.add%s  %-9s addresses: %7.3f ms for %.1f M lane-ops -> %6.1f G ops/s (%5.1f GB/s of payload)\n",
                   v4 ? ".v4.f32" : ".f32   ", pat ? "clustered" : "random", t, ops * 1e-6, ops / (t * 1e6), ops * (v4 ? 16 : 4) / (t * 1e6));
        }
    }
    return 0;
}
