// Microbenchmarks for the rooflines MEASURED_PEAKS.json lacks: FP32 FFMA, MUFU, L2 red.add.f32, smem RMW.
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <vector>
#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1);} } while (0)

__global__ void k_ffma(float* out, int iters) {
    float a = threadIdx.x * 1e-3f, b = 1.0001f, c = 0.5f, d = a + 1, e = a + 2, f = a + 3, g = a+4, h=a+5;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) { a = fmaf(a, b, c); d = fmaf(d, b, c); e = fmaf(e, b, c); f = fmaf(f, b, c); g = fmaf(g,b,c); h = fmaf(h,b,c);}
    }
    if (a + d + e + f + g + h == 12345.f) out[0] = a;
}
__global__ void k_mufu(float* out, int iters) {
    float a = 1.0f + threadIdx.x * 1e-3f, d = a + 1, e = a + 2, f = a + 3;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a));
            asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(d));
            asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(e));
            asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(f));
        }
    }
    if (a + d + e + f == 12345.f) out[0] = a;
}
// mix: 8 FFMA + 2 MUFU per "eval" (the kernel's arithmetic mix)
__global__ void k_mix(float* out, int iters) {
    float u = threadIdx.x * 1e-3f, acc = 0.f, acc2 = 0.f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            float x = u + j;
            float e2 = fmaf(-0.01f * x, x, -0.3f);
            float ba = fmaf(0.02f, x, 0.1f);
            float D = fmaf(0.5f, x, 4400.f);
            float rs; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rs) : "f"(D));
            float bar = ba * rs;
            e2 = fmaf(bar, bar, e2);
            float ex; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(ex) : "f"(e2));
            acc = fmaf(rs, ex, acc);
            u += 1e-4f;
        }
    }
    if (acc + acc2 == 12345.f) out[0] = acc;
}
// red.global.add.f32: each warp adds to 32 consecutive floats at a pseudo-random row offset in an image of M floats
template <int VEC>
__global__ void k_red(float* img, int M, int iters, int span /*floats per warp op*/, int nrep) {
    unsigned lane = threadIdx.x & 31;
    unsigned wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned state = wid * 2654435761u + 12345u;
    float* base = img + (size_t)(blockIdx.x % nrep) * M;
    for (int i = 0; i < iters; ++i) {
        state = state * 1664525u + 1013904223u;
        unsigned off = (state >> 8) % (unsigned)(M - 256);
        if (VEC == 1) {
            if ((int)lane < span) asm volatile("red.global.add.f32 [%0], %1;" :: "l"(base + off + lane), "f"(1.0f) : "memory");
        } else {
            off &= ~3u;
            if ((int)lane * 4 < span) asm volatile("red.global.add.v4.f32 [%0], {%1,%1,%1,%1};" :: "l"(base + off + lane * 4), "f"(1.0f) : "memory");
        }
    }
}
// smem non-atomic RMW (LDS + FADD + STS), each warp to its own region
__global__ void k_smem_rmw(float* out, int iters) {
    extern __shared__ float sm[];
    int n = 8192;
    for (int i = threadIdx.x; i < n; i += blockDim.x) sm[i] = 0.f;
    __syncthreads();
    unsigned lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned state = (blockIdx.x * 8 + w) * 2654435761u + 1u;
    float* mine = sm + w * 1024;
    for (int i = 0; i < iters; ++i) {
        state = state * 1664525u + 1013904223u;
        unsigned off = (state >> 8) % 992u;
        mine[off + lane] += 1.0f;
    }
    __syncthreads();
    if (sm[threadIdx.x] == 12345.f) out[0] = 1;
}
// smem atomicAdd float (CAS loop)
__global__ void k_smem_atomic(float* out, int iters) {
    extern __shared__ float sm[];
    int n = 8192;
    for (int i = threadIdx.x; i < n; i += blockDim.x) sm[i] = 0.f;
    __syncthreads();
    unsigned lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned state = (blockIdx.x * 8 + w) * 2654435761u + 1u;
    for (int i = 0; i < iters; ++i) {
        state = state * 1664525u + 1013904223u;
        unsigned off = (state >> 8) % 8160u;
        atomicAdd(&sm[off + lane], 1.0f);
    }
    __syncthreads();
    if (sm[threadIdx.x] == 12345.f) out[0] = 1;
}
// L1-cached gather loads like w: each warp loads 32 consecutive floats at random row offsets (image of M floats)
__global__ void k_ldg(const float* __restrict__ img, float* out, int M, int iters) {
    unsigned lane = threadIdx.x & 31;
    unsigned wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    unsigned state = wid * 2654435761u + 12345u;
    float acc = 0;
    for (int i = 0; i < iters; ++i) {
        state = state * 1664525u + 1013904223u;
        unsigned off = (state >> 8) % (unsigned)(M - 256);
        acc += __ldg(img + off + lane);
    }
    if (acc == 12345.f) out[0] = acc;
}

template <typename F> float timeit(F f, int reps = 5) {
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    f(); CK(cudaDeviceSynchronize());
    float best = 1e30f;
    for (int r = 0; r < reps; ++r) { cudaEventRecord(a); f(); cudaEventRecord(b); CK(cudaEventSynchronize(b)); float ms; cudaEventElapsedTime(&ms, a, b); if (ms < best) best = ms; }
    return best;
}

int main() {
    cudaDeviceProp prop; CK(cudaGetDeviceProperties(&prop, 0));
    int sms = prop.multiProcessorCount;
    printf("device %s SMs %d clock %d kHz\n", prop.name, sms, prop.clockRate);
    float* out; CK(cudaMalloc(&out, 1024));
    int blocks = sms * 8, threads = 256;
    {
        int iters = 4000; float ms = timeit([&] { k_ffma<<<blocks, threads>>>(out, iters); });
        double n = (double)blocks * threads * iters * 16 * 6;
        printf("FFMA: %.3f ms  %.3e FFMA lane-ops/s  (%.2f per clk per SM at 1.965GHz)\n", ms, n / (ms * 1e-3), n / (ms * 1e-3) / sms / 1.965e9);
    }
    {
        int iters = 2000; float ms = timeit([&] { k_mufu<<<blocks, threads>>>(out, iters); });
        double n = (double)blocks * threads * iters * 8 * 4;
        printf("MUFU: %.3f ms  %.3e MUFU lane-ops/s  (%.2f per clk per SM at 1.965GHz)\n", ms, n / (ms * 1e-3), n / (ms * 1e-3) / sms / 1.965e9);
    }
    {
        int iters = 2000; float ms = timeit([&] { k_mix<<<blocks, threads>>>(out, iters); });
        double n = (double)blocks * threads * iters * 8;
        printf("MIX (8 FP32 + 2 MUFU per eval): %.3f ms  %.3e evals/s  (%.2f per clk per SM at 1.965GHz)\n", ms, n / (ms * 1e-3), n / (ms * 1e-3) / sms / 1.965e9);
    }
    for (int M : {40000, 160000, 262144}) {
        for (int nrep : {1, 8, 32}) {
            float* img; CK(cudaMalloc(&img, sizeof(float) * (size_t)M * nrep)); CK(cudaMemset(img, 0, sizeof(float) * (size_t)M * nrep));
            for (int span : {32, 16, 8}) {
                int iters = 2000; float ms = timeit([&] { k_red<1><<<blocks, threads>>>(img, M, iters, span, nrep); });
                double n = (double)blocks * threads / 32 * iters;
                printf("RED.f32 M=%d nrep=%d span=%d: %.3f ms  %.3e warp-ops/s  %.3e adds/s\n", M, nrep, span, ms, n / (ms * 1e-3), n * span / (ms * 1e-3));
            }
            {
                int iters = 2000; float ms = timeit([&] { k_red<4><<<blocks, threads>>>(img, M, iters, 128, nrep); });
                double n = (double)blocks * threads / 32 * iters;
                printf("RED.v4.f32 M=%d nrep=%d span=128: %.3f ms  %.3e warp-ops/s  %.3e adds/s\n", M, nrep, ms, n / (ms * 1e-3), n * 128 / (ms * 1e-3));
                ms = timeit([&] { k_red<4><<<blocks, threads>>>(img, M, iters, 32, nrep); });
                printf("RED.v4.f32 M=%d nrep=%d span=32 (8 lanes): %.3f ms  %.3e warp-ops/s  %.3e adds/s\n", M, nrep, ms, n / (ms * 1e-3), n * 32 / (ms * 1e-3));
            }
            CK(cudaFree(img));
        }
    }
    {
        int iters = 20000; float ms = timeit([&] { k_smem_rmw<<<sms * 4, 256, 32768>>>(out, iters); });
        double n = (double)sms * 4 * 8 * iters * 32;
        printf("SMEM RMW (LDS+FADD+STS): %.3f ms %.3e adds/s (%.2f per clk per SM)\n", ms, n / (ms * 1e-3), n / (ms * 1e-3) / sms / 1.965e9);
        iters = 2000; ms = timeit([&] { k_smem_atomic<<<sms * 4, 256, 32768>>>(out, iters); });
        n = (double)sms * 4 * 8 * iters * 32;
        printf("SMEM atomicAdd f32 (CAS): %.3f ms %.3e adds/s (%.2f per clk per SM)\n", ms, n / (ms * 1e-3), n / (ms * 1e-3) / sms / 1.965e9);
    }
    for (int M : {40000, 262144}) {
        float* img; CK(cudaMalloc(&img, sizeof(float) * M)); CK(cudaMemset(img, 0, sizeof(float) * M));
        int iters = 4000; float ms = timeit([&] { k_ldg<<<blocks, threads>>>(img, out, M, iters); });
        double n = (double)blocks * threads / 32 * iters;
        printf("LDG 128B/warp M=%d: %.3f ms %.3e warp-loads/s (%.2f per clk per SM)\n", M, ms, n / (ms * 1e-3), n / (ms * 1e-3) / sms / 1.965e9);
        CK(cudaFree(img));
    }
    return 0;
}
