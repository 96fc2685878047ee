// bench_peaks.cu -- micro-benchmarks for the two roofline denominators of the zone
// kernel that MEASURED_PEAKS.json does not hold: plain (non-tensor) FP64 issue
// rate and shared-memory bandwidth, chip-wide on the device it runs on.
// Prints one JSON line.  Built and run by bench_peaks.py (beside bench.py, whose roofline
// denominators it measures); not part of the library.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>

#define CK(x)                                                                       \
    do {                                                                            \
        cudaError_t e = (x);                                                        \
        if (e != cudaSuccess) {                                                     \
            fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e));                 \
            return 1;                                                               \
        }                                                                           \
    } while (0)

// 8 independent chains per thread; OP 0: fma, 1: add, 2: mul
template <int OP>
__global__ void __launch_bounds__(512) fp64_kernel(double* out, int iters, double a, double b) {
    double v[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) v[q] = a + q * 1e-3 + threadIdx.x * 1e-6;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            if (OP == 0) v[q] = fma(v[q], a, b);
            if (OP == 1) v[q] = v[q] + b;
            if (OP == 2) v[q] = v[q] * a;
        }
    }
    double s = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += v[q];
    if (s == 123.456) out[0] = s;
}

// conflict-free LDS.64 (VEC = 1) or LDS.128 (VEC = 2) streaming over 32 KB
template <int VEC>
__global__ void __launch_bounds__(512) smem_kernel(unsigned long long* out, int iters) {
    __shared__ __align__(16) unsigned long long buf[4096];
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) buf[i] = i * 0x9E3779B97F4A7C15ull;
    __syncthreads();
    unsigned long long acc0 = 0, acc1 = 0;
    const int n = 4096 / VEC;
    int idx = threadIdx.x % n;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            unsigned long long x, y = 0;
            if (VEC == 1) {
                const unsigned addr = static_cast<unsigned>(__cvta_generic_to_shared(&buf[idx]));
                asm volatile("ld.volatile.shared.u64 %0, [%1];" : "=l"(x) : "r"(addr) : "memory");
            } else {
                const unsigned addr = static_cast<unsigned>(__cvta_generic_to_shared(&buf[2 * idx]));
                asm volatile("ld.volatile.shared.v2.u64 {%0, %1}, [%2];" : "=l"(x), "=l"(y) : "r"(addr) : "memory");
            }
            acc0 ^= x;
            acc1 ^= y;
            idx += 512;
            if (idx >= n) idx -= n;
        }
    }
    if ((acc0 ^ acc1) == 0x1234567ull) out[0] = acc0;
}

template <typename F>
static float time_ms(F launch) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    launch();
    cudaDeviceSynchronize();
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        launch();
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    return best;
}

int main() {
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, 0));
    const int sms = prop.multiProcessorCount;
    double* dout;
    CK(cudaMalloc(&dout, 64));
    const int blocks = sms * 4, threads = 512;
    const int iters = 20000;
    const double ops = double(blocks) * threads * iters * 8.0;
    const float t_fma = time_ms([&] { fp64_kernel<0><<<blocks, threads>>>(dout, iters, 1.0000001, 1e-9); });
    const float t_add = time_ms([&] { fp64_kernel<1><<<blocks, threads>>>(dout, iters, 1.0000001, 1e-9); });
    const float t_mul = time_ms([&] { fp64_kernel<2><<<blocks, threads>>>(dout, iters, 1.0000001, 1e-9); });
    const int siters = 4000;
    const double loads = double(blocks) * threads * siters * 8.0;
    auto* uout = reinterpret_cast<unsigned long long*>(dout);
    const float t_l64 = time_ms([&] { smem_kernel<1><<<blocks, threads>>>(uout, siters); });
    const float t_l128 = time_ms([&] { smem_kernel<2><<<blocks, threads>>>(uout, siters); });
    CK(cudaGetLastError());
    int clk_khz = 0;
    cudaDeviceGetAttribute(&clk_khz, cudaDevAttrClockRate, 0);
    printf("{\"gpu\": \"%s\", \"sms\": %d, \"clock_rate_mhz\": %.0f, "
           "\"fp64_fma_tinstr_s\": %.3f, \"fp64_add_tinstr_s\": %.3f, \"fp64_mul_tinstr_s\": %.3f, "
           "\"smem_lds64_tb_s\": %.3f, \"smem_lds128_tb_s\": %.3f}\n",
           prop.name, sms, clk_khz / 1e3, ops / t_fma / 1e9, ops / t_add / 1e9, ops / t_mul / 1e9,
           loads * 8 / t_l64 / 1e9, loads * 16 / t_l128 / 1e9);
    return 0;
}
