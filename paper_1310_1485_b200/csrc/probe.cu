// probe.cu -- micro-benchmarks of the two units that bound the FFT path on one SM: the FP64 FMA pipe
// and the shared-memory crossbar ("FP64 37.2 TFLOP/s is a model ... first GPU task: a
// DFMA-chain microbenchmark (and a 128-bit SMEM ld/st bandwidth one)").  Exported as
// gene_nl_probe_peaks (include/gene_nl_bench.h); bench.py uses it for the roofline denominators.
#include <cuda_runtime.h>

#include "../../include/gene_nl_bench.h"

namespace {

__global__ void __launch_bounds__(256) k_probe_dfma(double* out, int iters, double b, double c)
{
    double a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = 1.0 + 1e-3 * (threadIdx.x + 32 * j);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int j = 0; j < 8; ++j) a[j] = fma(a[j], b, c);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += a[j];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_probe_smem(double* out, int iters)
{
    extern __shared__ double2 buf[];
    const int t = threadIdx.x;
    buf[t] = make_double2(t, -t);
    buf[t + 256] = make_double2(0.5 * t, 1.0);
    __syncthreads();
    unsigned a0 = (unsigned)__cvta_generic_to_shared(buf + t);
    unsigned a1 = (unsigned)__cvta_generic_to_shared(buf + 256 + t);
    double x, y;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {  // conflict-free 128-bit load then store, ping-pong between halves
            asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(x), "=d"(y) : "r"(a0) : "memory");
            asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(a1), "d"(x), "d"(y) : "memory");
            asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(x), "=d"(y) : "r"(a1) : "memory");
            asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(a0), "d"(x), "d"(y) : "memory");
        }
    }
    out[blockIdx.x * blockDim.x + t] = x + y;
}

}  // namespace

extern "C" int gene_nl_probe_peaks(double* out3)
{
    if (!out3) return GENE_NL_EINVAL;
    int dev = 0, sms = 0, khz = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return GENE_NL_ECUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = sms * 8, threads = 256;
    double* buf = nullptr;
    if (cudaMalloc(&buf, sizeof(double) * blocks * threads) != cudaSuccess) return GENE_NL_ENOMEM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float ms = 0.f;
    double best_f = 0.0, best_s = 0.0;
    const int it_f = 4096, it_s = 2048;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        k_probe_dfma<<<blocks, threads>>>(buf, it_f, 1.0000001, 1e-9);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        double tf = 2.0 * 8 * 4 * (double)it_f * blocks * threads / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best_f) best_f = tf;
        cudaEventRecord(e0);
        k_probe_smem<<<blocks, threads, 512 * sizeof(double2)>>>(buf, it_s);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        double gbs = 16.0 * 16 * (double)it_s * blocks * threads / (ms * 1e-3) / 1e9;
        if (rep > 0 && gbs > best_s) best_s = gbs;
    }
    cudaError_t err = cudaDeviceSynchronize();
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    out3[0] = best_f;
    out3[1] = best_s;
    out3[2] = khz / 1000.0;
    return err == cudaSuccess ? GENE_NL_OK : GENE_NL_ECUDA;
}
