// fp64_probe.cu — what the plain fp64 pipe of this GPU delivers: dependent-DFMA latency and DFMA throughput per SM.
// DESIGN.md section 6 quotes these two numbers beside the HBM roofline (the step executes ~215 DP instructions per
// grid point); tests/test_gpu_parity.py builds and runs this file on the GPU box and prints its one JSON line.
// Not part of libdbec.so.
#include <cstdio>
#include <cuda_runtime.h>

__global__ void k_latency(double* out, long long* cyc, int n) {
    double a = out[0], b = 1.0000001, c = 1e-9;
    const long long t0 = clock64();
    for (int i = 0; i < n; ++i) {
#pragma unroll
        for (int k = 0; k < 16; ++k) a = fma(a, b, c);          // one dependent chain
    }
    const long long t1 = clock64();
    out[threadIdx.x] = a;
    if (threadIdx.x == 0) *cyc = t1 - t0;
}

template <int CH>
__global__ void __launch_bounds__(1024, 1) k_throughput(double* out, long long* cyc, int n) {
    double a[CH];
#pragma unroll
    for (int k = 0; k < CH; ++k) a[k] = out[0] + k;
    const double b = 1.0000001, c = 1e-9;
    __syncthreads();
    const long long t0 = clock64();
    for (int i = 0; i < n; ++i) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < CH; ++k) a[k] = fma(a[k], b, c);   // CH independent chains per thread
    }
    __syncthreads();
    const long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < CH; ++k) s += a[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

int main() {
    cudaDeviceProp p;
    cudaGetDeviceProperties(&p, 0);
    double* out; long long* cyc;
    cudaMalloc(&out, sizeof(double) * 1024 * p.multiProcessorCount);
    cudaMalloc(&cyc, sizeof(long long) * p.multiProcessorCount);
    cudaMemset(out, 0, sizeof(double) * 1024 * p.multiProcessorCount);
    long long h[1024];
    const int n = 4096;
    k_latency<<<1, 32>>>(out, cyc, n);
    k_latency<<<1, 32>>>(out, cyc, n);
    cudaMemcpy(h, cyc, sizeof(long long), cudaMemcpyDeviceToHost);
    const double lat = (double)h[0] / (16.0 * n);
    constexpr int CH = 8;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_throughput<CH><<<p.multiProcessorCount, 1024>>>(out, cyc, n);
    cudaEventRecord(e0);
    k_throughput<CH><<<p.multiProcessorCount, 1024>>>(out, cyc, n);
    cudaEventRecord(e1);
    cudaDeviceSynchronize();
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaMemcpy(h, cyc, sizeof(long long) * p.multiProcessorCount, cudaMemcpyDeviceToHost);
    long long cmax = 0;
    for (int i = 0; i < p.multiProcessorCount; ++i) cmax = h[i] > cmax ? h[i] : cmax;
    const double per_sm = 1024.0 * CH * 4.0 * n;                 // DFMAs one SM executed
    const double dfma_per_clk = per_sm / (double)cmax;
    const double tflops = 2.0 * per_sm * p.multiProcessorCount / (ms * 1e-3) / 1e12;
    const cudaError_t e = cudaGetLastError();
    printf("{\"gpu\": \"%s\", \"sms\": %d, \"dependent_dfma_latency_cycles\": %.2f, \"dfma_per_clk_per_sm\": %.2f, "
           "\"fp64_tflops_all_sms\": %.2f, \"kernel_ms\": %.4f, \"cuda_error\": %d}\n",
           p.name, p.multiProcessorCount, lat, dfma_per_clk, tflops, ms, (int)e);
    return e == cudaSuccess ? 0 : 1;
}
