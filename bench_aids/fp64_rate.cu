// Bench-side helper, NOT part of the product library: the plain FP64 ALU roofline of the device, measured with
// independent DFMA chains.  bench.py uses it as the denominator check of the "alu" roofline (MEASURED_PEAKS.json has
// no FP64 figure).  Built by __graft_entry__.build() into bench_aids/libgenga_bench_aids.so.
//
//   pattern 0: a = fma(a, m, c), m and c loop-invariant registers (operand reuse possible)
//   pattern 1: a_k = fma(a_k, b_k, c_k): three distinct register operands, no reuse
//   pattern 2: a_k = fma(a_k, b_k, imm): two distinct register operands
// The operands come from memory so that nothing folds; the result is stored so that nothing is dropped.
#include <cuda_runtime.h>
#include <stdint.h>

template <int PATTERN>
__global__ void __launch_bounds__(256, 2) fp64_rate_kernel(const double* __restrict__ in, double* __restrict__ out, int iters)
{
    const double m = in[0], c = in[1];
    double a[8], b[8], d[8];
#pragma unroll
    for (int k = 0; k < 8; k++) {
        a[k] = in[2] * (double)(threadIdx.x + k);
        b[k] = m - 1.0e-9 * (double)k;
        d[k] = c + 1.0e-9 * (double)k;
    }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < 8; u++) {
#pragma unroll
            for (int k = 0; k < 8; k++) {
                if (PATTERN == 0) a[k] = fma(a[k], m, c);
                if (PATTERN == 1) a[k] = fma(a[k], b[k], d[k]);
                if (PATTERN == 2) a[k] = fma(a[k], b[k], 1.0e-6);
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; k++) s += a[k];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// Runs `reps` + 1 launches (the first is a warm-up) of 8 CTAs x 256 threads per SM, 8 chains x iters x 8 DFMAs per
// thread, on `stream` of the current device; *dfma_per_s = the best launch's rate (one DFMA = 2 flops).
// Returns 0, -1 (bad argument) or the cudaError_t of the failing call.
extern "C" int bench_fp64_rate(int32_t pattern, int32_t iters, int32_t reps, void* stream, double* dfma_per_s)
{
    if (!dfma_per_s || iters < 1 || reps < 1 || pattern < 0 || pattern > 2) return -1;
    int dev = 0, sms = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return (int)e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return (int)e;
    const int blocks = 8 * sms, threads = 256;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    double* buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const double host_in[3] = {0.999999, 1.0e-6, 1.0e-3};
    float best = 0.0f;
    if ((e = cudaMalloc(&buf, ((size_t)blocks * threads + 4) * sizeof(double))) != cudaSuccess) goto done;
    if ((e = cudaMemcpyAsync(buf, host_in, sizeof(host_in), cudaMemcpyHostToDevice, st)) != cudaSuccess) goto done;
    if ((e = cudaEventCreate(&e0)) != cudaSuccess) goto done;
    if ((e = cudaEventCreate(&e1)) != cudaSuccess) goto done;
    for (int r = 0; r <= reps; r++) {
        if ((e = cudaEventRecord(e0, st)) != cudaSuccess) goto done;
        if (pattern == 0) fp64_rate_kernel<0><<<blocks, threads, 0, st>>>(buf, buf + 4, iters);
        if (pattern == 1) fp64_rate_kernel<1><<<blocks, threads, 0, st>>>(buf, buf + 4, iters);
        if (pattern == 2) fp64_rate_kernel<2><<<blocks, threads, 0, st>>>(buf, buf + 4, iters);
        if ((e = cudaGetLastError()) != cudaSuccess) goto done;
        if ((e = cudaEventRecord(e1, st)) != cudaSuccess) goto done;
        if ((e = cudaEventSynchronize(e1)) != cudaSuccess) goto done;
        float ms = 0.0f;
        if ((e = cudaEventElapsedTime(&ms, e0, e1)) != cudaSuccess) goto done;
        if (r > 0 && (best == 0.0f || ms < best)) best = ms;
    }
    *dfma_per_s = (double)blocks * threads * 64.0 * (double)iters / ((double)best * 1.0e-3);
done:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (buf) cudaFree(buf);
    return (int)e;
}
