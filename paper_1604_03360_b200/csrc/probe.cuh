// probe.cuh -- machine probe behind hydro_probe_fma_peak: a register-resident chain of independent fused
// multiply-adds on every SM.  Its sustained rate is the measured "alu" roofline denominator that bench.py
// reports next to the nominal 148 SM x 64 (fp64) or 128 (fp32) lanes x 2 flop x 1.965 GHz.
#pragma once
#include <cuda_runtime.h>

namespace hydro {

template <class T>
__global__ void __launch_bounds__(256) fma_chain_kernel(T* sink, int iters, T a, T b) {
    T x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = (T)(threadIdx.x + i) * (T)1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 16; ++rep) {
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = x[i] * a + b;  // contracted to one FMA each
        }
    }
    T s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    if (s == (T)123456789) sink[0] = s;  // never true: keeps the chain alive
}

template <class T>
int probe_impl(int millis, cudaStream_t st, double* out) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
    T* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(T)) != cudaSuccess) return -3;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = sms * 8, threads = 256;
    int iters = 2000;
    double best = 0.0;
    for (int pass = 0; pass < 3; ++pass) {
        cudaEventRecord(e0, st);
        fma_chain_kernel<T><<<blocks, threads, 0, st>>>(sink, iters, (T)0.999999, (T)1e-6);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(sink); return -3; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 8 * 16 * (double)iters * blocks * threads;
        const double tf = flops / (ms * 1e-3) / 1e12;
        if (pass > 0 && tf > best) best = tf;
        // aim the next pass at the requested duration
        if (ms > 0) {
            double want = (double)iters * millis / ms;
            if (want < 100) want = 100;
            if (want > 5e7) want = 5e7;
            iters = (int)want;
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    *out = best;
    return 0;
}

}  // namespace hydro

extern "C" int hydro_probe_fma_peak(int precision, int millis, void* cuda_stream, double* tflops_host) {
    if (!tflops_host || millis < 1 || (precision != 0 && precision != 1)) return HYDRO_EINVAL;
    const int rc = precision == 0 ? hydro::probe_impl<double>(millis, (cudaStream_t)cuda_stream, tflops_host)
                                  : hydro::probe_impl<float>(millis, (cudaStream_t)cuda_stream, tflops_host);
    return rc == 0 ? HYDRO_OK : HYDRO_ECUDA;
}
