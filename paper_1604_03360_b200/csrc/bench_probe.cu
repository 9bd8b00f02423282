// bench_probe.cu -- measurement helper of bench.py, NOT part of the product library or its ABI (include/hydro.h): a
// register-resident chain of independent fused multiply-adds on every SM.  Its sustained rate is the measured "alu"
// roofline denominator that bench.py reports next to the nominal 148 SM x 64 (fp64) or 128 (fp32) lanes x 2 flop x
// 1.965 GHz.  Built by paper_1604_03360_b200/build.py into libbench_probe.so and loaded by bench.py with ctypes:
//   int bench_probe_fma_peak(int precision /* 0 f64, 1 f32 */, int millis, void* cuda_stream,
//                            void* device_scratch /* >= 8 bytes, caller-owned */, double* tflops_host);
// returns 0, or -1 (bad argument) / -3 (CUDA error).
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
int probe_impl(int millis, cudaStream_t st, void* scratch, double* out) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
    T* sink = (T*)scratch;
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
        if (cudaEventSynchronize(e1) != cudaSuccess) return -3;
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
    *out = best;
    return 0;
}

}  // namespace hydro

extern "C" int bench_probe_fma_peak(int precision, int millis, void* cuda_stream, void* device_scratch,
                                    double* tflops_host) {
    if (!tflops_host || !device_scratch || millis < 1 || (precision != 0 && precision != 1)) return -1;
    return precision == 0 ? hydro::probe_impl<double>(millis, (cudaStream_t)cuda_stream, device_scratch, tflops_host)
                          : hydro::probe_impl<float>(millis, (cudaStream_t)cuda_stream, device_scratch, tflops_host);
}
