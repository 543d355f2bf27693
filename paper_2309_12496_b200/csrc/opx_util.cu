// Measurement utility of the C ABI: an FP32 FMA micro-benchmark that gives the roofline denominator
// of the ALU-bound propagation kernel as measured on the device at hand.
#include "opx_internal.cuh"

namespace opx {
namespace {

// 8 independent FMA chains per thread, 4096 FMAs each: pure FFMA issue, no memory traffic.
__global__ void __launch_bounds__(256) k_fma_peak(float* sink, float a, float b, int iters) {
    float x0 = threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            x0 = __fmaf_rn(x0, a, b); x1 = __fmaf_rn(x1, a, b); x2 = __fmaf_rn(x2, a, b); x3 = __fmaf_rn(x3, a, b);
            x4 = __fmaf_rn(x4, a, b); x5 = __fmaf_rn(x5, a, b); x6 = __fmaf_rn(x6, a, b); x7 = __fmaf_rn(x7, a, b);
        }
    }
    const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 12345.678f) sink[0] = s;      // never true: keeps the chains alive
}

}  // namespace
}  // namespace opx

extern "C" opx_status opx_measure_fp32_peak(double* tflops, void* d_scratch, void* cuda_stream) {
    using namespace opx;
    if (!tflops || !d_scratch) return fail(OPX_ERR_INVALID_ARG, "NULL argument");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (opx_status s = check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return s;
    if (opx_status s = check_cuda(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute")) return s;
    cudaEvent_t e0, e1;
    if (opx_status s = check_cuda(cudaEventCreate(&e0), "cudaEventCreate")) return s;
    if (opx_status s = check_cuda(cudaEventCreate(&e1), "cudaEventCreate")) { cudaEventDestroy(e0); return s; }
    const int iters = 2048, blocks = sms * 8;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {            // first repetition is the warm-up
        cudaEventRecord(e0, st);
        k_fma_peak<<<blocks, 256, 0, st>>>((float*)d_scratch, 0.999f, 0.001f, iters);
        count_launch(1);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return check_cuda(e, "opx_measure_fp32_peak"); }
        const double flop = 2.0 * 8.0 * 16.0 * (double)iters * 256.0 * (double)blocks;
        if (rep > 0 && ms > 0.f && flop / (ms * 1e-3) > best) best = flop / (ms * 1e-3);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    *tflops = best / 1e12;
    return OPX_OK;
}
