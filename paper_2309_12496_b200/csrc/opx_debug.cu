// Debugging and measurement exports (include/opx_debug.h): NOT part of the product boundary.  The all-triangle and
// binary-tree walks that tests compare the product walk with, the instrumented kernels behind the roofline model's work
// counts, per-kernel event timing, and an FP32 FMA micro-benchmark that gives the roofline denominator of the ALU-bound
// propagation kernel as measured on the device at hand.
#include "../../include/opx_debug.h"
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

using namespace opx;

extern "C" {

uint64_t opx_launch_count(void) { return launch_count(); }
const char* opx_last_kernel(void) { return last_kernel(); }

opx_status opx_propagate_brute(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                               const float* d_dirs, const float* d_wavelengths, uint64_t seed, const opx_hits* out,
                               uint32_t* d_hitmap, uint64_t* d_counters, void* cuda_stream) {
    return propagate_common(scene, kWalkBrute, n, nullptr, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, 0u, out, d_hitmap,
                            d_counters, cuda_stream);
}

opx_status opx_propagate_binary(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                                const float* d_dirs, const float* d_wavelengths, uint64_t seed, const opx_hits* out,
                                uint32_t* d_hitmap, uint64_t* d_counters, void* cuda_stream) {
    return propagate_common(scene, kWalkBinary, n, nullptr, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, 0u, out, d_hitmap,
                            d_counters, cuda_stream);
}

opx_status opx_profile_begin(opx_scene* scene, uint32_t max_calls) {
    if (!scene || max_calls == 0) return fail(OPX_ERR_INVALID_ARG, "scene is NULL or max_calls = 0");
    while (scene->prof_events.size() < 3ull * max_calls) {
        cudaEvent_t e;
        if (opx_status st = check_cuda(cudaEventCreate(&e), "cudaEventCreate")) return st;
        scene->prof_events.push_back(e);
    }
    scene->prof_max = max_calls;
    scene->prof_used = 0;
    return OPX_OK;
}

opx_status opx_profile_end(opx_scene* scene, float* ms_propagate, float* ms_bin, uint32_t* n_calls) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    const uint32_t used = scene->prof_used;
    scene->prof_max = 0;
    scene->prof_used = 0;
    if (n_calls) *n_calls = used;
    for (uint32_t k = 0; k < used; ++k) {
        cudaEvent_t* ev = &scene->prof_events[3 * k];
        if (opx_status st = check_cuda(cudaEventSynchronize(ev[2]), "cudaEventSynchronize")) return st;
        float a = 0.f, b = 0.f;
        if (opx_status st = check_cuda(cudaEventElapsedTime(&a, ev[0], ev[1]), "cudaEventElapsedTime")) return st;
        if (opx_status st = check_cuda(cudaEventElapsedTime(&b, ev[1], ev[2]), "cudaEventElapsedTime")) return st;
        if (ms_propagate) ms_propagate[k] = a;
        if (ms_bin) ms_bin[k] = b;
    }
    return OPX_OK;
}

opx_status opx_propagate_stats(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                               const float* d_dirs, const float* d_wavelengths, uint64_t seed, uint64_t* d_stats,
                               void* cuda_stream) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_propagate_stats before opx_bvh_build");
    if (n == 0) return OPX_OK;
    if (!d_origins || !d_dirs || !d_wavelengths || !d_stats) return fail(OPX_ERR_INVALID_ARG, "NULL pointer");
    return launch_stats(*scene, n, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, d_stats, (cudaStream_t)cuda_stream);
}

opx_status opx_propagate_packet_stats(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                                      const float* d_dirs, const float* d_wavelengths, uint64_t seed, const opx_hits* out,
                                      uint64_t* d_stats, void* cuda_stream) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_propagate_packet_stats before opx_bvh_build");
    if (n == 0) return OPX_OK;
    if (!d_origins || !d_dirs || !d_wavelengths || !d_stats || !out) return fail(OPX_ERR_INVALID_ARG, "NULL pointer");
    if (!out->pos || !out->dir || !out->pixel || !out->surface || !out->state || !out->bounces)
        return fail(OPX_ERR_INVALID_ARG, "NULL hit-record array");
    return launch_packet_stats(*scene, n, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, *out, d_stats, (cudaStream_t)cuda_stream);
}

opx_status opx_scene_wide_info(const opx_scene* scene, uint64_t* n_wide_nodes, uint64_t* capacity) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_scene_wide_info before opx_bvh_build");
    if (n_wide_nodes) {
        // the count lives on the device (the build does not read it back): this debug call waits for the device
        uint32_t c = 0;
        *n_wide_nodes = 0;
        if (scene->dev.wide_count) {
            if (opx_status st = check_cuda(cudaDeviceSynchronize(), "cudaDeviceSynchronize")) return st;
            if (opx_status st = check_cuda(cudaMemcpy(&c, scene->dev.wide_count, 4, cudaMemcpyDeviceToHost), "cudaMemcpy")) return st;
            *n_wide_nodes = c;
        }
    }
    if (capacity) *capacity = scene->layout.wide_node_capacity;
    return OPX_OK;
}

}  // extern "C"
