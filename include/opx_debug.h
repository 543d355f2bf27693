/* opx_debug.h -- debugging and measurement exports of libopx.so.  NOT part of the product boundary (include/opx.h):
 * nothing here is on the path a user calls; tests/ and bench.py use them to separate the arithmetic from the BVH, to
 * count the algorithmic work of a single ray for the roofline model, and to time kernels.  Conventions as in opx.h.
 */
#ifndef OPX_DEBUG_H_
#define OPX_DEBUG_H_

#include "opx.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Same computation with the closest hit found by testing EVERY triangle on the GPU (no BVH
 * traversal).  A debugging aid that separates the arithmetic of DESIGN.md section 3 from the BVH;
 * O(n x triangles), never timed. */
opx_status opx_propagate_brute(const opx_scene* scene, uint64_t n, uint64_t photon_id_base,
                               const float* d_origins, const float* d_dirs, const float* d_wavelengths,
                               uint64_t seed, const opx_hits* out, uint32_t* d_hitmap,
                               uint64_t* d_counters, void* cuda_stream);

/* opx_propagate with the packets walking the BINARY tree only (the 32-wide tree is ignored): the fallback that
 * incoherent packets, beam-stack overflows and scenes whose wide tree did not fit take in the product kernel, made
 * reachable for every photon so that tests can pin it on its own. */
opx_status opx_propagate_binary(const opx_scene* scene, uint64_t n, uint64_t photon_id_base,
                                const float* d_origins, const float* d_dirs, const float* d_wavelengths,
                                uint64_t seed, const opx_hits* out, uint32_t* d_hitmap,
                                uint64_t* d_counters, void* cuda_stream);

/* Per-kernel device times for a roofline report.  After opx_profile_begin(scene, max_calls) every
 * opx_propagate call on this scene records CUDA events around its two kernels (propagation; binning
 * + counters) on the call's stream, for at most max_calls calls.  opx_profile_end waits for those
 * events, writes the per-call durations in milliseconds to ms_propagate / ms_bin (each max_calls
 * floats, may be NULL), the number of recorded calls to n_calls, and switches recording off.  Not
 * thread-safe with concurrent opx_propagate calls on the same scene. */
opx_status opx_profile_begin(opx_scene* scene, uint32_t max_calls);
opx_status opx_profile_end(opx_scene* scene, float* ms_propagate, float* ms_bin, uint32_t* n_calls);

/* Work counters of the propagation kernel for the roofline model: runs the same
 * traversal with an instrumented kernel that writes no records and ADDS to d_stats (4 uint64,
 * DEVICE): [0] segments (closest-hit queries), [1] BVH nodes visited (two child boxes each),
 * [2] ray/triangle tests, [3] surface interactions.  Never timed. */
opx_status opx_propagate_stats(const opx_scene* scene, uint64_t n, uint64_t photon_id_base,
                               const float* d_origins, const float* d_dirs, const float* d_wavelengths,
                               uint64_t seed, uint64_t* d_stats, void* cuda_stream);

/* Work counters of the PRODUCT kernel (k_propagate_packet, instrumented instantiation): same records
 * as opx_propagate into `out` (DEVICE arrays of n), no binning, and ADDS to d_stats (8 uint64, DEVICE):
 * [0] packet-segments (one closest-hit query of a 32-photon packet) answered by beam traversal of the
 * 32-wide tree, [1] packet-segments answered by the per-lane walk of the binary tree (incoherent packets, stack
 * overflow, no wide tree), [2] wide nodes visited, [3] triangles handed to the lanes by beam traversal
 * (each is tested by every live lane), [4] beam-stack overflows, [5..7] reserved.  Never timed. */
opx_status opx_propagate_packet_stats(const opx_scene* scene, uint64_t n, uint64_t photon_id_base,
                                      const float* d_origins, const float* d_dirs, const float* d_wavelengths,
                                      uint64_t seed, const opx_hits* out, uint64_t* d_stats, void* cuda_stream);

/* Number of 32-wide nodes the last opx_bvh_build produced (0: the collapse did not fit its capacity and
 * packets walk the binary tree only) and the capacity reserved in the scene workspace. */
opx_status opx_scene_wide_info(const opx_scene* scene, uint64_t* n_wide_nodes, uint64_t* capacity);

/* FP32 FMA micro-benchmark (8 independent chains per thread, 8 blocks of 256 threads per SM, no memory
 * traffic): writes the best of three timed launches, in TFLOP/s (FMA = 2), to *tflops.  It is the
 * measured counterpart of the derived peak SMs x 128 lanes x 2 x clock that the roofline of the
 * ALU-bound propagation kernel is quoted against.  d_scratch: >= 4 device bytes.
 * Synchronises the stream. */
opx_status opx_measure_fp32_peak(double* tflops, void* d_scratch, void* cuda_stream);

/* Number of kernel launches the library has enqueued in this process (monotonic; for bench.py's
 * gpu_launches accounting). */
uint64_t opx_launch_count(void);

/* Name (as ncu prints it) of the propagation-kernel instantiation that the last opx_propagate* call on this thread
 * launched; "" before the first.  bench.py reports it as roofline.kernel. */
const char* opx_last_kernel(void);

#ifdef __cplusplus
}
#endif
#endif /* OPX_DEBUG_H_ */
