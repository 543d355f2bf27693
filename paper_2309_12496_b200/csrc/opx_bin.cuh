// k_bin: A11 hit binning + A12 counters.
#pragma once
#include "opx_device.cuh"

namespace opx {
namespace {

// ---------------------------------------------------------------- A11 hit binning + A12 counters
// One thread per photon; detected photons of a warp that share a pixel are merged with
// __match_any_sync so that a ring concentrated on a few hundred pixels costs one atomic per
// distinct pixel per warp.  Integer adds only, so the result does not depend on the order.
__global__ void __launch_bounds__(256) k_bin(const uint8_t* __restrict__ state, const uint8_t* __restrict__ bounces,
                                             const int32_t* __restrict__ pixel, uint64_t n,
                                             const unsigned long long* __restrict__ d_n, uint32_t* hitmap,
                                             unsigned long long* counters) {
    __shared__ unsigned int s_cnt[8];
    if (threadIdx.x < 8) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    if (d_n) n = min(n, (uint64_t)__ldg(d_n));
    unsigned int seg_local = 0;
    for (uint64_t base = (blockIdx.x * (uint64_t)blockDim.x + threadIdx.x) - lane; base < n; base += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t i = base + lane;
        const bool ok = i < n;
        const int st = ok ? (int)state[i] : 7;
        if (ok) seg_local += (unsigned int)bounces[i] + (st != OPX_BOUNCE_LIMIT ? 1u : 0u);
        const int key = (st == OPX_DETECTED) ? pixel[i] : -1 - lane;            // unique key for non-detected lanes
        const unsigned int peers = __match_any_sync(0xffffffffu, key);
        if (hitmap && st == OPX_DETECTED && lane == __ffs(peers) - 1) atomicAdd(&hitmap[key], (unsigned int)__popc(peers));
        for (int s = 0; s < 7; ++s) {
            const unsigned int m = __ballot_sync(0xffffffffu, st == s);
            if (lane == 0 && m) atomicAdd(&s_cnt[s], (unsigned int)__popc(m));
        }
    }
    for (int off = 16; off > 0; off >>= 1) seg_local += __shfl_xor_sync(0xffffffffu, seg_local, off);
    if (lane == 0 && seg_local) atomicAdd(&s_cnt[7], seg_local);
    __syncthreads();
    if (counters && threadIdx.x < 8 && s_cnt[threadIdx.x]) atomicAdd(&counters[threadIdx.x], (unsigned long long)s_cnt[threadIdx.x]);
}

}  // namespace
}  // namespace opx
