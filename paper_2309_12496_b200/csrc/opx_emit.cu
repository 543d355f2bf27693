// opx_emit_cherenkov: Cherenkov photons from charged-track steps, generated on the device straight into the arrays
// opx_propagate / opx_prefilter read (PAPER.md:71 cos(theta_c) = 1/(n beta),
// no intermediate files, everything memory-resident).
//
// One thread per photon: binary search of the photon's step in the prefix sums (the table is a few MB and stays in
// L2), one Philox4x32-10 block on stream 2 for position, wavelength and the first azimuth attempt, further blocks
// only for the 21 % of photons whose first disc sample is rejected.  IEEE operations only (no sin/cos): the bits are
// those of the CPU oracle.  28 B written per photon, nothing read but the step table.
#include "opx_device.cuh"

namespace opx {
namespace {

struct Words { uint32_t w0, w1, w2, w3; };

__device__ __forceinline__ Words philox4(uint64_t seed, uint64_t g, uint32_t a, uint32_t stream) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    uint32_t c0 = (uint32_t)g, c1 = (uint32_t)(g >> 32), c2 = a, c3 = stream;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return Words{c0, c1, c2, c3};
}

__device__ __forceinline__ float u01(uint32_t w) { return __fmul_rn((float)(w >> 8), 5.9604644775390625e-8f); }

__global__ void __launch_bounds__(256) k_emit_cherenkov(const opx_track_steps st, float n_index, float lambda1, float lambda2,
                                                        uint64_t n, uint64_t id_base, uint64_t seed,
                                                        float* __restrict__ origins, float* __restrict__ dirs,
                                                        float* __restrict__ wl) {
    // Step look-up.  The photons of a block are consecutive ids, so they sit in consecutive steps: warp 0 finds the step
    // of the block's first photon with a 32-ary search (4 dependent loads for 1e6 steps instead of 20), the block copies
    // the next 257 prefix sums to shared memory and every thread finishes with an 8-step binary search there.  A block
    // that spans more than 256 steps (long runs of steps without photons) falls back to the global binary search.
    __shared__ uint64_t s_first[257];
    __shared__ uint64_t s_base;
    const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    const uint64_t S = st.n_steps;
    if (threadIdx.x < 32) {
        const unsigned lane = threadIdx.x;
        const uint64_t g0 = id_base + blockIdx.x * (uint64_t)blockDim.x;
        uint64_t lo = 0, hi = S;                                   // invariant first[lo] <= g0 < first[hi]
        while (hi - lo > 1) {
            const uint64_t pos = lo + (((hi - lo) * (uint64_t)(lane + 1)) >> 5);       // in [lo, hi], non-decreasing in lane
            const bool le = pos == lo || (pos < hi && __ldg(st.first + pos) <= g0);
            const int k = __popc(__ballot_sync(0xffffffffu, le));                      // first[] is monotone: lanes 0..k-1 say yes
            const uint64_t nlo = __shfl_sync(0xffffffffu, pos, k > 0 ? k - 1 : 0), nhi = __shfl_sync(0xffffffffu, pos, k < 32 ? k : 31);
            lo = k > 0 ? nlo : lo; hi = k < 32 ? nhi : hi;
        }
        if (lane == 0) s_base = lo;
    }
    __syncthreads();
    const uint64_t base = s_base;
    for (unsigned j = threadIdx.x; j < 257u; j += blockDim.x) s_first[j] = __ldg(st.first + (base + j < S ? base + j : S));
    __syncthreads();
    if (i >= n) return;
    const uint64_t g = id_base + i;
    uint64_t lo;
    if (s_first[256] <= g && base + 256 < S) {
        lo = base + 256;                                           // first[lo] <= g < first[S]
        uint64_t hi = S;
        while (hi - lo > 1) {
            const uint64_t mid = lo + (hi - lo) / 2;
            if (__ldg(st.first + mid) <= g) lo = mid; else hi = mid;
        }
    } else {
        unsigned jl = 0, jh = 256;                                 // s_first[jl] <= g < s_first[jh] (entries past S repeat first[S] > g)
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const unsigned mid = (jl + jh) >> 1;
            if (s_first[mid] <= g) jl = mid; else jh = mid;
        }
        lo = base + jl;
    }
    const float* x = st.x + 3 * lo;
    const float* w = st.w + 3 * lo;
    const float wx = __ldg(w), wy = __ldg(w + 1), wz = __ldg(w + 2);
    Words r = philox4(seed, g, 0u, 2u);
    const float t = __fmul_rn(u01(r.w0), __ldg(st.length + lo));
    origins[3 * i] = __fmaf_rn(t, wx, __ldg(x)); origins[3 * i + 1] = __fmaf_rn(t, wy, __ldg(x + 1)); origins[3 * i + 2] = __fmaf_rn(t, wz, __ldg(x + 2));
    wl[i] = __fdiv_rn(__fmul_rn(lambda1, lambda2), __fmaf_rn(-u01(r.w1), __fsub_rn(lambda2, lambda1), lambda2));
    float c = __fdiv_rn(1.f, __fmul_rn(n_index, __ldg(st.beta + lo)));
    if (!(c < 1.f)) c = 1.f;
    const float sn = __fsqrt_rn(fmaxf(__fmaf_rn(-c, c, 1.f), 0.f));
    float cphi = 1.f, sphi = 0.f;
    for (uint32_t a = 0; a < 64u; ++a) {
        if (a > 0) r = philox4(seed, g, a, 2u);
        const float X = __fmaf_rn(2.f, u01(r.w2), -1.f), Y = __fmaf_rn(2.f, u01(r.w3), -1.f);
        const float q = __fmaf_rn(Y, Y, __fmul_rn(X, X));
        if (q > 0.f && q <= 1.f) {
            cphi = __fdiv_rn(__fsub_rn(__fmul_rn(X, X), __fmul_rn(Y, Y)), q);
            sphi = __fdiv_rn(__fmul_rn(__fmul_rn(2.f, X), Y), q);
            break;
        }
    }
    const float sg = wz >= 0.f ? 1.f : -1.f;
    const float k = __fdiv_rn(-1.f, __fadd_rn(sg, wz));
    const float b = __fmul_rn(__fmul_rn(wx, wy), k);
    const float e1x = __fmaf_rn(__fmul_rn(sg, wx), __fmul_rn(wx, k), 1.f), e1y = __fmul_rn(sg, b), e1z = __fmul_rn(-sg, wx);
    const float e2x = b, e2y = __fmaf_rn(wy, __fmul_rn(wy, k), sg), e2z = -wy;
    const float A = __fmul_rn(sn, cphi), B = __fmul_rn(sn, sphi);
    const float mx = __fmaf_rn(A, e1x, __fmaf_rn(B, e2x, __fmul_rn(c, wx)));
    const float my = __fmaf_rn(A, e1y, __fmaf_rn(B, e2y, __fmul_rn(c, wy)));
    const float mz = __fmaf_rn(A, e1z, __fmaf_rn(B, e2z, __fmul_rn(c, wz)));
    const float inv = __fdiv_rn(1.f, __fsqrt_rn(__fmaf_rn(mz, mz, __fmaf_rn(my, my, __fmul_rn(mx, mx)))));
    dirs[3 * i] = __fmul_rn(mx, inv); dirs[3 * i + 1] = __fmul_rn(my, inv); dirs[3 * i + 2] = __fmul_rn(mz, inv);
}

}  // namespace

opx_status launch_emit(const opx_track_steps& st, float n_index, float lambda1, float lambda2, uint64_t n, uint64_t id_base,
                       uint64_t seed, float* o, float* d, float* wl, cudaStream_t stream) {
    const uint64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffull) return fail(OPX_ERR_INVALID_ARG, "n too large for one launch");
    k_emit_cherenkov<<<(unsigned)blocks, 256, 0, stream>>>(st, n_index, lambda1, lambda2, n, id_base, seed, o, d, wl);
    count_launch(1);
    return check_cuda(cudaGetLastError(), "emit launch");
}

}  // namespace opx
