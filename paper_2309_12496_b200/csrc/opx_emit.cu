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

// ---- step look-up shared by the kernels below.  The photons a block handles are (a subset of) kSpan consecutive ids, so
// they sit in consecutive steps: warp 0 finds the step of the first id with a 32-ary search over the prefix sums (4
// dependent loads for 1e6 steps instead of 20), the block copies the next 257 prefix sums to shared memory and every
// thread finishes with an 8-step binary search there.  An id more than 256 steps further on (long runs of steps without
// photons) falls back to the global binary search.
struct StepWindow { uint64_t first[257]; uint64_t base; };

__device__ __forceinline__ void window_setup(StepWindow& sw, const opx_track_steps& st, uint64_t g0) {
    const uint64_t S = st.n_steps;
    if (threadIdx.x < 32) {
        const unsigned lane = threadIdx.x;
        uint64_t lo = 0, hi = S;                                   // invariant first[lo] <= g0 < first[hi]
        while (hi - lo > 1) {
            const uint64_t pos = lo + (((hi - lo) * (uint64_t)(lane + 1)) >> 5);       // in [lo, hi], non-decreasing in lane
            const bool le = pos == lo || (pos < hi && __ldg(st.first + pos) <= g0);
            const int k = __popc(__ballot_sync(0xffffffffu, le));                      // first[] is monotone: lanes 0..k-1 say yes
            const uint64_t nlo = __shfl_sync(0xffffffffu, pos, k > 0 ? k - 1 : 0), nhi = __shfl_sync(0xffffffffu, pos, k < 32 ? k : 31);
            lo = k > 0 ? nlo : lo; hi = k < 32 ? nhi : hi;
        }
        if (lane == 0) sw.base = lo;
    }
    __syncthreads();
    const uint64_t base = sw.base;
    for (unsigned j = threadIdx.x; j < 257u; j += blockDim.x) sw.first[j] = __ldg(st.first + (base + j < S ? base + j : S));
    __syncthreads();
}

// the LAST step s with first[s] <= g (steps without photons are skipped), for g >= the id the window was set up for
__device__ __forceinline__ uint64_t window_find(const StepWindow& sw, const opx_track_steps& st, uint64_t g) {
    const uint64_t S = st.n_steps, base = sw.base;
    if (sw.first[256] <= g && base + 256 < S) {
        uint64_t lo = base + 256, hi = S;                          // first[lo] <= g < first[S]
        while (hi - lo > 1) {
            const uint64_t mid = lo + (hi - lo) / 2;
            if (__ldg(st.first + mid) <= g) lo = mid; else hi = mid;
        }
        return lo;
    }
    unsigned jl = 0, jh = 256;                                     // first[jl] <= g < first[jh] (entries past S repeat first[S] > g)
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const unsigned mid = (jl + jh) >> 1;
        if (sw.first[mid] <= g) jl = mid; else jh = mid;
    }
    return base + jl;
}

// wavelength of photon g alone (word 1 of block 0): all the pre-propagation filter needs
__device__ __forceinline__ float emit_wavelength(uint64_t seed, uint64_t g, float lambda1, float lambda2) {
    const Words r = philox4(seed, g, 0u, 2u);
    return __fdiv_rn(__fmul_rn(lambda1, lambda2), __fmaf_rn(-u01(r.w1), __fsub_rn(lambda2, lambda1), lambda2));
}

// DESIGN.md 3.12 for photon g of step `s`, written to entry `q` of the output arrays
__device__ __forceinline__ void emit_photon(const opx_track_steps& st, uint64_t s, uint64_t g, uint64_t seed, float n_index,
                                            float lambda1, float lambda2, uint64_t q, float* __restrict__ origins,
                                            float* __restrict__ dirs, float* __restrict__ wl) {
    const float* x = st.x + 3 * s;
    const float* w = st.w + 3 * s;
    const float wx = __ldg(w), wy = __ldg(w + 1), wz = __ldg(w + 2);
    Words r = philox4(seed, g, 0u, 2u);
    const float t = __fmul_rn(u01(r.w0), __ldg(st.length + s));
    origins[3 * q] = __fmaf_rn(t, wx, __ldg(x)); origins[3 * q + 1] = __fmaf_rn(t, wy, __ldg(x + 1)); origins[3 * q + 2] = __fmaf_rn(t, wz, __ldg(x + 2));
    wl[q] = __fdiv_rn(__fmul_rn(lambda1, lambda2), __fmaf_rn(-u01(r.w1), __fsub_rn(lambda2, lambda1), lambda2));
    float c = __fdiv_rn(1.f, __fmul_rn(n_index, __ldg(st.beta + s)));
    if (!(c < 1.f)) c = 1.f;
    const float sn = __fsqrt_rn(fmaxf(__fmaf_rn(-c, c, 1.f), 0.f));
    float cphi = 1.f, sphi = 0.f;
    for (uint32_t a = 0; a < 64u; ++a) {
        if (a > 0) r = philox4(seed, g, a, 2u);
        const float X = __fmaf_rn(2.f, u01(r.w2), -1.f), Y = __fmaf_rn(2.f, u01(r.w3), -1.f);
        const float qq = __fmaf_rn(Y, Y, __fmul_rn(X, X));
        if (qq > 0.f && qq <= 1.f) {
            cphi = __fdiv_rn(__fsub_rn(__fmul_rn(X, X), __fmul_rn(Y, Y)), qq);
            sphi = __fdiv_rn(__fmul_rn(__fmul_rn(2.f, X), Y), qq);
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
    dirs[3 * q] = __fmul_rn(mx, inv); dirs[3 * q + 1] = __fmul_rn(my, inv); dirs[3 * q + 2] = __fmul_rn(mz, inv);
}

__global__ void __launch_bounds__(256) k_emit_cherenkov(const opx_track_steps st, float n_index, float lambda1, float lambda2,
                                                        uint64_t n, uint64_t id_base, uint64_t seed,
                                                        float* __restrict__ origins, float* __restrict__ dirs,
                                                        float* __restrict__ wl) {
    __shared__ StepWindow sw;
    const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    window_setup(sw, st, id_base + blockIdx.x * (uint64_t)blockDim.x);
    if (i >= n) return;
    const uint64_t g = id_base + i;
    emit_photon(st, window_find(sw, st, g), g, seed, n_index, lambda1, lambda2, i, origins, dirs, wl);
}

// ---------------------------------------------------------------- emission fused with the pre-propagation filter
// opx_emit_cherenkov_filtered = opx_emit_cherenkov followed by opx_prefilter, without ever writing the photons the
// filter discards (6 of 7 with the paper's efficiencies).  The filter needs only the wavelength, which
// is one Philox word and does not depend on the step:
//   k_emitf_mark     per photon: lambda, p = product of the efficiencies, the filter's draw on stream 1 (3.9); a mask word
//                    per warp, a survivor count per block of kFBlk ids.  Reads nothing, writes 1/8 B/photon.
//   k_prefilter_scan (opx_prefilter.cu) block offsets and the total.
//   k_emitf_compact  per block: the kept ids are listed densely in shared memory, then thread t emits the t-th survivor
//                    (full warps although only 1 id in 7 survives) straight to its final, stable position.
constexpr int kFBlk = 2048, kFThreads = 256, kFRounds = kFBlk / kFThreads, kFWords = kFBlk / 32;

__global__ void __launch_bounds__(kFThreads) k_emitf_mark(const SceneDev sc, const FilterFactors fa, float lambda1, float lambda2,
                                                          uint64_t n, uint64_t id_base, uint64_t seed,
                                                          uint32_t* __restrict__ words, uint32_t* __restrict__ block_count) {
    __shared__ uint32_t s_cnt[kFThreads / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t cnt = 0;
#pragma unroll
    for (int r = 0; r < kFRounds; ++r) {
        const uint64_t word = (uint64_t)blockIdx.x * kFWords + (uint64_t)(w * kFRounds + r);
        const uint64_t i = word * 32 + lane;
        bool keep = false;
        if (i < n) {
            const uint64_t g = id_base + i;
            keep = philox_uniform(seed, g, 0u, 1u) < filter_probability(sc, fa, emit_wavelength(seed, g, lambda1, lambda2));
        }
        const uint32_t mask = __ballot_sync(0xffffffffu, keep);
        if (lane == 0 && word * 32 < n) words[word] = mask;
        cnt += __popc(mask);
    }
    if (lane == 0) s_cnt[w] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int k = 0; k < kFThreads / 32; ++k) t += s_cnt[k];
        block_count[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(kFThreads) k_emitf_compact(const opx_track_steps st, float n_index, float lambda1, float lambda2,
                                                             uint64_t n, uint64_t id_base, uint64_t seed,
                                                             const uint32_t* __restrict__ words, const uint32_t* __restrict__ block_offset,
                                                             float* __restrict__ origins, float* __restrict__ dirs,
                                                             float* __restrict__ wl, uint32_t* __restrict__ oidx, uint64_t capacity) {
    __shared__ StepWindow sw;
    __shared__ uint32_t s_mask[kFWords], s_pre[kFWords + 1];
    __shared__ uint16_t s_list[kFBlk];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint64_t blk_base = (uint64_t)blockIdx.x * kFBlk;
    if (threadIdx.x < kFWords) {
        const uint64_t word = (uint64_t)blockIdx.x * kFWords + threadIdx.x;
        s_mask[threadIdx.x] = word * 32 < n ? __ldg(words + word) : 0u;
    }
    __syncthreads();
    if (w == 0) {       // exclusive prefix of the 64 word popcounts, two consecutive words per lane
        const uint32_t a = __popc(s_mask[2 * lane]), b = __popc(s_mask[2 * lane + 1]);
        uint32_t inc = a + b;
        for (int k = 1; k < 32; k <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, k); if (lane >= k) inc += y; }
        s_pre[2 * lane] = inc - a - b; s_pre[2 * lane + 1] = inc - b;
        if (lane == 31) s_pre[kFWords] = inc;
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kFRounds; ++r) {
        const int wi = w * kFRounds + r;
        const uint32_t mask = s_mask[wi];
        if ((mask >> lane) & 1u) s_list[s_pre[wi] + __popc(mask & ((1u << lane) - 1u))] = (uint16_t)(wi * 32 + lane);
    }
    window_setup(sw, st, id_base + blk_base);          // (its barriers also publish s_list)
    const uint32_t cnt = s_pre[kFWords];
    const uint64_t off = (uint64_t)__ldg(block_offset + blockIdx.x);
    for (uint32_t q = threadIdx.x; q < cnt; q += kFThreads) {
        if (off + q >= capacity) break;   // the out arrays are full: *d_n_kept still holds the true count
        const uint64_t i = blk_base + s_list[q], g = id_base + i;
        emit_photon(st, window_find(sw, st, g), g, seed, n_index, lambda1, lambda2, off + q, origins, dirs, wl);
        if (oidx) oidx[off + q] = (uint32_t)i;
    }
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

opx_status launch_emit_filtered(const SceneHost& s, const opx_track_steps& st, float n_index, float lambda1, float lambda2, uint64_t n,
                                uint64_t id_base, uint64_t seed, const uint32_t* factors, uint32_t n_factors, float* o, float* d,
                                float* wl, uint32_t* oidx, uint64_t capacity, uint64_t* d_n_kept, void* ws, cudaStream_t stream) {
    FilterFactors fa{};
    fa.n = n_factors;
    for (uint32_t k = 0; k < n_factors; ++k) { fa.m[k] = factors[k]; fa.mk[k] = s.mat_kinds[factors[k]]; }
    const uint64_t nb = (n + kFBlk - 1) / kFBlk;
    uint32_t* words = (uint32_t*)ws;
    uint32_t* counts = (uint32_t*)((char*)ws + align_up((size_t)nb * kFWords * 4, 256));
    k_emitf_mark<<<(unsigned)nb, kFThreads, 0, stream>>>(s.dev, fa, lambda1, lambda2, n, id_base, seed, words, counts);
    launch_prefilter_scan(counts, (uint32_t)nb, d_n_kept, stream);
    k_emitf_compact<<<(unsigned)nb, kFThreads, 0, stream>>>(st, n_index, lambda1, lambda2, n, id_base, seed, words, counts, o, d, wl, oidx, capacity);
    count_launch(3);
    return check_cuda(cudaGetLastError(), "emit+filter launch");
}

}  // namespace opx
