// opx_prefilter: the paper's pre-propagation efficiency filter, SURVEY 8(f) row f1.
//
// Three launches on the caller's stream, no host round trip:
//   k_prefilter_mark     one thread per photon: p = e_0(lambda) * e_1(lambda) * ... (left to right, fp32), one Philox
//                        draw on stream 1, keep iff u < p.  A warp writes its 32 decisions as one mask word and the
//                        CTA its number of survivors: 4 B/photon read, 1/8 B/photon written.
//   k_prefilter_scan     one CTA: exclusive scan of the per-CTA survivor counts in place; total -> *d_n_kept.
//   k_prefilter_compact  one CTA per kBlk photons: rank of every kept photon from the mask words (no second draw),
//                        survivors copied in input order (stable) - only their 28 input bytes are read.
// Integer ranks from integer masks: the output does not depend on scheduling.
#include "opx_device.cuh"

namespace opx {
namespace {

constexpr int kFThreads = 256;
constexpr int kFWarps = kFThreads / 32;
constexpr int kBlk = 2048;                      // photons per CTA
constexpr int kRounds = kBlk / kFThreads;       // 8 mask words per warp
constexpr int kWords = kBlk / 32;               // 64 mask words per CTA
using Factors = FilterFactors;

__global__ void __launch_bounds__(kFThreads) k_prefilter_mark(const SceneDev sc, const Factors fa, uint64_t n, uint64_t id_base,
                                                              const float* __restrict__ wl, uint64_t seed,
                                                              uint32_t* __restrict__ words, uint32_t* __restrict__ block_count) {
    __shared__ uint32_t s_cnt[kFWarps];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint64_t blk_base = (uint64_t)blockIdx.x * kBlk;
    uint32_t cnt = 0;
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        const uint64_t word = (uint64_t)blockIdx.x * kWords + (uint64_t)(w * kRounds + r);
        const uint64_t i = blk_base + (uint64_t)((w * kRounds + r) * 32 + lane);
        bool keep = false;
        if (i < n) {
            const float lambda = __ldcs(wl + i);
            const float p = filter_probability(sc, fa, lambda);
            keep = philox_uniform(seed, id_base + i, 0u, 1u) < p;
        }
        const uint32_t mask = __ballot_sync(0xffffffffu, keep);
        if (lane == 0 && word * 32 < n) words[word] = mask;
        cnt += __popc(mask);
    }
    if (lane == 0) s_cnt[w] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int k = 0; k < kFWarps; ++k) t += s_cnt[k];
        block_count[blockIdx.x] = t;
    }
}

// Exclusive scan of `count[0..nb)` in place by one CTA of 1024 threads; total to *total_out.
__global__ void __launch_bounds__(1024) k_prefilter_scan(uint32_t* __restrict__ count, uint32_t nb, unsigned long long* total_out) {
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_carry;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (uint32_t base = 0; base < nb; base += 1024) {
        const uint32_t i = base + threadIdx.x;
        const uint32_t v = i < nb ? count[i] : 0u;
        uint32_t inc = v;
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
        if (lane == 31) s_warp[w] = inc;
        __syncthreads();
        if (w == 0) {
            uint32_t x = s_warp[lane], xi = x;
            for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, xi, o); if (lane >= o) xi += y; }
            s_warp[lane] = xi - x;                       // exclusive prefix of the warp totals
        }
        __syncthreads();
        const uint32_t carry = s_carry;
        if (i < nb) count[i] = carry + s_warp[w] + inc - v;
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = carry + s_warp[w] + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total_out = (unsigned long long)s_carry;
}

__global__ void __launch_bounds__(kFThreads) k_prefilter_compact(uint64_t n, const float* __restrict__ o, const float* __restrict__ d,
                                                                 const float* __restrict__ wl, const uint32_t* __restrict__ words,
                                                                 const uint32_t* __restrict__ block_offset, float* __restrict__ oo,
                                                                 float* __restrict__ od, float* __restrict__ owl,
                                                                 uint32_t* __restrict__ oidx, uint64_t capacity) {
    __shared__ uint32_t s_mask[kWords];
    __shared__ uint32_t s_pre[kWords];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint64_t blk_base = (uint64_t)blockIdx.x * kBlk;
    if (threadIdx.x < kWords) {
        const uint64_t word = (uint64_t)blockIdx.x * kWords + threadIdx.x;
        s_mask[threadIdx.x] = word * 32 < n ? __ldg(words + word) : 0u;
    }
    __syncthreads();
    if (w == 0) {       // exclusive prefix of the 64 word popcounts, two consecutive words per lane
        const uint32_t a = __popc(s_mask[2 * lane]), b = __popc(s_mask[2 * lane + 1]);
        uint32_t inc = a + b;
        for (int k = 1; k < 32; k <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, k); if (lane >= k) inc += y; }
        s_pre[2 * lane] = inc - a - b; s_pre[2 * lane + 1] = inc - b;
    }
    __syncthreads();
    const uint64_t off = (uint64_t)__ldg(block_offset + blockIdx.x);
#pragma unroll
    for (int r = 0; r < kRounds; ++r) {
        const int wi = w * kRounds + r;
        const uint32_t mask = s_mask[wi];
        if (!((mask >> lane) & 1u)) continue;
        const uint64_t i = blk_base + (uint64_t)(wi * 32 + lane);
        const uint64_t q = off + s_pre[wi] + __popc(mask & ((1u << lane) - 1u));
        if (q >= capacity) continue;      // the out arrays are full: *d_n_kept still holds the true count
        const float ox = __ldcs(o + 3 * i), oy = __ldcs(o + 3 * i + 1), oz = __ldcs(o + 3 * i + 2);
        const float dx = __ldcs(d + 3 * i), dy = __ldcs(d + 3 * i + 1), dz = __ldcs(d + 3 * i + 2);
        oo[3 * q] = ox; oo[3 * q + 1] = oy; oo[3 * q + 2] = oz;
        od[3 * q] = dx; od[3 * q + 1] = dy; od[3 * q + 2] = dz;
        owl[q] = __ldg(wl + i);
        if (oidx) oidx[q] = (uint32_t)i;
    }
}

}  // namespace

void launch_prefilter_scan(uint32_t* counts, uint32_t nb, uint64_t* d_total, cudaStream_t stream) {
    k_prefilter_scan<<<1, 1024, 0, stream>>>(counts, nb, (unsigned long long*)d_total);
}

size_t prefilter_workspace_bytes(uint64_t n) {
    const uint64_t nb = (n + kBlk - 1) / kBlk;
    return align_up((size_t)nb * kWords * 4, 256) + align_up((size_t)nb * 4, 256) + 256;
}

opx_status launch_prefilter(const SceneHost& s, uint64_t n, uint64_t id_base, const float* o, const float* d, const float* wl,
                            uint64_t seed, const uint32_t* factors, uint32_t n_factors, float* oo, float* od, float* owl,
                            uint32_t* oidx, uint64_t capacity, uint64_t* d_n_kept, void* ws, cudaStream_t stream) {
    Factors fa{};
    fa.n = n_factors;
    for (uint32_t k = 0; k < n_factors; ++k) { fa.m[k] = factors[k]; fa.mk[k] = s.mat_kinds[factors[k]]; }
    const uint64_t nb = (n + kBlk - 1) / kBlk;
    uint32_t* words = (uint32_t*)ws;
    uint32_t* counts = (uint32_t*)((char*)ws + align_up((size_t)nb * kWords * 4, 256));
    k_prefilter_mark<<<(unsigned)nb, kFThreads, 0, stream>>>(s.dev, fa, n, id_base, wl, seed, words, counts);
    k_prefilter_scan<<<1, 1024, 0, stream>>>(counts, (uint32_t)nb, (unsigned long long*)d_n_kept);
    k_prefilter_compact<<<(unsigned)nb, kFThreads, 0, stream>>>(n, o, d, wl, words, counts, oo, od, owl, oidx, capacity);
    count_launch(3);
    return check_cuda(cudaGetLastError(), "prefilter launch");
}

}  // namespace opx

// ------------------------------------------------------------------ opx_prefilter_noalloc (include/opx.h)
// The filter for callers that have no device memory to give it and may not ask the driver for any: a Geant4 worker
// or an experiment-framework plug-in that was handed a fixed set of device buffers by the framework's own pool (the
// pool holds the whole card, so a cudaMalloc from inside the plug-in fails or is forbidden by the host code's rules),
// and event loops in which several worker threads keep their own streams busy on one GPU, where a cudaMalloc /
// cudaFree would make the whole device wait.  The mask words and per-CTA counts that opx_prefilter keeps in the
// caller's workspace live here in ONE array that is part of the library image: every GPU on which the library's code
// gets loaded holds these bytes from then until the process exits, whether or not the entry point is ever called.
#include <mutex>

namespace opx {
namespace {

constexpr uint64_t kNoAllocMaxPhotons = OPX_PREFILTER_NOALLOC_MAX_PHOTONS;
constexpr size_t kNoAllocBlocks = (size_t)((kNoAllocMaxPhotons + kBlk - 1) / kBlk);
// the layout launch_prefilter() carves out of a workspace: mask words, then per-CTA counts, then one spare line
constexpr size_t kNoAllocBytes = (kNoAllocBlocks * kWords * 4 + 255) / 256 * 256 + (kNoAllocBlocks * 4 + 255) / 256 * 256 + 256;
static_assert(kNoAllocBytes <= (size_t)(2u << 20) + (64u << 10), "the built-in scratch is meant to stay near 2 MiB");

// In HOST code this name is only a handle for the runtime's symbol table - it is not where the bytes are on the GPU,
// and handing it to a kernel would fault (or, where the GPU can reach host memory, quietly scribble over the host-side
// shadow).  Host code must go through noalloc_scratch() below.  Device code could name the array directly.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

constexpr int kMaxDevices = 64;
std::mutex g_noalloc_mutex;
void* g_noalloc_addr[kMaxDevices] = {};   // device address of g_noalloc_scratch on device k, looked up once

// Device address of the built-in scratch on the CURRENT device.  Each device has its own copy of the array at its own
// address, so the look-up is done once per device, with that device current, and remembered.  The look-up makes the
// runtime load this library's device code on that device if nothing has yet; it allocates nothing.
opx_status noalloc_scratch(void** out) {
    int dev = -1;
    if (cudaError_t e = cudaGetDevice(&dev)) return check_cuda(e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) return fail(OPX_ERR_UNSUPPORTED_DEVICE, "opx_prefilter_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[dev]) {
        void* p = nullptr;
        if (cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch)) return check_cuda(e, "cudaGetSymbolAddress(built-in prefilter scratch)");
        if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return fail(OPX_ERR_CUDA, "built-in prefilter scratch has no usable device address");
        g_noalloc_addr[dev] = p;
    }
    *out = g_noalloc_addr[dev];
    return OPX_OK;
}

}  // namespace
}  // namespace opx

extern "C" opx_status opx_prefilter_noalloc(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                                            const float* d_dirs, const float* d_wavelengths, uint64_t seed,
                                            const uint32_t* factors, uint32_t n_factors, float* d_out_origins,
                                            float* d_out_dirs, float* d_out_wavelengths, uint32_t* d_out_index,
                                            uint64_t out_capacity, uint64_t* d_n_kept, void* cuda_stream) {
    using namespace opx;
    auto off = [](const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) != 0; };
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_prefilter_noalloc before opx_bvh_build");
    if (!d_n_kept || off(d_n_kept, 8)) return fail(OPX_ERR_INVALID_ARG, "d_n_kept is NULL or misaligned");
    if (n > kNoAllocMaxPhotons)
        return fail(OPX_ERR_INVALID_ARG, "opx_prefilter_noalloc: n = " + std::to_string(n) + " photons is beyond the " +
                                             std::to_string(kNoAllocMaxPhotons) + " (OPX_PREFILTER_NOALLOC_MAX_PHOTONS) the built-in " +
                                             "scratch holds; split the call or use opx_prefilter with a workspace of your own");
    if (n_factors > 8 || (n_factors && !factors)) return fail(OPX_ERR_INVALID_ARG, "n_factors must be <= 8 and factors non-NULL");
    for (uint32_t k = 0; k < n_factors; ++k) {
        if (factors[k] >= scene->mat_kinds.size()) return fail(OPX_ERR_INVALID_ARG, "factor material index out of range");
        if ((scene->mat_kinds[factors[k]] & 0xffu) == OPX_MAT_ABSORBER) return fail(OPX_ERR_INVALID_ARG, "an absorber has no efficiency table");
    }
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_prefilter_noalloc")) return st;
    if (n == 0) return check_cuda(cudaMemsetAsync(d_n_kept, 0, 8, (cudaStream_t)cuda_stream), "cudaMemsetAsync");
    if (!d_origins || !d_dirs || !d_wavelengths || !d_out_origins || !d_out_dirs || !d_out_wavelengths)
        return fail(OPX_ERR_INVALID_ARG, "NULL photon pointer");
    if (off(d_origins, 4) || off(d_dirs, 4) || off(d_wavelengths, 4) || off(d_out_origins, 4) || off(d_out_dirs, 4) ||
        off(d_out_wavelengths, 4) || off(d_out_index, 4))
        return fail(OPX_ERR_INVALID_ARG, "misaligned pointer");
    if (d_out_origins == d_origins || d_out_dirs == d_dirs || d_out_wavelengths == d_wavelengths)
        return fail(OPX_ERR_INVALID_ARG, "out arrays must not alias the inputs");
    void* scratch = nullptr;
    if (opx_status st = noalloc_scratch(&scratch)) return st;
    // Nothing in the scratch has to start at zero: k_prefilter_mark writes every mask word and every per-CTA count that
    // k_prefilter_scan and k_prefilter_compact read for this n, so what the previous call left behind is never seen.
    return launch_prefilter(*scene, n, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, factors, n_factors, d_out_origins,
                            d_out_dirs, d_out_wavelengths, d_out_index, out_capacity, d_n_kept, scratch, (cudaStream_t)cuda_stream);
}
