// A5-A12 launchers: per-photon propagation and hit binning.
//   k_propagate_packet (opx_packet.cuh)  the product kernel: tile-sorted photons, warp-packet traversal
//   k_propagate_lane   (opx_lane.cuh)    per-thread traversal: instrumented / brute-force / tiny scenes
//   k_bin              (opx_bin.cuh)     A11 hit binning with warp-aggregated atomics + A12 counters
#include <atomic>

#include "opx_bin.cuh"
#include "opx_lane.cuh"
#include "opx_packet.cuh"

namespace opx {

using Big = PacketSmemT<512, 4>;      // 2048-photon tiles, 4 packets per warp: the general shape
using Small = PacketSmemT<512, 1>;    // 512-photon tiles, 1 packet per warp: calls too small to fill the machine
using Mid = PacketSmemT<256, 4>;      // 1024-photon tiles, 4 CTAs/SM: filtered (NO_EFFICIENCY) streams
using Wave = PacketSmemT<1024, 1>;    // one CTA per SM, one packet per warp, run-time tile size: a small call in a single wave
constexpr int kMaxDevices = 64;
static std::atomic<int> g_sms[kMaxDevices];      // SM count per device ordinal, 0 = not configured yet

// The dynamic shared memory limit of a kernel is an attribute per device (context): set once per device, at the first
// opx_bvh_build or launch on it, so that a later opx_propagate performs stream operations only (CUDA-graph capturable).
// The device's SM count, which decides the kernel shape of a small call, is looked up at the same time (*sms, may be NULL).
opx_status configure_device(int* sms) {
    int dev = 0;
    if (opx_status st = check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return st;
    if (dev < 0 || dev >= kMaxDevices) return fail(OPX_ERR_UNSUPPORTED_DEVICE, "device ordinal beyond 63");
    if (const int known = g_sms[dev].load(std::memory_order_acquire)) { if (sms) *sms = known; return OPX_OK; }
    int count = 0;
    cudaError_t e = cudaDeviceGetAttribute(&count, cudaDevAttrMultiProcessorCount, dev);
    if (!e && count < 1) return fail(OPX_ERR_UNSUPPORTED_DEVICE, "device reports no multiprocessors");
    if (!e) e = cudaFuncSetAttribute(k_propagate_packet<512, 4, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Big));
    if (!e) e = cudaFuncSetAttribute(k_propagate_packet<512, 4, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Big));
    if (!e) e = cudaFuncSetAttribute(k_propagate_packet<512, 1, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Small));
    if (!e) e = cudaFuncSetAttribute(k_propagate_packet<256, 4, 4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Mid));
    if (!e) e = cudaFuncSetAttribute(k_propagate_packet<1024, 1, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Wave));
    if (opx_status st = check_cuda(e, "cudaFuncSetAttribute")) return st;
    g_sms[dev].store(count, std::memory_order_release);      // two threads racing here both set the same attributes: harmless
    if (sms) *sms = count;
    return OPX_OK;
}

static opx_status launch_propagate_impl(const SceneHost& s, WalkMode mode, uint64_t n, const uint64_t* d_n, uint64_t id_base, const float* o,
                                        const float* d, const float* wl, uint64_t seed, uint32_t flags, const opx_hits& out,
                                        uint32_t* hitmap, uint64_t* counters, uint64_t* packet_stats, cudaStream_t stream,
                                        DetOut det = DetOut{}, uint64_t* det_tiles = nullptr) {
    SceneDev dev = s.dev;          // per-launch copy: flags and the optional device-side count ride in the kernel parameter
    dev.flags = flags;
    dev.d_n = (const unsigned long long*)d_n;
    if (mode == kWalkBinary) { dev.n_wnodes = 0; dev.flags |= kFlagPacketWalk; }      // debug: packets walk the binary tree only, as warps
    const bool brute = mode == kWalkBrute;
    cudaEvent_t* ev = nullptr;
    if (s.prof_used < s.prof_max) { ev = &s.prof_events[3 * (size_t)s.prof_used]; ++s.prof_used; }
    if (ev) cudaEventRecord(ev[0], stream);
    bool binned = false;         // A11/A12 done inside the propagation kernel
    if (det.id && (brute || s.dev.n_tri < 2)) return fail(OPX_ERR_BAD_STATE, "the detected-only output needs a scene with a hierarchy (two triangles or more)");
    if (brute || s.dev.n_tri < 2) {
        // debug mode, or a scene with fewer than two triangles (no hierarchy): test the triangle list directly
        const uint64_t blocks = (n + 127) / 128;
        if (blocks > 0x7fffffffull) return fail(OPX_ERR_INVALID_ARG, "n too large for one launch");
        k_propagate_lane<true, false><<<(unsigned)blocks, 128, 0, stream>>>(dev, n, id_base, o, d, wl, seed, out, nullptr);
        set_last_kernel("k_propagate_lane<1, 0>");
    } else {
        // Shapes (defined at the top of this file), re-measured on the final kernel of round 2: in-flight calls run fastest with
        // 2 x 512 threads per SM and 2048-photon tiles on every scene (toy scene C2 / C3: 1.158 / 1.210 ms per 1e7 photons
        // against 1.171 / 1.251 with 448 x 2 and 1.216 / 1.227 with 256 x 4; C4: 6.18 / 6.70 / 7.40 ms per 2e7).  A filtered
        // stream (NO_EFFICIENCY: 1 photon in 7-9 survives, so packets are wide and differ widely in cost; a tile's warps wait at
        // its barrier for the slowest packet) runs fastest with 4 CTAs of 256 threads and 1024-photon tiles on every scene (C4
        // survivors of 4e7 photons: 3.38 ms against 4.12 with 2 x 512; toy scene 0.280 against 0.320).
        int sm_count = 0;
        if (opx_status st = configure_device(&sm_count)) return st;
        const uint64_t kSMs = (uint64_t)sm_count;      // 148 on a B200; the thresholds below were measured there
        // A small call (the paper's own runs are 600 ... 6e5 photons) is latency-bound: its time is the dependent
        // chain of ONE packet times the packets a warp walks one after the other.  Up to 148 x 512 photons the 512-photon tiles
        // (one packet per warp) already put every packet in flight at once; from there to 148 x 1024 photons the call runs as a
        // single wave -- one CTA of up to 32 warps per SM, one packet per warp, the photons dealt out evenly over the SMs (tile
        // size = ceil(n / 148) rounded up to whole packets): measured 64 us against 82 us at 151 000 photons on the toy scene,
        // 74 against 81 at 1e5; below 148 x 512 photons the 1024-thread CTAs lose (80 us against 68 at 6000 photons).
        const bool wave = !packet_stats && n > kSMs * Small::kTile && n <= kSMs * Wave::kTile;
        uint32_t stride = 0;
        if (wave) stride = (uint32_t)(((n + kSMs - 1) / kSMs + 31) / 32 * 32);
        // measured crossover (kernel time vs n, both tile sizes): beyond one wave the 512-photon tiles still win on a large scene
        // (longer, latency-bound packets) up to about 2e5 photons; on a small scene the large tiles take over
        const uint64_t small_below = s.dev.n_tri < (1u << 18) ? kSMs * Small::kTile + 1 : 100ull * Big::kTile;
        const bool small = !packet_stats && !wave && n < small_below;
        const bool mid = !packet_stats && !wave && !small && (flags & OPX_FLAG_NO_EFFICIENCY);
        const uint64_t tile = wave ? stride : small ? Small::kTile : (mid ? Mid::kTile : Big::kTile);
        const uint64_t tiles = (n + tile - 1) / tile;
        if (tiles > 0x7fffffffull) return fail(OPX_ERR_INVALID_ARG, "n too large for one launch");
        if (det_tiles) *det_tiles = tiles;
        if (packet_stats) k_propagate_packet<512, 4, 2, true><<<(unsigned)tiles, 512, sizeof(Big), stream>>>(dev, n, id_base, o, d, wl, seed, out, nullptr, nullptr, (unsigned long long*)packet_stats, det, 0u);
        else if (wave) k_propagate_packet<1024, 1, 1, false><<<(unsigned)tiles, 1024, sizeof(Wave), stream>>>(dev, n, id_base, o, d, wl, seed, out, hitmap, (unsigned long long*)counters, nullptr, det, stride);
        else if (mid) k_propagate_packet<256, 4, 4, false><<<(unsigned)tiles, 256, sizeof(Mid), stream>>>(dev, n, id_base, o, d, wl, seed, out, hitmap, (unsigned long long*)counters, nullptr, det, 0u);
        else if (small) k_propagate_packet<512, 1, 2, false><<<(unsigned)tiles, 512, sizeof(Small), stream>>>(dev, n, id_base, o, d, wl, seed, out, hitmap, (unsigned long long*)counters, nullptr, det, 0u);
        else k_propagate_packet<512, 4, 2, false><<<(unsigned)tiles, 512, sizeof(Big), stream>>>(dev, n, id_base, o, d, wl, seed, out, hitmap, (unsigned long long*)counters, nullptr, det, 0u);
        // the names ncu prints for these instantiations
        set_last_kernel(packet_stats ? "k_propagate_packet<512, 4, 2, 1>" : wave ? "k_propagate_packet<1024, 1, 1, 0>" : mid ? "k_propagate_packet<256, 4, 4, 0>"
                        : small ? "k_propagate_packet<512, 1, 2, 0>" : "k_propagate_packet<512, 4, 2, 0>");
        binned = !packet_stats;
    }
    count_launch(1);
    if (ev) cudaEventRecord(ev[1], stream);
    if (!binned && (hitmap || counters)) {
        const uint64_t bb = (n + 255) / 256;
        int sm_count = 0;
        if (opx_status st = configure_device(&sm_count)) return st;
        const unsigned grid = (unsigned)(bb < (uint64_t)sm_count * 8 ? bb : (uint64_t)sm_count * 8);
        k_bin<<<grid, 256, 0, stream>>>(out.state, out.bounces, out.pixel, n, (const unsigned long long*)d_n, hitmap, (unsigned long long*)counters);
        count_launch(1);
    }
    if (ev) cudaEventRecord(ev[2], stream);
    return check_cuda(cudaGetLastError(), "propagate launch");
}

opx_status launch_propagate(const SceneHost& s, WalkMode mode, uint64_t n, const uint64_t* d_n, uint64_t id_base, const float* o,
                            const float* d, const float* wl, uint64_t seed, uint32_t flags, const opx_hits& out, uint32_t* hitmap,
                            uint64_t* counters, cudaStream_t stream) {
    return launch_propagate_impl(s, mode, n, d_n, id_base, o, d, wl, seed, flags, out, hitmap, counters, nullptr, stream);
}

// Workspace of a detected-only launch: the counter of the staging list, the tile table (16 B) and the staging offsets (8 B)
// per tile of the smallest tile size, and a staging list of `capacity` entries.
struct DetWorkspace { unsigned long long* count; ulonglong2* table; unsigned long long* src; DetOut stage; size_t bytes; };
static DetWorkspace det_workspace(void* ws, uint64_t n, uint64_t capacity) {
    // the smallest fixed tile size bounds the tile count of every shape: the single-wave shape runs only where it makes tiles
    // of more than Small::kTile photons (n > SMs x Small::kTile dealt out over SMs tiles)
    const uint64_t tiles = (n + Small::kTile - 1) / Small::kTile + 1;
    char* p = (char*)ws;
    auto take = [&](size_t bytes) { char* r = p; p += align_up(bytes, 256); return r; };
    DetWorkspace w{};
    w.count = (unsigned long long*)take(256);
    w.table = (ulonglong2*)take(tiles * 16);
    w.src = (unsigned long long*)take(tiles * 8);
    w.stage.id = (unsigned long long*)take(capacity * 8); w.stage.pixel = (int32_t*)take(capacity * 4);
    w.stage.pos = (float*)take(capacity * 12); w.stage.dir = (float*)take(capacity * 12);
    w.stage.capacity = capacity; w.stage.stage_count = w.count; w.stage.tile_table = w.table;
    w.bytes = (size_t)(p - (char*)ws);
    return w;
}
size_t detected_workspace_bytes(uint64_t n, uint64_t capacity) { return det_workspace(nullptr, n, capacity).bytes; }

opx_status launch_propagate_detected(const SceneHost& s, uint64_t n, const uint64_t* d_n, uint64_t id_base, const float* o,
                                     const float* d, const float* wl, uint64_t seed, uint32_t flags, const opx_detected& list,
                                     uint64_t capacity, uint64_t* d_n_detected, const uint32_t* d_index, void* workspace, uint32_t* hitmap,
                                     uint64_t* counters, cudaStream_t stream) {
    DetWorkspace w = det_workspace(workspace, n, capacity);
    w.stage.index = d_index;
    // the counter and the whole tile table start at zero: tiles beyond a device-side photon count never run and must read (0, 0)
    if (opx_status st = check_cuda(cudaMemsetAsync(w.count, 0, (size_t)((char*)w.src - (char*)w.count), stream), "cudaMemsetAsync")) return st;
    uint64_t tiles = 0;
    if (opx_status st = launch_propagate_impl(s, kWalkProduct, n, d_n, id_base, o, d, wl, seed, flags, opx_hits{}, hitmap, counters, nullptr,
                                              stream, w.stage, &tiles)) return st;
    k_det_scan<<<1, 1024, 0, stream>>>(w.table, w.src, tiles, capacity, (unsigned long long*)d_n_detected, w.count);
    DetOut out{(unsigned long long*)list.id, list.pixel, list.pos, list.dir, capacity, nullptr, nullptr, nullptr};
    k_det_gather<<<(unsigned)((tiles * 32 + 255) / 256), 256, 0, stream>>>(w.table, w.src, tiles, w.stage, out);
    count_launch(2);
    return check_cuda(cudaGetLastError(), "detected-list launch");
}

opx_status launch_packet_stats(const SceneHost& s, uint64_t n, uint64_t id_base, const float* o, const float* d,
                               const float* wl, uint64_t seed, const opx_hits& out, uint64_t* stats, cudaStream_t stream) {
    if (s.dev.n_tri < 2) return fail(OPX_ERR_BAD_STATE, "no hierarchy to instrument (fewer than two triangles)");
    return launch_propagate_impl(s, kWalkProduct, n, nullptr, id_base, o, d, wl, seed, 0u, out, nullptr, nullptr, stats, stream);
}

opx_status launch_stats(const SceneHost& s, uint64_t n, uint64_t id_base, const float* o, const float* d, const float* wl,
                        uint64_t seed, uint64_t* stats, cudaStream_t stream) {
    const uint64_t blocks = (n + 127) / 128;
    if (blocks > 0x7fffffffull) return fail(OPX_ERR_INVALID_ARG, "n too large for one launch");
    if (s.dev.n_tri < 2) return fail(OPX_ERR_BAD_STATE, "no hierarchy to instrument (fewer than two triangles)");
    k_propagate_lane<false, true><<<(unsigned)blocks, 128, 0, stream>>>(s.dev, n, id_base, o, d, wl, seed, opx_hits{}, (unsigned long long*)stats);
    count_launch(1);
    return check_cuda(cudaGetLastError(), "stats launch");
}

}  // namespace opx
