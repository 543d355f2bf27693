// k_propagate_packet: the product kernel for A5-A10.
//
// One CTA owns a tile of kTile consecutive photons:
//   1. stage   the tile's inputs are copied to shared memory by three TMA bulk copies (cp.async.bulk) that one thread
//              issues (a ragged or misaligned tile falls back to coalesced streaming loads);
//   2. sort    photons are ordered by a 12-bit pseudo-angle of their direction about the tile's mean
//              direction (Cherenkov photons of a track lie on a cone = a ring in the octahedral
//              plane), with a 2-pass 6-bit radix sort in shared memory;
//   3. trace   every warp takes groups of 32 neighbouring photons and walks the 32-wide tree as ONE packet bounded by a
//              beam (opx_beam.cuh): lane k tests child k of a wide node, control flow is uniform, the stack is the
//              warp's in shared memory.  A packet too incoherent for a beam is walked per lane through the binary
//              tree (closest_hit_own).  Each lane intersects its own ray with the contract test against the triangles
//              its ray's box test leaves, so results are exactly the per-photon results of DESIGN.md section 2;
//   4. store   records are written back into the photon's own shared-memory slot and the tile leaves by six TMA bulk
//              stores (or coalesced streaming stores for a ragged / misaligned tile).
#pragma once
#include "opx_beam.cuh"
#include "opx_device.cuh"

namespace opx {
namespace {

constexpr int kPktStack = 96;                        // depth bound of the Karras tree (see opx_lane.cuh)
constexpr int kStackSmem = kPktStack - 32;
constexpr int kRadixBits = 6, kRadix = 1 << kRadixBits;      // 2 passes over the 12-bit key

// (A fifth shape, 1024 threads x 1 photon with a run-time tile stride, spreads a call of at most 148 x 1024 photons over all
// SMs with every packet in flight at once: opx_propagate.cu.)
// The kernel is compiled for two tile sizes on 512 threads: kItems = 4 photons per thread, 2048-photon tiles (the
// product shape: the more photons of a ring a tile holds, the narrower its packets; each warp walks 4 packets), and
// kItems = 1, 512-photon tiles where each warp walks ONE packet, for calls too small to fill the machine with large
// tiles: four times the CTAs and a quarter of the latency (the paper's own runs are 600 ... 6e5 photons).
template <int kPktThreads, int kItems>
struct PacketSmemT {
    static constexpr int kPktWarps = kPktThreads / 32;
    static constexpr int kTile = kItems * kPktThreads;
    float o[kTile * 3];          // in: origins            out: hit positions
    float d[kTile * 3];          // in: directions         out: arrival directions
    float wl[kTile];             // in: wavelengths        out: pixel ids (int bits)
    int surface[kTile];          // sort scratch (second key buffer), then out: surface ids
    uint32_t key[kTile];         // (angle12 << 16) | index in tile, sorted (ping-pong with `surface`)
    uint8_t state[kTile];
    uint8_t bounces[kTile];
    union {
        int stack[kPktWarps][kStackSmem];        // traversal: stack entries >= 32 of each warp
        uint32_t cnt[kRadix][kPktWarps];         // sort: radix counters [digit][warp]
    };
    float beam_tn[kPktWarps][kBeamStackWords];        // beam traversal: entry bounds of the stacked wide nodes (refs alias `stack`)
    float4 cull[kPktWarps][2 * kCullSlots];      // beam traversal: candidate boxes of the node a warp is culling (opx_beam.cuh)
    float red[kPktWarps][3];
    float bcast[3];
    uint32_t scan_tot[kPktWarps < 8 ? 8 : kPktWarps];    // sort: per-warp totals; store phase: the 8 state counters
    int next_group;              // dynamic hand-out of packet groups to warps
    alignas(8) unsigned long long mbar;          // completion barrier of the bulk loads of the staging phase
};
static_assert(sizeof(int) * kStackSmem >= sizeof(uint32_t) * kRadix, "radix counters alias the stack overflow area");
static_assert(kBeamStackWords <= kStackSmem && kBeamStack + 8 <= kBeamStackWords, "the beam stack refs (and the parked beam behind them) alias the binary walk's overflow area");

// ---- TMA bulk copies (cp.async.bulk, 1-D): a full tile's inputs and records are contiguous 16-byte-aligned blocks, so one
// elected thread moves them between global and shared memory instead of 512 threads looping over float4s.
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity) {
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "OPX_WAIT_%=:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 "@p bra OPX_DONE_%=;\n"
                 "bra OPX_WAIT_%=;\n"
                 "OPX_DONE_%=:\n"
                 "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// Photon inputs and records are touched once: an evict-first L2 policy keeps them from pushing the BVH out of L2.
__device__ __forceinline__ uint64_t l2_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, void* bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_u32(dst)), "l"(__cvta_generic_to_global(src)), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, uint32_t bytes, uint64_t pol) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                 ::"l"(__cvta_generic_to_global(dst)), "r"(smem_u32(src)), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

// Second and third step of a detected-only launch (the first is the store phase of k_propagate_packet).  `stage` holds the
// detected photons tile by tile in the order the tiles finished, table[b] = (offset, count) of tile b.
// k_det_scan (one CTA): exclusive prefix of the staged counts in tile order -> table[b].x becomes the tile's position in the
// caller's list (after the entries already there), table[b].y keeps the staged count, the staging offset moves to src[b];
// *n_detected grows by the TRUE number of detections.  A tile's chunk is staged only as far as the staging area reaches
// (capacity entries, like the list): an overflow therefore implies *n_detected > capacity, which is how the caller learns
// that the list is incomplete.
__global__ void __launch_bounds__(1024) k_det_scan(ulonglong2* table, unsigned long long* src, unsigned long long tiles,
                                                   unsigned long long stage_capacity, unsigned long long* n_detected,
                                                   unsigned long long* stage_count) {
    __shared__ unsigned long long s_warp[32];
    __shared__ unsigned long long s_run;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_run = 0ull;
    __syncthreads();
    const unsigned long long list_base = *n_detected;
    for (unsigned long long b0 = 0; b0 < tiles; b0 += 1024) {
        const unsigned long long b = b0 + threadIdx.x;
        ulonglong2 e = make_ulonglong2(0ull, 0ull);
        if (b < tiles) e = table[b];
        const unsigned long long staged = e.x >= stage_capacity ? 0ull : (e.x + e.y > stage_capacity ? stage_capacity - e.x : e.y);
        unsigned long long inc = staged;
        for (int o2 = 1; o2 < 32; o2 <<= 1) { const unsigned long long y = __shfl_up_sync(0xffffffffu, inc, o2); if (lane >= o2) inc += y; }
        if (lane == 31) s_warp[w] = inc;
        __syncthreads();
        unsigned long long before = s_run;
        for (int k = 0; k < w; ++k) before += s_warp[k];
        if (b < tiles) { src[b] = e.x; table[b] = make_ulonglong2(list_base + before + inc - staged, staged); }
        __syncthreads();
        if (threadIdx.x == 1023) s_run = before + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) { *n_detected = list_base + *stage_count; *stage_count = 0ull; }
}

// One warp per tile: copies the tile's staged chunk to its place in the caller's list (entries beyond the capacity dropped).
__global__ void __launch_bounds__(256) k_det_gather(const ulonglong2* __restrict__ table, const unsigned long long* __restrict__ src,
                                                    unsigned long long tiles, DetOut stage, DetOut out) {
    const unsigned long long b = (blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x) >> 5;
    if (b >= tiles) return;
    const int lane = threadIdx.x & 31;
    const ulonglong2 e = table[b];
    const unsigned long long from = src[b];
    for (unsigned long long k = lane; k < e.y; k += 32) {
        const unsigned long long r = e.x + k, q = from + k;
        if (r >= out.capacity) break;
        out.id[r] = stage.id[q]; out.pixel[r] = stage.pixel[q];
        out.pos[3 * r] = stage.pos[3 * q]; out.pos[3 * r + 1] = stage.pos[3 * q + 1]; out.pos[3 * r + 2] = stage.pos[3 * q + 2];
        out.dir[3 * r] = stage.dir[3 * q]; out.dir[3 * r + 1] = stage.dir[3 * q + 1]; out.dir[3 * r + 2] = stage.dir[3 * q + 2];
    }
}

// Octahedral map of a direction to [-1,1]^2 (NaN-safe: garbage maps to 0,0).
__device__ __forceinline__ void octa(float dx, float dy, float dz, float& u, float& v) {
    const float s = fabsf(dx) + fabsf(dy) + fabsf(dz);
    const float inv = (s > 0.f && s < kInf) ? 1.f / s : 0.f;
    u = dx * inv; v = dy * inv;
    if (dz < 0.f) {
        const float uu = (1.f - fabsf(v)) * (u >= 0.f ? 1.f : -1.f), vv = (1.f - fabsf(u)) * (v >= 0.f ? 1.f : -1.f);
        u = uu; v = vv;
    }
    if (!(fabsf(u) <= 1.f)) u = 0.f;
    if (!(fabsf(v) <= 1.f)) v = 0.f;
}

template <int kPktThreads, int kItems>
__device__ __forceinline__ void block_sum3(PacketSmemT<kPktThreads, kItems>& sm, float x, float y, float z, float& sx, float& sy, float& sz) {
    constexpr int kPktWarps = kPktThreads / 32;
    for (int off = 16; off > 0; off >>= 1) {
        x += __shfl_xor_sync(0xffffffffu, x, off); y += __shfl_xor_sync(0xffffffffu, y, off); z += __shfl_xor_sync(0xffffffffu, z, off);
    }
    if ((threadIdx.x & 31) == 0) { sm.red[threadIdx.x >> 5][0] = x; sm.red[threadIdx.x >> 5][1] = y; sm.red[threadIdx.x >> 5][2] = z; }
    __syncthreads();
    if (threadIdx.x < 3) {
        float r = 0.f;
        for (int w = 0; w < kPktWarps; ++w) r += sm.red[w][threadIdx.x];
        sm.bcast[threadIdx.x] = r;
    }
    __syncthreads();
    sx = sm.bcast[0]; sy = sm.bcast[1]; sz = sm.bcast[2];
}

// One stable radix pass (kRadixBits bits) src -> dst over kTile packed keys.  Warp w owns the
// 32*kItems consecutive entries [w*32*kItems, ...) and ranks them in kItems rounds with
// per-bit ballots; the kRadix x kPktWarps counters are scanned in (digit, warp) order.
template <int kPktThreads, int kItems>
__device__ __forceinline__ void smem_radix_pass(PacketSmemT<kPktThreads, kItems>& sm, const uint32_t* src, uint32_t* dst, int shift) {
    constexpr int kPktWarps = kPktThreads / 32;
    constexpr int kCnt = kRadix * kPktWarps, kPer = kCnt / kPktThreads;   // 1024 counters, 2 per thread
    static_assert(kCnt % kPktThreads == 0, "counter scan layout");
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t* cnt = &sm.cnt[0][0];
#pragma unroll
    for (int k = 0; k < kPer; ++k) cnt[k * kPktThreads + threadIdx.x] = 0;
    __syncthreads();
    uint32_t val[kItems], off[kItems];
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
        val[r] = src[w * (32 * kItems) + r * 32 + lane];
        const uint32_t dgt = (val[r] >> shift) & (kRadix - 1);
        // lanes with the same digit, from one ballot per digit bit (measured faster than __match_any_sync, whose latency
        // grows with the number of distinct values: here nearly 32 of them)
        uint32_t peers = 0xffffffffu;
#pragma unroll
        for (int b = 0; b < kRadixBits; ++b) {
            const bool bit = (dgt >> b) & 1u;
            const uint32_t bal = __ballot_sync(0xffffffffu, bit);
            peers &= bit ? bal : ~bal;
        }
        const int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (lane == leader) { old = sm.cnt[dgt][w]; sm.cnt[dgt][w] = old + __popc(peers); }
        old = __shfl_sync(0xffffffffu, old, leader);
        off[r] = old + __popc(peers & ((1u << lane) - 1u));
        __syncwarp();
    }
    __syncthreads();
    {   // exclusive scan: thread t owns counters [t*kPer, t*kPer + kPer)
        uint32_t c[kPer], sum = 0;
#pragma unroll
        for (int k = 0; k < kPer; ++k) { c[k] = cnt[threadIdx.x * kPer + k]; sum += c[k]; }
        uint32_t inc = sum;
        for (int o2 = 1; o2 < 32; o2 <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o2); if (lane >= o2) inc += y; }
        if (lane == 31) sm.scan_tot[w] = inc;
        __syncthreads();
        uint32_t run = inc - sum;
        for (int k = 0; k < w; ++k) run += sm.scan_tot[k];
#pragma unroll
        for (int k = 0; k < kPer; ++k) { cnt[threadIdx.x * kPer + k] = run; run += c[k]; }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kItems; ++r) dst[sm.cnt[(val[r] >> shift) & (kRadix - 1)][w] + off[r]] = val[r];
    __syncthreads();
}

// Closest hit of 32 rays walked as one packet.  `alive` lanes carry a ray; the others follow along
// without ever hitting anything.  All control flow is warp-uniform.  kOct = 0..7: every alive lane's
// direction lies in that sign octant (specialised slab test); kOct = 8: mixed signs (generic test).
struct PacketStack { int stk = 0, sp = 0; };   // stk: entry `lane` of the warp's stack (entries >= 32 in shared memory)

constexpr int kDone = 0x7fffffff;

// Walks internal nodes from `ref` until the packet reaches a leaf (returns its ref < 0) or the
// traversal is finished (returns kDone).  This small loop is the only code specialised per octant.
// kOct = 9: generic test with per-ray slack `e` (some lane's origin lies beyond SceneDev::origin_limit).
template <int kOct>
__device__ __forceinline__ int descend(const SceneDev& sc, const Slab& sl, float e, float tcap, int ref, PacketStack& st, int lane, int* s_stack) {
    for (;;) {
        if (ref < 0) return ref;
        const NodeDev* nd = sc.nodes + ref;
        const float4 q0 = __ldg(&nd->q0), q1 = __ldg(&nd->q1), q2 = __ldg(&nd->q2);
        const int4 q3 = __ldg(&nd->q3);
        float n0, f0, n1, f1;
        if (kOct < 8) slab2_oct<kOct>(sl, q0, q1, q2, tcap, n0, f0, n1, f1);
        else if (kOct == 8) slab2(sl, q0, q1, q2, tcap, n0, f0, n1, f1);
        else slab2_slack(sl, e, q0, q1, q2, tcap, n0, f0, n1, f1);
        const bool hit0 = n0 <= f0, hit1 = n1 <= f1;
        const unsigned b0 = __ballot_sync(0xffffffffu, hit0), b1 = __ballot_sync(0xffffffffu, hit1);
        if (b0 && b1) {
            // order by majority vote of the lanes: a lane prefers child 1 if it enters it first
            const unsigned p1 = __ballot_sync(0xffffffffu, hit1 && (!hit0 || n1 < n0));
            const bool one_first = 2 * __popc(p1) > __popc(b0 | b1);
            const int far = one_first ? q3.x : q3.y;
            if (st.sp < 32) { if (lane == st.sp) st.stk = far; } else s_stack[st.sp - 32] = far;
            ++st.sp;
            ref = one_first ? q3.y : q3.x;
            continue;
        }
        if (b0) { ref = q3.x; continue; }
        if (b1) { ref = q3.y; continue; }
        if (st.sp == 0) return kDone;
        --st.sp;
        ref = st.sp < 32 ? __shfl_sync(0xffffffffu, st.stk, st.sp) : s_stack[st.sp - 32];
    }
}

// `oct` (warp-uniform) = 0..7: every alive lane's direction lies in that sign octant; 8: mixed signs; 9: mixed signs and
// per-ray slack e (an origin beyond SceneDev::origin_limit).
__device__ __forceinline__ Hit closest_hit_packet(const SceneDev& sc, const RayR& rw, const Slab& sl, float e, float tmin, int last_j,
                                                  bool alive, int lane, int* s_stack, int oct) {
    Hit h{kInf, -1, 0x7fffffff};
    float tcap = alive ? kInf : -1.f;
    PacketStack st;
    int ref = 0;
    for (;;) {
        ref = oct == 9 ? descend<9>(sc, sl, e, tcap, ref, st, lane, s_stack) : descend<8>(sc, sl, e, tcap, ref, st, lane, s_stack);
        if (ref == kDone) break;
        consider_rot(sc, rw, ~ref, tmin, last_j, h);
        if (alive) tcap = h.t;
        if (st.sp == 0) break;
        --st.sp;
        ref = st.sp < 32 ? __shfl_sync(0xffffffffu, st.stk, st.sp) : s_stack[st.sp - 32];
    }
    return h;
}

// Closest hit of ONE ray with a private stack (the walk of opx_lane.cuh on the packet kernels' rotated triangle records): what
// the lanes of a packet do when the packet is too incoherent for a beam.  Lanes then walk different subtrees and most of the
// warp idles, but each ray's walk is ~40 dependent node visits instead of the ~1000 of a warp that visits the union of 32
// unrelated walks one node after the other -- and an incoherent packet is a matter of latency (it holds up its tile), not
// of throughput (1 packet-segment in 250 on the C4 scene).
__device__ __forceinline__ Hit closest_hit_own(const SceneDev& sc, const RayR& rr, const Slab& sl, float e, float tmin, int last_j) {
    Hit h{kInf, -1, 0x7fffffff};
    int stack_ref[kPktStack];
    float stack_t[kPktStack];
    int sp = 0, ref = 0;
    for (;;) {
        if (ref >= 0) {
            const NodeDev* nd = sc.nodes + ref;
            const float4 q0 = __ldg(&nd->q0), q1 = __ldg(&nd->q1), q2 = __ldg(&nd->q2);
            const int4 q3 = __ldg(&nd->q3);
            float n0, f0, n1, f1;
            slab2_slack(sl, e, q0, q1, q2, h.t, n0, f0, n1, f1);
            const bool hit0 = n0 <= f0, hit1 = n1 <= f1;
            if (hit0 && hit1) {
                int near = q3.x, far = q3.y;
                float tf = n1;
                if (n1 < n0) { near = q3.y; far = q3.x; tf = n0; }
                stack_ref[sp] = far; stack_t[sp] = tf; ++sp;
                ref = near;
                continue;
            }
            if (hit0) { ref = q3.x; continue; }
            if (hit1) { ref = q3.y; continue; }
        } else {
            consider_rot(sc, rr, ~ref, tmin, last_j, h);
        }
        bool found = false;
        while (sp > 0) {
            --sp;
            if (stack_t[sp] <= h.t) { ref = stack_ref[sp]; found = true; break; }
        }
        if (!found) break;
    }
    return h;
}

// The photon arrays of a tile in shared memory (inputs, then the segment in flight, then the record: section 8.3).
struct TileView { float* o; float* d; float* wl; int* surface; const uint32_t* key; uint8_t* state; uint8_t* bounces; };

// One packet: the 32 photons at sorted positions [32 gidx, 32 gidx + 32) of tile `t` (m photons; photon i of the tile is
// global photon id0 + i) are walked segment by segment until each has reached its terminal state; records replace the
// photons' segments in their shared-memory slots.  s_ref / s_tn / s_cb: the warp's traversal scratch.
template <bool kStats>
__device__ __forceinline__ void trace_packet(const SceneDev& sc, const TileView& t, int m, int gidx, uint64_t id0, uint64_t seed, bool have_wide,
                                             int lane, int* s_ref, float* s_tn, float4* s_cb, BeamStats& bstats, unsigned long long* stats) {
    const int slot = gidx * 32 + lane;
    bool alive = slot < m;
    const int i = alive ? (int)(t.key[slot] & 0xffffu) : 0;
    // Only the bounce count and the triangle just left stay in registers across the traversal: the segment
    // (origin, direction) lives in the photon's own shared-memory slot (rewritten after each reflection; nobody
    // else reads or writes that slot), wavelength and id are re-read at each interaction, and the record
    // replaces the segment in the slot the moment the photon terminates.
    const float* so = t.o + 3 * i;
    const float* sd = t.d + 3 * i;
    uint32_t nb = 0;
    int last = -1, last_j = -1;      // the triangle just left: global id (the record's) and leaf-order index (the walk's)
    while (__any_sync(0xffffffffu, alive)) {
        const float tmin = nb == 0 ? 0.f : sc.t_min;
        Hit h;
        RayR rw;
        bool done = false;
        {
            const float ox = so[0], oy = so[1], oz = so[2], dx = sd[0], dy = sd[1], dz = sd[2];
            rw = ray_setup_rot(so, sd, sc.n_tri);
            Beam bm;
            float s;
            const unsigned tris_before = bstats.tris, visits_before = bstats.visits;
            if (have_wide && beam_setup(sc, ox, oy, oz, dx, dy, dz, tmin, alive, bm, s)) {     // coherent packet: one beam through the 32-wide tree
                done = bm.mixed ? closest_hit_beam<true, kStats>(sc, rw, bm, s, tmin, last_j, alive, lane, so, sd, s_ref, s_tn, s_cb, h, bstats)
                                : closest_hit_beam<false, kStats>(sc, rw, bm, s, tmin, last_j, alive, lane, so, sd, s_ref, s_tn, s_cb, h, bstats);
                if (kStats && done) {
                    ++bstats.beam_segments;
                    const unsigned dt = bstats.tris - tris_before, dv = bstats.visits - visits_before;
                    const int bucket = min(15, 32 - __clz(dt));
                    const int bb = min(3, (int)__shfl_sync(0xffffffffu, nb, __ffs(__ballot_sync(0xffffffffu, alive)) - 1));
                    if (lane == 0) {
                        atomicAdd(&stats[8 + bucket], 1ull); atomicAdd(&stats[24 + bucket], (unsigned long long)dt);
                        atomicAdd(&stats[40 + bb], 1ull); atomicAdd(&stats[44 + bb], (unsigned long long)dt);
                        atomicAdd(&stats[48 + bb], (unsigned long long)dv);
                    }
                }
            }
        }
        if (!done) {
            if (kStats) ++bstats.fallback_segments;
            const float ox = so[0], oy = so[1], oz = so[2], dx = sd[0], dy = sd[1], dz = sd[2];
            const Slab sl = slab_setup(ox, oy, oz, dx, dy, dz);
            // every box is widened by the ray's own rounding slack, which matters for an origin beyond origin_limit only (8.2)
            const float far_o = fmaxf(fmaxf(fabsf(ox), fabsf(oy)), fabsf(oz));
            if (sc.flags & kFlagPacketWalk) {            // debug (opx_propagate_binary): the warp walks the binary tree as one packet
                const bool far = __any_sync(0xffffffffu, alive && !(far_o < sc.origin_limit));
                h = closest_hit_packet(sc, rw, sl, far_o * 9.5367431640625e-7f, tmin, last_j, alive, lane, s_ref, far ? 9 : 8);
            } else {
                h = Hit{kInf, -1, 0x7fffffff};
                if (alive) h = closest_hit_own(sc, rw, sl, far_o * 9.5367431640625e-7f, tmin, last_j);
            }
        }
        if (alive) {
            Photon p;
            photon_init(p, so[0], so[1], so[2], sd[0], sd[1], sd[2], t.wl[i], id0 + (uint64_t)i);
            p.b = nb; p.last = last;
            alive = interact(sc, h, rw, p, seed);
            t.d[3 * i] = p.dx; t.d[3 * i + 1] = p.dy; t.d[3 * i + 2] = p.dz;
            if (alive) {
                t.o[3 * i] = p.ox; t.o[3 * i + 1] = p.oy; t.o[3 * i + 2] = p.oz;
                nb = p.b; last = p.last; last_j = h.j;
            } else {
                t.o[3 * i] = p.px; t.o[3 * i + 1] = p.py; t.o[3 * i + 2] = p.pz;
                t.wl[i] = __int_as_float(p.pixel);
                t.surface[i] = p.surface;
                t.state[i] = (uint8_t)p.state; t.bounces[i] = (uint8_t)p.b;
            }
        }
    }
}

template <int kPktThreads, int kItems, int kPktCtas, bool kStats>
__global__ void __launch_bounds__(kPktThreads, kPktCtas) k_propagate_packet(const SceneDev sc, uint64_t n, uint64_t id_base,
                                                                     const float* __restrict__ origins,
                                                                     const float* __restrict__ dirs,
                                                                     const float* __restrict__ wl, uint64_t seed, opx_hits out,
                                                                     uint32_t* hitmap, unsigned long long* counters,
                                                                     unsigned long long* stats, const DetOut det, uint32_t tile_stride) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using PacketSmem = PacketSmemT<kPktThreads, kItems>;
    constexpr int kPktWarps = PacketSmem::kPktWarps, kTile = PacketSmem::kTile;
    PacketSmem& sm = *reinterpret_cast<PacketSmem*>(smem_raw);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    // opaque to the compiler from here on: it otherwise re-derives both (and every shared-memory address built on them) from
    // the thread id inside the node and cull loops -- S2R + shifts + address arithmetic at every node -- to save two registers
    asm volatile("" : "+r"(lane), "+r"(w));
    // photons per tile: kTile, or fewer (a multiple of 32) when a small call is spread over all SMs (launch_propagate)
    const uint32_t stride = tile_stride ? tile_stride : (uint32_t)kTile;
    const uint64_t tile_base = (uint64_t)blockIdx.x * stride;
    if (sc.d_n) n = min(n, (uint64_t)__ldg(sc.d_n));       // photon count left on the device by opx_prefilter
    if (tile_base >= n) return;
    const int m = (int)min((uint64_t)stride, n - tile_base);
    if (threadIdx.x == 0) sm.next_group = 0;

    // 1. stage the tile (read once).  A full tile whose three input blocks are 16-byte aligned is fetched by three TMA bulk
    //    copies issued by one thread; anything else (the ragged last tile, odd slices) by coalesced streaming loads.
    const bool bulk_in = m == kTile && aligned16(origins + 3 * tile_base) && aligned16(dirs + 3 * tile_base) && aligned16(wl + tile_base);
    if (bulk_in) {
        if (threadIdx.x == 0) mbar_init(&sm.mbar, 1);
        __syncthreads();
        if (threadIdx.x == 0) {
            const uint64_t pol = l2_evict_first();
            mbar_expect_tx(&sm.mbar, (uint32_t)(kTile * 28));
            bulk_g2s(sm.o, origins + 3 * tile_base, kTile * 12, &sm.mbar, pol);
            bulk_g2s(sm.d, dirs + 3 * tile_base, kTile * 12, &sm.mbar, pol);
            bulk_g2s(sm.wl, wl + tile_base, kTile * 4, &sm.mbar, pol);
        }
        mbar_wait(&sm.mbar, 0);
    } else {
        for (int k = threadIdx.x; k < 3 * m; k += kPktThreads) {
            sm.o[k] = __ldcs(origins + 3 * tile_base + k);
            sm.d[k] = __ldcs(dirs + 3 * tile_base + k);
        }
        for (int k = threadIdx.x; k < m; k += kPktThreads) sm.wl[k] = __ldcs(wl + tile_base + k);
        __syncthreads();
    }

    // 2. sort key: (run of the tile the photon belongs to, 10-bit pseudo-angle of its direction about
    //    the run's mean direction in the octahedral plane).  A run is a stretch of consecutive photons
    //    without a jump of the origin (> 16 x the tile's mean jump): photons arrive in generation order,
    //    so a jump is where the next charged track starts, and its cone has a different axis.
    {
        float u[kItems], v[kItems], jump[kItems];
        float su = 0.f, sv = 0.f, sj = 0.f;
#pragma unroll
        for (int r = 0; r < kItems; ++r) {
            const int i = r * kPktThreads + threadIdx.x;
            u[r] = 0.f; v[r] = 0.f; jump[r] = 0.f;
            if (i < m) {
                octa(sm.d[3 * i], sm.d[3 * i + 1], sm.d[3 * i + 2], u[r], v[r]); su += u[r]; sv += v[r];
                if (i > 0) {
                    const float j = fmaxf(fmaxf(fabsf(sm.o[3 * i] - sm.o[3 * i - 3]), fabsf(sm.o[3 * i + 1] - sm.o[3 * i - 2])),
                                          fabsf(sm.o[3 * i + 2] - sm.o[3 * i - 1]));
                    if (j < kInf) { jump[r] = j; sj += j; }
                }
            }
        }
        float cu, cv, cj;
        block_sum3(sm, su, sv, sj, cu, cv, cj);
        const float thr = 16.f * cj / (float)m;
        bool flag[kItems];
        bool any = false;
#pragma unroll
        for (int r = 0; r < kItems; ++r) { flag[r] = jump[r] > thr; any |= flag[r]; }
        uint32_t run[kItems] = {};
        float cur[kItems], cvr[kItems];
#pragma unroll
        for (int r = 0; r < kItems; ++r) { cur[r] = cu / (float)m; cvr[r] = cv / (float)m; }
        if (__syncthreads_or(any)) {      // rare: the tile holds photons of more than one track
            uint32_t* chunk = &sm.cnt[0][0];                       // kItems x kPktWarps jump counts, in tile order
            float* rs = reinterpret_cast<float*>(chunk + kItems * kPktWarps);      // 4 runs x (sum u, sum v, count)
            unsigned bal[kItems];
#pragma unroll
            for (int r = 0; r < kItems; ++r) {
                bal[r] = __ballot_sync(0xffffffffu, flag[r]);
                if (lane == 0) chunk[r * kPktWarps + w] = __popc(bal[r]);
            }
            if (threadIdx.x < 12) rs[threadIdx.x] = 0.f;
            __syncthreads();
            {   // exclusive prefix of the kItems x kPktWarps (<= 128) jump counts, once, by warp 0
                constexpr int kC = kItems * kPktWarps;
                static_assert(kC <= 128, "four chunk counts per lane of warp 0");
                if (w == 0) {
                    uint32_t c4[4], sum = 0;
#pragma unroll
                    for (int k = 0; k < 4; ++k) { c4[k] = 4 * lane + k < kC ? chunk[4 * lane + k] : 0u; sum += c4[k]; }
                    uint32_t inc = sum;
                    for (int o2 = 1; o2 < 32; o2 <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o2); if (lane >= o2) inc += y; }
                    uint32_t runsum = inc - sum;
#pragma unroll
                    for (int k = 0; k < 4; ++k) { if (4 * lane + k < kC) chunk[4 * lane + k] = runsum; runsum += c4[k]; }
                }
                __syncthreads();
            }
#pragma unroll
            for (int r = 0; r < kItems; ++r) {
                const uint32_t before = chunk[r * kPktWarps + w];
                run[r] = min(3u, before + __popc(bal[r] & (0xffffffffu >> (31 - lane))));
                // sums per run.  A warp's 32 photons are consecutive, so all but the warps that hold a track boundary belong to one
                // run: those add once per warp (2048 threads adding floats to three words one by one serialise on a
                // compare-and-swap loop)
                const bool in = r * kPktThreads + (int)threadIdx.x < m;
                const uint32_t run0 = __shfl_sync(0xffffffffu, run[r], 0);
                if (__all_sync(0xffffffffu, run[r] == run0)) {
                    float a = in ? u[r] : 0.f, b = in ? v[r] : 0.f, c = in ? 1.f : 0.f;
                    for (int off = 16; off > 0; off >>= 1) {
                        a += __shfl_xor_sync(0xffffffffu, a, off); b += __shfl_xor_sync(0xffffffffu, b, off); c += __shfl_xor_sync(0xffffffffu, c, off);
                    }
                    if (lane == 0) { atomicAdd(&rs[3 * run0], a); atomicAdd(&rs[3 * run0 + 1], b); atomicAdd(&rs[3 * run0 + 2], c); }
                } else if (in) {
                    atomicAdd(&rs[3 * run[r]], u[r]); atomicAdd(&rs[3 * run[r] + 1], v[r]); atomicAdd(&rs[3 * run[r] + 2], 1.f);
                }
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < kItems; ++r) {
                const float cnt = fmaxf(rs[3 * run[r] + 2], 1.f);
                cur[r] = rs[3 * run[r]] / cnt; cvr[r] = rs[3 * run[r] + 1] / cnt;
            }
            __syncthreads();
        }
#pragma unroll
        for (int r = 0; r < kItems; ++r) {
            const int i = r * kPktThreads + threadIdx.x;
            uint32_t key = 0xfffu;
            if (i < m) {
                const float du = u[r] - cur[r], dv = v[r] - cvr[r];
                const float a = fabsf(du) + fabsf(dv);
                const float pp = a > 0.f ? dv / a : 0.f;                     // diamond angle in [0,4)
                const float ang = du >= 0.f ? (dv >= 0.f ? pp : 4.f + pp) : 2.f - pp;
                key = (run[r] << 10) | min(1023u, (uint32_t)(ang * 256.f));
            }
            sm.key[i] = (key << 16) | (uint32_t)i;
        }
        __syncthreads();
        uint32_t* alt = reinterpret_cast<uint32_t*>(sm.surface);
        smem_radix_pass(sm, sm.key, alt, 16);
        smem_radix_pass(sm, alt, sm.key, 22);
    }

    const bool have_wide = sc.n_wnodes && __ldg(sc.wide_count) != 0u;      // the build's verdict on the 32-wide tree (warp-uniform)
    // 3. each warp takes groups of 32 neighbouring photons and walks them as a packet
    //    (groups are handed out dynamically so that a slow packet does not hold up its warp's share)
    const int groups = (m + 31) >> 5;
    BeamStats bstats;
    const TileView tv{sm.o, sm.d, sm.wl, sm.surface, sm.key, sm.state, sm.bounces};
    for (;;) {
        int gidx = 0;
        if (lane == 0) gidx = atomicAdd(&sm.next_group, 1);
        gidx = __shfl_sync(0xffffffffu, gidx, 0);
        if (gidx >= groups) break;
        trace_packet<kStats>(sc, tv, m, gidx, id_base + tile_base, seed, have_wide, lane, sm.stack[w], sm.beam_tn[w], sm.cull[w], bstats, stats);
    }
    __syncthreads();
    if (kStats) {
        if (lane == 0) {
            atomicAdd(&stats[0], (unsigned long long)bstats.beam_segments); atomicAdd(&stats[1], (unsigned long long)bstats.fallback_segments);
            atomicAdd(&stats[2], (unsigned long long)bstats.visits); atomicAdd(&stats[3], (unsigned long long)bstats.tris);
            atomicAdd(&stats[4], (unsigned long long)bstats.overflows); atomicAdd(&stats[5], (unsigned long long)bstats.culls);
            atomicAdd(&stats[6], (unsigned long long)bstats.cands); atomicAdd(&stats[7], (unsigned long long)bstats.pairs);
        }
    }

    // 4a. A11 + A12 for this tile, straight from shared memory (what k_bin does for the other kernels).  Integer adds only.
    if (hitmap || counters) {
        uint32_t* s_cnt = sm.scan_tot;                       // 8 of its kPktWarps words; free since the sort
        if (threadIdx.x < 8) s_cnt[threadIdx.x] = 0;
        __syncthreads();
        unsigned seg = 0, acc = 0;                           // acc: seven 4-bit per-state counts of this thread (<= kItems each)
        static_assert(kItems <= 7, "4-bit state counts per thread, 8-bit per warp");
        for (int k = threadIdx.x; k < kTile; k += kPktThreads) {           // uniform trip count: warp collectives inside
            const bool ok = k < m;
            const int st = ok ? (int)sm.state[k] : 7;
            if (ok) { seg += (unsigned)sm.bounces[k] + (st != OPX_BOUNCE_LIMIT ? 1u : 0u); acc += 1u << (4 * st); }
            if (hitmap) {
                // one atomic per detected photon, except when all detected photons of the warp share a pixel (a focused spot:
                // the case that would serialise on one address), which costs one atomic per warp.  A full __match_any_sync
                // merge of equal pixels was measured at 3 % of the kernel on C2, where a ring spreads over ~700 pixels.
                const bool det = st == OPX_DETECTED;
                const unsigned dm = __ballot_sync(0xffffffffu, det);
                if (dm) {
                    const int pix = det ? __float_as_int(sm.wl[k]) : 0;
                    const int lead = __ffs(dm) - 1;
                    const int first = __shfl_sync(0xffffffffu, pix, lead);
                    const unsigned same = __ballot_sync(0xffffffffu, det && pix == first);
                    if (same == dm) { if (lane == lead) atomicAdd(&hitmap[first], (unsigned)__popc(dm)); }
                    else if (det) atomicAdd(&hitmap[pix], 1u);
                }
            }
        }
        if (counters) {
            // widen the 4-bit fields to 8 bits (a warp sums to <= 32 * kItems = 128 per state) and add across the warp
            const unsigned lo4 = (acc & 0xfu) | ((acc & 0xf0u) << 4) | ((acc & 0xf00u) << 8) | ((acc & 0xf000u) << 12);       // states 0..3
            const unsigned hi4 = ((acc >> 16) & 0xfu) | ((acc >> 12) & 0xf00u) | ((acc >> 8) & 0xf0000u);                    // states 4..6
            const unsigned a = __reduce_add_sync(0xffffffffu, lo4), b = __reduce_add_sync(0xffffffffu, hi4);
            seg = __reduce_add_sync(0xffffffffu, seg);
            if (lane < 4) { const unsigned c = (a >> (8 * lane)) & 0xffu; if (c) atomicAdd(&s_cnt[lane], c); }
            else if (lane < 7) { const unsigned c = (b >> (8 * (lane - 4))) & 0xffu; if (c) atomicAdd(&s_cnt[lane], c); }
            else if (lane == 7 && seg) atomicAdd(&s_cnt[7], seg);
            __syncthreads();
            if (threadIdx.x < 8 && s_cnt[threadIdx.x]) atomicAdd(&counters[threadIdx.x], (unsigned long long)s_cnt[threadIdx.x]);
        }
    }

    // 4b. detected-only output (opx_propagate_detected): the tile's DETECTED photons go, in id order, to a staging list at an
    //     offset taken from a global counter (so tiles land in the order they finish and nobody waits for anybody), and the
    //     tile notes (offset, count) in a table; k_det_scan / k_det_gather then move the chunks to the caller's list in tile
    //     order = photon-id order.  (A single-pass look-back scan inside this kernel was measured first: on the C4 scene,
    //     where tile times differ by a factor of several, finished CTAs spinning for their predecessors halved the rate.)
    if (det.id) {
        constexpr int kChunks = kTile / 32;                  // <= 64: two per lane of warp 0
        static_assert(kChunks <= 64 && kTile % 32 == 0, "chunk scan layout");
        uint32_t* s_chunk = &sm.cnt[0][0];                   // free since the traversal ended (aliases the warps' stacks)
        unsigned long long* s_base = reinterpret_cast<unsigned long long*>(s_chunk + 64);
        __syncthreads();
        for (int k = threadIdx.x; k < kTile; k += kPktThreads) {
            const unsigned dm = __ballot_sync(0xffffffffu, k < m && sm.state[k] == OPX_DETECTED);
            if (lane == 0) s_chunk[k >> 5] = __popc(dm);
        }
        __syncthreads();
        if (w == 0) {
            const uint32_t c0 = 2 * lane < kChunks ? s_chunk[2 * lane] : 0u, c1 = 2 * lane + 1 < kChunks ? s_chunk[2 * lane + 1] : 0u;
            uint32_t inc = c0 + c1;
            for (int o2 = 1; o2 < 32; o2 <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o2); if (lane >= o2) inc += y; }
            const uint32_t total = __shfl_sync(0xffffffffu, inc, 31);
            if (2 * lane < kChunks) s_chunk[2 * lane] = inc - c0 - c1;
            if (2 * lane + 1 < kChunks) s_chunk[2 * lane + 1] = inc - c1;
            if (lane == 0) {
                const unsigned long long off = total ? atomicAdd(det.stage_count, (unsigned long long)total) : 0ull;
                det.tile_table[blockIdx.x] = make_ulonglong2(off, (unsigned long long)total);
                *s_base = off;
            }
        }
        __syncthreads();
        const unsigned long long base = *s_base;
        for (int k = threadIdx.x; k < kTile; k += kPktThreads) {
            const bool isdet = k < m && sm.state[k] == OPX_DETECTED;
            const unsigned dm = __ballot_sync(0xffffffffu, isdet);
            const unsigned long long r = base + s_chunk[k >> 5] + __popc(dm & ((1u << lane) - 1u));
            if (isdet && r < det.capacity) {
                det.id[r] = id_base + (det.index ? (uint64_t)__ldg(det.index + tile_base + k) : tile_base + (uint64_t)k);
                det.pixel[r] = __float_as_int(sm.wl[k]);
                det.pos[3 * r] = sm.o[3 * k]; det.pos[3 * r + 1] = sm.o[3 * k + 1]; det.pos[3 * r + 2] = sm.o[3 * k + 2];
                det.dir[3 * r] = sm.d[3 * k]; det.dir[3 * r + 1] = sm.d[3 * k + 1]; det.dir[3 * r + 2] = sm.d[3 * k + 2];
            }
        }
        return;            // a detected-only launch writes no per-photon records
    }

    // 4. write the tile's records: six TMA bulk stores by one thread for a full, aligned tile, else coalesced streaming stores
    const bool bulk_out = m == kTile && aligned16(out.pos + 3 * tile_base) && aligned16(out.dir + 3 * tile_base) &&
                          aligned16(out.pixel + tile_base) && aligned16(out.surface + tile_base) && aligned16(out.state + tile_base) &&
                          aligned16(out.bounces + tile_base);
    if (bulk_out) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // this thread's record writes -> visible to the TMA engine
        __syncthreads();
        if (threadIdx.x == 0) {
            const uint64_t pol = l2_evict_first();
            bulk_s2g(out.pos + 3 * tile_base, sm.o, kTile * 12, pol);
            bulk_s2g(out.dir + 3 * tile_base, sm.d, kTile * 12, pol);
            bulk_s2g(out.pixel + tile_base, sm.wl, kTile * 4, pol);
            bulk_s2g(out.surface + tile_base, sm.surface, kTile * 4, pol);
            bulk_s2g(out.state + tile_base, sm.state, kTile, pol);
            bulk_s2g(out.bounces + tile_base, sm.bounces, kTile, pol);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); // shared memory must outlive the reads: the CTA ends after this
        }
        return;
    }
    for (int k = threadIdx.x; k < 3 * m; k += kPktThreads) {
        __stcs(out.pos + 3 * tile_base + k, sm.o[k]);
        __stcs(out.dir + 3 * tile_base + k, sm.d[k]);
    }
    for (int k = threadIdx.x; k < m; k += kPktThreads) {
        __stcs(out.pixel + tile_base + k, __float_as_int(sm.wl[k]));
        __stcs(out.surface + tile_base + k, sm.surface[k]);
    }
    for (int k = threadIdx.x; k < m; k += kPktThreads) { out.state[tile_base + k] = sm.state[k]; out.bounces[tile_base + k] = sm.bounces[k]; }
}

}  // namespace
}  // namespace opx
