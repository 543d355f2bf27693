// A1-A4: GPU LBVH build.
//   k_bounds     scene AABB by block reduction + ordered-int atomics
//   k_morton     63-bit Morton key (21 bits/axis) of each triangle's AABB centre
//   k_radix_*    LSD radix sort of (key, triangle), 8 bits per pass, stable
//   k_pack_tris  triangles gathered into leaf (sorted) order, 3 x float4 each
//   k_hierarchy  Karras 2012: one thread per internal node, delta = clz(ki ^ kj), index tie-break
//   k_refit      padded leaf boxes, bottom-up union with per-node arrival counters
// The BVH is not part of the parity contract (the oracle has none); what is, is that traversal
// never culls a triangle the contract test of DESIGN.md 3.3 accepts -- hence the padding here.
#include <cfloat>
#include <cmath>
#include <mutex>

#include "opx_internal.cuh"

namespace opx {

namespace {

#ifndef OPX_BEAM_WIDTH
#define OPX_BEAM_WIDTH 4.f
#endif
constexpr float kBeamWidthInTriangles = OPX_BEAM_WIDTH;    // beam_max_width = this x the typical triangle size
constexpr int kSortBlock = 256;
constexpr int kSortItems = 8;
constexpr int kSortTile = kSortBlock * kSortItems;  // 2048 keys per block per pass

struct BuildTmp {
    float* tri_in;        // T x 9, global id order
    int32_t* surf_in;     // T
    float* normals_in;    // T x 3
    uint64_t* keys[2];    // ping-pong
    uint32_t* idx[2];
    uint32_t* hist;       // 256 x n_sort_blocks
    uint32_t* bounds;     // 6 ordered-int floats: min xyz, max xyz
    uint32_t* flags;      // T-1 arrival counters
    int2* queue[2];       // collapse tasks (binary node, wide node), ping-pong per level
    uint32_t* wcount;     // collapse counters: n_in, n_out, n_wide_nodes, overflow
};

__host__ __device__ inline size_t sort_blocks(size_t T) { return (T + kSortTile - 1) / kSortTile; }

// float <-> order-preserving uint32
__device__ inline uint32_t f2ord(float f) {
    const uint32_t b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ inline float ord2f(uint32_t u) {
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u);
}

__global__ void k_init_bounds(uint32_t* bounds) {
    if (threadIdx.x < 3) bounds[threadIdx.x] = 0xffffffffu;
    else if (threadIdx.x < 6) bounds[threadIdx.x] = 0u;
}

__global__ void __launch_bounds__(256) k_bounds(const float* __restrict__ tri, uint32_t T, uint32_t* bounds) {
    float lo[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, hi[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
    for (uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x; i < (uint64_t)T * 3; i += (uint64_t)gridDim.x * blockDim.x) {
        for (int c = 0; c < 3; ++c) {
            const float v = tri[3 * i + c];
            lo[c] = fminf(lo[c], v); hi[c] = fmaxf(hi[c], v);
        }
    }
    for (int c = 0; c < 3; ++c) {
        for (int off = 16; off > 0; off >>= 1) {
            lo[c] = fminf(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], off));
            hi[c] = fmaxf(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], off));
        }
    }
    if ((threadIdx.x & 31) == 0) {
        for (int c = 0; c < 3; ++c) {
            atomicMin(&bounds[c], f2ord(lo[c]));
            atomicMax(&bounds[3 + c], f2ord(hi[c]));
        }
    }
}

__device__ inline uint64_t spread21(uint32_t v) {  // 21 bits -> every third bit
    uint64_t x = v & 0x1fffffu;
    x = (x | (x << 32)) & 0x1f00000000ffffull;
    x = (x | (x << 16)) & 0x1f0000ff0000ffull;
    x = (x | (x << 8)) & 0x100f00f00f00f00full;
    x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
    x = (x | (x << 2)) & 0x1249249249249249ull;
    return x;
}

__global__ void __launch_bounds__(256) k_morton(const float* __restrict__ tri, uint32_t T, const uint32_t* __restrict__ bounds,
                                                uint64_t* keys, uint32_t* idx) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= T) return;
    uint32_t q[3];
    for (int c = 0; c < 3; ++c) {
        const float smin = ord2f(bounds[c]), smax = ord2f(bounds[3 + c]);
        const float a = tri[9 * (size_t)i + c], b = tri[9 * (size_t)i + 3 + c], d = tri[9 * (size_t)i + 6 + c];
        const float centre = 0.5f * (fminf(a, fminf(b, d)) + fmaxf(a, fmaxf(b, d)));
        const float ext = smax - smin;
        const float s = ext > 0.f ? 2097152.f / ext : 0.f;
        float f = (centre - smin) * s;
        f = fminf(fmaxf(f, 0.f), 2097151.f);
        q[c] = (uint32_t)f;
    }
    keys[i] = (spread21(q[0]) << 2) | (spread21(q[1]) << 1) | spread21(q[2]);
    idx[i] = i;
}

// ------------------------------------------------------------------------------------ radix sort
__global__ void __launch_bounds__(kSortBlock) k_radix_hist(const uint64_t* __restrict__ keys, uint32_t T, int shift,
                                                           uint32_t* hist, uint32_t n_blocks) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * kSortTile;
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t i = base + r * kSortBlock + threadIdx.x;
        if (i < T) atomicAdd(&h[(uint32_t)(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * n_blocks + blockIdx.x] = h[threadIdx.x];
}

// One block of 32 warps: exclusive scan of hist[digit][block] in (digit, block) order.  A warp owns 8 digits; its lanes stride
// over the blocks (coalesced) and scan them 32 at a time.
__global__ void __launch_bounds__(1024) k_radix_scan(uint32_t* hist, uint32_t n_blocks) {
    __shared__ uint32_t tot[256];
    const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (uint32_t d = w; d < 256; d += 32) {
        uint32_t sum = 0;
        for (uint32_t b = lane; b < n_blocks; b += 32) sum += hist[(size_t)d * n_blocks + b];
        sum = __reduce_add_sync(0xffffffffu, sum);
        if (lane == 0) tot[d] = sum;
    }
    __syncthreads();
    if (w == 0) {      // exclusive scan of the 256 digit totals: 8 per lane
        uint32_t c[8], sum = 0;
        for (int k = 0; k < 8; ++k) { c[k] = tot[8 * lane + k]; sum += c[k]; }
        uint32_t inc = sum;
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (uint32_t)o) inc += y; }
        uint32_t run = inc - sum;
        for (int k = 0; k < 8; ++k) { tot[8 * lane + k] = run; run += c[k]; }
    }
    __syncthreads();
    for (uint32_t d = w; d < 256; d += 32) {
        uint32_t run = tot[d];
        for (uint32_t b0 = 0; b0 < n_blocks; b0 += 32) {
            const uint32_t b = b0 + lane;
            const uint32_t t = b < n_blocks ? hist[(size_t)d * n_blocks + b] : 0u;
            uint32_t inc = t;
            for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= (uint32_t)o) inc += y; }
            if (b < n_blocks) hist[(size_t)d * n_blocks + b] = run + inc - t;
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
}

// Stable scatter.  Warp w of the block owns the 256 consecutive keys [tile + 256 w, tile + 256 w + 256)
// and ranks them in 8 rounds of 32 with __match_any_sync; warps are ordered by a per-digit scan.
__global__ void __launch_bounds__(kSortBlock) k_radix_scatter(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ idx_in,
                                                              uint64_t* keys_out, uint32_t* idx_out, uint32_t T, int shift,
                                                              const uint32_t* __restrict__ hist, uint32_t n_blocks) {
    constexpr int kWarps = kSortBlock / 32;
    __shared__ uint32_t cnt[kWarps][256];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int k = threadIdx.x; k < kWarps * 256; k += kSortBlock) (&cnt[0][0])[k] = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * kSortTile + w * (32 * kSortItems);
    uint64_t key[kSortItems];
    uint32_t val[kSortItems], off[kSortItems];
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t i = base + r * 32 + lane;
        const bool ok = i < T;
        key[r] = ok ? keys_in[i] : 0;
        val[r] = ok ? idx_in[i] : 0;
        const uint32_t dgt = ok ? ((uint32_t)(key[r] >> shift) & 255u) : 0xffffffffu;
        const uint32_t peers = __match_any_sync(0xffffffffu, dgt);
        const int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (ok && lane == leader) { old = cnt[w][dgt]; cnt[w][dgt] = old + __popc(peers); }
        old = __shfl_sync(0xffffffffu, old, leader);
        off[r] = old + __popc(peers & ((1u << lane) - 1u));
        __syncwarp();
    }
    __syncthreads();
    {   // thread d: exclusive scan over warps of cnt[*][d], plus the block's global offset for digit d
        const uint32_t d = threadIdx.x;
        uint32_t run = hist[(size_t)d * n_blocks + blockIdx.x];
        for (int k = 0; k < kWarps; ++k) { const uint32_t t = cnt[k][d]; cnt[k][d] = run; run += t; }
    }
    __syncthreads();
    for (int r = 0; r < kSortItems; ++r) {
        const uint32_t i = base + r * 32 + lane;
        if (i < T) {
            const uint32_t dgt = (uint32_t)(key[r] >> shift) & 255u;
            const uint32_t dst = cnt[w][dgt] + off[r];
            keys_out[dst] = key[r];
            idx_out[dst] = val[r];
        }
    }
}

// --------------------------------------------------------------------------------- pack triangles
__global__ void __launch_bounds__(256) k_pack_tris(const float* __restrict__ tri, const int32_t* __restrict__ surf,
                                                   const float* __restrict__ nrm, const uint32_t* __restrict__ idx,
                                                   uint32_t T, float4* tris_out, float4* normals_out) {
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= T) return;
    const uint32_t g = idx[j];
    const float* v = tri + 9 * (size_t)g;
    const int32_t s = surf[g];
    // three rotations of the record, one array after the other (SceneDev::tris): (x, y, z), (y, z, x), (z, x, y)
    for (uint32_t r = 0; r < 3; ++r) {
        float4* o = tris_out + 3 * ((size_t)r * T + j);
        const uint32_t c0 = r, c1 = (r + 1) % 3, c2 = (r + 2) % 3;
        o[0] = make_float4(v[c0], v[c1], v[c2], __int_as_float((int)g));
        o[1] = make_float4(v[3 + c0], v[3 + c1], v[3 + c2], __int_as_float(s));
        o[2] = make_float4(v[6 + c0], v[6 + c1], v[6 + c2], 0.f);
    }
    normals_out[j] = make_float4(nrm[3 * (size_t)g], nrm[3 * (size_t)g + 1], nrm[3 * (size_t)g + 2], __int_as_float(s));
}

// ------------------------------------------------------------------------------- Karras hierarchy
__device__ inline int delta(const uint64_t* __restrict__ keys, int T, int i, int j) {
    if (j < 0 || j >= T) return -1;
    const uint64_t a = keys[i], b = keys[j];
    if (a != b) return __clzll((long long)(a ^ b));
    return 64 + __clz(i ^ j);      // equal keys: fall back to the index so that the tree stays balanced
}

__global__ void __launch_bounds__(256) k_hierarchy(const uint64_t* __restrict__ keys, int T, NodeDev* nodes, int* parents) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= T - 1) return;
    const int d = (delta(keys, T, i, i + 1) - delta(keys, T, i, i - 1)) >= 0 ? 1 : -1;
    const int dmin = delta(keys, T, i, i - d);
    int lmax = 2;
    while (delta(keys, T, i, i + lmax * d) > dmin) lmax <<= 1;
    int l = 0;
    for (int t = lmax >> 1; t >= 1; t >>= 1)
        if (delta(keys, T, i, i + (l + t) * d) > dmin) l += t;
    const int j = i + l * d;
    const int dnode = delta(keys, T, i, j);
    int s = 0;
    for (int t = (l + 1) >> 1;; t = (t + 1) >> 1) {
        if (delta(keys, T, i, i + (s + t) * d) > dnode) s += t;
        if (t == 1) break;
    }
    const int gamma = i + s * d + min(d, 0);
    const int lo = min(i, j), hi = max(i, j);
    const int left = (lo == gamma) ? ~gamma : gamma;
    const int right = (hi == gamma + 1) ? ~(gamma + 1) : gamma + 1;
    nodes[i].q3 = make_int4(left, right, l + 1, 0);      // .z: leaves below this node
    parents[left >= 0 ? left : (T - 1 + ~left)] = i;
    parents[right >= 0 ? right : (T - 1 + ~right)] = i;
    if (i == 0) parents[0] = -1;
}

// -------------------------------------------------------------------------------------- refit
__device__ inline void store_child_box(NodeDev* node, int slot, const float lo[3], const float hi[3]) {
    float* f = reinterpret_cast<float*>(node);
    float* p = f + slot * 6;      // slot 0: floats 0..5, slot 1: floats 6..11 (lo.xyz, hi.xyz)
    p[0] = lo[0]; p[1] = lo[1]; p[2] = lo[2]; p[3] = hi[0]; p[4] = hi[1]; p[5] = hi[2];
}

__global__ void __launch_bounds__(256) k_refit(const float4* __restrict__ tris, int T, float pad, NodeDev* nodes,
                                               const int* __restrict__ parents, uint32_t* flags) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= T) return;
    const float4 a = tris[3 * (size_t)j], b = tris[3 * (size_t)j + 1], c = tris[3 * (size_t)j + 2];
    float lo[3] = {fminf(a.x, fminf(b.x, c.x)), fminf(a.y, fminf(b.y, c.y)), fminf(a.z, fminf(b.z, c.z))};
    float hi[3] = {fmaxf(a.x, fmaxf(b.x, c.x)), fmaxf(a.y, fmaxf(b.y, c.y)), fmaxf(a.z, fmaxf(b.z, c.z))};
    // padding: `pad` = 2^-16 of the largest scene coordinate covers the rounding of vertex - origin, of the
    // shear and of the slab arithmetic; 2^-10 of the triangle's own extent covers the one error that grows with the
    // triangle: at grazing incidence the contract's barycentric weights lose accuracy and the hit point o + t d can sit
    // up to sqrt(3 x 2^-23) = 6e-4 of the triangle's size off its plane
    pad += 9.765625e-4f * fmaxf(hi[0] - lo[0], fmaxf(hi[1] - lo[1], hi[2] - lo[2]));
    for (int k = 0; k < 3; ++k) { lo[k] -= pad; hi[k] += pad; }
    int child = ~j;
    int p = parents[T - 1 + j];
    while (p >= 0) {
        NodeDev* node = nodes + p;
        const int slot = (node->q3.x == child) ? 0 : 1;
        store_child_box(node, slot, lo, hi);
        __threadfence();
        if (atomicAdd(&flags[p], 1u) == 0u) return;       // first to arrive: the sibling finishes the job
        const volatile float* o = reinterpret_cast<const volatile float*>(node) + (1 - slot) * 6;
        for (int k = 0; k < 3; ++k) { lo[k] = fminf(lo[k], o[k]); hi[k] = fmaxf(hi[k], o[3 + k]); }
        child = p;
        p = parents[p];
    }
}

// ------------------------------------------------------------------- collapse to the 32-wide tree
// One warp per wide node, one launch per level.  A task (b, w) turns the binary subtree rooted at b
// into wide node w: lane k holds child k; the child with the largest box (among those with more
// than 32 leaves -- smaller subtrees become full bottom nodes later) is replaced by its two
// children until 32 slots are used; then the smallest remaining subtrees are expanded all the way to
// their triangles while they fit.  Children that are still binary subtrees become tasks of the next
// level.  A subtree of at most 32 leaves expands completely into triangle children.
struct WEntry { int ref; int cnt; float lo[3], hi[3]; };

__device__ inline void take_child(const NodeDev* __restrict__ bn, int node, int slot, WEntry& e) {
    const NodeDev* nd = bn + node;
    const float* f = reinterpret_cast<const float*>(nd) + slot * 6;
    e.lo[0] = f[0]; e.lo[1] = f[1]; e.lo[2] = f[2]; e.hi[0] = f[3]; e.hi[1] = f[4]; e.hi[2] = f[5];
    e.ref = slot == 0 ? nd->q3.x : nd->q3.y;
    e.cnt = e.ref >= 0 ? bn[e.ref].q3.z : 1;
}

__device__ __forceinline__ void collapse_level(const NodeDev* __restrict__ bn, const int2* q_in, uint32_t n_in, int2* q_out, uint32_t* n_out,
                                               WNodeDev* wn, uint32_t* n_wn, uint32_t cap_wn, uint32_t* overflow) {
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const uint32_t warps = gridDim.x * (blockDim.x >> 5);
    for (uint32_t task = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); task < n_in; task += warps) {
        const int2 tk = __ldcg(&q_in[task]);      // written by other SMs one level earlier: not through L1
        const int b = tk.x, w = tk.y;
        WEntry e; e.ref = 0x7fffffff; e.cnt = 0;
        bool valid = false;
        if (lane < 2) { take_child(bn, b, lane, e); valid = true; }
        const bool bottom = bn[b].q3.z <= kWide;
        int count = 2;
        while (count < kWide) {
            uint32_t key = 0;
            if (valid && e.ref >= 0 && e.ref != 0x7fffffff && (bottom || e.cnt > kWide)) {
                const float ex = e.hi[0] - e.lo[0], ey = e.hi[1] - e.lo[1], ez = e.hi[2] - e.lo[2];
                key = __float_as_uint(fmaxf(ex * ey + ey * ez + ez * ex, 0.f)) + 1u;
            }
            const uint32_t best = __reduce_max_sync(full, key);
            if (best == 0) break;
            const int L = __ffs(__ballot_sync(full, key == best)) - 1;
            const int r = __shfl_sync(full, e.ref, L);
            if (lane == L) take_child(bn, r, 0, e);
            if (lane == count) { take_child(bn, r, 1, e); valid = true; }
            ++count;
        }
        if (!bottom) {
            for (;;) {   // fill: expand the smallest remaining subtree completely while it fits
                const bool cand = valid && e.ref >= 0 && e.cnt <= kWide;
                const int cmin = __reduce_min_sync(full, cand ? e.cnt : 0x7fffffff);
                if (cmin == 0x7fffffff || count + cmin - 1 > kWide) break;
                const int L = __ffs(__ballot_sync(full, cand && e.cnt == cmin)) - 1;
                bool mine = lane == L;       // entries of the subtree being expanded
                for (;;) {
                    const unsigned m = __ballot_sync(full, mine && e.ref >= 0);
                    if (!m) break;
                    const int P = __ffs(m) - 1;
                    const int r = __shfl_sync(full, e.ref, P);
                    if (lane == P) take_child(bn, r, 0, e);
                    if (lane == count) { take_child(bn, r, 1, e); valid = true; mine = true; }
                    ++count;
                }
            }
        }
        // children that are still binary subtrees become wide nodes of the next level
        const bool internal = valid && e.ref >= 0;
        const unsigned m = __ballot_sync(full, internal);
        const int k = __popc(m);
        bool ok = true;
        if (k) {
            uint32_t base = 0, qbase = 0;
            if (lane == 0) { base = atomicAdd(n_wn, (uint32_t)k); qbase = atomicAdd(n_out, (uint32_t)k); }
            base = __shfl_sync(full, base, 0); qbase = __shfl_sync(full, qbase, 0);
            if (base + k > cap_wn) { ok = false; if (lane == 0) *overflow = 1u; }
            else if (internal) {
                const int rank = __popc(m & ((1u << lane) - 1u));
                q_out[qbase + rank] = make_int2(e.ref, (int)(base + rank));
                e.ref = (int)(base + rank);
            }
        }
        if (!ok) continue;
        WNodeDev* o = wn + w;
        const float inf = __int_as_float(0x7f800000);
        for (int a = 0; a < 3; ++a) { o->lo[a][lane] = valid ? e.lo[a] : inf; o->hi[a][lane] = valid ? e.hi[a] : -inf; }
        o->ref[lane] = valid ? e.ref : 0x7fffffff;
    }
}

// Barrier across the CTAs of a grid that is resident as a whole.  k_collapse_all is launched with cudaLaunchCooperativeKernel
// (launch_collapse below), so the runtime refuses a grid that could not be co-resident instead of letting it spin for ever;
// where cooperative launches are not available the kernel runs as ONE CTA, for which the barrier is a __syncthreads.
// bar[0] counts arrivals, bar[1] is the generation.
__device__ __forceinline__ void grid_barrier(uint32_t* bar) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const uint32_t gen = atomicAdd(&bar[1], 0u);
        if (atomicAdd(&bar[0], 1u) == gridDim.x - 1) { atomicExch(&bar[0], 0u); __threadfence(); atomicAdd(&bar[1], 1u); }
        else while (atomicAdd(&bar[1], 0u) == gen) { }
        __threadfence();
    }
    __syncthreads();
}

// The whole collapse in ONE launch: the levels of the 32-wide tree are produced one after the other with a grid barrier in
// between, the size of each level being known on the device only.  counters: [0] tasks of this level, [1] tasks of the next,
// [2] wide nodes so far, [3] capacity overflow, [4..5] the barrier.  On exit *wide_count = number of wide nodes, or 0 if the
// tree outgrew its capacity or is deeper than the level loop (packets then walk the binary tree).  The host reads nothing
// back: opx_bvh_build returns after enqueueing.
__global__ void __launch_bounds__(256, 2) k_collapse_all(const NodeDev* __restrict__ bn, int2* q0, int2* q1, uint32_t* counters, WNodeDev* wn,
                                                      uint32_t cap_wn, uint32_t* wide_count) {
    int2* q_in = q0;
    int2* q_out = q1;
    for (int level = 0; level < 128; ++level) {
        const uint32_t n_in = level == 0 ? 1u : atomicAdd(&counters[0], 0u);
        if (n_in == 0u) break;                                   // the same value in every CTA (set before the last barrier)
        collapse_level(bn, q_in, n_in, q_out, counters + 1, wn, counters + 2, cap_wn, counters + 3);
        grid_barrier(counters + 4);
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            const uint32_t next = atomicAdd(&counters[1], 0u);
            atomicExch(&counters[0], atomicAdd(&counters[3], 0u) ? 0u : next);      // overflow: stop
            atomicExch(&counters[1], 0u);
        }
        grid_barrier(counters + 4);
        int2* t = q_in; q_in = q_out; q_out = t;
    }
    // counters[0] != 0 here: the level loop ran out with tasks still pending (a tree deeper than 128 wide levels) - no wide tree
    if (blockIdx.x == 0 && threadIdx.x == 0)
        *wide_count = (atomicAdd(&counters[3], 0u) || atomicAdd(&counters[0], 0u)) ? 0u : atomicAdd(&counters[2], 0u);
}

__global__ void k_collapse_init(int2* q, uint32_t* counters) {
    q[0] = make_int2(0, 0);
    counters[0] = 1u; counters[1] = 0u; counters[2] = 1u; counters[3] = 0u; counters[4] = 0u; counters[5] = 0u;
}

// Largest grid of k_collapse_all that is resident as a whole on the current device (at most two CTAs per SM: more only adds
// arrivals at the barrier), and whether the device takes cooperative launches; queried once per device.
constexpr int kCollapseThreads = 256;
struct CollapseShape { int max_grid = 0; bool cooperative = false; bool known = false; };
std::mutex g_collapse_mutex;
CollapseShape g_collapse_shape[64];

opx_status collapse_shape(CollapseShape* out) {
    int dev = 0;
    if (cudaError_t e = cudaGetDevice(&dev)) return check_cuda(e, "cudaGetDevice");
    if (dev < 0 || dev >= 64) return fail(OPX_ERR_UNSUPPORTED_DEVICE, "device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_collapse_mutex);
    CollapseShape& c = g_collapse_shape[dev];
    if (!c.known) {
        int coop = 0, sms = 0, per_sm = 0;
        cudaError_t e;
        if ((e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev)) ||
            (e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) ||
            (e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_collapse_all, kCollapseThreads, 0)))
            return check_cuda(e, "k_collapse_all occupancy query");
        c.cooperative = coop != 0 && per_sm >= 1 && sms >= 1;
        c.max_grid = c.cooperative ? std::min(per_sm, 2) * sms : 1;
        c.known = true;
    }
    *out = c;
    return OPX_OK;
}

// One launch for all levels.  Cooperative: the runtime checks that the grid fits on the device (or the MIG slice / SM partition
// the context really has) and returns an error otherwise, so a wrong guess is an OPX_ERR_CUDA, never a hang.
opx_status launch_collapse(const NodeDev* nodes, int2* q0, int2* q1, uint32_t* counters, WNodeDev* wnodes, uint32_t cap,
                           uint32_t* wide_count, size_t wanted_grid, cudaStream_t stream) {
    CollapseShape shape;
    if (opx_status st = collapse_shape(&shape)) return st;
    const uint32_t grid = (uint32_t)std::max<size_t>(1, std::min<size_t>(wanted_grid, (size_t)shape.max_grid));
    if (shape.cooperative) {
        void* args[] = {(void*)&nodes, (void*)&q0, (void*)&q1, (void*)&counters, (void*)&wnodes, (void*)&cap, (void*)&wide_count};
        return check_cuda(cudaLaunchCooperativeKernel((const void*)k_collapse_all, dim3(grid), dim3(kCollapseThreads), args, 0, stream),
                          "k_collapse_all (cooperative launch)");
    }
    k_collapse_all<<<1, kCollapseThreads, 0, stream>>>(nodes, q0, q1, counters, wnodes, cap, wide_count);
    return check_cuda(cudaGetLastError(), "k_collapse_all (single CTA)");
}

}  // namespace

size_t wide_node_capacity(size_t T) { return T >= 2 ? T / 8 + 64 : 1; }

// ------------------------------------------------------------------------------------- layout
void compute_layout(const SceneHost& s, opx_scene_layout* lay, size_t* tmp_bytes) {
    const size_t T = s.tri_surface.size();
    const size_t n_nodes = T > 1 ? T - 1 : 1;
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t r = off; off += align_up(bytes ? bytes : 16, 256); return r; };
    lay->nodes = take(n_nodes * sizeof(NodeDev));
    lay->triangles = take((T ? T : 1) * 48 * 3);      // three rotations of the record (opx_device.cuh: RayR)
    lay->normals = take((T ? T : 1) * 16);
    lay->surfaces = take(s.surfaces.size() * 8);
    lay->mat_kinds = take(s.mat_kinds.size() * 4);
    lay->tables = take(s.tables.size() * 4);
    lay->frames = take(s.frames.size() * sizeof(FrameDev));
    lay->sorted_keys = take(T * 8);
    lay->parents = take((2 * T + 1) * 4);
    lay->wide_node_capacity = wide_node_capacity(T);
    lay->wide_nodes = take(lay->wide_node_capacity * sizeof(WNodeDev));
    lay->wide_count = take(4);
    lay->vertex_normals = take(s.tri_vnormals.size() * 4);
    lay->total_bytes = off;
    if (tmp_bytes) {
        size_t t = 0;
        auto tk = [&](size_t bytes) { t += align_up(bytes ? bytes : 16, 256); };
        tk(T * 36); tk(T * 4); tk(T * 12);
        tk(T * 8); tk(T * 4); tk(T * 4);            // second key buffer, two index buffers
        tk(256 * sort_blocks(T) * 4); tk(64); tk(T * 4);
        tk(wide_node_capacity(T) * 8); tk(wide_node_capacity(T) * 8); tk(64);      // collapse queues + counters
        *tmp_bytes = t;
    }
}

// Scene constants the build needs, computed once when the scene is created (host only).
void compute_scene_stats(SceneHost& s) {
    const size_t T = s.tri_surface.size();
    // padding of the leaf boxes: 2^-16 of the largest |coordinate| (>= 128 ulp there), at least 1e-6
    float maxabs = 0.f;
    for (float v : s.tri) { const float a = std::fabs(v); if (a > maxabs) maxabs = a; }
    s.leaf_pad = fmaxf(maxabs * (1.0f / 65536.0f), 1e-6f);
    s.max_abs = maxabs;
    // typical triangle size (log-mean of the largest AABB extent) and scene extent: a beam much wider
    // than the triangles it meets gains nothing over per-ray box tests
    double logsum = 0.0;
    float slo[3] = {FLT_MAX, FLT_MAX, FLT_MAX}, shi[3] = {-FLT_MAX, -FLT_MAX, -FLT_MAX};
    for (size_t t = 0; t < T; ++t) {
        const float* v = &s.tri[9 * t];
        float ext = 0.f;
        for (int c = 0; c < 3; ++c) {
            const float lo = std::fmin(v[c], std::fmin(v[3 + c], v[6 + c])), hi = std::fmax(v[c], std::fmax(v[3 + c], v[6 + c]));
            ext = std::fmax(ext, hi - lo);
            slo[c] = std::fmin(slo[c], lo); shi[c] = std::fmax(shi[c], hi);
        }
        logsum += std::log2((double)std::fmax(ext, 1e-20f));
    }
    s.tri_size = T ? (float)std::exp2(logsum / (double)T) : 0.f;
    s.scene_ext = T ? std::fmax(shi[0] - slo[0], std::fmax(shi[1] - slo[1], shi[2] - slo[2])) : 0.f;

}

opx_status build_bvh(SceneHost& s, void* d_scene_ws, void* d_tmp_ws, cudaStream_t stream) {
    const size_t T = s.tri_surface.size();
    const opx_scene_layout& lay = s.layout;
    char* ws = (char*)d_scene_ws;
    NodeDev* nodes = (NodeDev*)(ws + lay.nodes);
    float4* tris = (float4*)(ws + lay.triangles);
    float4* normals = (float4*)(ws + lay.normals);
    int2* surfaces = (int2*)(ws + lay.surfaces);
    uint32_t* mat_kinds = (uint32_t*)(ws + lay.mat_kinds);
    float* tables = (float*)(ws + lay.tables);
    FrameDev* frames = (FrameDev*)(ws + lay.frames);
    uint64_t* sorted_keys = (uint64_t*)(ws + lay.sorted_keys);
    int* parents = (int*)(ws + lay.parents);

    BuildTmp tmp;
    {
        char* p = (char*)d_tmp_ws;
        auto take = [&](size_t bytes) { char* r = p; p += align_up(bytes ? bytes : 16, 256); return r; };
        tmp.tri_in = (float*)take(T * 36); tmp.surf_in = (int32_t*)take(T * 4); tmp.normals_in = (float*)take(T * 12);
        tmp.keys[0] = sorted_keys; tmp.keys[1] = (uint64_t*)take(T * 8);
        tmp.idx[0] = (uint32_t*)take(T * 4); tmp.idx[1] = (uint32_t*)take(T * 4);
        tmp.hist = (uint32_t*)take(256 * sort_blocks(T) * 4); tmp.bounds = (uint32_t*)take(64); tmp.flags = (uint32_t*)take(T * 4);
        tmp.queue[0] = (int2*)take(wide_node_capacity(T) * 8); tmp.queue[1] = (int2*)take(wide_node_capacity(T) * 8);
        tmp.wcount = (uint32_t*)take(64);
    }
    auto up = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
        if (!bytes) return cudaSuccess;
        return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, stream);
    };
    cudaError_t e;
    if ((e = up(tmp.tri_in, s.tri.data(), T * 36)) || (e = up(tmp.surf_in, s.tri_surface.data(), T * 4)) ||
        (e = up(tmp.normals_in, s.normals.data(), T * 12)) || (e = up(surfaces, s.surfaces.data(), s.surfaces.size() * 8)) ||
        (e = up(mat_kinds, s.mat_kinds.data(), s.mat_kinds.size() * 4)) || (e = up(tables, s.tables.data(), s.tables.size() * 4)) ||
        (e = up(frames, s.frames.data(), s.frames.size() * sizeof(FrameDev))) ||
        (e = up(ws + lay.vertex_normals, s.tri_vnormals.data(), s.tri_vnormals.size() * 4)))
        return check_cuda(e, "scene upload");

    if (opx_status st = configure_device()) return st;
    const float pad = s.leaf_pad, tri_size = s.tri_size, scene_ext = s.scene_ext;      // scene constants (compute_scene_stats)

    const int Ti = (int)T;
    if (T >= 2) {
        const uint32_t nsb = (uint32_t)sort_blocks(T);
        const uint32_t g256 = (uint32_t)((T + 255) / 256);
        k_init_bounds<<<1, 32, 0, stream>>>(tmp.bounds);
        k_bounds<<<min(g256, 1184u), 256, 0, stream>>>(tmp.tri_in, (uint32_t)T, tmp.bounds);
        k_morton<<<g256, 256, 0, stream>>>(tmp.tri_in, (uint32_t)T, tmp.bounds, tmp.keys[0], tmp.idx[0]);
        count_launch(3);
        int cur = 0;
        for (int shift = 0; shift < 64; shift += 8) {
            k_radix_hist<<<nsb, kSortBlock, 0, stream>>>(tmp.keys[cur], (uint32_t)T, shift, tmp.hist, nsb);
            k_radix_scan<<<1, 1024, 0, stream>>>(tmp.hist, nsb);
            k_radix_scatter<<<nsb, kSortBlock, 0, stream>>>(tmp.keys[cur], tmp.idx[cur], tmp.keys[cur ^ 1], tmp.idx[cur ^ 1],
                                                           (uint32_t)T, shift, tmp.hist, nsb);
            count_launch(3);
            cur ^= 1;
        }
        // 8 passes: the sorted keys are back in keys[0] == sorted_keys, indices in idx[0]
        k_pack_tris<<<g256, 256, 0, stream>>>(tmp.tri_in, tmp.surf_in, tmp.normals_in, tmp.idx[0], (uint32_t)T, tris, normals);
        k_hierarchy<<<(uint32_t)((T - 1 + 255) / 256), 256, 0, stream>>>(sorted_keys, Ti, nodes, parents);
        if ((e = cudaMemsetAsync(tmp.flags, 0, T * 4, stream))) return check_cuda(e, "memset flags");
        k_refit<<<g256, 256, 0, stream>>>(tris, Ti, pad, nodes, parents, tmp.flags);
        count_launch(3);
        // collapse into the 32-wide tree: one launch for all levels (k_collapse_all), nothing read back
        WNodeDev* wnodes = (WNodeDev*)(ws + lay.wide_nodes);
        const uint32_t cap = (uint32_t)lay.wide_node_capacity;
        k_collapse_init<<<1, 1, 0, stream>>>(tmp.queue[0], tmp.wcount);
        if (opx_status st = launch_collapse(nodes, tmp.queue[0], tmp.queue[1], tmp.wcount, wnodes, cap, (uint32_t*)(ws + lay.wide_count),
                                            (lay.wide_node_capacity + 7) / 8, stream))
            return st;
        count_launch(2);
    } else {
        if ((e = cudaMemsetAsync(ws + lay.wide_count, 0, 4, stream))) return check_cuda(e, "memset wide count");
        if (T == 1) {
            // a single triangle needs no hierarchy: propagate tests it directly (see launch_propagate)
            uint64_t zero_key = 0;
            uint32_t zero_idx = 0;
            if ((e = up(sorted_keys, &zero_key, 8)) || (e = up(tmp.idx[0], &zero_idx, 4))) return check_cuda(e, "tiny upload");
            k_pack_tris<<<1, 32, 0, stream>>>(tmp.tri_in, tmp.surf_in, tmp.normals_in, tmp.idx[0], 1u, tris, normals);
            count_launch(1);
        }
    }
    if ((e = cudaGetLastError())) return check_cuda(e, "BVH build launch");
    // No synchronisation: the uploads above left from pageable host memory, which cudaMemcpyAsync stages before it returns,
    // so the scene's host arrays are no longer referenced; everything else is stream-ordered.

    SceneDev& d = s.dev;
    d.wnodes = (const WNodeDev*)(ws + lay.wide_nodes); d.n_wnodes = T >= 2 ? (uint32_t)lay.wide_node_capacity : 0u;
    d.wide_count = (const uint32_t*)(ws + lay.wide_count);
    d.nodes = nodes; d.tris = tris; d.normals = normals; d.surfaces = surfaces; d.mat_kinds = mat_kinds;
    d.tables = tables; d.frames = frames;
    d.vnormals = s.tri_vnormals.empty() ? nullptr : (const float*)(ws + lay.vertex_normals);
    d.n_tri = (uint32_t)T; d.n_nodes = (uint32_t)(T > 1 ? T - 1 : 1);
    d.n_lambda = s.params.n_lambda; d.max_bounces = s.params.max_bounces;
    d.beam_max_width = kBeamWidthInTriangles * tri_size;
    d.beam_max_spread = scene_ext > 0.f ? d.beam_max_width / (0.5f * scene_ext) : 0.f;
    d.lambda_min = s.params.lambda_min_nm; d.inv_dlambda = s.inv_dlambda; d.t_min = s.params.t_min_mm;
    d.inv_bin = s.inv_bin; d.flags = 0; d.d_n = nullptr;
    d.origin_limit = 4.f * fmaxf(s.max_abs, 1.f);
    return OPX_OK;
}

}  // namespace opx
