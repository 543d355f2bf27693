// Beam traversal of the 32-wide tree: the 32 rays of a packet are bounded by
// ONE beam -- an axis-aligned box that moves linearly with the ray parameter -- and lane k tests child
// k of a wide node against that beam, so 32 boxes cost what one box costs in a per-ray walk.  Only the
// triangles whose (padded) box the beam enters are tested, by every lane against its own ray with the
// contract test of DESIGN.md 3.3, so the result is exactly the per-photon closest hit.
//
// Beam.  Every member ray is re-based on a common plane x_K = c (K = dominant axis of the packet,
// c = the rear-most member origin along K): o'_i = o_i + s_i d_i with s_i = (c - o_iK) / d_iK <= 0, and
// t' = t - s_i.  For t' >= 0 all member rays lie inside
//     [omin_a + t' dmin_a,  omax_a + t' dmax_a]        per axis a,
// with omin/omax/dmin/dmax the (slightly widened) extremes of o'_i and d_i over the members.  A box
// [lo, hi] can only be entered by a member while, on every axis,
//     (1) omax_a + t' dmax_a >= lo_a     and     (2) omin_a + t' dmin_a <= hi_a,
// each of which is a lower or an upper bound on t' depending on the sign of dmax_a / dmin_a.  The
// interval they leave, clipped to [tlo, thi] with tlo = min_i(tmin - s_i) and thi = max_i(t_best_i - s_i),
// is empty  =>  no member ray can hit anything in the box closer than its current best hit (ties kept).
//
// Per-lane cull.  When the beam enters many triangle boxes of a node (a packet's footprint covers more
// facets than one ray crosses), every lane first slab-tests ITS OWN ray against those boxes (the planes
// sit in the registers of the lane that owns the child and are broadcast by shuffle) and then tests
// only the triangles whose box its ray enters: the leaf loop runs max-over-lanes instead of
// sum-over-lanes iterations.
#pragma once
#include "opx_device.cuh"

namespace opx {
namespace {

constexpr int kBeamStack = 56;            // per warp, in shared memory; overflow => fall back to the binary walk
constexpr int kBeamStackWords = 64;       // words reserved per array: the last 8 of each hold the parked beam (closest_hit_beam)
#ifndef OPX_CULL_MIN
#define OPX_CULL_MIN 4
#endif
constexpr int kCullMin = OPX_CULL_MIN;   // per-lane cull when the beam enters at least this many triangle boxes of a node
#ifndef OPX_CULL_SLOTS
#define OPX_CULL_SLOTS 16
#endif
constexpr int kCullSlots = OPX_CULL_SLOTS;   // candidate boxes a warp stages in shared memory per culling round
#ifndef OPX_RECULL
#define OPX_RECULL 0                          // 1: per-lane candidates nearest-first, re-tested against the current best hit
#endif

struct Beam {
    // entry bound of axis a: fma(near_a, rn_a, cn_a); exit bound: fma(far_a, rf_a, cf_a), where
    // (near, far) = (lo, hi) of the child box, swapped on an axis where all member directions are negative.
    // On an axis where the member directions have both signs (mixed), both planes give ENTRY bounds.
    float rn[3], cn[3], rf[3], cf[3];
    unsigned neg;                         // bit a: near plane of axis a is hi
    unsigned mixed;                       // bit a: axis a is mixed
    float tlo;
};

struct BeamStats { unsigned visits = 0, tris = 0, beam_segments = 0, fallback_segments = 0, overflows = 0, culls = 0, cands = 0, pairs = 0; };

__device__ __forceinline__ int f2ordi(float f) { const int i = __float_as_int(f); return i ^ ((i >> 31) & 0x7fffffff); }
__device__ __forceinline__ float ordi2f(int i) { return __int_as_float(i ^ ((i >> 31) & 0x7fffffff)); }
__device__ __forceinline__ float warp_min(float v) { return ordi2f(__reduce_min_sync(0xffffffffu, f2ordi(v))); }
__device__ __forceinline__ float warp_max(float v) { return ordi2f(__reduce_max_sync(0xffffffffu, f2ordi(v))); }
// min / max of floats known to be >= 0 (or +inf): their bit patterns order like the values
__device__ __forceinline__ float warp_min_pos(float v) { return __int_as_float(__reduce_min_sync(0xffffffffu, __float_as_int(v))); }
__device__ __forceinline__ float warp_max_pos(float v) { return __int_as_float(__reduce_max_sync(0xffffffffu, __float_as_int(v))); }
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// Builds the beam of the alive lanes.  Returns false (warp-uniform) when the packet is not coherent
// enough for a beam: some alive ray is non-finite, runs against the packet's dominant axis or nearly
// perpendicular to it, or a re-based origin / a direction lies further than the scene's limits
// (SceneDev::beam_max_width, beam_max_spread) from the leader's.  `s` is the lane's re-basing offset
// (t = t' + s).
//
// The extremes are taken on keys  k = x - (x_leader - W)  in [0, 2W]  (W = the limit): non-negative
// floats order like their bit patterns, so each extreme is one integer warp reduction; a negative
// key (bit pattern < 0), a key > 2W or a NaN (bit pattern > that of 2W) marks a packet that is too wide.
__device__ __forceinline__ bool beam_setup(const SceneDev& sc, float ox, float oy, float oz, float dx, float dy, float dz, float tmin, bool alive,
                                           Beam& bm, float& s) {
    const unsigned full = 0xffffffffu;
    const unsigned am = __ballot_sync(full, alive);
    const int leader = __ffs(am) - 1;
    const int src = alive ? (int)(threadIdx.x & 31) : leader;     // a lane without a ray stands in for the leader
    dx = __shfl_sync(full, dx, src); dy = __shfl_sync(full, dy, src); dz = __shfl_sync(full, dz, src);
    ox = __shfl_sync(full, ox, src); oy = __shfl_sync(full, oy, src); oz = __shfl_sync(full, oz, src);
    const float lx = __shfl_sync(full, dx, leader), ly = __shfl_sync(full, dy, leader), lz = __shfl_sync(full, dz, leader);
    int K = 0; float lk = lx;
    if (fabsf(ly) > fabsf(lk)) { K = 1; lk = ly; }
    if (fabsf(lz) > fabsf(lk)) { K = 2; lk = lz; }
    const float dK = K == 0 ? dx : (K == 1 ? dy : dz), oK = K == 0 ? ox : (K == 1 ? oy : oz);
    const float sumabs = fabsf(ox) + fabsf(oy) + fabsf(oz) + fabsf(dx) + fabsf(dy) + fabsf(dz);
    // sumabs bounds |o|_inf: an origin beyond origin_limit (4 x the scene's largest coordinate) leaves the error budget of
    // the padded boxes and takes the binary walk with per-ray slack
    const bool member = sumabs < sc.origin_limit && (lk > 0.f ? dK >= 0.25f : dK <= -0.25f);     // NaN fails both
    if (!__all_sync(full, member)) return false;
    // rear-most origin along K
    const float c = lk > 0.f ? warp_min(oK) : warp_max(oK);
    s = fminf((c - oK) * rcp_approx(dK), 0.f);
    const float px = __fmaf_rn(s, dx, ox), py = __fmaf_rn(s, dy, oy), pz = __fmaf_rn(s, dz, oz);
    const float W = sc.beam_max_width, S = sc.beam_max_spread;
    const float bx = __shfl_sync(full, px, leader) - W, by = __shfl_sync(full, py, leader) - W, bz = __shfl_sync(full, pz, leader) - W;
    const float ex = lx - S, ey = ly - S, ez = lz - S;
    const float kx = px - bx, ky = py - by, kz = pz - bz, jx = dx - ex, jy = dy - ey, jz = dz - ez;
    float omin[3], omax[3], dmin[3], dmax[3];
    omin[0] = warp_min_pos(kx); omax[0] = warp_max_pos(kx); omin[1] = warp_min_pos(ky); omax[1] = warp_max_pos(ky);
    omin[2] = warp_min_pos(kz); omax[2] = warp_max_pos(kz);
    dmin[0] = warp_min_pos(jx); dmax[0] = warp_max_pos(jx); dmin[1] = warp_min_pos(jy); dmax[1] = warp_max_pos(jy);
    dmin[2] = warp_min_pos(jz); dmax[2] = warp_max_pos(jz);
    const int lim_o = __float_as_int(2.f * W), lim_d = __float_as_int(2.f * S);
    bool ok = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        ok = ok && __float_as_int(omin[a]) >= 0 && __float_as_int(omax[a]) <= lim_o && __float_as_int(dmin[a]) >= 0 &&
             __float_as_int(dmax[a]) <= lim_d;
    }
    if (!ok) return false;
    bm.tlo = warp_min_pos(alive ? tmin - s : kInf);      // tmin >= 0 and s <= 0
    const float base_o[3] = {bx, by, bz}, base_d[3] = {ex, ey, ez};
    // widen: keys, re-based origins and their sums carry a few ulp of rounding, directions a few ulp of 1
    const float scale = fmaxf(fmaxf(fabsf(bx), fabsf(by)), fmaxf(fabsf(bz), 4.f * W));
    const float eo = scale * 3.8146973e-6f + 1e-30f;      // 2^-18 of the largest |coordinate|
    bm.mixed = 0u; bm.neg = 0u;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float lo_o = (omin[a] + base_o[a]) - eo, hi_o = (omax[a] + base_o[a]) + eo;
        float lo_d = (dmin[a] + base_d[a]) - 2e-6f, hi_d = (dmax[a] + base_d[a]) + 2e-6f;
        if (fabsf(hi_d) < 1e-9f) hi_d = 1e-9f;             // widening only
        if (fabsf(lo_d) < 1e-9f) lo_d = -1e-9f;
        // constraint 1: hi_o + t hi_d >= lo  ->  bound fma(lo, r1, c1);  2: lo_o + t lo_d <= hi  ->  fma(hi, r2, c2).
        // The approximate reciprocals are off by <= 2 ulp: far inside the padding of the boxes.
        const float r1 = rcp_approx(hi_d), r2 = rcp_approx(lo_d);
        const float c1 = -hi_o * r1, c2 = -lo_o * r2;
        const bool neg = hi_d < 0.f;                       // all negative: 2 bounds the entry (plane hi), 1 the exit (plane lo)
        bm.rn[a] = neg ? r2 : r1; bm.cn[a] = neg ? c2 : c1;
        bm.rf[a] = neg ? r1 : r2; bm.cf[a] = neg ? c1 : c2;
        if (neg) bm.neg |= 1u << a;
        else if (!(lo_d > 0.f)) bm.mixed |= 1u << a;       // mixed: (lo, r1, c1) and (hi, r2, c2) are both entry bounds
    }
    return true;
}

// Closest hit of the packet by beam traversal.  Returns false (warp-uniform) if the shared-memory
// stack overflowed: the caller then redoes the segment with the per-lane walk of the binary tree.
// (so, sd) point at the lane's own segment in shared memory (origin, direction; not re-based): the per-lane cull
// reads it back from there, so the segment does not occupy registers during the walk.
// s_cb: 2 x kCullSlots float4 of the warp: the candidate boxes of the node being culled, (near planes, child ref) and
// (far planes, -), written by the lanes that own the candidates and read back by every lane with uniform addresses
// (two broadcast 16-byte loads per candidate instead of six shuffles).
template <bool kMixed, bool kStats>
__device__ __forceinline__ bool closest_hit_beam(const SceneDev& sc, const RayR& rr, Beam bm, float s, float tmin, int last_j,
                                                 bool alive, int lane, const float* so, const float* sd,
                                                 int* s_ref, float* s_tn, float4* s_cb, Hit& h, BeamStats& stats) {
    const unsigned full = 0xffffffffu;
    h = Hit{kInf, -1, 0x7fffffff};
    float thi = kInf;
    int sp = 0, ref = 0;
    const unsigned lt = (1u << lane) - 1u;
    // The beam is read at every node and in no leaf phase, and the leaf phases need many registers of their own: it is parked
    // in shared memory (the 8 words behind each stack array) and read back after every leaf phase, so that it occupies no
    // register while triangles are tested -- left to itself the compiler kept it in local memory and re-read it at EVERY node.
    float4* s_beam = reinterpret_cast<float4*>(s_ref + kBeamStack);
    float4* s_beam2 = reinterpret_cast<float4*>(s_tn + kBeamStack);
    if (lane == 0) {
        s_beam[0] = make_float4(bm.rn[0], bm.rn[1], bm.rn[2], bm.tlo);
        s_beam[1] = make_float4(bm.cn[0], bm.cn[1], bm.cn[2], __uint_as_float(bm.neg | (bm.mixed << 3)));
        s_beam2[0] = make_float4(bm.rf[0], bm.rf[1], bm.rf[2], 0.f);
        s_beam2[1] = make_float4(bm.cf[0], bm.cf[1], bm.cf[2], 0.f);
    }
    __syncwarp();
    for (;;) {
        const bool ngx = bm.neg & 1u, ngy = bm.neg & 2u, ngz = bm.neg & 4u;
        if (kStats) ++stats.visits;
        const float* nd = reinterpret_cast<const float*>(sc.wnodes + ref) + lane;
        const float lox = __ldg(nd + kWOffLo), loy = __ldg(nd + kWOffLo + kWide), loz = __ldg(nd + kWOffLo + 2 * kWide);
        const float hix = __ldg(nd + kWOffHi), hiy = __ldg(nd + kWOffHi + kWide), hiz = __ldg(nd + kWOffHi + 2 * kWide);
        const int cref = __float_as_int(__ldg(nd + kWOffRef));
        const float nx = ngx ? hix : lox, ny = ngy ? hiy : loy, nz = ngz ? hiz : loz;
        const float fx = ngx ? lox : hix, fy = ngy ? loy : hiy, fz = ngz ? loz : hiz;
        const float ax = __fmaf_rn(nx, bm.rn[0], bm.cn[0]), ay = __fmaf_rn(ny, bm.rn[1], bm.cn[1]), az = __fmaf_rn(nz, bm.rn[2], bm.cn[2]);
        const float bx = __fmaf_rn(fx, bm.rf[0], bm.cf[0]), by = __fmaf_rn(fy, bm.rf[1], bm.cf[1]), bz = __fmaf_rn(fz, bm.rf[2], bm.cf[2]);
        float tn = fmaxf(fmaxf(ax, ay), fmaxf(az, bm.tlo)), tf = thi;
        if (kMixed) {
            if (bm.mixed & 1u) tn = fmaxf(tn, bx); else tf = fminf(tf, bx);
            if (bm.mixed & 2u) tn = fmaxf(tn, by); else tf = fminf(tf, by);
            if (bm.mixed & 4u) tn = fmaxf(tn, bz); else tf = fminf(tf, bz);
        } else {
            tf = fminf(fminf(bx, by), fminf(bz, tf));
        }
        const bool hit = tn <= tf;
        const unsigned mt = __ballot_sync(full, hit && cref < 0);
        if (mt) {
            if (kStats) stats.cands += __popc(mt);
            if (kMixed || __popc(mt) < kCullMin) {
                // no per-lane cull (warp-uniform): one uniform pass over the candidates, no votes, no per-lane bit scans
                if (kStats) stats.pairs += __popc(mt) * __popc(__ballot_sync(full, alive));
                unsigned m = mt;
                do {
                    const int L = __ffs(m) - 1;
                    m &= m - 1u;
                    const int j = ~__shfl_sync(full, cref, L);
                    if (kStats) ++stats.tris;
                    if (alive) consider_rot(sc, rr, j, tmin, last_j, h);
                } while (m);
            } else {
                // per-lane cull: own ray against the candidate boxes (all member rays share the beam's sign octant, so
                // near/far are the same planes for every lane).  Approximate reciprocals: see slab_setup.
                if (kStats) ++stats.culls;
                const float ix = rcp_approx(sd[0]), iy = rcp_approx(sd[1]), iz = rcp_approx(sd[2]);
                const float qx = -so[0] * ix, qy = -so[1] * iy, qz = -so[2] * iz;
                unsigned rem = mt;
                do {                                     // kCullSlots candidates at a time (one round unless the node holds more)
                    const int rank = __popc(rem & lt);
                    const bool put = ((rem >> lane) & 1u) && rank < kCullSlots;
                    if (put) {
                        s_cb[rank] = make_float4(nx, ny, nz, __int_as_float(cref));
                        s_cb[kCullSlots + rank] = make_float4(fx, fy, fz, 0.f);
                    }
                    const int cnt = min(__popc(rem), kCullSlots);
                    rem &= ~__ballot_sync(full, put);
                    __syncwarp();
                    const float cap = alive ? h.t : -1.f;
                    unsigned mine = 0u;                  // the candidates (slots) this lane still has to test
#if OPX_RECULL
                    float near_en = kInf;                // the candidate whose box this lane's ray enters first
                    int near_c = 0;
#endif
#pragma unroll
                    for (int c = 0; c < kCullSlots; ++c) {       // unrolled: slot addresses and mask bits are immediates
                        if (c >= cnt) break;
                        const float4 n4 = s_cb[c], f4 = s_cb[kCullSlots + c];
                        const float e0 = __fmaf_rn(n4.x, ix, qx), e1 = __fmaf_rn(n4.y, iy, qy), e2 = __fmaf_rn(n4.z, iz, qz);
                        const float x0 = __fmaf_rn(f4.x, ix, qx), x1 = __fmaf_rn(f4.y, iy, qy), x2 = __fmaf_rn(f4.z, iz, qz);
                        const float en = fmaxf(fmaxf(e0, e1), fmaxf(e2, 0.f)), exi = fminf(fminf(x0, x1), fminf(x2, cap));
                        if (en <= exi && ~__float_as_int(n4.w) != last_j) {
                            mine |= 1u << c;
#if OPX_RECULL
                            if (en < near_en) { near_en = en; near_c = c; }
#endif
                        }
                    }
#if OPX_RECULL
                    // Nearest box first, and every later candidate is tested against the lane's CURRENT best hit before its
                    // triangle is fetched: a hit on the facet in front (a mirror) drops the candidates whose boxes begin
                    // behind it (its backing plate).  The box test is the cull's own (entry bound <= best t, ties kept), so
                    // the surviving set still holds every triangle that could win.  The warp iterates while ANY lane has a
                    // candidate left: lanes skip their pruned candidates without spending an iteration of the warp on them.
                    unsigned tested = 0u, t_iter = 0u;
                    int c = near_c;
                    for (;;) {
                        int j = -1;
                        while (mine) {
                            mine &= ~(1u << c);
                            const float4 n4 = s_cb[c];
                            const float en = fmaxf(fmaxf(__fmaf_rn(n4.x, ix, qx), __fmaf_rn(n4.y, iy, qy)), __fmaf_rn(n4.z, iz, qz));
                            c = __ffs(mine) - 1;
                            if (en <= h.t) { j = ~__float_as_int(n4.w); break; }
                        }
                        if (!__any_sync(full, j >= 0)) break;
                        if (kStats) { ++t_iter; tested += j >= 0; }
                        if (j >= 0) consider_rot(sc, rr, j, tmin, last_j, h);
                    }
                    if (kStats) { stats.pairs += __reduce_add_sync(full, tested); stats.tris += t_iter; }
#else
                    if (kStats) {
                        stats.pairs += __reduce_add_sync(full, (unsigned)__popc(mine));
                        stats.tris += __reduce_max_sync(full, (unsigned)__popc(mine));
                    }
                    while (mine) {                       // per-lane trip count: the warp runs max-over-lanes iterations
                        const int c = __ffs(mine) - 1;
                        mine &= mine - 1u;
                        consider_rot(sc, rr, ~__float_as_int(s_cb[c].w), tmin, last_j, h);
                    }
#endif
                    __syncwarp();
                } while (rem);
            }
            thi = warp_max_pos(alive ? h.t - s : 0.f);            // h.t > 0 >= s: the bounds are positive, their bit patterns order like the values
            {
                const float4 a = s_beam[0], b = s_beam[1], c = s_beam2[0], d = s_beam2[1];
                bm.rn[0] = a.x; bm.rn[1] = a.y; bm.rn[2] = a.z; bm.tlo = a.w;
                bm.cn[0] = b.x; bm.cn[1] = b.y; bm.cn[2] = b.z; bm.neg = __float_as_uint(b.w) & 7u; bm.mixed = __float_as_uint(b.w) >> 3;
                bm.rf[0] = c.x; bm.rf[1] = c.y; bm.rf[2] = c.z; bm.cf[0] = d.x; bm.cf[1] = d.y; bm.cf[2] = d.z;
            }
        }
        const bool go = hit && cref >= 0 && tn <= thi;
        const unsigned mn = __ballot_sync(full, go);
        if (mn) {
            // nearest child next, the others onto the stack with their entry bounds (tn >= 0: bit patterns order like values)
            int L = __ffs(mn) - 1;
            if (mn & (mn - 1u)) {          // several children: the one the beam enters first
                const int kmin = __reduce_min_sync(full, go ? __float_as_int(tn) : 0x7fffffff);
                L = __ffs(__ballot_sync(full, go && __float_as_int(tn) == kmin)) - 1;
            }
            const unsigned rest = mn & ~(1u << L);
            if (rest) {
                const int k = __popc(rest);
                if (sp + k > kBeamStack) { if (kStats) ++stats.overflows; return false; }
                if ((rest >> lane) & 1u) { const int pos = sp + __popc(rest & lt); s_ref[pos] = cref; s_tn[pos] = tn; }
                sp += k;
                __syncwarp();
            }
            ref = __shfl_sync(full, cref, L);
            continue;
        }
        for (;;) {
            if (sp == 0) return true;
            --sp;
            const float t = s_tn[sp];
            if (t <= thi) { ref = s_ref[sp]; break; }
        }
        __syncwarp();
    }
}

}  // namespace
}  // namespace opx
