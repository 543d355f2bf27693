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
//     omax_a + t' dmax_a >= lo_a     and     omin_a + t' dmin_a <= hi_a,
// each of which is a lower or an upper bound on t' depending on the sign of dmax_a / dmin_a.  The
// interval they leave, clipped to [tlo, thi] with tlo = min_i(tmin - s_i) and thi = max_i(t_best_i - s_i),
// is empty  =>  no member ray can hit anything in the box closer than its current best hit (ties kept).
#pragma once
#include "opx_device.cuh"

namespace opx {
namespace {

constexpr int kBeamStack = 64;            // per warp, in shared memory; overflow => fall back to the binary walk

struct Beam {
    // entry bound per axis: fma(plane[offN_a], rn_a, cn_a); exit bound: fma(plane[offF_a], rf_a, cf_a).
    // On an axis where the member directions have both signs (mixed), both planes give ENTRY bounds.
    float rn[3], cn[3], rf[3], cf[3];
    int offN[3], offF[3];                 // word offsets of the two planes inside a WNodeDev (lane added by the caller)
    unsigned mixed;                       // bit a: axis a is mixed
    float tlo;
};

struct BeamStats { unsigned visits = 0, tris = 0, beam_segments = 0, fallback_segments = 0, overflows = 0; };

__device__ __forceinline__ int f2ordi(float f) { const int i = __float_as_int(f); return i ^ ((i >> 31) & 0x7fffffff); }
__device__ __forceinline__ float ordi2f(int i) { return __int_as_float(i ^ ((i >> 31) & 0x7fffffff)); }
__device__ __forceinline__ float warp_min(float v) { return ordi2f(__reduce_min_sync(0xffffffffu, f2ordi(v))); }
__device__ __forceinline__ float warp_max(float v) { return ordi2f(__reduce_max_sync(0xffffffffu, f2ordi(v))); }

// Builds the beam of the alive lanes.  Returns false (warp-uniform) when the packet is not coherent
// enough for a beam: some alive ray is non-finite, runs against the packet's dominant axis or nearly
// perpendicular to it, or the re-based origins / the directions spread by more than the scene's limits
// (SceneDev::beam_max_width, beam_max_spread).  `s` is the lane's re-basing offset (t = t' + s).
__device__ __forceinline__ bool beam_setup(const SceneDev& sc, float ox, float oy, float oz, float dx, float dy, float dz, float tmin, bool alive,
                                           Beam& bm, float& s) {
    const unsigned full = 0xffffffffu;
    const unsigned am = __ballot_sync(full, alive);
    const int leader = __ffs(am) - 1;
    // dominant axis of the leader's direction
    const float lx = __shfl_sync(full, dx, leader), ly = __shfl_sync(full, dy, leader), lz = __shfl_sync(full, dz, leader);
    int K = 0; float lk = lx;
    if (fabsf(ly) > fabsf(lk)) { K = 1; lk = ly; }
    if (fabsf(lz) > fabsf(lk)) { K = 2; lk = lz; }
    const float dK = K == 0 ? dx : (K == 1 ? dy : dz), oK = K == 0 ? ox : (K == 1 ? oy : oz);
    const float sumabs = fabsf(ox) + fabsf(oy) + fabsf(oz) + fabsf(dx) + fabsf(dy) + fabsf(dz);
    const bool member = alive && sumabs < kInf && (lk > 0.f ? dK >= 0.25f : dK <= -0.25f);     // NaN fails both
    if (__ballot_sync(full, alive && !member)) return false;
    // rear-most origin along K
    const float c = lk > 0.f ? warp_min(alive ? oK : kInf) : warp_max(alive ? oK : -kInf);
    s = alive ? __fdividef(c - oK, dK) : 0.f;
    s = fminf(s, 0.f);
    const float px = __fmaf_rn(s, dx, ox), py = __fmaf_rn(s, dy, oy), pz = __fmaf_rn(s, dz, oz);
    float omin[3], omax[3], dmin[3], dmax[3];
    omin[0] = warp_min(alive ? px : kInf); omax[0] = warp_max(alive ? px : -kInf);
    omin[1] = warp_min(alive ? py : kInf); omax[1] = warp_max(alive ? py : -kInf);
    omin[2] = warp_min(alive ? pz : kInf); omax[2] = warp_max(alive ? pz : -kInf);
    dmin[0] = warp_min(alive ? dx : kInf); dmax[0] = warp_max(alive ? dx : -kInf);
    dmin[1] = warp_min(alive ? dy : kInf); dmax[1] = warp_max(alive ? dy : -kInf);
    dmin[2] = warp_min(alive ? dz : kInf); dmax[2] = warp_max(alive ? dz : -kInf);
    bm.tlo = fmaxf(warp_min(alive ? tmin - s : kInf), 0.f);
    // widen: re-based origins carry a few ulp of rounding, directions a few ulp of 1
    float scale = 0.f;
#pragma unroll
    for (int a = 0; a < 3; ++a) scale = fmaxf(scale, fmaxf(fabsf(omin[a]), fabsf(omax[a])));
    const float eo = scale * 1.9073486e-6f + 1e-30f;      // 2^-19 of the largest |coordinate|
    bool ok = true;
    bm.mixed = 0u;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (dmax[a] - dmin[a] > sc.beam_max_spread || omax[a] - omin[a] > sc.beam_max_width) ok = false;
        const float lo_o = omin[a] - eo, hi_o = omax[a] + eo;
        float lo_d = dmin[a] - 1e-6f, hi_d = dmax[a] + 1e-6f;
        if (fabsf(hi_d) < 1e-9f) hi_d = 1e-9f;             // widening only
        if (fabsf(lo_d) < 1e-9f) lo_d = -1e-9f;
        const float r1 = 1.f / hi_d, r2 = 1.f / lo_d;      // constraint 1: omax + t dmax >= lo;  2: omin + t dmin <= hi
        const float c1 = -hi_o * r1, c2 = -lo_o * r2;
        if (lo_d > 0.f) {             // all positive: 1 bounds the entry (uses lo), 2 the exit (uses hi)
            bm.rn[a] = r1; bm.cn[a] = c1; bm.offN[a] = kWOffLo + a * kWide;
            bm.rf[a] = r2; bm.cf[a] = c2; bm.offF[a] = kWOffHi + a * kWide;
        } else if (hi_d < 0.f) {      // all negative: 2 bounds the entry (uses hi), 1 the exit (uses lo)
            bm.rn[a] = r2; bm.cn[a] = c2; bm.offN[a] = kWOffHi + a * kWide;
            bm.rf[a] = r1; bm.cf[a] = c1; bm.offF[a] = kWOffLo + a * kWide;
        } else {                      // mixed: both are entry bounds, no exit bound
            bm.rn[a] = r1; bm.cn[a] = c1; bm.offN[a] = kWOffLo + a * kWide;
            bm.rf[a] = r2; bm.cf[a] = c2; bm.offF[a] = kWOffHi + a * kWide;
            bm.mixed |= 1u << a;
        }
    }
    return ok;
}

// Closest hit of the packet by beam traversal.  Returns false (warp-uniform) if the shared-memory
// stack overflowed: the caller then redoes the segment with the binary packet walk.
template <bool kMixed, bool kStats>
__device__ __forceinline__ bool closest_hit_beam(const SceneDev& sc, const RayW& rw, const Beam& bm, float s, float tmin, int last,
                                                 bool alive, int lane, int* s_ref, float* s_tn, Hit& h, BeamStats& stats) {
    const unsigned full = 0xffffffffu;
    h = Hit{kInf, -1, 0x7fffffff};
    float thi = kInf;
    int sp = 0, ref = 0;
    const unsigned lt = (1u << lane) - 1u;
    for (;;) {
        if (kStats) ++stats.visits;
        const float* nd = reinterpret_cast<const float*>(sc.wnodes + ref) + lane;
        const float nx = __ldg(nd + bm.offN[0]), ny = __ldg(nd + bm.offN[1]), nz = __ldg(nd + bm.offN[2]);
        const float fx = __ldg(nd + bm.offF[0]), fy = __ldg(nd + bm.offF[1]), fz = __ldg(nd + bm.offF[2]);
        const int cref = __float_as_int(__ldg(nd + kWOffRef));
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
        unsigned mt = __ballot_sync(full, hit && cref < 0);
        if (mt) {
            do {
                const int L = __ffs(mt) - 1;
                mt &= mt - 1;
                const int j = ~__shfl_sync(full, cref, L);
                if (kStats) ++stats.tris;
                if (alive) consider(sc, rw, j, tmin, last, h);
            } while (mt);
            thi = warp_max(alive ? h.t - s : -kInf);
        }
        const bool go = hit && cref >= 0 && tn <= thi;
        const unsigned mn = __ballot_sync(full, go);
        if (mn) {
            // nearest child next, the others onto the stack with their entry bounds
            const int kmin = __reduce_min_sync(full, go ? f2ordi(tn) : 0x7fffffff);
            const int L = __ffs(__ballot_sync(full, go && f2ordi(tn) == kmin)) - 1;
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
