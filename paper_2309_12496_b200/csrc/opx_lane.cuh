// k_propagate_lane: one photon per thread with a private traversal stack.  Used for the instrumented
// build that counts the algorithmic work of a single ray (opx_propagate_stats), for the all-triangle
// debug mode (opx_propagate_brute) and for scenes without a hierarchy (fewer than two triangles).
#pragma once
#include "opx_device.cuh"

namespace opx {
namespace {

constexpr int kStack = 96;   // >= depth bound of a Karras tree over 63-bit keys + 32-bit index tie-break

struct Work { unsigned int nodes = 0, tris = 0; };   // instrumented build only

// ------------------------------------------------------------------------- per-lane traversal
template <bool kStats>
// e: per-ray slack of the box test (2^-20 |origin|_inf), negligible for origins inside the scene.
__device__ __forceinline__ Hit closest_hit_lane(const SceneDev& sc, const RayW& rw, const Slab& sl, float e, float tmin, int last, Work& work) {
    Hit h{kInf, -1, 0x7fffffff};
    int stack_ref[kStack];
    float stack_t[kStack];
    int sp = 0;
    int ref = 0;
    for (;;) {
        if (ref >= 0) {
            if (kStats) ++work.nodes;
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
            if (kStats) ++work.tris;
            consider(sc, rw, ~ref, tmin, last, h);
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

__device__ __forceinline__ Hit closest_hit_brute(const SceneDev& sc, const RayW& rw, float tmin, int last) {
    Hit h{kInf, -1, 0x7fffffff};
    for (uint32_t j = 0; j < sc.n_tri; ++j) consider(sc, rw, (int)j, tmin, last, h);
    return h;
}

template <bool kBrute, bool kStats>
__global__ void __launch_bounds__(128) k_propagate_lane(const SceneDev sc, uint64_t n, uint64_t id_base,
                                                        const float* __restrict__ origins, const float* __restrict__ dirs,
                                                        const float* __restrict__ wl, uint64_t seed, opx_hits out,
                                                        unsigned long long* stats) {
    const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    if (sc.d_n) n = min(n, (uint64_t)__ldg(sc.d_n));
    if (i >= n) return;
    Photon p;
    photon_init(p, origins[3 * i], origins[3 * i + 1], origins[3 * i + 2], dirs[3 * i], dirs[3 * i + 1], dirs[3 * i + 2], wl[i], id_base + i);
    Work work;
    unsigned int segments = 0, interactions = 0;
    for (;;) {
        const RayW rw = ray_setup(p.ox, p.oy, p.oz, p.dx, p.dy, p.dz);
        const float tmin = p.b == 0 ? 0.f : sc.t_min;
        Hit h;
        if (kBrute) h = closest_hit_brute(sc, rw, tmin, p.last);
        else h = closest_hit_lane<kStats>(sc, rw, slab_setup(p.ox, p.oy, p.oz, p.dx, p.dy, p.dz),
                                          fmaxf(fmaxf(fabsf(p.ox), fabsf(p.oy)), fabsf(p.oz)) * 9.5367431640625e-7f, tmin, p.last, work);
        if (kStats) { ++segments; if (h.j >= 0) ++interactions; }
        if (!interact(sc, h, rw, p, seed)) break;
    }
    if (kStats) {
        const unsigned int mask = __activemask();
        const unsigned int v[4] = {segments, work.nodes, work.tris, interactions};
        for (int k = 0; k < 4; ++k) {
            const unsigned int sum = __reduce_add_sync(mask, v[k]);
            if ((threadIdx.x & 31) == (unsigned)(__ffs(mask) - 1)) atomicAdd(&stats[k], (unsigned long long)sum);
        }
        return;
    }
    store_record(out, i, p);
}

}  // namespace
}  // namespace opx
