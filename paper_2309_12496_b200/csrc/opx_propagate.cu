// A5-A12: per-photon propagation (k_propagate), hit binning + counters (k_bin).
// Arithmetic follows DESIGN.md section 3 operation by operation: every contract operation is an
// explicit round-to-nearest intrinsic (__fmul_rn, __fsub_rn, __fmaf_rn, __fdiv_rn), so the result
// does not depend on the compiler's contraction choices.  Shares nothing with oracle/.
#include "opx_internal.cuh"

namespace opx {

namespace {

constexpr float kInf = __builtin_huge_valf();
constexpr int kStack = 96;   // >= depth bound of a Karras tree over 63-bit keys + 32-bit index tie-break

// ---------------------------------------------------------------------------- Philox4x32-10 (3.1)
__device__ __forceinline__ float philox_uniform(uint64_t seed, uint64_t g, uint32_t b) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    uint32_t c0 = (uint32_t)g, c1 = (uint32_t)(g >> 32), c2 = b, c3 = 0u;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return __fmul_rn((float)(c0 >> 8), 5.9604644775390625e-8f);   // 2^-24, exact
}

// ------------------------------------------------------------------------------ table lookup (3.2)
__device__ __forceinline__ float table_lerp(const float* __restrict__ y, uint32_t n_lambda, float lambda_min,
                                            float inv_dl, float lambda) {
    const float x = __fmul_rn(__fsub_rn(lambda, lambda_min), inv_dl);
    const float xf = floorf(x);
    int j;
    if (!(xf >= 0.f)) j = 0;
    else if (xf > (float)(n_lambda - 2)) j = (int)n_lambda - 2;
    else j = (int)xf;
    float f = __fsub_rn(x, (float)j);
    if (!(f >= 0.f)) f = 0.f;
    if (f > 1.f) f = 1.f;
    const float y0 = __ldg(y + j), y1 = __ldg(y + j + 1);
    return __fmaf_rn(f, __fsub_rn(y1, y0), y0);
}

// ------------------------------------------------------------------------------- ray set-up (3.3)
struct RayW {                 // watertight-test constants of one segment
    float okx, oky, okz;      // origin permuted to (kx, ky, kz)
    float Sx, Sy, Sz;
    int kx, ky, kz;
};

__device__ __forceinline__ float sel3(float x, float y, float z, int k) { return k == 0 ? x : (k == 1 ? y : z); }

__device__ __forceinline__ RayW ray_setup(float ox, float oy, float oz, float dx, float dy, float dz) {
    RayW r;
    int kz = 0;
    float best = fabsf(dx);
    if (fabsf(dy) > best) { kz = 1; best = fabsf(dy); }
    if (fabsf(dz) > best) { kz = 2; }
    int kx = kz == 2 ? 0 : kz + 1;
    int ky = kx == 2 ? 0 : kx + 1;
    const float dkz = sel3(dx, dy, dz, kz);
    if (dkz < 0.f) { const int t = kx; kx = ky; ky = t; }
    r.kx = kx; r.ky = ky; r.kz = kz;
    r.Sx = __fdiv_rn(sel3(dx, dy, dz, kx), dkz);
    r.Sy = __fdiv_rn(sel3(dx, dy, dz, ky), dkz);
    r.Sz = __fdiv_rn(1.f, dkz);
    r.okx = sel3(ox, oy, oz, kx); r.oky = sel3(ox, oy, oz, ky); r.okz = sel3(ox, oy, oz, kz);
    return r;
}

// Contract triangle test.  Returns true with t when the triangle is hit at finite t > tmin.
__device__ __forceinline__ bool tri_test(const RayW& r, const float4 a, const float4 b, const float4 c, float tmin, float& t_out) {
    const float Akx = __fsub_rn(sel3(a.x, a.y, a.z, r.kx), r.okx), Aky = __fsub_rn(sel3(a.x, a.y, a.z, r.ky), r.oky), Akz = __fsub_rn(sel3(a.x, a.y, a.z, r.kz), r.okz);
    const float Bkx = __fsub_rn(sel3(b.x, b.y, b.z, r.kx), r.okx), Bky = __fsub_rn(sel3(b.x, b.y, b.z, r.ky), r.oky), Bkz = __fsub_rn(sel3(b.x, b.y, b.z, r.kz), r.okz);
    const float Ckx = __fsub_rn(sel3(c.x, c.y, c.z, r.kx), r.okx), Cky = __fsub_rn(sel3(c.x, c.y, c.z, r.ky), r.oky), Ckz = __fsub_rn(sel3(c.x, c.y, c.z, r.kz), r.okz);
    const float Ax = __fmaf_rn(-r.Sx, Akz, Akx), Ay = __fmaf_rn(-r.Sy, Akz, Aky);
    const float Bx = __fmaf_rn(-r.Sx, Bkz, Bkx), By = __fmaf_rn(-r.Sy, Bkz, Bky);
    const float Cx = __fmaf_rn(-r.Sx, Ckz, Ckx), Cy = __fmaf_rn(-r.Sy, Ckz, Cky);
    const float U = __fsub_rn(__fmul_rn(Cx, By), __fmul_rn(Cy, Bx));
    const float V = __fsub_rn(__fmul_rn(Ax, Cy), __fmul_rn(Ay, Cx));
    const float W = __fsub_rn(__fmul_rn(Bx, Ay), __fmul_rn(By, Ax));
    float t;
    if (U == 0.f || V == 0.f || W == 0.f) {
        const double Ud = __dsub_rn(__dmul_rn((double)Cx, (double)By), __dmul_rn((double)Cy, (double)Bx));
        const double Vd = __dsub_rn(__dmul_rn((double)Ax, (double)Cy), __dmul_rn((double)Ay, (double)Cx));
        const double Wd = __dsub_rn(__dmul_rn((double)Bx, (double)Ay), __dmul_rn((double)By, (double)Ax));
        if ((Ud < 0.0 || Vd < 0.0 || Wd < 0.0) && (Ud > 0.0 || Vd > 0.0 || Wd > 0.0)) return false;
        const double det = __dadd_rn(__dadd_rn(Ud, Vd), Wd);
        if (det == 0.0) return false;
        const double Az = (double)__fmul_rn(r.Sz, Akz), Bz = (double)__fmul_rn(r.Sz, Bkz), Cz = (double)__fmul_rn(r.Sz, Ckz);
        const double T = __fma_rn(Wd, Cz, __fma_rn(Vd, Bz, __dmul_rn(Ud, Az)));
        t = __double2float_rn(__ddiv_rn(T, det));
    } else {
        if ((U < 0.f || V < 0.f || W < 0.f) && (U > 0.f || V > 0.f || W > 0.f)) return false;
        const float det = __fadd_rn(__fadd_rn(U, V), W);
        if (det == 0.f) return false;
        const float Az = __fmul_rn(r.Sz, Akz), Bz = __fmul_rn(r.Sz, Bkz), Cz = __fmul_rn(r.Sz, Ckz);
        const float T = __fmaf_rn(W, Cz, __fmaf_rn(V, Bz, __fmul_rn(U, Az)));
        t = __fdiv_rn(T, det);
    }
    if (!(fabsf(t) < kInf) || !(t > tmin)) return false;      // NaN and +-inf rejected
    t_out = t;
    return true;
}

struct Hit { float t; int j; int gid; };   // j: leaf-order index; gid: global triangle id
struct Work { unsigned int nodes = 0, tris = 0; };   // instrumented build only

__device__ __forceinline__ void consider(const SceneDev& sc, const RayW& rw, int j, float tmin, int last, Hit& h) {
    const float4 a = __ldg(sc.tris + 3 * (size_t)j), b = __ldg(sc.tris + 3 * (size_t)j + 1), c = __ldg(sc.tris + 3 * (size_t)j + 2);
    const int gid = __float_as_int(a.w);
    if (gid == last) return;
    float t;
    if (!tri_test(rw, a, b, c, tmin, t)) return;
    if (t < h.t || (t == h.t && gid < h.gid)) { h.t = t; h.j = j; h.gid = gid; }
}

// Closest hit through the BVH: near child first, cull on t_entry > t_best (ties kept so that the
// (t, id) tie-break sees every candidate).  Boxes are padded at build time, which is
// what makes the cheap fma slab test conservative with respect to the contract triangle test.
template <bool kStats>
__device__ __forceinline__ Hit closest_hit_bvh(const SceneDev& sc, const RayW& rw, float ox, float oy, float oz,
                                               float dx, float dy, float dz, float tmin, int last, Work& work) {
    Hit h{kInf, -1, 0x7fffffff};
    const float ix = __fdiv_rn(1.f, dx), iy = __fdiv_rn(1.f, dy), iz = __fdiv_rn(1.f, dz);
    const float px = -ox * ix, py = -oy * iy, pz = -oz * iz;
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
            // child 0: lo = (q0.x,q0.y,q0.z) hi = (q0.w,q1.x,q1.y); child 1: lo = (q1.z,q1.w,q2.x) hi = (q2.y,q2.z,q2.w)
            float a, b;
            a = __fmaf_rn(q0.x, ix, px); b = __fmaf_rn(q0.w, ix, px);
            float n0 = fminf(a, b), f0 = fmaxf(a, b);
            a = __fmaf_rn(q0.y, iy, py); b = __fmaf_rn(q1.x, iy, py);
            n0 = fmaxf(n0, fminf(a, b)); f0 = fminf(f0, fmaxf(a, b));
            a = __fmaf_rn(q0.z, iz, pz); b = __fmaf_rn(q1.y, iz, pz);
            n0 = fmaxf(n0, fminf(a, b)); f0 = fminf(f0, fmaxf(a, b));
            a = __fmaf_rn(q1.z, ix, px); b = __fmaf_rn(q2.y, ix, px);
            float n1 = fminf(a, b), f1 = fmaxf(a, b);
            a = __fmaf_rn(q1.w, iy, py); b = __fmaf_rn(q2.z, iy, py);
            n1 = fmaxf(n1, fminf(a, b)); f1 = fminf(f1, fmaxf(a, b));
            a = __fmaf_rn(q2.x, iz, pz); b = __fmaf_rn(q2.w, iz, pz);
            n1 = fmaxf(n1, fminf(a, b)); f1 = fminf(f1, fmaxf(a, b));
            n0 = fmaxf(n0, 0.f); n1 = fmaxf(n1, 0.f);
            f0 = fminf(f0, h.t) * 1.0000004f; f1 = fminf(f1, h.t) * 1.0000004f;
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
        // pop
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

// ------------------------------------------------------------------------------ the photon loop
template <bool kBrute, bool kStats>
__global__ void __launch_bounds__(128) k_propagate(const SceneDev sc, uint64_t n, uint64_t id_base,
                                                   const float* __restrict__ origins, const float* __restrict__ dirs,
                                                   const float* __restrict__ wl, uint64_t seed, opx_hits out,
                                                   unsigned long long* stats) {
    const uint64_t i = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    float ox = origins[3 * i], oy = origins[3 * i + 1], oz = origins[3 * i + 2];
    float dx = dirs[3 * i], dy = dirs[3 * i + 1], dz = dirs[3 * i + 2];
    const float lambda = wl[i];
    const uint64_t g = id_base + i;
    uint32_t b = 0;
    int last = -1;
    int state, surface = -1, pixel = -1;
    float px = ox, py = oy, pz = oz;
    Work work;
    unsigned int segments = 0, interactions = 0;
    for (;;) {
        const RayW rw = ray_setup(ox, oy, oz, dx, dy, dz);
        const float tmin = b == 0 ? 0.f : sc.t_min;
        const Hit h = kBrute ? closest_hit_brute(sc, rw, tmin, last)
                             : closest_hit_bvh<kStats>(sc, rw, ox, oy, oz, dx, dy, dz, tmin, last, work);
        if (kStats) { ++segments; if (h.j >= 0) ++interactions; }
        if (h.j < 0) { state = OPX_ESCAPED; px = ox; py = oy; pz = oz; surface = -1; break; }
        px = __fmaf_rn(h.t, dx, ox); py = __fmaf_rn(h.t, dy, oy); pz = __fmaf_rn(h.t, dz, oz);
        const float4 nrm = __ldg(sc.normals + h.j);
        surface = __float_as_int(nrm.w);
        const int2 sf = __ldg(sc.surfaces + surface);
        const uint32_t kind = __ldg(sc.mat_kinds + sf.x);
        const float* table = sc.tables + (size_t)sf.x * sc.n_lambda;
        if (kind == OPX_MAT_ABSORBER) { state = OPX_ABSORBED_SURFACE; break; }
        if (kind == OPX_MAT_MIRROR) {
            const float u = philox_uniform(seed, g, b);
            if (!(u < table_lerp(table, sc.n_lambda, sc.lambda_min, sc.inv_dlambda, lambda))) { state = OPX_ABSORBED_MIRROR; break; }
            const float c = __fmaf_rn(dz, nrm.z, __fmaf_rn(dy, nrm.y, __fmul_rn(dx, nrm.x)));   // 3.5
            const float m2c = __fmul_rn(-2.f, c);
            dx = __fmaf_rn(m2c, nrm.x, dx); dy = __fmaf_rn(m2c, nrm.y, dy); dz = __fmaf_rn(m2c, nrm.z, dz);
            ox = px; oy = py; oz = pz; last = h.gid; ++b;
            if (b == sc.max_bounces) { state = OPX_BOUNCE_LIMIT; break; }
            continue;
        }
        // detector (3.6)
        const FrameDev* f = sc.frames + sf.y;
        const float4 f0 = __ldg(reinterpret_cast<const float4*>(f)), f1 = __ldg(reinterpret_cast<const float4*>(f) + 1),
                     f2 = __ldg(reinterpret_cast<const float4*>(f) + 2);
        const uint4 f3 = __ldg(reinterpret_cast<const uint4*>(f) + 3);
        const float qx = __fsub_rn(px, f0.x), qy = __fsub_rn(py, f0.y), qz = __fsub_rn(pz, f0.z);
        const float ca = __fmaf_rn(qz, f1.y, __fmaf_rn(qy, f1.x, __fmul_rn(qx, f0.w)));
        const float cb = __fmaf_rn(qz, f2.x, __fmaf_rn(qy, f1.w, __fmul_rn(qx, f1.z)));
        const float fu = floorf(__fmul_rn(ca, f2.y)), fv = floorf(__fmul_rn(cb, f2.z));
        if (!(fu >= 0.f) || !(fv >= 0.f) || !(fu < (float)f3.x) || !(fv < (float)f3.y)) { state = OPX_DETECTOR_DEAD; break; }
        pixel = (int)(f3.z + (uint32_t)fv * f3.x + (uint32_t)fu);
        const float u = philox_uniform(seed, g, b);
        state = (u < table_lerp(table, sc.n_lambda, sc.lambda_min, sc.inv_dlambda, lambda)) ? OPX_DETECTED : OPX_QE_REJECTED;
        break;
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
    out.pos[3 * i] = px; out.pos[3 * i + 1] = py; out.pos[3 * i + 2] = pz;
    out.dir[3 * i] = dx; out.dir[3 * i + 1] = dy; out.dir[3 * i + 2] = dz;
    out.pixel[i] = pixel; out.surface[i] = surface;
    out.state[i] = (uint8_t)state; out.bounces[i] = (uint8_t)b;
}

// ---------------------------------------------------------------- A11 hit binning + A12 counters
// One thread per photon; detected photons of a warp that share a pixel are merged with
// __match_any_sync so that a ring concentrated on a few hundred pixels costs one atomic per
// distinct pixel per warp.  Integer adds only, so the result does not depend on the order.
__global__ void __launch_bounds__(256) k_bin(const uint8_t* __restrict__ state, const uint8_t* __restrict__ bounces,
                                             const int32_t* __restrict__ pixel, uint64_t n, uint32_t* hitmap,
                                             unsigned long long* counters) {
    __shared__ unsigned int s_cnt[8];
    if (threadIdx.x < 8) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
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

opx_status launch_propagate(const SceneHost& s, bool brute, uint64_t n, uint64_t id_base, const float* o, const float* d,
                            const float* wl, uint64_t seed, const opx_hits& out, uint32_t* hitmap, uint64_t* counters,
                            cudaStream_t stream) {
    const uint64_t blocks = (n + 127) / 128;
    if (blocks > 0x7fffffffull) return fail(OPX_ERR_INVALID_ARG, "n too large for one launch");
    cudaEvent_t* ev = nullptr;
    if (s.prof_used < s.prof_max) { ev = &s.prof_events[3 * (size_t)s.prof_used]; ++s.prof_used; }
    if (ev) cudaEventRecord(ev[0], stream);
    // a scene with fewer than two triangles has no hierarchy: test the triangle list directly
    if (brute || s.dev.n_tri < 2) k_propagate<true, false><<<(unsigned)blocks, 128, 0, stream>>>(s.dev, n, id_base, o, d, wl, seed, out, nullptr);
    else k_propagate<false, false><<<(unsigned)blocks, 128, 0, stream>>>(s.dev, n, id_base, o, d, wl, seed, out, nullptr);
    count_launch(1);
    if (ev) cudaEventRecord(ev[1], stream);
    if (hitmap || counters) {
        const uint64_t bb = (n + 255) / 256;
        const unsigned grid = (unsigned)(bb < 148ull * 8 ? bb : 148ull * 8);
        k_bin<<<grid, 256, 0, stream>>>(out.state, out.bounces, out.pixel, n, hitmap, (unsigned long long*)counters);
        count_launch(1);
    }
    if (ev) cudaEventRecord(ev[2], stream);
    return check_cuda(cudaGetLastError(), "propagate launch");
}

opx_status launch_stats(const SceneHost& s, uint64_t n, uint64_t id_base, const float* o, const float* d, const float* wl,
                        uint64_t seed, uint64_t* stats, cudaStream_t stream) {
    const uint64_t blocks = (n + 127) / 128;
    if (blocks > 0x7fffffffull) return fail(OPX_ERR_INVALID_ARG, "n too large for one launch");
    if (s.dev.n_tri < 2) return fail(OPX_ERR_BAD_STATE, "no hierarchy to instrument (fewer than two triangles)");
    k_propagate<false, true><<<(unsigned)blocks, 128, 0, stream>>>(s.dev, n, id_base, o, d, wl, seed, opx_hits{}, (unsigned long long*)stats);
    count_launch(1);
    return check_cuda(cudaGetLastError(), "stats launch");
}

}  // namespace opx
