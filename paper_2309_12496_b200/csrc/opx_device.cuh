// Device functions of the arithmetic contract, shared by the propagation kernels
// of opx_propagate.cu.  Every contract operation is an explicit round-to-nearest intrinsic
// (__fmul_rn, __fsub_rn, __fmaf_rn, __fdiv_rn): the result does not depend on contraction choices.
#pragma once
#include "opx_internal.cuh"

namespace opx {

__device__ constexpr float kInf = __builtin_huge_valf();

// ---------------------------------------------------------------------------- Philox4x32-10 (3.1)
// `stream` is counter word 3: 0 = in-flight draws (3.1), 1 = the pre-propagation filter (3.9).
__device__ __forceinline__ float philox_uniform(uint64_t seed, uint64_t g, uint32_t b, uint32_t stream = 0u) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    uint32_t c0 = (uint32_t)g, c1 = (uint32_t)(g >> 32), c2 = b, c3 = stream;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;     // one IMAD.WIDE each
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
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

// ------------------------------------------------------------------------ histogram lookup (3.8)
__device__ __forceinline__ float table_hist(const float* __restrict__ y, uint32_t n_lambda, float lambda_min,
                                            float inv_bin, float lambda) {
    const float xf = floorf(__fmul_rn(__fsub_rn(lambda, lambda_min), inv_bin));
    int j;
    if (!(xf >= 0.f)) j = 0;
    else if (xf > (float)(n_lambda - 1)) j = (int)n_lambda - 1;
    else j = (int)xf;
    return __ldg(y + j);
}

// e_m(lambda): efficiency of material m in its own table form; mk = mat_kinds[m] (kind | interp << 8).
__device__ __forceinline__ float table_value(const SceneDev& sc, uint32_t m, uint32_t mk, float lambda) {
    const float* y = sc.tables + (size_t)m * sc.n_lambda;
    if ((mk >> 8) == OPX_TABLE_HISTOGRAM) return table_hist(y, sc.n_lambda, sc.lambda_min, sc.inv_bin, lambda);
    return table_lerp(y, sc.n_lambda, sc.lambda_min, sc.inv_dlambda, lambda);
}

// --------------------------------------------------------------------- pre-propagation filter (3.9)
constexpr int kMaxFactors = 8;
struct FilterFactors { uint32_t m[kMaxFactors]; uint32_t mk[kMaxFactors]; uint32_t n; };   // material indices, their mat_kinds words

// p = e_0(lambda) * e_1(lambda) * ... left to right in fp32 (1 for an empty list)
__device__ __forceinline__ float filter_probability(const SceneDev& sc, const FilterFactors& fa, float lambda) {
    float p = 1.f;
#pragma unroll
    for (uint32_t k = 0; k < (uint32_t)kMaxFactors; ++k) {       // unrolled: the factor list is read with constant indices
        if (k >= fa.n) break;
        const float e = table_value(sc, fa.m[k], fa.mk[k], lambda);
        p = k == 0 ? e : __fmul_rn(p, e);
    }
    return p;
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

// The same set-up for a segment stored as o[3], d[3] in (shared) memory: the permuted components are fetched with
// indexed loads instead of register selects.  Same values, same operations.
__device__ __forceinline__ RayW ray_setup_mem(const float* o, const float* d) {
    RayW r;
    const float dx = d[0], dy = d[1], dz = d[2];
    int kz = 0;
    float best = fabsf(dx);
    if (fabsf(dy) > best) { kz = 1; best = fabsf(dy); }
    if (fabsf(dz) > best) { kz = 2; }
    int kx = kz == 2 ? 0 : kz + 1;
    int ky = kx == 2 ? 0 : kx + 1;
    const float dkz = d[kz];
    if (dkz < 0.f) { const int t = kx; kx = ky; ky = t; }
    r.kx = kx; r.ky = ky; r.kz = kz;
    r.Sx = __fdiv_rn(d[kx], dkz);
    r.Sy = __fdiv_rn(d[ky], dkz);
    r.Sz = __fdiv_rn(1.f, dkz);
    r.okx = o[kx]; r.oky = o[ky]; r.okz = o[kz];
    return r;
}

// Packet kernels: the same constants WITHOUT the exchange of kx and ky for a negative d[kz], and with the triangle record
// read from the copy whose components are already rotated to (kx, ky, kz) = (kz+1, kz+2, kz) mod 3 (SceneDev::tris holds the
// three rotations one after the other), so that a vertex is one 16-byte load and no component is ever selected.
// Dropping the exchange changes no result bit: with kx and ky exchanged, Sx <-> Sy and (Ax, Ay) <-> (Ay, Ax) for every
// vertex, so each edge function U = Cx By - Cy Bx (two rounded products, one rounded difference) turns into exactly -U;
// likewise det -> -det and T -> -T (every fma operand pair changes one sign), so t = T / det, the zero tests, the
// both-signs rejection and the fp64 branch are unchanged; the shading normal m -> -m gives n -> -n, and the reflection
// fma(-2 (d.n), n, d) is even in n operation by operation.  tests/test_gpu_parity.py compares this path with the oracle, which
// does exchange, and with the per-lane kernel of opx_lane.cuh, which does too.
struct RayR {
    float okx, oky, okz;      // origin permuted to (kx, ky, kz)
    float Sx, Sy, Sz;
    uint32_t toff;            // float4 offset of the rotation of the triangle array this ray reads: kx * 3 * n_tri
};

__device__ __forceinline__ RayR ray_setup_rot(const float* o, const float* d, uint32_t n_tri) {
    RayR r;
    const float dx = d[0], dy = d[1], dz = d[2];
    int kz = 0;
    float best = fabsf(dx);
    if (fabsf(dy) > best) { kz = 1; best = fabsf(dy); }
    if (fabsf(dz) > best) { kz = 2; }
    const int kx = kz == 2 ? 0 : kz + 1;
    const int ky = kx == 2 ? 0 : kx + 1;
    const float dkz = d[kz];
    r.Sx = __fdiv_rn(d[kx], dkz);
    r.Sy = __fdiv_rn(d[ky], dkz);
    r.Sz = __fdiv_rn(1.f, dkz);
    r.okx = o[kx]; r.oky = o[ky]; r.okz = o[kz];
    r.toff = (uint32_t)kx * 3u * n_tri;      // rotation 0 = (x, y, z) for kz = 2, 1 = (y, z, x) for kz = 0, 2 = (z, x, y) for kz = 1
    return r;
}

// The exact-zero branch of the contract test: all three edge functions recomputed as differences of exact
// fp64 products, sign test, determinant and T in fp64.  Out of line on purpose: it runs for rays through a vertex or along
// an edge only, and inlined into every leaf loop it was a third of their code.
static __device__ __noinline__ bool tri_test_exact(float Ax, float Ay, float Bx, float By, float Cx, float Cy, float Az, float Bz, float Cz, float& t) {
    const double Ud = __dsub_rn(__dmul_rn((double)Cx, (double)By), __dmul_rn((double)Cy, (double)Bx));
    const double Vd = __dsub_rn(__dmul_rn((double)Ax, (double)Cy), __dmul_rn((double)Ay, (double)Cx));
    const double Wd = __dsub_rn(__dmul_rn((double)Bx, (double)Ay), __dmul_rn((double)By, (double)Ax));
    if ((Ud < 0.0 || Vd < 0.0 || Wd < 0.0) && (Ud > 0.0 || Vd > 0.0 || Wd > 0.0)) return false;
    const double det = __dadd_rn(__dadd_rn(Ud, Vd), Wd);
    if (det == 0.0) return false;
    const double T = __fma_rn(Wd, (double)Cz, __fma_rn(Vd, (double)Bz, __dmul_rn(Ud, (double)Az)));
    t = __double2float_rn(__ddiv_rn(T, det));
    return true;
}

// Contract triangle test on vertex components already permuted to (kx, ky, kz) and shifted to the ray
// origin (A = a - o, ...).  Returns true with t when the triangle is hit at finite t > tmin.
// Ray: RayW or RayR (only Sx, Sy, Sz are read).
template <class Ray>
__device__ __forceinline__ bool tri_test(const Ray& r, float Akx, float Aky, float Akz, float Bkx, float Bky, float Bkz,
                                         float Ckx, float Cky, float Ckz, float tmin, float& t_out) {
    const float Ax = __fmaf_rn(-r.Sx, Akz, Akx), Ay = __fmaf_rn(-r.Sy, Akz, Aky);
    const float Bx = __fmaf_rn(-r.Sx, Bkz, Bkx), By = __fmaf_rn(-r.Sy, Bkz, Bky);
    const float Cx = __fmaf_rn(-r.Sx, Ckz, Ckx), Cy = __fmaf_rn(-r.Sy, Ckz, Cky);
    const float U = __fsub_rn(__fmul_rn(Cx, By), __fmul_rn(Cy, Bx));
    const float V = __fsub_rn(__fmul_rn(Ax, Cy), __fmul_rn(Ay, Cx));
    const float W = __fsub_rn(__fmul_rn(Bx, Ay), __fmul_rn(By, Ax));
    float t;
    if (U == 0.f || V == 0.f || W == 0.f) {
        if (!tri_test_exact(Ax, Ay, Bx, By, Cx, Cy, __fmul_rn(r.Sz, Akz), __fmul_rn(r.Sz, Bkz), __fmul_rn(r.Sz, Ckz), t)) return false;
    } else {
        // (U<0 || V<0 || W<0) && (U>0 || V>0 || W>0): fminf/fmaxf skip a NaN operand exactly as the comparisons do
        if (fminf(fminf(U, V), W) < 0.f && fmaxf(fmaxf(U, V), W) > 0.f) return false;
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

// Tests leaf-order triangle j and keeps the lexicographic minimum of (t, global id).  The vertex
// components are fetched already permuted (per-lane offsets kx, ky, kz into the 48-byte record: the
// lanes of a warp read the same sectors), so no register selects are needed.
__device__ __forceinline__ void consider(const SceneDev& sc, const RayW& rw, int j, float tmin, int last, Hit& h) {
    const float* t = reinterpret_cast<const float*>(sc.tris + 3 * (size_t)j);
    const int gid = __float_as_int(__ldg(t + 3));      // all ten loads are issued before the first use: one latency, not two
    const float Akx = __fsub_rn(__ldg(t + rw.kx), rw.okx), Aky = __fsub_rn(__ldg(t + rw.ky), rw.oky), Akz = __fsub_rn(__ldg(t + rw.kz), rw.okz);
    const float Bkx = __fsub_rn(__ldg(t + 4 + rw.kx), rw.okx), Bky = __fsub_rn(__ldg(t + 4 + rw.ky), rw.oky), Bkz = __fsub_rn(__ldg(t + 4 + rw.kz), rw.okz);
    const float Ckx = __fsub_rn(__ldg(t + 8 + rw.kx), rw.okx), Cky = __fsub_rn(__ldg(t + 8 + rw.ky), rw.oky), Ckz = __fsub_rn(__ldg(t + 8 + rw.kz), rw.okz);
    if (gid == last) return;
    float tt;
    if (!tri_test(rw, Akx, Aky, Akz, Bkx, Bky, Bkz, Ckx, Cky, Ckz, tmin, tt)) return;
    if (tt < h.t || (tt == h.t && gid < h.gid)) { h.t = tt; h.j = j; h.gid = gid; }
}

// The same for a packet kernel's ray: three 16-byte loads from the ray's rotation of the triangle array; the triangle just
// left is recognised by its leaf-order index, so no load sits in front of the test.
__device__ __forceinline__ void consider_rot(const SceneDev& sc, const RayR& r, int j, float tmin, int last_j, Hit& h) {
    const float4* t = sc.tris + (r.toff + 3u * (uint32_t)j);
    const float4 a = __ldg(t), b = __ldg(t + 1), c = __ldg(t + 2);
    if (j == last_j) return;
    float tt;
    if (!tri_test(r, __fsub_rn(a.x, r.okx), __fsub_rn(a.y, r.oky), __fsub_rn(a.z, r.okz), __fsub_rn(b.x, r.okx), __fsub_rn(b.y, r.oky),
                  __fsub_rn(b.z, r.okz), __fsub_rn(c.x, r.okx), __fsub_rn(c.y, r.oky), __fsub_rn(c.z, r.okz), tmin, tt)) return;
    const int gid = __float_as_int(a.w);
    if (tt < h.t || (tt == h.t && gid < h.gid)) { h.t = tt; h.j = j; h.gid = gid; }
}

// Shading normal of DESIGN.md 3.11 for the hit on leaf-order triangle j (global id gid): the vertex normals weighted by
// the fp32 edge functions U, V, W of 3.3, recomputed here for the one winning triangle (same operations on the same
// inputs as tri_test, hence the same bits) so that the traversal loop does not have to carry them.  Returns false when
// the face normal applies (no vertex normals on this triangle, or a degenerate sum).
__device__ __forceinline__ bool shading_normal(const SceneDev& sc, const RayW& r, int j, int gid, float& nx, float& ny, float& nz) {
    const float* t = reinterpret_cast<const float*>(sc.tris + 3 * (size_t)j);
    const float Akx = __fsub_rn(__ldg(t + r.kx), r.okx), Aky = __fsub_rn(__ldg(t + r.ky), r.oky), Akz = __fsub_rn(__ldg(t + r.kz), r.okz);
    const float Bkx = __fsub_rn(__ldg(t + 4 + r.kx), r.okx), Bky = __fsub_rn(__ldg(t + 4 + r.ky), r.oky), Bkz = __fsub_rn(__ldg(t + 4 + r.kz), r.okz);
    const float Ckx = __fsub_rn(__ldg(t + 8 + r.kx), r.okx), Cky = __fsub_rn(__ldg(t + 8 + r.ky), r.oky), Ckz = __fsub_rn(__ldg(t + 8 + r.kz), r.okz);
    const float Ax = __fmaf_rn(-r.Sx, Akz, Akx), Ay = __fmaf_rn(-r.Sy, Akz, Aky);
    const float Bx = __fmaf_rn(-r.Sx, Bkz, Bkx), By = __fmaf_rn(-r.Sy, Bkz, Bky);
    const float Cx = __fmaf_rn(-r.Sx, Ckz, Ckx), Cy = __fmaf_rn(-r.Sy, Ckz, Cky);
    const float U = __fsub_rn(__fmul_rn(Cx, By), __fmul_rn(Cy, Bx));
    const float V = __fsub_rn(__fmul_rn(Ax, Cy), __fmul_rn(Ay, Cx));
    const float W = __fsub_rn(__fmul_rn(Bx, Ay), __fmul_rn(By, Ax));
    const float* vn = sc.vnormals + 9 * (size_t)gid;
    const float mx = __fmaf_rn(W, __ldg(vn + 6), __fmaf_rn(V, __ldg(vn + 3), __fmul_rn(U, __ldg(vn + 0))));
    const float my = __fmaf_rn(W, __ldg(vn + 7), __fmaf_rn(V, __ldg(vn + 4), __fmul_rn(U, __ldg(vn + 1))));
    const float mz = __fmaf_rn(W, __ldg(vn + 8), __fmaf_rn(V, __ldg(vn + 5), __fmul_rn(U, __ldg(vn + 2))));
    const float len2 = __fmaf_rn(mz, mz, __fmaf_rn(my, my, __fmul_rn(mx, mx)));
    if (!(len2 > 0.f) || !(len2 < kInf)) return false;
    const float inv = __fdiv_rn(1.f, __fsqrt_rn(len2));
    nx = __fmul_rn(mx, inv); ny = __fmul_rn(my, inv); nz = __fmul_rn(mz, inv);
    return true;
}

__device__ __forceinline__ bool shading_normal(const SceneDev& sc, const RayR& r, int j, int gid, float& nx, float& ny, float& nz) {
    const float4* t = sc.tris + (r.toff + 3u * (uint32_t)j);
    const float4 a = __ldg(t), b = __ldg(t + 1), c = __ldg(t + 2);
    const float Akx = __fsub_rn(a.x, r.okx), Aky = __fsub_rn(a.y, r.oky), Akz = __fsub_rn(a.z, r.okz);
    const float Bkx = __fsub_rn(b.x, r.okx), Bky = __fsub_rn(b.y, r.oky), Bkz = __fsub_rn(b.z, r.okz);
    const float Ckx = __fsub_rn(c.x, r.okx), Cky = __fsub_rn(c.y, r.oky), Ckz = __fsub_rn(c.z, r.okz);
    const float Ax = __fmaf_rn(-r.Sx, Akz, Akx), Ay = __fmaf_rn(-r.Sy, Akz, Aky);
    const float Bx = __fmaf_rn(-r.Sx, Bkz, Bkx), By = __fmaf_rn(-r.Sy, Bkz, Bky);
    const float Cx = __fmaf_rn(-r.Sx, Ckz, Ckx), Cy = __fmaf_rn(-r.Sy, Ckz, Cky);
    const float U = __fsub_rn(__fmul_rn(Cx, By), __fmul_rn(Cy, Bx));
    const float V = __fsub_rn(__fmul_rn(Ax, Cy), __fmul_rn(Ay, Cx));
    const float W = __fsub_rn(__fmul_rn(Bx, Ay), __fmul_rn(By, Ax));
    const float* vn = sc.vnormals + 9 * (size_t)gid;
    const float mx = __fmaf_rn(W, __ldg(vn + 6), __fmaf_rn(V, __ldg(vn + 3), __fmul_rn(U, __ldg(vn + 0))));
    const float my = __fmaf_rn(W, __ldg(vn + 7), __fmaf_rn(V, __ldg(vn + 4), __fmul_rn(U, __ldg(vn + 1))));
    const float mz = __fmaf_rn(W, __ldg(vn + 8), __fmaf_rn(V, __ldg(vn + 5), __fmul_rn(U, __ldg(vn + 2))));
    const float len2 = __fmaf_rn(mz, mz, __fmaf_rn(my, my, __fmul_rn(mx, mx)));
    if (!(len2 > 0.f) || !(len2 < kInf)) return false;
    const float inv = __fdiv_rn(1.f, __fsqrt_rn(len2));
    nx = __fmul_rn(mx, inv); ny = __fmul_rn(my, inv); nz = __fmul_rn(mz, inv);
    return true;
}

// ------------------------------------------------------------------- photon state + interaction
struct Photon {
    float ox, oy, oz, dx, dy, dz;      // current segment
    float px, py, pz;                   // record position
    float lambda;
    uint64_t g;                         // global photon id
    uint32_t b;                         // reflections so far
    int last, state, surface, pixel;
};

__device__ __forceinline__ void photon_init(Photon& p, float ox, float oy, float oz, float dx, float dy, float dz,
                                            float lambda, uint64_t g) {
    p.ox = ox; p.oy = oy; p.oz = oz; p.dx = dx; p.dy = dy; p.dz = dz; p.px = ox; p.py = oy; p.pz = oz;
    p.lambda = lambda; p.g = g; p.b = 0; p.last = -1; p.state = -1; p.surface = -1; p.pixel = -1;
}

// Applies the outcome of one closest-hit query.  Returns true when the photon
// was reflected and continues with a new segment; otherwise p.state holds the terminal state.
// rw: the watertight-test constants of the segment that produced h (needed for the shading normal only).
template <class Ray>
__device__ __forceinline__ bool interact(const SceneDev& sc, const Hit& h, const Ray& rw, Photon& p, uint64_t seed) {
    if (h.j < 0) { p.state = OPX_ESCAPED; p.px = p.ox; p.py = p.oy; p.pz = p.oz; p.surface = -1; return false; }
    p.px = __fmaf_rn(h.t, p.dx, p.ox); p.py = __fmaf_rn(h.t, p.dy, p.oy); p.pz = __fmaf_rn(h.t, p.dz, p.oz);   // 3.7
    const float4 nrm = __ldg(sc.normals + h.j);
    p.surface = __float_as_int(nrm.w);
    const int2 sf = __ldg(sc.surfaces + p.surface);
    const uint32_t mk = __ldg(sc.mat_kinds + sf.x), kind = mk & 0xffu;
    const bool draw = !(sc.flags & OPX_FLAG_NO_EFFICIENCY);                                       // 3.10
    if (kind == OPX_MAT_ABSORBER) { p.state = OPX_ABSORBED_SURFACE; return false; }
    if (kind == OPX_MAT_MIRROR) {
        if (draw && !(philox_uniform(seed, p.g, p.b) < table_value(sc, (uint32_t)sf.x, mk, p.lambda))) { p.state = OPX_ABSORBED_MIRROR; return false; }
        float nx = nrm.x, ny = nrm.y, nz = nrm.z;
        if (sc.vnormals) shading_normal(sc, rw, h.j, h.gid, nx, ny, nz);                           // 3.11 (face normal kept on false)
        const float c = __fmaf_rn(p.dz, nz, __fmaf_rn(p.dy, ny, __fmul_rn(p.dx, nx)));             // 3.5
        const float m2c = __fmul_rn(-2.f, c);
        p.dx = __fmaf_rn(m2c, nx, p.dx); p.dy = __fmaf_rn(m2c, ny, p.dy); p.dz = __fmaf_rn(m2c, nz, p.dz);
        p.ox = p.px; p.oy = p.py; p.oz = p.pz; p.last = h.gid; ++p.b;
        if (p.b == sc.max_bounces) { p.state = OPX_BOUNCE_LIMIT; return false; }
        return true;
    }
    // detector (3.6)
    const float4* f = reinterpret_cast<const float4*>(sc.frames + sf.y);
    const float4 f0 = __ldg(f), f1 = __ldg(f + 1), f2 = __ldg(f + 2);
    const uint4 f3 = __ldg(reinterpret_cast<const uint4*>(f) + 3);
    const float qx = __fsub_rn(p.px, f0.x), qy = __fsub_rn(p.py, f0.y), qz = __fsub_rn(p.pz, f0.z);
    const float ca = __fmaf_rn(qz, f1.y, __fmaf_rn(qy, f1.x, __fmul_rn(qx, f0.w)));
    const float cb = __fmaf_rn(qz, f2.x, __fmaf_rn(qy, f1.w, __fmul_rn(qx, f1.z)));
    const float fu = floorf(__fmul_rn(ca, f2.y)), fv = floorf(__fmul_rn(cb, f2.z));
    if (!(fu >= 0.f) || !(fv >= 0.f) || !(fu < (float)f3.x) || !(fv < (float)f3.y)) { p.state = OPX_DETECTOR_DEAD; return false; }
    p.pixel = (int)(f3.z + (uint32_t)fv * f3.x + (uint32_t)fu);
    p.state = (!draw || philox_uniform(seed, p.g, p.b) < table_value(sc, (uint32_t)sf.x, mk, p.lambda)) ? OPX_DETECTED : OPX_QE_REJECTED;
    return false;
}

__device__ __forceinline__ void store_record(const opx_hits& out, uint64_t i, const Photon& p) {
    out.pos[3 * i] = p.px; out.pos[3 * i + 1] = p.py; out.pos[3 * i + 2] = p.pz;
    out.dir[3 * i] = p.dx; out.dir[3 * i + 1] = p.dy; out.dir[3 * i + 2] = p.dz;
    out.pixel[i] = p.pixel; out.surface[i] = p.surface;
    out.state[i] = (uint8_t)p.state; out.bounces[i] = (uint8_t)p.b;
}

// Slab test of one segment against the two child boxes of a node.  px = -o*inv_d.  The boxes are
// padded at build time (2^-16 of the largest scene coordinate + 2^-10 of the triangle's
// own extent), which is what makes this cheap form (approximate reciprocal, one fma per plane, no
// re-scaling of the exit distance) conservative with respect to tri_test for origins inside
// SceneDev::origin_limit; rays that start further out add their own slack (slab2_slack).
struct Slab { float ix, iy, iz, px, py, pz; };

// 1/d for the slab test, finite for every finite d: a component of +-0 (or a denormal) would give ix = +-inf and
// px = -o*ix = -+inf, and fma(plane, ix, px) = inf - inf = NaN whenever plane and origin share a sign -- the NaN-skipping
// fminf/fmaxf would then EMPTY the interval of a box the ray runs through.  With |d| clamped to 1e-30 (sign kept, so a
// component of -0 still belongs to the negative octant, see dir_octant) the planes of that axis land at -+1e30-ish: the
// axis constrains nothing when the origin is between the planes and rejects the box when it is not, which is what a ray
// parallel to the slab must do.  NaN stays NaN: every comparison fails and the ray hits no box.
__device__ __forceinline__ float slab_rcp(float d) {
    return __fdividef(1.f, fabsf(d) < 1e-30f ? copysignf(1e-30f, d) : d);
}

__device__ __forceinline__ Slab slab_setup(float ox, float oy, float oz, float dx, float dy, float dz) {
    Slab s;
    s.ix = slab_rcp(dx); s.iy = slab_rcp(dy); s.iz = slab_rcp(dz);
    s.px = -ox * s.ix; s.py = -oy * s.iy; s.pz = -oz * s.iz;
    return s;
}

// Sign octant of a direction from the SIGN BITS (bit a set = component a negative, -0 included): the octant-specialised
// slab test picks the entry plane by this, and slab_rcp keeps the sign of a zero, so the two always agree.
__device__ __forceinline__ int dir_octant(float dx, float dy, float dz) {
    return (int)(((unsigned)__float_as_int(dx) >> 31) | (((unsigned)__float_as_int(dy) >> 31) << 1) | (((unsigned)__float_as_int(dz) >> 31) << 2));
}

// child 0: lo = (q0.x,q0.y,q0.z) hi = (q0.w,q1.x,q1.y); child 1: lo = (q1.z,q1.w,q2.x) hi = (q2.y,q2.z,q2.w).
// tcap = t_best (or a negative number for a lane that must not hit anything).
__device__ __forceinline__ void slab2(const Slab& s, const float4 q0, const float4 q1, const float4 q2, float tcap,
                                      float& n0, float& f0, float& n1, float& f1) {
    float a, b;
    a = __fmaf_rn(q0.x, s.ix, s.px); b = __fmaf_rn(q0.w, s.ix, s.px);
    n0 = fminf(a, b); f0 = fmaxf(a, b);
    a = __fmaf_rn(q0.y, s.iy, s.py); b = __fmaf_rn(q1.x, s.iy, s.py);
    n0 = fmaxf(n0, fminf(a, b)); f0 = fminf(f0, fmaxf(a, b));
    a = __fmaf_rn(q0.z, s.iz, s.pz); b = __fmaf_rn(q1.y, s.iz, s.pz);
    n0 = fmaxf(n0, fminf(a, b)); f0 = fminf(f0, fmaxf(a, b));
    a = __fmaf_rn(q1.z, s.ix, s.px); b = __fmaf_rn(q2.y, s.ix, s.px);
    n1 = fminf(a, b); f1 = fmaxf(a, b);
    a = __fmaf_rn(q1.w, s.iy, s.py); b = __fmaf_rn(q2.z, s.iy, s.py);
    n1 = fmaxf(n1, fminf(a, b)); f1 = fminf(f1, fmaxf(a, b));
    a = __fmaf_rn(q2.x, s.iz, s.pz); b = __fmaf_rn(q2.w, s.iz, s.pz);
    n1 = fmaxf(n1, fminf(a, b)); f1 = fminf(f1, fmaxf(a, b));
    n0 = fmaxf(n0, 0.f); n1 = fmaxf(n1, 0.f);
    f0 = fminf(f0, tcap); f1 = fminf(f1, tcap);
}

// slab2 for a ray whose origin lies outside SceneDev::origin_limit: the contract test works on
// vertex - origin, whose rounding grows with |origin|, so the triangles it accepts may lie up to e = 2^-20 |origin|_inf
// outside their padded boxes.  Every box is widened by e on the fly: e |i_a| in the ray parameter of axis a.
__device__ __forceinline__ void slab2_slack(const Slab& s, float e, const float4 q0, const float4 q1, const float4 q2, float tcap,
                                            float& n0, float& f0, float& n1, float& f1) {
    const float ex = e * fabsf(s.ix), ey = e * fabsf(s.iy), ez = e * fabsf(s.iz);
    float a, b;
    a = __fmaf_rn(q0.x, s.ix, s.px); b = __fmaf_rn(q0.w, s.ix, s.px);
    n0 = fminf(a, b) - ex; f0 = fmaxf(a, b) + ex;
    a = __fmaf_rn(q0.y, s.iy, s.py); b = __fmaf_rn(q1.x, s.iy, s.py);
    n0 = fmaxf(n0, fminf(a, b) - ey); f0 = fminf(f0, fmaxf(a, b) + ey);
    a = __fmaf_rn(q0.z, s.iz, s.pz); b = __fmaf_rn(q1.y, s.iz, s.pz);
    n0 = fmaxf(n0, fminf(a, b) - ez); f0 = fminf(f0, fmaxf(a, b) + ez);
    a = __fmaf_rn(q1.z, s.ix, s.px); b = __fmaf_rn(q2.y, s.ix, s.px);
    n1 = fminf(a, b) - ex; f1 = fmaxf(a, b) + ex;
    a = __fmaf_rn(q1.w, s.iy, s.py); b = __fmaf_rn(q2.z, s.iy, s.py);
    n1 = fmaxf(n1, fminf(a, b) - ey); f1 = fminf(f1, fmaxf(a, b) + ey);
    a = __fmaf_rn(q2.x, s.iz, s.pz); b = __fmaf_rn(q2.w, s.iz, s.pz);
    n1 = fmaxf(n1, fminf(a, b) - ez); f1 = fminf(f1, fmaxf(a, b) + ez);
    n0 = fmaxf(n0, 0.f); n1 = fmaxf(n1, 0.f);
    f0 = fminf(f0, tcap); f1 = fminf(f1, tcap);
}

// The same test when the signs of the direction components are known at compile time (kOct bit 0/1/2
// set = dx/dy/dz negative): the entry plane of each axis is known, so no min/max per axis is needed.
template <int kOct>
__device__ __forceinline__ void slab2_oct(const Slab& s, const float4 q0, const float4 q1, const float4 q2, float tcap,
                                          float& n0, float& f0, float& n1, float& f1) {
    constexpr bool sx = kOct & 1, sy = kOct & 2, sz = kOct & 4;
    const float lx0 = q0.x, ly0 = q0.y, lz0 = q0.z, hx0 = q0.w, hy0 = q1.x, hz0 = q1.y;
    const float lx1 = q1.z, ly1 = q1.w, lz1 = q2.x, hx1 = q2.y, hy1 = q2.z, hz1 = q2.w;
    n0 = fmaxf(fmaxf(__fmaf_rn(sx ? hx0 : lx0, s.ix, s.px), __fmaf_rn(sy ? hy0 : ly0, s.iy, s.py)),
               fmaxf(__fmaf_rn(sz ? hz0 : lz0, s.iz, s.pz), 0.f));
    f0 = fminf(fminf(__fmaf_rn(sx ? lx0 : hx0, s.ix, s.px), __fmaf_rn(sy ? ly0 : hy0, s.iy, s.py)),
               fminf(__fmaf_rn(sz ? lz0 : hz0, s.iz, s.pz), tcap));
    n1 = fmaxf(fmaxf(__fmaf_rn(sx ? hx1 : lx1, s.ix, s.px), __fmaf_rn(sy ? hy1 : ly1, s.iy, s.py)),
               fmaxf(__fmaf_rn(sz ? hz1 : lz1, s.iz, s.pz), 0.f));
    f1 = fminf(fminf(__fmaf_rn(sx ? lx1 : hx1, s.ix, s.px), __fmaf_rn(sy ? ly1 : hy1, s.iy, s.py)),
               fminf(__fmaf_rn(sz ? lz1 : hz1, s.iz, s.pz), tcap));
}

}  // namespace opx
