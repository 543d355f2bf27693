// ============================================================================================
// ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT.
//
// A plain, slow, scalar CPU restatement of the per-photon optical propagation of
// arXiv:2309.12496 ("Optical Photon Simulation with Mitsuba3"), written from PAPER.md and from
// DESIGN.md section 3 (the arithmetic contract), sharing no code with the CUDA path.  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
// load or call it.
//
// What it computes (PAPER.md line numbers):
//   * emitter: one ray per entry of the input position/momentum arrays, constant weight, no cone
//     (section 4.2 "photon_emitter");
//   * closest hit against triangle meshes grouped per material -- here by
//     BRUTE FORCE over every triangle, the plain definition of "closest hit"; there is no
//     acceleration structure anywhere in this file;
//   * mirrors reflect specularly with wavelength-dependent reflectivity,
//     the detector accepts with a wavelength-dependent quantum efficiency, both by accept-reject
//     (PAPER.md:117-119), applied in flight per interaction as the paper proposes at PAPER.md:197;
//   * the detector records the global hit position and the 2-D pixel coordinate from
//     the corner point A along the two in-plane unit vectors (PAPER.md:127, 135 / Fig. 4).
//
// Modes: Real = float follows the fp32 arithmetic contract operation by operation (bit parity with
// the GPU is judged against this mode); Real = double runs the same algorithm in fp64 (truth for
// closed forms).  An analytic-sphere tracer for the toy RICH (config 0) is at the bottom.
//
// Pins (tests/test_oracle_pins.py): Philox known answers, law of reflection, table lookup at
// nodes, pixel map edges, brute-force vs analytic plane/sphere, focal ring (R/2) tan(theta_c),
// conservation, binomial counts, permutation invariance.  Nothing here is "parity unpinned".
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -mfma -fPIC -shared (see oracle/build.py).
// ============================================================================================
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

namespace {

enum State : uint8_t {
    DETECTED = 0, QE_REJECTED = 1, ABSORBED_SURFACE = 2, ABSORBED_MIRROR = 3,
    DETECTOR_DEAD = 4, BOUNCE_LIMIT = 5, ESCAPED = 6
};
enum MatKind : uint32_t { MAT_ABSORBER = 0, MAT_MIRROR = 1, MAT_DETECTOR = 2 };

// ------------------------------------------------------------------------------- Philox4x32-10
// Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11.
// DESIGN.md section 3.1.  The method's "accept-reject" needs one uniform per surface
// interaction; keyed so that the draw depends only on (seed, photon id, bounce).
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// u(seed, g, b) in [0,1): 24 high bits of word 0, exactly representable in fp32.
// Counter word 3 names the stream: 0 = in-flight draws of the propagation, 1 = the pre-propagation filter
// (DESIGN.md 3.9), so the two never share a random number.
float uniform_draw(uint64_t seed, uint64_t g, uint32_t b, uint32_t stream = 0u) {
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    const uint32_t ctr[4] = {(uint32_t)g, (uint32_t)(g >> 32), b, stream};
    uint32_t r[4];
    philox4x32_10(ctr, key, r);
    return (float)(r[0] >> 8) * 0x1.0p-24f;
}

// ------------------------------------------------------------------------- small real helpers
template <typename R> inline R rfma(R a, R b, R c);
template <> inline float rfma<float>(float a, float b, float c) { return __builtin_fmaf(a, b, c); }
template <> inline double rfma<double>(double a, double b, double c) { return __builtin_fma(a, b, c); }

template <typename R> struct Vec3 { R x, y, z;  R operator[](int i) const { return i == 0 ? x : (i == 1 ? y : z); } };

// ------------------------------------------------------------------------------ table lookup
// DESIGN.md 3.2.  Efficiency at wavelength lambda from a uniform n_lambda-point grid, piecewise
// linear, clamped to the end values (PAPER.md:117-119 uses histograms of the measured curves;
// BASELINE.json config 1 fixes 64-point piecewise-linear tables).
template <typename R>
R table_lerp(const float* y, uint32_t n_lambda, R lambda_min, R inv_dlambda, R lambda) {
    const R x = (lambda - lambda_min) * inv_dlambda;
    const R xf = std::floor(x);
    int j;                                                     // j = clamp(floor(x), 0, n_lambda-2)
    if (!(xf >= (R)0)) j = 0;                                  // also catches NaN
    else if (xf > (R)(n_lambda - 2)) j = (int)n_lambda - 2;
    else j = (int)xf;
    R f = x - (R)j;                                            // f = clamp(x - j, 0, 1)
    if (!(f >= (R)0)) f = (R)0;
    if (f > (R)1) f = (R)1;
    const R y0 = (R)y[j], y1 = (R)y[j + 1];
    return rfma<R>(f, y1 - y0, y0);
}

// DESIGN.md 3.8.  The paper's own table form: "histograms of 33 nm bin width" (QE) and
// "bins of 25 nm" (reflectivity).  The n_lambda values are the contents of n_lambda equal bins that tile
// [lambda_min, lambda_max]; a wavelength takes the content of its bin, the end bins extend outwards.
template <typename R>
R table_histogram(const float* y, uint32_t n_lambda, R lambda_min, R inv_bin, R lambda) {
    const R xf = std::floor((lambda - lambda_min) * inv_bin);
    int j;                                                     // j = clamp(floor(x), 0, n_lambda-1)
    if (!(xf >= (R)0)) j = 0;                                  // also catches NaN
    else if (xf > (R)(n_lambda - 1)) j = (int)n_lambda - 1;
    else j = (int)xf;
    return (R)y[j];
}

enum TableInterp : uint32_t { TABLE_LINEAR = 0, TABLE_HISTOGRAM = 1 };

// Efficiency of one material at lambda in its own table form.  The grid constants are computed in double and
// rounded once to Real: inv_dlambda = (n-1)/(max-min) for the linear form, inv_bin = n/(max-min) for bins.
template <typename R>
R table_value(const float* y, uint32_t n_lambda, uint32_t interp, float lambda_min, float lambda_max, R lambda) {
    const double span = (double)lambda_max - (double)lambda_min;
    if (interp == TABLE_HISTOGRAM) return table_histogram<R>(y, n_lambda, (R)lambda_min, (R)((double)n_lambda / span), lambda);
    return table_lerp<R>(y, n_lambda, (R)lambda_min, (R)((double)(n_lambda - 1) / span), lambda);
}

// ------------------------------------------------------------------------ ray / triangle test
// DESIGN.md 3.3.  Watertight test (after Woop, Benthin, Wald, JCGT 2(1) 2013, restated): shear the
// triangle into a ray space whose z axis is the ray, evaluate the three 2-D edge functions, fall
// back to exact products in double when one of them is exactly zero.
template <typename R> struct RaySetup {
    Vec3<R> o;  int kx, ky, kz;  R Sx, Sy, Sz;
};

template <typename R> RaySetup<R> ray_setup(const Vec3<R>& o, const Vec3<R>& d) {
    RaySetup<R> rs;
    rs.o = o;
    int kz = 0;                                                // argmax |d_i|, lowest index on ties
    R best = std::fabs(d.x);
    if (std::fabs(d.y) > best) { kz = 1; best = std::fabs(d.y); }
    if (std::fabs(d.z) > best) { kz = 2; }
    int kx = (kz + 1) % 3, ky = (kx + 1) % 3;
    if (d[kz] < (R)0) { const int t = kx; kx = ky; ky = t; }
    rs.kx = kx; rs.ky = ky; rs.kz = kz;
    rs.Sx = d[kx] / d[kz];
    rs.Sy = d[ky] / d[kz];
    rs.Sz = (R)1 / d[kz];
    return rs;
}

// Returns true and t when the ray hits triangle (a,b,c) with t > tmin and t finite.
// uvw (optional) receives the edge functions U, V, W as computed in Real: the unnormalised barycentric
// weights of a, b, c at the hit (they sum to det), used by the shading normal of DESIGN.md 3.11.
template <typename R>
bool hit_triangle(const RaySetup<R>& rs, const Vec3<R>& a, const Vec3<R>& b, const Vec3<R>& c,
                  R tmin, R* t_out, R* uvw = nullptr) {
    const Vec3<R> A{a.x - rs.o.x, a.y - rs.o.y, a.z - rs.o.z};
    const Vec3<R> B{b.x - rs.o.x, b.y - rs.o.y, b.z - rs.o.z};
    const Vec3<R> C{c.x - rs.o.x, c.y - rs.o.y, c.z - rs.o.z};
    const R Ax = rfma<R>(-rs.Sx, A[rs.kz], A[rs.kx]), Ay = rfma<R>(-rs.Sy, A[rs.kz], A[rs.ky]);
    const R Bx = rfma<R>(-rs.Sx, B[rs.kz], B[rs.kx]), By = rfma<R>(-rs.Sy, B[rs.kz], B[rs.ky]);
    const R Cx = rfma<R>(-rs.Sx, C[rs.kz], C[rs.kx]), Cy = rfma<R>(-rs.Sy, C[rs.kz], C[rs.ky]);
    // Edge functions: two rounded products and one rounded difference, deliberately NOT fused, so
    // that the two triangles sharing an edge compute exactly opposite values (watertightness).
    const R U = Cx * By - Cy * Bx;
    const R V = Ax * Cy - Ay * Cx;
    const R W = Bx * Ay - By * Ax;
    const R Az = rs.Sz * A[rs.kz], Bz = rs.Sz * B[rs.kz], Cz = rs.Sz * C[rs.kz];
    R t;
    if (sizeof(R) == sizeof(float) && (U == (R)0 || V == (R)0 || W == (R)0)) {
        // fp32 contract only: edge functions recomputed from exact double products, kept in double
        // for the sign test, the sum and the distance.
        const double Ud = (double)Cx * (double)By - (double)Cy * (double)Bx;
        const double Vd = (double)Ax * (double)Cy - (double)Ay * (double)Cx;
        const double Wd = (double)Bx * (double)Ay - (double)By * (double)Ax;
        if ((Ud < 0 || Vd < 0 || Wd < 0) && (Ud > 0 || Vd > 0 || Wd > 0)) return false;
        const double det = (Ud + Vd) + Wd;
        if (det == 0) return false;
        const double T = __builtin_fma(Wd, (double)Cz, __builtin_fma(Vd, (double)Bz, Ud * (double)Az));
        t = (R)(T / det);
    } else {
        if ((U < (R)0 || V < (R)0 || W < (R)0) && (U > (R)0 || V > (R)0 || W > (R)0)) return false;
        const R det = (U + V) + W;
        if (det == (R)0) return false;
        const R T = rfma<R>(W, Cz, rfma<R>(V, Bz, U * Az));
        t = T / det;
    }
    if (!std::isfinite(t) || !(t > tmin)) return false;
    *t_out = t;
    if (uvw) { uvw[0] = U; uvw[1] = V; uvw[2] = W; }
    return true;
}

// --------------------------------------------------------------------------------- reflection
// DESIGN.md 3.5.  Specular mirror: d' = d - 2 (d.n) n with the geometric face
// normal; even in n, so the orientation of n does not matter; no renormalisation.
template <typename R> Vec3<R> reflect(const Vec3<R>& d, const Vec3<R>& n) {
    const R c = rfma<R>(d.z, n.z, rfma<R>(d.y, n.y, d.x * n.x));
    const R m2c = (R)(-2) * c;
    return Vec3<R>{rfma<R>(m2c, n.x, d.x), rfma<R>(m2c, n.y, d.y), rfma<R>(m2c, n.z, d.z)};
}

// Face normal: normalise((b-a) x (c-a)) in double, rounded once to Real.
template <typename R> Vec3<R> face_normal(const float* v /*9*/) {
    const double e1x = (double)v[3] - (double)v[0], e1y = (double)v[4] - (double)v[1], e1z = (double)v[5] - (double)v[2];
    const double e2x = (double)v[6] - (double)v[0], e2y = (double)v[7] - (double)v[1], e2z = (double)v[8] - (double)v[2];
    const double nx = e1y * e2z - e1z * e2y, ny = e1z * e2x - e1x * e2z, nz = e1x * e2y - e1y * e2x;
    const double len = std::sqrt((nx * nx + ny * ny) + nz * nz);
    if (!(len > 0.0)) return Vec3<R>{(R)0, (R)0, (R)0};
    return Vec3<R>{(R)(nx / len), (R)(ny / len), (R)(nz / len)};
}

// DESIGN.md 3.11.  Shading normal of a mesh that carries vertex normals (an OBJ file's `vn` records; the paper
// exports its mirrors as OBJ meshes, whose facets blur the ring): the vertex
// normals na, nb, nc weighted by the edge functions of the hit (U weighs a, V weighs b, W weighs c; their common
// factor 1/det drops out of the normalisation, and the sign it may carry does not matter to a reflection),
//     m = fma(W, nc, fma(V, nb, U na)),   n = m * (1 / sqrt(fma(mz, mz, fma(my, my, mx mx)))).
// A zero or non-finite length (a mesh without vertex normals has them all zero) falls back to the face normal.
template <typename R>
Vec3<R> shading_normal(const R* uvw, const float* vn /*9: na, nb, nc*/, const Vec3<R>& face) {
    const R U = uvw[0], V = uvw[1], W = uvw[2];
    const R mx = rfma<R>(W, (R)vn[6], rfma<R>(V, (R)vn[3], U * (R)vn[0]));
    const R my = rfma<R>(W, (R)vn[7], rfma<R>(V, (R)vn[4], U * (R)vn[1]));
    const R mz = rfma<R>(W, (R)vn[8], rfma<R>(V, (R)vn[5], U * (R)vn[2]));
    const R len2 = rfma<R>(mz, mz, rfma<R>(my, my, mx * mx));
    if (!(len2 > (R)0) || !std::isfinite(len2)) return face;
    const R inv = (R)1 / std::sqrt(len2);
    return Vec3<R>{mx * inv, my * inv, mz * inv};
}

// ---------------------------------------------------------------------------------- pixel map
// DESIGN.md 3.6.  2-D detector coordinate relative to the corner A along the in-plane unit vectors
// ("2D coordinates relative to the bottom left corner", Fig. 4).
struct Frame {          // corner A, in-plane unit vectors u, v, pitches, grid size, first pixel id (plain data)
    float A[3], u[3], v[3], pitch_u, pitch_v;
    uint32_t nu, nv, pixel_base;
};

template <typename R>
bool pixel_map(const Frame& f, const Vec3<R>& p, int32_t* iu_out, int32_t* iv_out) {
    const R qx = p.x - (R)f.A[0], qy = p.y - (R)f.A[1], qz = p.z - (R)f.A[2];
    const R a = rfma<R>(qz, (R)f.u[2], rfma<R>(qy, (R)f.u[1], qx * (R)f.u[0]));
    const R b = rfma<R>(qz, (R)f.v[2], rfma<R>(qy, (R)f.v[1], qx * (R)f.v[0]));
    const R inv_pu = (R)(1.0 / (double)f.pitch_u), inv_pv = (R)(1.0 / (double)f.pitch_v);
    const R fu = std::floor(a * inv_pu), fv = std::floor(b * inv_pv);
    *iu_out = -1; *iv_out = -1;
    if (!(fu >= (R)0) || !(fv >= (R)0) || !(fu < (R)f.nu) || !(fv < (R)f.nv)) return false;
    *iu_out = (int32_t)fu; *iv_out = (int32_t)fv;
    return true;
}

// -------------------------------------------------------------------------------- scene view
struct SceneView {
    const float* tri;              // T x 9: a, b, c
    const int32_t* tri_surface;    // T
    uint64_t n_tri;
    const uint32_t* surf_material; // S
    const int32_t* surf_frame;     // S, -1 unless detector
    uint32_t n_surf;
    const uint32_t* mat_kind;      // M
    const float* mat_table;        // M x n_lambda
    uint32_t n_mat, n_lambda;
    float lambda_min, lambda_max;
    const Frame* frames; uint32_t n_frames;
    uint32_t max_bounces; float t_min;
    const uint32_t* mat_interp;    // M table forms (TableInterp), NULL = all linear
    uint32_t flags;                // FLAG_NO_EFFICIENCY: surfaces act with probability 1, no random draws
    const float* tri_vnormal;      // T x 9 vertex normals (na, nb, nc) or NULL: mirrors reflect about the face normal
};
enum : uint32_t { FLAG_NO_EFFICIENCY = 1u };

struct Record { double pos[3], dir[3]; int32_t pixel, surface, tri; uint8_t state, bounces; uint32_t segments; };

// ------------------------------------------------------------------- one photon, start to end
// DESIGN.md section 2 (the algorithm) -- follows SURVEY.md 8(c) step by step.
template <typename R>
Record trace_photon(const SceneView& sc, const std::vector<Vec3<R>>& normals, uint64_t seed,
                    uint64_t g, const float* o_in, const float* d_in, float lambda_in) {
    Vec3<R> o{(R)o_in[0], (R)o_in[1], (R)o_in[2]}, d{(R)d_in[0], (R)d_in[1], (R)d_in[2]};
    const R lambda = (R)lambda_in;
    const bool draw = !(sc.flags & FLAG_NO_EFFICIENCY);        // efficiencies already applied (3.9)
    uint32_t b = 0;
    int64_t last = -1;
    Record rec{};
    rec.pixel = -1; rec.surface = -1; rec.tri = -1; rec.segments = 0;
    for (;;) {
        // closest hit: lexicographic minimum of (t_k, k) over ALL triangles k != last
        const RaySetup<R> rs = ray_setup<R>(o, d);
        const R tmin = (b == 0) ? (R)0 : (R)sc.t_min;
        R t_best = std::numeric_limits<R>::infinity();
        int64_t k_best = -1;
        R uvw_best[3] = {(R)0, (R)0, (R)0};
        for (uint64_t k = 0; k < sc.n_tri; ++k) {
            if ((int64_t)k == last) continue;
            const float* v = sc.tri + 9 * k;
            R t, uvw[3];
            if (!hit_triangle<R>(rs, Vec3<R>{(R)v[0], (R)v[1], (R)v[2]}, Vec3<R>{(R)v[3], (R)v[4], (R)v[5]},
                                 Vec3<R>{(R)v[6], (R)v[7], (R)v[8]}, tmin, &t, uvw)) continue;
            if (t < t_best) {                                      // ascending k: ties keep the lower id
                t_best = t; k_best = (int64_t)k;
                uvw_best[0] = uvw[0]; uvw_best[1] = uvw[1]; uvw_best[2] = uvw[2];
            }
        }
        rec.segments++;
        if (k_best < 0) {
            rec.state = ESCAPED; rec.pos[0] = o.x; rec.pos[1] = o.y; rec.pos[2] = o.z;
            rec.dir[0] = d.x; rec.dir[1] = d.y; rec.dir[2] = d.z; rec.surface = -1; rec.pixel = -1;
            break;
        }
        const Vec3<R> p{rfma<R>(t_best, d.x, o.x), rfma<R>(t_best, d.y, o.y), rfma<R>(t_best, d.z, o.z)};
        const int32_t s = sc.tri_surface[k_best];
        const uint32_t m = sc.surf_material[s];
        const uint32_t kind = sc.mat_kind[m];
        const float* table = sc.mat_table + (size_t)m * sc.n_lambda;
        rec.surface = s; rec.tri = (int32_t)k_best;
        rec.pos[0] = p.x; rec.pos[1] = p.y; rec.pos[2] = p.z;
        rec.dir[0] = d.x; rec.dir[1] = d.y; rec.dir[2] = d.z;
        if (kind == MAT_ABSORBER) { rec.state = ABSORBED_SURFACE; break; }
        const uint32_t interp = sc.mat_interp ? sc.mat_interp[m] : (uint32_t)TABLE_LINEAR;
        if (kind == MAT_MIRROR) {
            if (draw) {
                const R u = (R)uniform_draw(seed, g, b);
                if (!(u < table_value<R>(table, sc.n_lambda, interp, sc.lambda_min, sc.lambda_max, lambda))) {
                    rec.state = ABSORBED_MIRROR; break;
                }
            }
            d = reflect<R>(d, sc.tri_vnormal ? shading_normal<R>(uvw_best, sc.tri_vnormal + 9 * k_best, normals[k_best])
                                             : normals[k_best]);
            o = p; last = k_best; b++;
            if (b == sc.max_bounces) {
                rec.state = BOUNCE_LIMIT; rec.dir[0] = d.x; rec.dir[1] = d.y; rec.dir[2] = d.z; break;
            }
            continue;
        }
        // detector
        int32_t iu, iv;
        const Frame& f = sc.frames[sc.surf_frame[s]];
        if (!pixel_map<R>(f, p, &iu, &iv)) { rec.state = DETECTOR_DEAD; rec.pixel = -1; break; }
        rec.pixel = (int32_t)(f.pixel_base + (uint32_t)iv * f.nu + (uint32_t)iu);
        if (!draw) { rec.state = DETECTED; break; }
        const R u = (R)uniform_draw(seed, g, b);
        rec.state = (u < table_value<R>(table, sc.n_lambda, interp, sc.lambda_min, sc.lambda_max, lambda)) ? DETECTED : QE_REJECTED;
        break;
    }
    rec.bounces = (uint8_t)b;
    return rec;
}

struct Outputs {
    double* pos; double* dir; int32_t* pixel; int32_t* surface; int32_t* tri;
    uint8_t* state; uint8_t* bounces; uint32_t* segments; uint32_t* hitmap; uint64_t* counters;
};

template <typename R>
void trace_all(const SceneView& sc, uint64_t n, const uint64_t* ids, uint64_t id_base,
               const float* origins, const float* dirs, const float* wl, uint64_t seed,
               const Outputs& out, int n_threads) {
    std::vector<Vec3<R>> normals(sc.n_tri);
    for (uint64_t k = 0; k < sc.n_tri; ++k) normals[k] = face_normal<R>(sc.tri + 9 * k);
    if (n_threads < 1) n_threads = 1;
    std::vector<std::thread> pool;
    for (int w = 0; w < n_threads; ++w) {
        pool.emplace_back([&, w]() {
            for (uint64_t i = (uint64_t)w; i < n; i += (uint64_t)n_threads) {
                const uint64_t g = ids ? ids[i] : id_base + i;
                const Record r = trace_photon<R>(sc, normals, seed, g, origins + 3 * i, dirs + 3 * i, wl[i]);
                for (int c = 0; c < 3; ++c) { out.pos[3 * i + c] = r.pos[c]; out.dir[3 * i + c] = r.dir[c]; }
                out.pixel[i] = r.pixel; out.surface[i] = r.surface; out.tri[i] = r.tri;
                out.state[i] = r.state; out.bounces[i] = r.bounces; out.segments[i] = r.segments;
            }
        });
    }
    for (auto& th : pool) th.join();
    // hit-map and counters: plain serial histogram of the per-photon records
    for (uint64_t i = 0; i < n; ++i) {
        out.counters[out.state[i]] += 1;
        out.counters[7] += out.segments[i];
        if (out.state[i] == DETECTED) out.hitmap[out.pixel[i]] += 1;
    }
}

}  // namespace

// ============================================================================== C interface
extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
float oracle_uniform(uint64_t seed, uint64_t g, uint32_t b) { return uniform_draw(seed, g, b); }

double oracle_table_lerp(int fp64, const float* y, uint32_t n_lambda, float lmin, float lmax, float lambda) {
    const double inv = (double)(n_lambda - 1) / ((double)lmax - (double)lmin);
    if (fp64) return table_lerp<double>(y, n_lambda, (double)lmin, inv, (double)lambda);
    return (double)table_lerp<float>(y, n_lambda, lmin, (float)inv, lambda);
}

void oracle_reflect(int fp64, const double* d, const double* n, double* out) {
    if (fp64) { auto r = reflect<double>({d[0], d[1], d[2]}, {n[0], n[1], n[2]}); out[0] = r.x; out[1] = r.y; out[2] = r.z; }
    else { auto r = reflect<float>({(float)d[0], (float)d[1], (float)d[2]}, {(float)n[0], (float)n[1], (float)n[2]});
           out[0] = r.x; out[1] = r.y; out[2] = r.z; }
}

void oracle_face_normal(const float* v9, double* out) {
    auto n = face_normal<double>(v9); out[0] = n.x; out[1] = n.y; out[2] = n.z;
}

int oracle_pixel_map(int fp64, const Frame* f, const double* p, int32_t* iu, int32_t* iv) {
    if (fp64) return pixel_map<double>(*f, {p[0], p[1], p[2]}, iu, iv) ? 1 : 0;
    return pixel_map<float>(*f, {(float)p[0], (float)p[1], (float)p[2]}, iu, iv) ? 1 : 0;
}

int oracle_hit_triangle(int fp64, const float* o, const float* d, const float* v9, double tmin, double* t) {
    if (fp64) {
        auto rs = ray_setup<double>({o[0], o[1], o[2]}, {d[0], d[1], d[2]});
        double tt; const bool h = hit_triangle<double>(rs, {v9[0], v9[1], v9[2]}, {v9[3], v9[4], v9[5]}, {v9[6], v9[7], v9[8]}, tmin, &tt);
        if (h) *t = tt;
        return h;
    }
    auto rs = ray_setup<float>({o[0], o[1], o[2]}, {d[0], d[1], d[2]});
    float tt; const bool h = hit_triangle<float>(rs, {v9[0], v9[1], v9[2]}, {v9[3], v9[4], v9[5]}, {v9[6], v9[7], v9[8]}, (float)tmin, &tt);
    if (h) *t = tt;
    return h;
}

// Trace n photons through a triangle scene.  counters: 8 uint64 (+=): one per terminal state 0..6,
// [7] = closest-hit queries (segments).  hitmap: n_pixels uint32 (+=).  ids == NULL => global id =
// id_base + i.
int oracle_trace_mesh_ex2(int fp64, const uint32_t* mat_interp, uint32_t flags, const float* tri_vnormal,
                      const float* tri, const int32_t* tri_surface, uint64_t n_tri,
                      const uint32_t* surf_material, const int32_t* surf_frame, uint32_t n_surf,
                      const uint32_t* mat_kind, const float* mat_table, uint32_t n_mat, uint32_t n_lambda,
                      float lambda_min, float lambda_max, const Frame* frames, uint32_t n_frames,
                      uint32_t max_bounces, float t_min,
                      uint64_t n, const uint64_t* ids, uint64_t id_base,
                      const float* origins, const float* dirs, const float* wl, uint64_t seed,
                      double* pos, double* dir, int32_t* pixel, int32_t* surface, int32_t* tri_out,
                      uint8_t* state, uint8_t* bounces, uint32_t* segments, uint32_t* hitmap,
                      uint64_t* counters, int n_threads) {
    if (n_lambda < 2 || !(lambda_max > lambda_min)) return 1;
    for (uint64_t k = 0; k < n_tri; ++k) if (tri_surface[k] < 0 || (uint32_t)tri_surface[k] >= n_surf) return 2;
    for (uint32_t s = 0; s < n_surf; ++s) {
        if (surf_material[s] >= n_mat) return 3;
        if (mat_kind[surf_material[s]] == MAT_DETECTOR && (surf_frame[s] < 0 || (uint32_t)surf_frame[s] >= n_frames)) return 4;
    }
    if (mat_interp) for (uint32_t m = 0; m < n_mat; ++m) if (mat_interp[m] > TABLE_HISTOGRAM) return 5;
    SceneView sc{tri, tri_surface, n_tri, surf_material, surf_frame, n_surf, mat_kind, mat_table, n_mat,
                 n_lambda, lambda_min, lambda_max, frames, n_frames, max_bounces, t_min, mat_interp, flags, tri_vnormal};
    Outputs out{pos, dir, pixel, surface, tri_out, state, bounces, segments, hitmap, counters};
    if (fp64) trace_all<double>(sc, n, ids, id_base, origins, dirs, wl, seed, out, n_threads);
    else trace_all<float>(sc, n, ids, id_base, origins, dirs, wl, seed, out, n_threads);
    return 0;
}

// Shading normal at the point where the ray (o, d) meets triangle v9 with vertex normals n9.
// Returns 0 on a miss; uvw (3, may be NULL) receives the edge functions.
int oracle_shading_normal(int fp64, const float* o, const float* d, const float* v9, const float* n9, double* out, double* uvw_out) {
    if (fp64) {
        auto rs = ray_setup<double>({o[0], o[1], o[2]}, {d[0], d[1], d[2]});
        double t, uvw[3];
        if (!hit_triangle<double>(rs, {v9[0], v9[1], v9[2]}, {v9[3], v9[4], v9[5]}, {v9[6], v9[7], v9[8]}, 0.0, &t, uvw)) return 0;
        const auto nn = shading_normal<double>(uvw, n9, face_normal<double>(v9));
        out[0] = nn.x; out[1] = nn.y; out[2] = nn.z;
        if (uvw_out) { uvw_out[0] = uvw[0]; uvw_out[1] = uvw[1]; uvw_out[2] = uvw[2]; }
        return 1;
    }
    auto rs = ray_setup<float>({o[0], o[1], o[2]}, {d[0], d[1], d[2]});
    float t, uvw[3];
    if (!hit_triangle<float>(rs, {v9[0], v9[1], v9[2]}, {v9[3], v9[4], v9[5]}, {v9[6], v9[7], v9[8]}, 0.f, &t, uvw)) return 0;
    const auto nn = shading_normal<float>(uvw, n9, face_normal<float>(v9));
    out[0] = nn.x; out[1] = nn.y; out[2] = nn.z;
    if (uvw_out) { uvw_out[0] = uvw[0]; uvw_out[1] = uvw[1]; uvw_out[2] = uvw[2]; }
    return 1;
}

double oracle_table_value(int fp64, const float* y, uint32_t n_lambda, uint32_t interp, float lmin, float lmax, float lambda) {
    if (fp64) return table_value<double>(y, n_lambda, interp, lmin, lmax, (double)lambda);
    return (double)table_value<float>(y, n_lambda, interp, lmin, lmax, lambda);
}
float oracle_uniform_stream(uint64_t seed, uint64_t g, uint32_t b, uint32_t stream) { return uniform_draw(seed, g, b, stream); }

// Pre-propagation efficiency filter, the paper's own method ("For each photon, with its
// specific wavelength, an accept-reject algorithm was used to model the three efficiencies before propagation
// ... any discarded photons would not be detected").  DESIGN.md 3.9: ONE draw per photon,
// u = U(seed, g, 0; stream 1), against the product of the listed materials' efficiencies at the photon's
// wavelength, p = (..(e_0 * e_1) * e_2 ..) multiplied left to right in fp32; the photon is kept iff u < p.
// keep[i] = 1/0; kept_index receives the indices of the kept photons in input order (stable compaction);
// returns their number.  prob (may be NULL) receives p per photon.
uint64_t oracle_prefilter(const float* mat_table, const uint32_t* mat_interp, uint32_t n_mat, uint32_t n_lambda,
                          float lambda_min, float lambda_max, const uint32_t* factors, uint32_t n_factors,
                          uint64_t n, uint64_t id_base, const float* wl, uint64_t seed,
                          uint8_t* keep, uint32_t* kept_index, float* prob) {
    uint64_t kept = 0;
    for (uint64_t i = 0; i < n; ++i) {
        float p = 1.0f;
        for (uint32_t k = 0; k < n_factors; ++k) {
            const uint32_t m = factors[k];
            if (m >= n_mat) return ~0ull;
            const float e = table_value<float>(mat_table + (size_t)m * n_lambda, n_lambda,
                                               mat_interp ? mat_interp[m] : (uint32_t)TABLE_LINEAR, lambda_min, lambda_max, wl[i]);
            p = (k == 0) ? e : p * e;
        }
        const float u = uniform_draw(seed, id_base + i, 0u, 1u);
        const bool k = u < p;
        if (prob) prob[i] = p;
        keep[i] = k ? 1 : 0;
        if (k) kept_index[kept++] = (uint32_t)i;
    }
    return kept;
}

// ------------------------------------------------------- Cherenkov emission from track steps (row f4)
// DESIGN.md 3.12.  "The Cherenkov angle theta_c ... cos(theta_c) = 1/(n beta)"; photons are emitted
// uniformly along the step, uniformly in azimuth about the track, with a wavelength density ~ 1/lambda^2.  The paper
// leaves this to Geant4 and wants it memory-resident; here it is step by step in fp32, with the
// azimuth drawn by Marsaglia's disc method so that no transcendental function is involved.
// Step s: x (3), w (3, unit), L, beta; first (S+1) = exclusive prefix sum of the photon counts.
// Photon g = id_base + i for i in [0, n) -> origins, dirs (n x 3), wl (n).  Returns 0, or 1 if some g has no step.
int oracle_emit_cherenkov(uint64_t n_steps, const float* step_x, const float* step_w, const float* step_len,
                          const float* step_beta, const uint64_t* first, float n_index, float lambda1, float lambda2,
                          uint64_t n, uint64_t id_base, uint64_t seed, float* origins, float* dirs, float* wl) {
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (uint64_t i = 0; i < n; ++i) {
        const uint64_t g = id_base + i;
        if (n_steps == 0 || g >= first[n_steps]) return 1;
        // the step with first[s] <= g < first[s+1]: the LAST s with first[s] <= g (steps without photons are skipped)
        uint64_t lo = 0, hi = n_steps;                           // invariant: first[lo] <= g < first[hi]
        while (hi - lo > 1) { const uint64_t mid = lo + (hi - lo) / 2; if (first[mid] <= g) lo = mid; else hi = mid; }
        const uint64_t s = lo;
        const float* x = step_x + 3 * s;
        const float* w = step_w + 3 * s;
        auto block = [&](uint32_t a, float* u) {
            const uint32_t ctr[4] = {(uint32_t)g, (uint32_t)(g >> 32), a, 2u};
            uint32_t r[4];
            philox4x32_10(ctr, key, r);
            for (int k = 0; k < 4; ++k) u[k] = (float)(r[k] >> 8) * 0x1.0p-24f;
        };
        float u[4];
        block(0u, u);
        const float t = u[0] * step_len[s];
        for (int a = 0; a < 3; ++a) origins[3 * i + a] = __builtin_fmaf(t, w[a], x[a]);
        wl[i] = (lambda1 * lambda2) / __builtin_fmaf(-u[1], lambda2 - lambda1, lambda2);
        float c = 1.0f / (n_index * step_beta[s]);
        if (!(c < 1.0f)) c = 1.0f;
        const float sn = std::sqrt(std::fmax(__builtin_fmaf(-c, c, 1.0f), 0.0f));
        float cphi = 1.0f, sphi = 0.0f;
        for (uint32_t a = 0; a < 64u; ++a) {
            if (a > 0) block(a, u);
            const float X = __builtin_fmaf(2.0f, u[2], -1.0f), Y = __builtin_fmaf(2.0f, u[3], -1.0f);
            const float q = __builtin_fmaf(Y, Y, X * X);
            if (q > 0.0f && q <= 1.0f) { cphi = (X * X - Y * Y) / q; sphi = ((2.0f * X) * Y) / q; break; }
        }
        const float sg = (w[2] >= 0.0f) ? 1.0f : -1.0f;
        const float k = -1.0f / (sg + w[2]);
        const float b = (w[0] * w[1]) * k;
        const float e1[3] = {__builtin_fmaf(sg * w[0], w[0] * k, 1.0f), sg * b, -sg * w[0]};
        const float e2[3] = {b, __builtin_fmaf(w[1], w[1] * k, sg), -w[1]};
        const float A = sn * cphi, B = sn * sphi;
        float m[3];
        for (int a = 0; a < 3; ++a) m[a] = __builtin_fmaf(A, e1[a], __builtin_fmaf(B, e2[a], c * w[a]));
        const float len2 = __builtin_fmaf(m[2], m[2], __builtin_fmaf(m[1], m[1], m[0] * m[0]));
        const float inv = 1.0f / std::sqrt(len2);
        for (int a = 0; a < 3; ++a) dirs[3 * i + a] = m[a] * inv;
    }
    return 0;
}

// ------------------------------------------------------------------- analytic toy RICH (fp64)
// Config 0 of BASELINE.json with the mirror as an exact sphere: cap of the sphere (centre C, radius
// R) whose points P satisfy |(P-V).ex| <= half, |(P-V).ey| <= half and (P-V).a < R (the hemisphere
// of the vertex V); one detector rectangle (centre D, in-plane unit vectors du, dv, half-sizes hu,
// hv) with its pixel frame; an axis-aligned absorbing box [lo,hi] seen from inside.  Same state
// machine, same Philox stream, everything in double.  Pins the mesh tracer (P3, P5, P6, P8).
int oracle_trace_analytic_toy(const double* C, double R, const double* V, const double* ex, const double* ey,
                              const double* a, double half,
                              const double* D, const double* du, const double* dv, double hu, double hv,
                              const Frame* frame, const double* box_lo, const double* box_hi,
                              const float* refl_table, const float* qe_table, uint32_t n_lambda,
                              float lambda_min, float lambda_max, uint32_t max_bounces, double t_min,
                              uint64_t n, uint64_t id_base, const float* origins, const float* dirs,
                              const float* wl, uint64_t seed,
                              double* pos, double* dir, int32_t* pixel, int32_t* surface, uint8_t* state,
                              uint8_t* bounces) {
    auto dot = [](const double* p, const double* q) { return p[0] * q[0] + p[1] * q[1] + p[2] * q[2]; };
    const double inv_dl = (double)(n_lambda - 1) / ((double)lambda_max - (double)lambda_min);
    double dn[3] = {du[1] * dv[2] - du[2] * dv[1], du[2] * dv[0] - du[0] * dv[2], du[0] * dv[1] - du[1] * dv[0]};
    for (uint64_t i = 0; i < n; ++i) {
        double o[3] = {origins[3 * i], origins[3 * i + 1], origins[3 * i + 2]};
        double d[3] = {dirs[3 * i], dirs[3 * i + 1], dirs[3 * i + 2]};
        const double lambda = wl[i];
        uint32_t b = 0; int last = -1;                          // surfaces: 0 mirror, 1 detector, 2 box
        uint8_t st = ESCAPED; int32_t surf = -1, pix = -1; double p[3] = {o[0], o[1], o[2]};
        for (;;) {
            const double tmin = b == 0 ? 0.0 : t_min;
            double tb = std::numeric_limits<double>::infinity(); int kb = -1;
            {   // sphere: |o + t d - C|^2 = R^2, both roots, restricted to the cap
                const double oc[3] = {o[0] - C[0], o[1] - C[1], o[2] - C[2]};
                const double A2 = dot(d, d), Bh = dot(oc, d), Cc = dot(oc, oc) - R * R;
                const double disc = Bh * Bh - A2 * Cc;
                if (disc >= 0.0 && last != 0) {
                    const double sq = std::sqrt(disc);
                    const double roots[2] = {(-Bh - sq) / A2, (-Bh + sq) / A2};
                    for (double t : roots) {
                        if (!(t > tmin) || !(t < tb)) continue;
                        const double q[3] = {o[0] + t * d[0] - V[0], o[1] + t * d[1] - V[1], o[2] + t * d[2] - V[2]};
                        if (std::fabs(dot(q, ex)) <= half && std::fabs(dot(q, ey)) <= half && dot(q, a) < R) { tb = t; kb = 0; }
                    }
                }
            }
            {   // detector rectangle
                const double denom = dot(d, dn);
                if (denom != 0.0 && last != 1) {
                    const double od[3] = {D[0] - o[0], D[1] - o[1], D[2] - o[2]};
                    const double t = dot(od, dn) / denom;
                    if (t > tmin && t < tb) {
                        const double q[3] = {o[0] + t * d[0] - D[0], o[1] + t * d[1] - D[1], o[2] + t * d[2] - D[2]};
                        if (std::fabs(dot(q, du)) <= hu && std::fabs(dot(q, dv)) <= hv) { tb = t; kb = 1; }
                    }
                }
            }
            if (box_lo) {   // box from inside: nearest exit plane
                double texit = std::numeric_limits<double>::infinity();
                for (int c = 0; c < 3; ++c) {
                    if (d[c] > 0) texit = std::fmin(texit, (box_hi[c] - o[c]) / d[c]);
                    else if (d[c] < 0) texit = std::fmin(texit, (box_lo[c] - o[c]) / d[c]);
                }
                if (texit > tmin && texit < tb) { tb = texit; kb = 2; }
            }
            if (kb < 0) { st = ESCAPED; surf = -1; p[0] = o[0]; p[1] = o[1]; p[2] = o[2]; break; }
            for (int c = 0; c < 3; ++c) p[c] = o[c] + tb * d[c];
            surf = kb;
            if (kb == 2) { st = ABSORBED_SURFACE; break; }
            if (kb == 0) {
                const double u = (double)uniform_draw(seed, id_base + i, b);
                if (!(u < table_lerp<double>(refl_table, n_lambda, (double)lambda_min, inv_dl, lambda))) { st = ABSORBED_MIRROR; break; }
                double nn[3] = {(C[0] - p[0]) / R, (C[1] - p[1]) / R, (C[2] - p[2]) / R};
                const double c2 = 2.0 * dot(d, nn);
                for (int c = 0; c < 3; ++c) { d[c] -= c2 * nn[c]; o[c] = p[c]; }
                last = 0; b++;
                if (b == max_bounces) { st = BOUNCE_LIMIT; break; }
                continue;
            }
            int32_t iu, iv;
            if (!pixel_map<double>(*frame, {p[0], p[1], p[2]}, &iu, &iv)) { st = DETECTOR_DEAD; pix = -1; break; }
            pix = (int32_t)(frame->pixel_base + (uint32_t)iv * frame->nu + (uint32_t)iu);
            const double u = (double)uniform_draw(seed, id_base + i, b);
            st = (u < table_lerp<double>(qe_table, n_lambda, (double)lambda_min, inv_dl, lambda)) ? DETECTED : QE_REJECTED;
            break;
        }
        for (int c = 0; c < 3; ++c) { pos[3 * i + c] = p[c]; dir[3 * i + c] = d[c]; }
        pixel[i] = pix; surface[i] = surf; state[i] = st; bounces[i] = (uint8_t)b;
    }
    return 0;
}

}  // extern "C"
