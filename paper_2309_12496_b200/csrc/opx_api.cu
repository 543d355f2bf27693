// C-ABI entry points of libopx.so (include/opx.h): argument validation, scene flattening (A0),
// workspace accounting, error reporting and the host-buffer streaming form of propagate.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "opx_internal.cuh"

namespace opx {

static thread_local std::string g_last_error;
static std::atomic<uint64_t> g_launches{0};

opx_status fail(opx_status st, const std::string& msg) {
    g_last_error = msg;
    return st;
}

opx_status check_cuda(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return OPX_OK;
    return fail(OPX_ERR_CUDA, std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")");
}

void count_launch(uint64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
uint64_t launch_count() { return g_launches.load(std::memory_order_relaxed); }
static thread_local const char* g_last_kernel = "";
void set_last_kernel(const char* name) { g_last_kernel = name; }
const char* last_kernel() { return g_last_kernel; }

// n = normalise((b-a) x (c-a)) in fp64, rounded once; zero-area triangle => 0.
static void face_normal(const float* v, float* out) {
    const double ux = (double)v[3] - (double)v[0], uy = (double)v[4] - (double)v[1], uz = (double)v[5] - (double)v[2];
    const double wx = (double)v[6] - (double)v[0], wy = (double)v[7] - (double)v[1], wz = (double)v[8] - (double)v[2];
    const double cx = uy * wz - uz * wy, cy = uz * wx - ux * wz, cz = ux * wy - uy * wx;
    const double len = std::sqrt((cx * cx + cy * cy) + cz * cz);
    if (!(len > 0.0)) { out[0] = out[1] = out[2] = 0.f; return; }
    out[0] = (float)(cx / len); out[1] = (float)(cy / len); out[2] = (float)(cz / len);
}

opx_status device_ok() {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return check_cuda(e, "cudaGetDevice");
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return check_cuda(e, "cudaDeviceGetAttribute");
    if (major != 10) return fail(OPX_ERR_UNSUPPORTED_DEVICE, "libopx.so is built for sm_100a only (compute capability 10.x)");
    return OPX_OK;
}

static bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) != 0; }

opx_status propagate_common(const opx_scene* scene, WalkMode mode, uint64_t n, const uint64_t* d_n, uint64_t base,
                                   const float* o, const float* d, const float* wl, uint64_t seed, uint32_t flags,
                                   const opx_hits* out, uint32_t* hitmap, uint64_t* counters, void* stream) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_propagate before opx_bvh_build");
    if (n == 0) return OPX_OK;
    if (!o || !d || !wl || !out) return fail(OPX_ERR_INVALID_ARG, "NULL photon/record pointer");
    if (!out->pos || !out->dir || !out->pixel || !out->surface || !out->state || !out->bounces)
        return fail(OPX_ERR_INVALID_ARG, "NULL hit-record array");
    if (!hitmap && scene->n_pixels) return fail(OPX_ERR_INVALID_ARG, "d_hitmap is NULL but the scene has pixels");
    if (misaligned(o, 4) || misaligned(d, 4) || misaligned(wl, 4) || misaligned(out->pos, 4) || misaligned(out->dir, 4) ||
        misaligned(out->pixel, 4) || misaligned(out->surface, 4) || misaligned(hitmap, 4) || misaligned(counters, 8))
        return fail(OPX_ERR_INVALID_ARG, "misaligned pointer");
    if (n > (1ull << 40)) return fail(OPX_ERR_INVALID_ARG, "n too large for one call");
    if (flags & ~(uint32_t)OPX_FLAG_NO_EFFICIENCY) return fail(OPX_ERR_INVALID_ARG, "unknown flag");
    if (misaligned(d_n, 8)) return fail(OPX_ERR_INVALID_ARG, "misaligned d_n");
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_propagate")) return st;
    return launch_propagate(*scene, mode, n, d_n, base, o, d, wl, seed, flags, *out, hitmap, counters, (cudaStream_t)stream);
}

}  // namespace opx

using namespace opx;

extern "C" {

const char* opx_last_error(void) { return g_last_error.c_str(); }
const char* opx_version(void) { return "opx 0.1 (sm_100a)"; }

opx_status opx_scene_create(const opx_scene_params* params, const opx_mesh* meshes, uint32_t n_meshes,
                            const opx_material* materials, uint32_t n_materials,
                            const opx_pixel_frame* frames, uint32_t n_frames, opx_scene** out) {
    if (!params || !out) return fail(OPX_ERR_INVALID_ARG, "params/out is NULL");
    *out = nullptr;
    if ((n_meshes && !meshes) || (n_materials && !materials) || (n_frames && !frames))
        return fail(OPX_ERR_INVALID_ARG, "array pointer is NULL with a non-zero count");
    if (params->n_lambda < 2) return fail(OPX_ERR_INVALID_ARG, "n_lambda must be >= 2");
    if (!(params->lambda_max_nm > params->lambda_min_nm)) return fail(OPX_ERR_INVALID_ARG, "lambda_max must exceed lambda_min");
    if (params->max_bounces < 1 || params->max_bounces > 255) return fail(OPX_ERR_INVALID_ARG, "max_bounces must be in 1..255");
    if (!(params->t_min_mm >= 0.f)) return fail(OPX_ERR_INVALID_ARG, "t_min_mm must be >= 0");

    auto* s = new opx_scene();
    s->params = *params;
    s->inv_dlambda = (float)((double)(params->n_lambda - 1) / ((double)params->lambda_max_nm - (double)params->lambda_min_nm));
    s->inv_bin = (float)((double)params->n_lambda / ((double)params->lambda_max_nm - (double)params->lambda_min_nm));
    auto bail = [&](const std::string& m) { delete s; return fail(OPX_ERR_INVALID_ARG, m); };

    s->mat_kinds.resize(n_materials);
    s->tables.assign((size_t)n_materials * params->n_lambda, 0.f);
    for (uint32_t m = 0; m < n_materials; ++m) {
        if (materials[m].kind > OPX_MAT_DETECTOR) return bail("material kind out of range");
        if (materials[m].interp > OPX_TABLE_HISTOGRAM) return bail("material table form out of range");
        s->mat_kinds[m] = materials[m].kind | (materials[m].interp << 8);
        if (materials[m].kind == OPX_MAT_ABSORBER) continue;
        if (!materials[m].table) return bail("mirror/detector material without a table");
        for (uint32_t j = 0; j < params->n_lambda; ++j) {
            const float y = materials[m].table[j];
            if (!(y >= 0.f && y <= 1.f)) return bail("table value outside [0,1]");
            s->tables[(size_t)m * params->n_lambda + j] = y;
        }
    }
    s->frames.resize(n_frames);
    for (uint32_t f = 0; f < n_frames; ++f) {
        const opx_pixel_frame& in = frames[f];
        if (!(in.pitch_u > 0.f) || !(in.pitch_v > 0.f)) return bail("pixel pitch must be > 0");
        if (in.nu == 0 || in.nv == 0) return bail("pixel grid must be at least 1x1");
        const uint64_t end = (uint64_t)in.pixel_base + (uint64_t)in.nu * in.nv;
        if (end > 0x7fffffffull) return bail("pixel ids must fit in int32");
        FrameDev& o = s->frames[f];
        o.Ax = in.A[0]; o.Ay = in.A[1]; o.Az = in.A[2];
        o.ux = in.u[0]; o.uy = in.u[1]; o.uz = in.u[2];
        o.vx = in.v[0]; o.vy = in.v[1]; o.vz = in.v[2];
        o.inv_pitch_u = (float)(1.0 / (double)in.pitch_u);   // rounded once from fp64
        o.inv_pitch_v = (float)(1.0 / (double)in.pitch_v);
        o.pad0 = 0.f; o.nu = in.nu; o.nv = in.nv; o.pixel_base = in.pixel_base; o.pad1 = 0;
        if (end > s->n_pixels) s->n_pixels = end;
    }
    uint64_t total = 0;
    for (uint32_t k = 0; k < n_meshes; ++k) total += meshes[k].n_triangles;
    if (total > (1ull << 28)) { return bail("too many triangles (limit 2^28: 32-bit offsets into the three rotations of the triangle array)"); }
    s->tri.reserve(total * 9);
    s->tri_surface.reserve(total);
    s->surfaces.resize(n_meshes);
    bool any_vn = false;
    for (uint32_t k = 0; k < n_meshes; ++k) any_vn = any_vn || (meshes[k].vertex_normals && meshes[k].n_triangles);
    if (any_vn) s->tri_vnormals.reserve(total * 9);
    for (uint32_t k = 0; k < n_meshes; ++k) {
        const opx_mesh& m = meshes[k];
        if (m.material >= n_materials) return bail("mesh material index out of range");
        const bool det = (s->mat_kinds[m.material] & 0xffu) == OPX_MAT_DETECTOR;
        if (det && (m.pixel_frame < 0 || (uint32_t)m.pixel_frame >= n_frames)) return bail("detector mesh needs a valid pixel frame");
        s->surfaces[k] = make_int2((int)m.material, det ? m.pixel_frame : -1);
        if (m.n_triangles && (!m.vertices || !m.indices)) return bail("mesh vertices/indices is NULL");
        for (uint32_t t = 0; t < m.n_triangles; ++t) {
            for (int c = 0; c < 3; ++c) {
                const uint32_t vi = m.indices[3 * (size_t)t + c];
                if (vi >= m.n_vertices) return bail("vertex index out of range");
                const float* v = m.vertices + 3 * (size_t)vi;
                s->tri.push_back(v[0]); s->tri.push_back(v[1]); s->tri.push_back(v[2]);
                if (any_vn) {
                    for (int a = 0; a < 3; ++a) {
                        const float x = m.vertex_normals ? m.vertex_normals[3 * (size_t)vi + a] : 0.f;
                        if (!std::isfinite(x)) return bail("vertex normal component is not finite");
                        s->tri_vnormals.push_back(x);
                    }
                }
            }
            s->tri_surface.push_back((int32_t)k);
        }
    }
    s->normals.resize(total * 3);
    for (uint64_t t = 0; t < total; ++t) face_normal(&s->tri[9 * t], &s->normals[3 * t]);
    compute_scene_stats(*s);
    compute_layout(*s, &s->layout, nullptr);
    *out = s;
    return OPX_OK;
}

opx_status opx_scene_workspace_bytes(const opx_scene* scene, size_t* scene_bytes, size_t* build_tmp_bytes) {
    if (!scene || !scene_bytes || !build_tmp_bytes) return fail(OPX_ERR_INVALID_ARG, "NULL argument");
    opx_scene_layout lay;
    size_t tmp = 0;
    compute_layout(*scene, &lay, &tmp);
    *scene_bytes = (size_t)lay.total_bytes;
    *build_tmp_bytes = tmp;
    return OPX_OK;
}

opx_status opx_bvh_build(opx_scene* scene, void* d_scene_ws, size_t scene_bytes, void* d_tmp_ws,
                         size_t tmp_bytes, void* cuda_stream) {
    if (!scene || !d_scene_ws || !d_tmp_ws) return fail(OPX_ERR_INVALID_ARG, "NULL argument");
    if (misaligned(d_scene_ws, 256) || misaligned(d_tmp_ws, 256)) return fail(OPX_ERR_INVALID_ARG, "workspaces must be 256-byte aligned");
    if (opx_status st = device_ok()) return st;
    opx_scene_layout lay;
    size_t tmp = 0;
    compute_layout(*scene, &lay, &tmp);
    if (scene_bytes < lay.total_bytes || tmp_bytes < tmp) return fail(OPX_ERR_WORKSPACE_TOO_SMALL, "workspace too small (see opx_scene_workspace_bytes)");
    scene->built = false;
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_bvh_build")) return st;
    if (opx_status st = build_bvh(*scene, d_scene_ws, d_tmp_ws, (cudaStream_t)cuda_stream)) return st;
    scene->d_scene_ws = d_scene_ws;
    scene->scene_bytes = scene_bytes;
    scene->built = true;
    drop_host_pipe_of_other_device(*scene);      // a rebuild on another GPU: the streams of the host-buffer calls follow
    return OPX_OK;
}

opx_status opx_propagate(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                         const float* d_dirs, const float* d_wavelengths, uint64_t seed, const opx_hits* out,
                         uint32_t* d_hitmap, uint64_t* d_counters, void* cuda_stream) {
    return propagate_common(scene, kWalkProduct, n, nullptr, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, 0u, out, d_hitmap,
                            d_counters, cuda_stream);
}

opx_status opx_propagate_flags(const opx_scene* scene, uint64_t n, const uint64_t* d_n, uint64_t photon_id_base,
                               const float* d_origins, const float* d_dirs, const float* d_wavelengths,
                               uint64_t seed, uint32_t flags, const opx_hits* out, uint32_t* d_hitmap,
                               uint64_t* d_counters, void* cuda_stream) {
    return propagate_common(scene, kWalkProduct, n, d_n, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, flags, out, d_hitmap,
                            d_counters, cuda_stream);
}

opx_status opx_prefilter_workspace_bytes(uint64_t n, size_t* bytes) {
    if (!bytes) return fail(OPX_ERR_INVALID_ARG, "bytes is NULL");
    if (n > 0xffffffffull) return fail(OPX_ERR_INVALID_ARG, "n must be <= 2^32 - 1");
    *bytes = prefilter_workspace_bytes(n);
    return OPX_OK;
}

opx_status opx_prefilter(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                         const float* d_dirs, const float* d_wavelengths, uint64_t seed,
                         const uint32_t* factors, uint32_t n_factors,
                         float* d_out_origins, float* d_out_dirs, float* d_out_wavelengths, uint32_t* d_out_index,
                         uint64_t out_capacity, uint64_t* d_n_kept, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_prefilter before opx_bvh_build");
    if (!d_n_kept || misaligned(d_n_kept, 8)) return fail(OPX_ERR_INVALID_ARG, "d_n_kept is NULL or misaligned");
    if (n > 0xffffffffull) return fail(OPX_ERR_INVALID_ARG, "n must be <= 2^32 - 1");
    if (n_factors > 8 || (n_factors && !factors)) return fail(OPX_ERR_INVALID_ARG, "n_factors must be <= 8 and factors non-NULL");
    for (uint32_t k = 0; k < n_factors; ++k) {
        if (factors[k] >= scene->mat_kinds.size()) return fail(OPX_ERR_INVALID_ARG, "factor material index out of range");
        if ((scene->mat_kinds[factors[k]] & 0xffu) == OPX_MAT_ABSORBER) return fail(OPX_ERR_INVALID_ARG, "an absorber has no efficiency table");
    }
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_prefilter")) return st;
    if (n == 0) return check_cuda(cudaMemsetAsync(d_n_kept, 0, 8, (cudaStream_t)cuda_stream), "cudaMemsetAsync");
    if (!d_origins || !d_dirs || !d_wavelengths || !d_out_origins || !d_out_dirs || !d_out_wavelengths || !d_workspace)
        return fail(OPX_ERR_INVALID_ARG, "NULL photon/workspace pointer");
    if (misaligned(d_origins, 4) || misaligned(d_dirs, 4) || misaligned(d_wavelengths, 4) || misaligned(d_out_origins, 4) ||
        misaligned(d_out_dirs, 4) || misaligned(d_out_wavelengths, 4) || misaligned(d_out_index, 4) || misaligned(d_workspace, 256))
        return fail(OPX_ERR_INVALID_ARG, "misaligned pointer");
    if (d_out_origins == d_origins || d_out_dirs == d_dirs || d_out_wavelengths == d_wavelengths)
        return fail(OPX_ERR_INVALID_ARG, "out arrays must not alias the inputs");
    if (workspace_bytes < prefilter_workspace_bytes(n)) return fail(OPX_ERR_WORKSPACE_TOO_SMALL, "workspace too small (see opx_prefilter_workspace_bytes)");
    return launch_prefilter(*scene, n, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, factors, n_factors, d_out_origins,
                            d_out_dirs, d_out_wavelengths, d_out_index, out_capacity, d_n_kept, d_workspace, (cudaStream_t)cuda_stream);
}

opx_status opx_emit_cherenkov(const opx_track_steps* steps, uint64_t n_total, float n_index, float lambda1_nm,
                              float lambda2_nm, uint64_t n, uint64_t photon_id_base, uint64_t seed, float* d_origins,
                              float* d_dirs, float* d_wavelengths, void* cuda_stream) {
    if (!steps) return fail(OPX_ERR_INVALID_ARG, "steps is NULL");
    if (!(lambda1_nm > 0.f) || !(lambda2_nm > lambda1_nm) || !std::isfinite(lambda2_nm) || !std::isfinite(n_index))
        return fail(OPX_ERR_INVALID_ARG, "need 0 < lambda1 < lambda2 and a finite refractive index");
    if (n == 0) return OPX_OK;
    if (steps->n_steps == 0 || !steps->x || !steps->w || !steps->length || !steps->beta || !steps->first)
        return fail(OPX_ERR_INVALID_ARG, "empty or NULL step table");
    if (photon_id_base > n_total || n > n_total - photon_id_base) return fail(OPX_ERR_INVALID_ARG, "photon ids beyond first[n_steps]");
    if (!d_origins || !d_dirs || !d_wavelengths) return fail(OPX_ERR_INVALID_ARG, "NULL output array");
    if (misaligned(d_origins, 4) || misaligned(d_dirs, 4) || misaligned(d_wavelengths, 4) || misaligned(steps->first, 8) ||
        misaligned(steps->x, 4) || misaligned(steps->w, 4) || misaligned(steps->length, 4) || misaligned(steps->beta, 4))
        return fail(OPX_ERR_INVALID_ARG, "misaligned pointer");
    if (opx_status st = device_ok()) return st;
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_emit_cherenkov")) return st;
    return launch_emit(*steps, n_index, lambda1_nm, lambda2_nm, n, photon_id_base, seed, d_origins, d_dirs, d_wavelengths,
                       (cudaStream_t)cuda_stream);
}

opx_status opx_emit_cherenkov_filtered(const opx_scene* scene, const opx_track_steps* steps, uint64_t n_total, float n_index,
                                       float lambda1_nm, float lambda2_nm, uint64_t n, uint64_t photon_id_base, uint64_t seed,
                                       const uint32_t* factors, uint32_t n_factors, float* d_out_origins, float* d_out_dirs,
                                       float* d_out_wavelengths, uint32_t* d_out_index, uint64_t out_capacity, uint64_t* d_n_kept,
                                       void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!scene || !steps) return fail(OPX_ERR_INVALID_ARG, "scene/steps is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_emit_cherenkov_filtered before opx_bvh_build");
    if (!d_n_kept || misaligned(d_n_kept, 8)) return fail(OPX_ERR_INVALID_ARG, "d_n_kept is NULL or misaligned");
    if (!(lambda1_nm > 0.f) || !(lambda2_nm > lambda1_nm) || !std::isfinite(lambda2_nm) || !std::isfinite(n_index))
        return fail(OPX_ERR_INVALID_ARG, "need 0 < lambda1 < lambda2 and a finite refractive index");
    if (n > 0xffffffffull) return fail(OPX_ERR_INVALID_ARG, "n must be <= 2^32 - 1");
    if (n_factors > 8 || (n_factors && !factors)) return fail(OPX_ERR_INVALID_ARG, "n_factors must be <= 8 and factors non-NULL");
    for (uint32_t k = 0; k < n_factors; ++k) {
        if (factors[k] >= scene->mat_kinds.size()) return fail(OPX_ERR_INVALID_ARG, "factor material index out of range");
        if ((scene->mat_kinds[factors[k]] & 0xffu) == OPX_MAT_ABSORBER) return fail(OPX_ERR_INVALID_ARG, "an absorber has no efficiency table");
    }
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_emit_cherenkov_filtered")) return st;
    if (n == 0) return check_cuda(cudaMemsetAsync(d_n_kept, 0, 8, (cudaStream_t)cuda_stream), "cudaMemsetAsync");
    if (steps->n_steps == 0 || !steps->x || !steps->w || !steps->length || !steps->beta || !steps->first)
        return fail(OPX_ERR_INVALID_ARG, "empty or NULL step table");
    if (photon_id_base > n_total || n > n_total - photon_id_base) return fail(OPX_ERR_INVALID_ARG, "photon ids beyond first[n_steps]");
    if (!d_out_origins || !d_out_dirs || !d_out_wavelengths || !d_workspace) return fail(OPX_ERR_INVALID_ARG, "NULL output/workspace pointer");
    if (misaligned(d_out_origins, 4) || misaligned(d_out_dirs, 4) || misaligned(d_out_wavelengths, 4) || misaligned(d_out_index, 4) ||
        misaligned(d_workspace, 256) || misaligned(steps->first, 8) || misaligned(steps->x, 4) || misaligned(steps->w, 4) ||
        misaligned(steps->length, 4) || misaligned(steps->beta, 4))
        return fail(OPX_ERR_INVALID_ARG, "misaligned pointer");
    if (workspace_bytes < prefilter_workspace_bytes(n)) return fail(OPX_ERR_WORKSPACE_TOO_SMALL, "workspace too small (see opx_prefilter_workspace_bytes)");
    return launch_emit_filtered(*scene, *steps, n_index, lambda1_nm, lambda2_nm, n, photon_id_base, seed, factors, n_factors,
                                d_out_origins, d_out_dirs, d_out_wavelengths, d_out_index, out_capacity, d_n_kept, d_workspace, (cudaStream_t)cuda_stream);
}

// ------------------------------------------------------------------------- detected-only output
opx_status opx_propagate_detected_workspace_bytes(uint64_t n, uint64_t capacity, size_t* bytes) {
    if (!bytes) return fail(OPX_ERR_INVALID_ARG, "bytes is NULL");
    *bytes = detected_workspace_bytes(n, capacity);
    return OPX_OK;
}

opx_status opx_propagate_detected(const opx_scene* scene, uint64_t n, const uint64_t* d_n, uint64_t photon_id_base,
                                  const float* d_origins, const float* d_dirs, const float* d_wavelengths, uint64_t seed,
                                  uint32_t flags, const uint32_t* d_index, const opx_detected* out, uint64_t capacity,
                                  uint64_t* d_n_detected, void* d_workspace, size_t workspace_bytes, uint32_t* d_hitmap,
                                  uint64_t* d_counters, void* cuda_stream) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_propagate_detected before opx_bvh_build");
    if (flags & ~(uint32_t)OPX_FLAG_NO_EFFICIENCY) return fail(OPX_ERR_INVALID_ARG, "unknown flag");
    if (!d_n_detected || misaligned(d_n_detected, 8)) return fail(OPX_ERR_INVALID_ARG, "d_n_detected is NULL or misaligned");
    if (n == 0) return OPX_OK;
    if (!d_origins || !d_dirs || !d_wavelengths || !out || !d_workspace) return fail(OPX_ERR_INVALID_ARG, "NULL photon/list/workspace pointer");
    if (capacity && (!out->id || !out->pixel || !out->pos || !out->dir)) return fail(OPX_ERR_INVALID_ARG, "NULL list array");
    if (!capacity) return fail(OPX_ERR_INVALID_ARG, "capacity = 0");
    if (!d_hitmap && scene->n_pixels) return fail(OPX_ERR_INVALID_ARG, "d_hitmap is NULL but the scene has pixels");
    if (misaligned(d_origins, 4) || misaligned(d_dirs, 4) || misaligned(d_wavelengths, 4) || misaligned(out->id, 8) ||
        misaligned(out->pixel, 4) || misaligned(out->pos, 4) || misaligned(out->dir, 4) || misaligned(d_hitmap, 4) ||
        misaligned(d_counters, 8) || misaligned(d_n, 8) || misaligned(d_index, 4) || misaligned(d_workspace, 256))
        return fail(OPX_ERR_INVALID_ARG, "misaligned pointer");
    if (workspace_bytes < detected_workspace_bytes(n, capacity)) return fail(OPX_ERR_WORKSPACE_TOO_SMALL, "workspace too small (see opx_propagate_detected_workspace_bytes)");
    if (scene->tri_surface.size() < 2) return fail(OPX_ERR_BAD_STATE, "the detected-only output needs a scene of two triangles or more");
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_propagate_detected")) return st;
    return launch_propagate_detected(*scene, n, d_n, photon_id_base, d_origins, d_dirs, d_wavelengths, seed, flags, *out, capacity,
                                     d_n_detected, d_index, d_workspace, d_hitmap, d_counters, (cudaStream_t)cuda_stream);
}

// ------------------------------------------------------------------------- host-buffer streaming
// Device staging per slot (kSlots slots, one stream each): inputs 28 B/photon, records 34 B/photon.  Three slots let the
// upload of chunk k+2 run while chunk k+1 computes and chunk k downloads, so neither copy engine waits for a buffer.
#ifndef OPX_HOST_SLOTS
#define OPX_HOST_SLOTS 3
#endif
static constexpr int kSlots = OPX_HOST_SLOTS;
static_assert(kSlots >= 2, "the host-buffer calls alternate between at least two slots / events");
}  // extern "C"

namespace opx {
struct HostPipe {
    cudaStream_t st[kSlots]{};
    cudaEvent_t done[kSlots]{}, kernel[kSlots]{}, start{};
    int device = -1;
    std::mutex busy;              // one host-buffer call per scene at a time (the calls synchronise anyway)
};
void destroy_host_pipe(HostPipe* p) {
    if (!p) return;
    for (int k = 0; k < kSlots; ++k) {
        if (p->st[k]) cudaStreamDestroy(p->st[k]);
        if (p->done[k]) cudaEventDestroy(p->done[k]);
        if (p->kernel[k]) cudaEventDestroy(p->kernel[k]);
    }
    if (p->start) cudaEventDestroy(p->start);
    delete p;
}
static std::mutex g_pipe_mutex;
void drop_host_pipe_of_other_device(const SceneHost& s) {
    std::lock_guard<std::mutex> lock(g_pipe_mutex);
    int dev = 0;
    if (!s.pipe || cudaGetDevice(&dev) != cudaSuccess || s.pipe->device == dev) return;
    destroy_host_pipe(s.pipe);
    s.pipe = nullptr;
}
// The scene's pipe, created on its first host-buffer call (streams and events are not created per call).
static opx_status host_pipe(const SceneHost& s, HostPipe** out) {
    std::lock_guard<std::mutex> lock(g_pipe_mutex);
    int dev = 0;
    if (opx_status st = check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return st;
    // never torn down here: another thread may be inside propagate_host_impl with these streams (opx_bvh_build, which needs the
    // scene to itself anyway, drops the pipe when the scene moves to another device)
    if (s.pipe && s.pipe->device != dev)
        return fail(OPX_ERR_BAD_STATE, "host-buffer call with another device current than the one this scene's host-buffer calls started on");
    if (!s.pipe) {
        HostPipe* p = new HostPipe;
        p->device = dev;
        cudaError_t e = cudaEventCreateWithFlags(&p->start, cudaEventDisableTiming);
        for (int k = 0; k < kSlots && e == cudaSuccess; ++k) {
            e = cudaStreamCreateWithFlags(&p->st[k], cudaStreamNonBlocking);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->done[k], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->kernel[k], cudaEventDisableTiming);
        }
        if (e != cudaSuccess) { destroy_host_pipe(p); return check_cuda(e, "creating the streams of the host-buffer path"); }
        s.pipe = p;
    }
    *out = s.pipe;
    return OPX_OK;
}

static size_t slot_bytes(uint64_t chunk, bool records) {
    size_t b = 0;
    b += align_up(chunk * 12, 256) * (records ? 4 : 2);   // origins, dirs (, pos, dir)
    b += align_up(chunk * 4, 256) * (records ? 3 : 1);    // wavelengths (, pixel, surface)
    if (records) b += align_up(chunk, 256) * 2;           // state, bounces
    return b;
}
static size_t host_workspace_bytes(const SceneHost& s, uint64_t chunk, bool records, uint64_t capacity) {
    size_t b = kSlots * slot_bytes(chunk, records) + align_up(s.n_pixels * 4 + 4, 256) + 256;
    // the device copy of the list + the workspace of the detected-only launches (one: the chunks' kernels run one after another)
    if (!records) b += align_up(capacity * 8, 256) + align_up(capacity * 4, 256) + 2 * align_up(capacity * 12, 256) + 256 + detected_workspace_bytes(chunk, capacity);
    return b;
}

// Both host-buffer calls: h_out (per-photon records) or h_det (detected-only list), never both.
static opx_status propagate_host_impl(const SceneHost& scene, uint64_t n, uint64_t photon_id_base, const float* h_origins,
                                      const float* h_dirs, const float* h_wavelengths, uint64_t seed, uint32_t flags,
                                      const opx_hits* h_out, const opx_detected* h_det, uint64_t capacity, uint64_t* h_n_detected,
                                      uint32_t* h_hitmap, uint64_t* h_counters, void* d_workspace, uint64_t chunk, cudaStream_t main) {
    const bool records = h_out != nullptr;
    HostPipe* pipe = nullptr;
    if (opx_status st = host_pipe(scene, &pipe)) return st;
    std::lock_guard<std::mutex> lock(pipe->busy);
    struct Slot { float *o, *d, *wl, *pos, *dir; int32_t *pixel, *surface; uint8_t *state, *bounces; };
    Slot slot[kSlots];
    char* p = (char*)d_workspace;
    auto take = [&](size_t bytes) { char* r = p; p += align_up(bytes, 256); return r; };
    for (int k = 0; k < kSlots; ++k) {
        Slot& s = slot[k];
        s = Slot{};
        s.o = (float*)take(chunk * 12); s.d = (float*)take(chunk * 12); s.wl = (float*)take(chunk * 4);
        if (records) {
            s.pos = (float*)take(chunk * 12); s.dir = (float*)take(chunk * 12);
            s.pixel = (int32_t*)take(chunk * 4); s.surface = (int32_t*)take(chunk * 4);
            s.state = (uint8_t*)take(chunk); s.bounces = (uint8_t*)take(chunk);
        }
    }
    uint32_t* d_hitmap = (uint32_t*)take(scene.n_pixels * 4 + 4);
    uint64_t* d_counters = (uint64_t*)take(64);           // [0..7] counters, then the detected list's length
    uint64_t* d_n_det = d_counters + 8;
    take(64);
    opx_detected det{};
    void* det_ws = nullptr;
    if (!records) {
        det.id = (uint64_t*)take(capacity * 8); det.pixel = (int32_t*)take(capacity * 4);
        det.pos = (float*)take(capacity * 12); det.dir = (float*)take(capacity * 12);
        det_ws = take(detected_workspace_bytes(chunk, capacity));
    }

    cudaError_t err = cudaSuccess;
    auto ck = [&](cudaError_t e) { if (e != cudaSuccess && err == cudaSuccess) err = e; };
    opx_status st = OPX_OK;
    // fork: the slot streams wait for whatever preceded on the caller's stream
    ck(cudaMemsetAsync(d_hitmap, 0, scene.n_pixels * 4 + 4, main));
    ck(cudaMemsetAsync(d_counters, 0, 128, main));
    ck(cudaEventRecord(pipe->start, main));
    for (int k = 0; k < kSlots; ++k) ck(cudaStreamWaitEvent(pipe->st[k], pipe->start, 0));

    uint64_t done = 0;
    int k = 0, prev = -1;
    // Chunk schedule: the first upload and the last download cannot overlap anything, so the stream is ramped up
    // (chunk/8, chunk/8, chunk/4, chunk/2, then full chunks) and ramped down (halving the remainder, floor chunk/8).
    const uint64_t small = chunk >= 8 ? chunk / 8 : 1;
    uint32_t issued = 0;
    while (done < n && st == OPX_OK && err == cudaSuccess) {
        uint64_t m = chunk;
        if (issued < 2) m = small; else if (issued == 2) m = chunk / 4 ? chunk / 4 : 1; else if (issued == 3) m = chunk / 2 ? chunk / 2 : 1;
        const uint64_t left = n - done;
        if (left < 2 * m) { const uint64_t half = (left + 1) / 2; m = half > small ? half : (left < small ? left : small); }
        if (m > left) m = left;
        ++issued;
        Slot& s = slot[k];
        cudaStream_t sst = pipe->st[k];
        ck(cudaMemcpyAsync(s.o, h_origins + 3 * done, m * 12, cudaMemcpyHostToDevice, sst));
        ck(cudaMemcpyAsync(s.d, h_dirs + 3 * done, m * 12, cudaMemcpyHostToDevice, sst));
        ck(cudaMemcpyAsync(s.wl, h_wavelengths + done, m * 4, cudaMemcpyHostToDevice, sst));
        if (records) {
            opx_hits dev_out{s.pos, s.dir, s.pixel, s.surface, s.state, s.bounces};
            st = launch_propagate(scene, kWalkProduct, m, nullptr, photon_id_base + done, s.o, s.d, s.wl, seed, flags, dev_out, d_hitmap,
                                  d_counters, sst);
            ck(cudaMemcpyAsync(h_out->pos + 3 * done, s.pos, m * 12, cudaMemcpyDeviceToHost, sst));
            ck(cudaMemcpyAsync(h_out->dir + 3 * done, s.dir, m * 12, cudaMemcpyDeviceToHost, sst));
            ck(cudaMemcpyAsync(h_out->pixel + done, s.pixel, m * 4, cudaMemcpyDeviceToHost, sst));
            ck(cudaMemcpyAsync(h_out->surface + done, s.surface, m * 4, cudaMemcpyDeviceToHost, sst));
            ck(cudaMemcpyAsync(h_out->state + done, s.state, m, cudaMemcpyDeviceToHost, sst));
            ck(cudaMemcpyAsync(h_out->bounces + done, s.bounces, m, cudaMemcpyDeviceToHost, sst));
        } else {
            // the chunks append to one list: a chunk's kernel starts after the previous chunk's (they would not overlap much
            // anyway: the uploads are what the pipeline waits for)
            if (prev >= 0) ck(cudaStreamWaitEvent(sst, pipe->kernel[prev], 0));
            st = launch_propagate_detected(scene, m, nullptr, photon_id_base + done, s.o, s.d, s.wl, seed, flags, det, capacity, d_n_det, nullptr,
                                           det_ws, d_hitmap, d_counters, sst);
            ck(cudaEventRecord(pipe->kernel[k], sst));
            prev = k;
        }
        done += m;
        k = (k + 1) % kSlots;
    }
    // join
    for (int j = 0; j < kSlots; ++j) { ck(cudaEventRecord(pipe->done[j], pipe->st[j])); ck(cudaStreamWaitEvent(main, pipe->done[j], 0)); }
    std::vector<uint32_t> hm(scene.n_pixels);
    uint64_t cnt[9] = {0};
    if (scene.n_pixels) ck(cudaMemcpyAsync(hm.data(), d_hitmap, scene.n_pixels * 4, cudaMemcpyDeviceToHost, main));
    ck(cudaMemcpyAsync(cnt, d_counters, 72, cudaMemcpyDeviceToHost, main));
    ck(cudaStreamSynchronize(main));
    if (!records && st == OPX_OK && err == cudaSuccess) {
        const uint64_t have = cnt[8] < capacity ? cnt[8] : capacity;
        if (have) {
            ck(cudaMemcpyAsync(h_det->id, det.id, have * 8, cudaMemcpyDeviceToHost, main));
            ck(cudaMemcpyAsync(h_det->pixel, det.pixel, have * 4, cudaMemcpyDeviceToHost, main));
            ck(cudaMemcpyAsync(h_det->pos, det.pos, have * 12, cudaMemcpyDeviceToHost, main));
            ck(cudaMemcpyAsync(h_det->dir, det.dir, have * 12, cudaMemcpyDeviceToHost, main));
            ck(cudaStreamSynchronize(main));
        }
        *h_n_detected = cnt[8];
    }
    if (st != OPX_OK) { cudaStreamSynchronize(main); return st; }
    if (err != cudaSuccess) { cudaStreamSynchronize(main); return check_cuda(err, "opx_propagate_host"); }
    for (uint64_t i = 0; i < scene.n_pixels; ++i) h_hitmap[i] += hm[i];
    if (h_counters) for (int i = 0; i < 8; ++i) h_counters[i] += cnt[i];
    return OPX_OK;
}
}  // namespace opx

extern "C" {
using namespace opx;

opx_status opx_propagate_host_workspace_bytes(const opx_scene* scene, uint64_t chunk, size_t* bytes) {
    if (!scene || !bytes || chunk == 0) return fail(OPX_ERR_INVALID_ARG, "NULL argument or chunk = 0");
    *bytes = host_workspace_bytes(*scene, chunk, true, 0);
    return OPX_OK;
}

opx_status opx_propagate_host_detected_workspace_bytes(const opx_scene* scene, uint64_t chunk, uint64_t capacity, size_t* bytes) {
    if (!scene || !bytes || chunk == 0 || capacity == 0) return fail(OPX_ERR_INVALID_ARG, "NULL argument, chunk = 0 or capacity = 0");
    *bytes = host_workspace_bytes(*scene, chunk, false, capacity);
    return OPX_OK;
}

opx_status opx_propagate_host(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* h_origins,
                              const float* h_dirs, const float* h_wavelengths, uint64_t seed, const opx_hits* h_out,
                              uint32_t* h_hitmap, uint64_t* h_counters, void* d_workspace, size_t workspace_bytes,
                              uint64_t chunk, void* cuda_stream) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_propagate_host before opx_bvh_build");
    if (n == 0) return OPX_OK;
    if (!h_origins || !h_dirs || !h_wavelengths || !h_out || !d_workspace || chunk == 0)
        return fail(OPX_ERR_INVALID_ARG, "NULL argument or chunk = 0");
    if (!h_out->pos || !h_out->dir || !h_out->pixel || !h_out->surface || !h_out->state || !h_out->bounces)
        return fail(OPX_ERR_INVALID_ARG, "NULL hit-record array");
    if (!h_hitmap && scene->n_pixels) return fail(OPX_ERR_INVALID_ARG, "h_hitmap is NULL but the scene has pixels");
    if (misaligned(d_workspace, 256)) return fail(OPX_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    if (workspace_bytes < host_workspace_bytes(*scene, chunk, true, 0)) return fail(OPX_ERR_WORKSPACE_TOO_SMALL, "workspace too small (see opx_propagate_host_workspace_bytes)");
    if (opx_status st = device_ok()) return st;
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_propagate_host")) return st;
    return propagate_host_impl(*scene, n, photon_id_base, h_origins, h_dirs, h_wavelengths, seed, 0u, h_out, nullptr, 0, nullptr, h_hitmap,
                               h_counters, d_workspace, chunk, (cudaStream_t)cuda_stream);
}

opx_status opx_propagate_host_detected(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* h_origins,
                                       const float* h_dirs, const float* h_wavelengths, uint64_t seed, uint32_t flags,
                                       const opx_detected* h_out, uint64_t capacity, uint64_t* h_n_detected, uint32_t* h_hitmap,
                                       uint64_t* h_counters, void* d_workspace, size_t workspace_bytes, uint64_t chunk, void* cuda_stream) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_propagate_host_detected before opx_bvh_build");
    if (flags & ~(uint32_t)OPX_FLAG_NO_EFFICIENCY) return fail(OPX_ERR_INVALID_ARG, "unknown flag");
    if (!h_n_detected) return fail(OPX_ERR_INVALID_ARG, "h_n_detected is NULL");
    *h_n_detected = 0;
    if (n == 0) return OPX_OK;
    if (!h_origins || !h_dirs || !h_wavelengths || !h_out || !d_workspace || chunk == 0 || capacity == 0)
        return fail(OPX_ERR_INVALID_ARG, "NULL argument, chunk = 0 or capacity = 0");
    if (!h_out->id || !h_out->pixel || !h_out->pos || !h_out->dir) return fail(OPX_ERR_INVALID_ARG, "NULL list array");
    if (!h_hitmap && scene->n_pixels) return fail(OPX_ERR_INVALID_ARG, "h_hitmap is NULL but the scene has pixels");
    if (scene->tri_surface.size() < 2) return fail(OPX_ERR_BAD_STATE, "the detected-only output needs a scene of two triangles or more");
    if (misaligned(d_workspace, 256)) return fail(OPX_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    if (workspace_bytes < host_workspace_bytes(*scene, chunk, false, capacity)) return fail(OPX_ERR_WORKSPACE_TOO_SMALL, "workspace too small (see opx_propagate_host_detected_workspace_bytes)");
    if (opx_status st = device_ok()) return st;
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_propagate_host_detected")) return st;
    return propagate_host_impl(*scene, n, photon_id_base, h_origins, h_dirs, h_wavelengths, seed, flags, nullptr, h_out, capacity,
                               h_n_detected, h_hitmap, h_counters, d_workspace, chunk, (cudaStream_t)cuda_stream);
}

// ------------------------------------------------------------------------- from track steps (host) to detected photons (host)
static size_t tracks_workspace_bytes(const SceneHost& s, uint64_t n_steps, uint64_t chunk, uint64_t capacity) {
    size_t b = 2 * align_up(n_steps * 12, 256) + 2 * align_up(n_steps * 4, 256) + align_up((n_steps + 1) * 8, 256);     // step table
    b += 2 * align_up(chunk * 12, 256) + 2 * align_up(chunk * 4, 256) + 256;                                          // photons of a chunk, index, count
    b += prefilter_workspace_bytes(chunk) + detected_workspace_bytes(chunk, capacity);
    b += align_up(capacity * 8, 256) + align_up(capacity * 4, 256) + 2 * align_up(capacity * 12, 256);               // the list on the device
    b += align_up(s.n_pixels * 4 + 4, 256) + 256;
    return b;
}

opx_status opx_tracks_host_detected_workspace_bytes(const opx_scene* scene, uint64_t n_steps, uint64_t chunk, uint64_t capacity, size_t* bytes) {
    if (!scene || !bytes || chunk == 0 || capacity == 0 || chunk > 0xffffffffull) return fail(OPX_ERR_INVALID_ARG, "NULL argument, chunk = 0, chunk > 2^32 - 1 or capacity = 0");
    *bytes = tracks_workspace_bytes(*scene, n_steps, chunk, capacity);
    return OPX_OK;
}

opx_status opx_tracks_host_detected(const opx_scene* scene, const opx_track_steps* h_steps, uint64_t n_total, float n_index, float lambda1_nm,
                                    float lambda2_nm, uint64_t n, uint64_t photon_id_base, uint64_t seed, const uint32_t* factors,
                                    uint32_t n_factors, const opx_detected* h_out, uint64_t capacity, uint64_t* h_n_detected,
                                    uint32_t* h_hitmap, uint64_t* h_counters, void* d_workspace, size_t workspace_bytes, uint64_t chunk,
                                    void* cuda_stream) {
    if (!scene || !h_steps) return fail(OPX_ERR_INVALID_ARG, "scene/steps is NULL");
    if (!scene->built) return fail(OPX_ERR_BAD_STATE, "opx_tracks_host_detected before opx_bvh_build");
    if (!h_n_detected) return fail(OPX_ERR_INVALID_ARG, "h_n_detected is NULL");
    *h_n_detected = 0;
    if (!(lambda1_nm > 0.f) || !(lambda2_nm > lambda1_nm) || !std::isfinite(lambda2_nm) || !std::isfinite(n_index))
        return fail(OPX_ERR_INVALID_ARG, "need 0 < lambda1 < lambda2 and a finite refractive index");
    if (n_factors > 8 || (n_factors && !factors)) return fail(OPX_ERR_INVALID_ARG, "n_factors must be <= 8 and factors non-NULL");
    for (uint32_t k = 0; k < n_factors; ++k) {
        if (factors[k] >= scene->mat_kinds.size()) return fail(OPX_ERR_INVALID_ARG, "factor material index out of range");
        if ((scene->mat_kinds[factors[k]] & 0xffu) == OPX_MAT_ABSORBER) return fail(OPX_ERR_INVALID_ARG, "an absorber has no efficiency table");
    }
    if (n == 0) return OPX_OK;
    const uint64_t S = h_steps->n_steps;
    if (S == 0 || !h_steps->x || !h_steps->w || !h_steps->length || !h_steps->beta || !h_steps->first)
        return fail(OPX_ERR_INVALID_ARG, "empty or NULL step table");
    if (photon_id_base > n_total || n > n_total - photon_id_base) return fail(OPX_ERR_INVALID_ARG, "photon ids beyond first[n_steps]");
    if (!h_out || !h_out->id || !h_out->pixel || !h_out->pos || !h_out->dir || !d_workspace || chunk == 0 || capacity == 0 || chunk > 0xffffffffull)
        return fail(OPX_ERR_INVALID_ARG, "NULL argument, chunk = 0, chunk > 2^32 - 1 or capacity = 0");
    if (!h_hitmap && scene->n_pixels) return fail(OPX_ERR_INVALID_ARG, "h_hitmap is NULL but the scene has pixels");
    if (scene->tri_surface.size() < 2) return fail(OPX_ERR_BAD_STATE, "the detected-only output needs a scene of two triangles or more");
    if (misaligned(d_workspace, 256)) return fail(OPX_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
    if (workspace_bytes < tracks_workspace_bytes(*scene, S, chunk, capacity)) return fail(OPX_ERR_WORKSPACE_TOO_SMALL, "workspace too small (see opx_tracks_host_detected_workspace_bytes)");
    if (opx_status st = device_ok()) return st;
    if (opx_status st = check_cuda(cudaGetLastError(), "pending CUDA error before opx_tracks_host_detected")) return st;

    cudaStream_t main = (cudaStream_t)cuda_stream;
    char* p = (char*)d_workspace;
    auto take = [&](size_t bytes) { char* r = p; p += align_up(bytes, 256); return r; };
    float* dx = (float*)take(S * 12); float* dw = (float*)take(S * 12); float* dl = (float*)take(S * 4); float* db = (float*)take(S * 4);
    uint64_t* df = (uint64_t*)take((S + 1) * 8);
    float* po = (float*)take(chunk * 12); float* pd = (float*)take(chunk * 12); float* pw = (float*)take(chunk * 4);
    uint32_t* pidx = (uint32_t*)take(chunk * 4);
    uint64_t* d_n_kept = (uint64_t*)take(256);
    void* pf_ws = take(prefilter_workspace_bytes(chunk));
    void* det_ws = take(detected_workspace_bytes(chunk, capacity));
    opx_detected det{(uint64_t*)take(capacity * 8), (int32_t*)take(capacity * 4), (float*)take(capacity * 12), (float*)take(capacity * 12)};
    uint32_t* d_hitmap = (uint32_t*)take(scene->n_pixels * 4 + 4);
    uint64_t* d_counters = (uint64_t*)take(128);
    uint64_t* d_n_det = d_counters + 8;

    // The step table goes up in slices on a side stream while the chunks before it are being traced: chunk k's emission needs
    // only the steps its photon ids fall into (a photon depends on its step's data, not on the step's index, so the kernels get
    // the slice as a table of its own), and the host knows which those are from first[].  The first kernel starts after the
    // first slice (a few MB) instead of after the whole table.
    HostPipe* pipe = nullptr;
    if (opx_status st0 = host_pipe(*scene, &pipe)) return st0;
    std::lock_guard<std::mutex> lock(pipe->busy);
    cudaStream_t up = pipe->st[0];
    cudaEvent_t slice_up = pipe->done[0];
    cudaError_t err = cudaSuccess;
    auto ck = [&](cudaError_t e) { if (e != cudaSuccess && err == cudaSuccess) err = e; };
    ck(cudaEventRecord(pipe->start, main));                  // the side stream starts after whatever used the workspace before
    ck(cudaStreamWaitEvent(up, pipe->start, 0));
    ck(cudaMemsetAsync(d_hitmap, 0, scene->n_pixels * 4 + 4, main));
    ck(cudaMemsetAsync(d_counters, 0, 128, main));
    const uint64_t* hf = h_steps->first;
    uint64_t uploaded = 0;                                   // steps [0, uploaded) and first[0 .. uploaded] are on their way
    bool first_slice = true;
    opx_status st = OPX_OK;
    // Chunk sizes: at most `chunk`; the first three are short (2^20, 2^22, 2^24 photons) so that tracing starts after a small
    // slice of the table, and a long last chunk leaves 2^22 photons to a chunk of their own so that little of the list is
    // still on the device when the last kernel ends.  Any chunking gives the same list (ids key the random streams).
    std::vector<uint64_t> sizes;
    for (uint64_t left = n; left;) {
        uint64_t c = chunk < left ? chunk : left;
        if (sizes.size() < 3) c = std::min<uint64_t>(c, 1ull << (20 + 2 * sizes.size()));
        if (c == left && c > (1ull << 24)) c -= 1ull << 22;
        sizes.push_back(c);
        left -= c;
    }
    // The list goes down chunk by chunk on a second side stream: once chunk k is queued the host reads the list's length as
    // chunk k-1 left it (a copy parked in a slot of its own, so that chunk k's scan cannot be seen half-way) and sends the
    // new entries on their way while chunk k runs.  Entries below `capacity` are never rewritten by a later chunk.
    cudaStream_t down = pipe->st[1];
    uint64_t* d_len = d_counters + 9;                        // 4 slots: the list's length after chunk k, k mod 4
    uint64_t downloaded = 0;
    auto fetch = [&](uint64_t upto) {
        const uint64_t hi = upto < capacity ? upto : capacity;
        if (hi <= downloaded) return;
        const uint64_t a = downloaded, c = hi - a;
        ck(cudaMemcpyAsync(h_out->id + a, det.id + a, c * 8, cudaMemcpyDeviceToHost, down));
        ck(cudaMemcpyAsync(h_out->pixel + a, det.pixel + a, c * 4, cudaMemcpyDeviceToHost, down));
        ck(cudaMemcpyAsync(h_out->pos + 3 * a, det.pos + 3 * a, c * 12, cudaMemcpyDeviceToHost, down));
        ck(cudaMemcpyAsync(h_out->dir + 3 * a, det.dir + 3 * a, c * 12, cudaMemcpyDeviceToHost, down));
        downloaded = hi;
    };
    uint64_t done = 0;
    for (size_t k = 0; k < sizes.size() && st == OPX_OK && err == cudaSuccess; done += sizes[k], ++k) {
        const uint64_t m = sizes[k];
        const uint64_t base = photon_id_base + done;
        // steps of this chunk: s_lo = the last step with first[s] <= base, s_hi = the first step with first[s] > base + m - 1
        const uint64_t s_lo = (uint64_t)(std::upper_bound(hf, hf + S + 1, base) - hf) - 1;
        uint64_t s_hi = (uint64_t)(std::upper_bound(hf, hf + S + 1, base + m - 1) - hf);
        if (s_lo >= S || hf[0] > base) { st = fail(OPX_ERR_INVALID_ARG, "first[] does not cover the photon ids (first[0] must be 0, first[n_steps] = n_total)"); break; }
        if (s_hi > S) s_hi = S;
        const uint64_t from = first_slice ? s_lo : uploaded;      // a call that starts in the middle of the table skips what lies before
        if (s_hi > from || first_slice) {
            const uint64_t cnt_steps = s_hi - from;
            ck(cudaMemcpyAsync(dx + 3 * from, h_steps->x + 3 * from, cnt_steps * 12, cudaMemcpyHostToDevice, up));
            ck(cudaMemcpyAsync(dw + 3 * from, h_steps->w + 3 * from, cnt_steps * 12, cudaMemcpyHostToDevice, up));
            ck(cudaMemcpyAsync(dl + from, h_steps->length + from, cnt_steps * 4, cudaMemcpyHostToDevice, up));
            ck(cudaMemcpyAsync(db + from, h_steps->beta + from, cnt_steps * 4, cudaMemcpyHostToDevice, up));
            const uint64_t f0 = first_slice ? from : from + 1;    // first[from] went up with the slice before
            ck(cudaMemcpyAsync(df + f0, hf + f0, (s_hi + 1 - f0) * 8, cudaMemcpyHostToDevice, up));
            ck(cudaEventRecord(slice_up, up));
            ck(cudaStreamWaitEvent(main, slice_up, 0));      // waits for THIS record; the event is recorded again for the next slice
            uploaded = s_hi;
            first_slice = false;
        }
        const opx_track_steps dsteps{dx + 3 * s_lo, dw + 3 * s_lo, dl + s_lo, db + s_lo, df + s_lo, s_hi - s_lo};
        if (n_factors) {
            st = launch_emit_filtered(*scene, dsteps, n_index, lambda1_nm, lambda2_nm, m, base, seed, factors, n_factors, po, pd, pw, pidx, m,
                                      d_n_kept, pf_ws, main);
            if (st == OPX_OK)
                st = launch_propagate_detected(*scene, m, d_n_kept, base, po, pd, pw, seed, OPX_FLAG_NO_EFFICIENCY, det, capacity, d_n_det, pidx,
                                               det_ws, d_hitmap, d_counters, main);
        } else {
            st = launch_emit(dsteps, n_index, lambda1_nm, lambda2_nm, m, base, seed, po, pd, pw, main);
            if (st == OPX_OK)
                st = launch_propagate_detected(*scene, m, nullptr, base, po, pd, pw, seed, 0u, det, capacity, d_n_det, nullptr, det_ws, d_hitmap,
                                               d_counters, main);
        }
        if (st != OPX_OK) break;
        ck(cudaMemcpyAsync(d_len + (k & 3), d_n_det, 8, cudaMemcpyDeviceToDevice, main));
        ck(cudaEventRecord(pipe->kernel[k % kSlots], main));
        if (k >= 1) {
            uint64_t len = 0;
            ck(cudaStreamWaitEvent(down, pipe->kernel[(k - 1) % kSlots], 0));
            ck(cudaMemcpyAsync(&len, d_len + ((k - 1) & 3), 8, cudaMemcpyDeviceToHost, down));
            ck(cudaStreamSynchronize(down));                 // chunk k-1 has ended; chunk k is queued or running
            if (err == cudaSuccess) fetch(len);
        }
    }
    std::vector<uint32_t> hm(scene->n_pixels);
    uint64_t cnt[9] = {0};
    if (scene->n_pixels) ck(cudaMemcpyAsync(hm.data(), d_hitmap, scene->n_pixels * 4, cudaMemcpyDeviceToHost, main));
    ck(cudaMemcpyAsync(cnt, d_counters, 72, cudaMemcpyDeviceToHost, main));
    ck(cudaStreamSynchronize(main));
    if (st == OPX_OK && err == cudaSuccess) {
        fetch(cnt[8]);                                       // what the last chunk added
        *h_n_detected = cnt[8];
    }
    ck(cudaStreamSynchronize(down));                         // the side streams are idle when the call returns, whatever happened
    ck(cudaStreamSynchronize(up));
    if (st != OPX_OK) return st;
    if (err != cudaSuccess) return check_cuda(err, "opx_tracks_host_detected");
    for (uint64_t i = 0; i < scene->n_pixels; ++i) h_hitmap[i] += hm[i];
    if (h_counters) for (int i = 0; i < 8; ++i) h_counters[i] += cnt[i];
    return OPX_OK;
}

opx_status opx_scene_info(const opx_scene* scene, uint64_t* n_triangles, uint64_t* n_nodes, uint64_t* n_pixels,
                          uint64_t* n_surfaces) {
    if (!scene) return fail(OPX_ERR_INVALID_ARG, "scene is NULL");
    const uint64_t T = scene->tri_surface.size();
    if (n_triangles) *n_triangles = T;
    if (n_nodes) *n_nodes = T > 1 ? T - 1 : 1;
    if (n_pixels) *n_pixels = scene->n_pixels;
    if (n_surfaces) *n_surfaces = scene->surfaces.size();
    return OPX_OK;
}

opx_status opx_scene_get_layout(const opx_scene* scene, opx_scene_layout* out) {
    if (!scene || !out) return fail(OPX_ERR_INVALID_ARG, "NULL argument");
    *out = scene->layout;
    return OPX_OK;
}

void opx_scene_destroy(opx_scene* scene) { delete scene; }

}  // extern "C"
