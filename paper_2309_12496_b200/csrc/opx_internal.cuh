// Internal declarations shared by the translation units of libopx.so (CUDA path only).
// Written from DESIGN.md sections 2, 3 and 8; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/opx.h"

namespace opx {

// ------------------------------------------------------------------ device-side scene description
struct alignas(16) FrameDev {  // 64 B
    float Ax, Ay, Az, ux;
    float uy, uz, vx, vy;
    float vz, inv_pitch_u, inv_pitch_v, pad0;
    uint32_t nu, nv, pixel_base, pad1;
};

// BVH node, 64 B: boxes of the two children and their references.
//   q0 = (c0.lo.x, c0.lo.y, c0.lo.z, c0.hi.x)
//   q1 = (c0.hi.y, c0.hi.z, c1.lo.x, c1.lo.y)
//   q2 = (c1.lo.z, c1.hi.x, c1.hi.y, c1.hi.z)
//   q3 = (child0, child1, 0, 0) as int bits; child >= 0: internal node index; child < 0: leaf ~child
//   q3.z = number of leaves (triangles) below this node
struct alignas(16) NodeDev { float4 q0, q1, q2; int4 q3; };

// Wide BVH node, 896 B: up to 32 children in SoA so that lane k of a warp reads child k with seven
// coalesced 128-byte loads.  ref >= 0: wide node index; ref < 0: ~(leaf-order triangle index).
// Unused slots hold an empty box (lo = +inf, hi = -inf) that no beam can enter.
constexpr int kWide = 32;
struct alignas(128) WNodeDev { float lo[3][kWide]; float hi[3][kWide]; int ref[kWide]; };
constexpr int kWOffLo = 0, kWOffHi = 3 * kWide, kWOffRef = 6 * kWide;      // word offsets inside a WNodeDev

// Everything the propagation kernels need, passed by value as a kernel parameter.
struct SceneDev {
    const NodeDev* nodes;      // n_nodes
    const WNodeDev* wnodes;    // the 32-wide tree (n_wnodes = its capacity, 0: none was built)
    const uint32_t* wide_count; // device word the build leaves behind: number of wide nodes, 0 = the collapse did not fit (packets then
                               // walk the binary tree); read by the kernels, so opx_bvh_build never has to wait for it
    const float4* tris;        // 3 per triangle, leaf order: (a.xyz, id bits) (b.xyz, surface bits) (c.xyz, 0); then the same array with
                               // the components rotated to (y, z, x), then to (z, x, y)   (packet kernels: RayR::toff)
    const float4* normals;     // leaf order: n.xyz, surface id bits
    const float* vnormals;     // 9 per triangle (na, nb, nc), GLOBAL id order; NULL when no mesh carries vertex normals (3.11)
    const int2* surfaces;      // (material, frame)
    const uint32_t* mat_kinds; // opx_mat_kind | opx_table_interp << 8
    const float* tables;       // n_materials x n_lambda
    const FrameDev* frames;
    uint32_t n_tri, n_nodes, n_wnodes, n_lambda, max_bounces;
    float lambda_min, inv_dlambda, t_min;
    float inv_bin;             // histogram tables: n_lambda / (lambda_max - lambda_min)
    uint32_t flags;            // opx_flags of this launch (set per call, 0 in the stored copy)
    const unsigned long long* d_n;   // optional device-side photon count of this launch (min(n, *d_n) photons), else NULL
    float beam_max_width, beam_max_spread;   // packets wider than this (origins [mm] / directions) walk the binary tree
    float origin_limit;        // 4 x the largest |vertex coordinate|: a ray whose |o|_inf reaches this is walked with per-ray slack
};

struct Layout : opx_scene_layout {};
constexpr uint32_t kFlagPacketWalk = 1u << 16;   // internal launch flag (debug): incoherent packets walk the binary tree as a warp, not per lane

// A list of detected photons (opx_detected) as the kernels see it.  Inside a detected-only launch of the propagation kernel
// it describes the STAGING list of that launch (opx_packet.cuh, step 4b): tiles append their chunks at offsets taken from
// *stage_count and note them in tile_table.
struct DetOut {
    unsigned long long* id;      // NULL: this launch writes no detected list
    int32_t* pixel;
    float* pos;
    float* dir;
    unsigned long long capacity;
    unsigned long long* stage_count;   // entries handed out so far (zero at launch)
    ulonglong2* tile_table;            // (staging offset, count) per tile
    const uint32_t* index;             // optional: entry i of this launch is photon id_base + index[i] (the survivors of a filter)
};

// Streams and events of the host-buffer calls (opx_propagate_host*), created once per scene at the first such call.
struct HostPipe;
void destroy_host_pipe(HostPipe* p);
struct SceneHost;
void drop_host_pipe_of_other_device(const SceneHost& s);   // opx_bvh_build only: needs the scene to itself

// ------------------------------------------------------------------------------ host-side scene
struct SceneHost {
    opx_scene_params params{};
    std::vector<float> tri;          // T x 9, global id order
    std::vector<int32_t> tri_surface;
    std::vector<float> normals;      // T x 3, contract 3.4
    std::vector<float> tri_vnormals; // T x 9 (zeros for meshes without vertex normals), empty when no mesh has any
    std::vector<int2> surfaces;      // material, frame
    std::vector<uint32_t> mat_kinds;
    std::vector<float> tables;       // M x n_lambda
    std::vector<FrameDev> frames;
    uint64_t n_pixels = 0;
    float inv_dlambda = 0.f, inv_bin = 0.f;
    float leaf_pad = 1e-6f, tri_size = 0.f, scene_ext = 0.f, max_abs = 0.f;   // compute_scene_stats: box padding, typical triangle size, extent, largest |coordinate|
    // set by opx_bvh_build
    bool built = false;
    void* d_scene_ws = nullptr;
    size_t scene_bytes = 0;
    SceneDev dev{};
    opx_scene_layout layout{};
    // opx_profile_begin/end: event triples (start, after propagate, after bin), one per call
    mutable std::vector<cudaEvent_t> prof_events;
    mutable uint32_t prof_max = 0, prof_used = 0;
    mutable HostPipe* pipe = nullptr;
    ~SceneHost() { for (cudaEvent_t e : prof_events) cudaEventDestroy(e); destroy_host_pipe(pipe); }
};

// error plumbing (opx_api.cu)
opx_status fail(opx_status st, const std::string& msg);
opx_status check_cuda(cudaError_t e, const char* what);
void count_launch(uint64_t n = 1);
uint64_t launch_count();
void set_last_kernel(const char* name);   // name of the propagation kernel instantiation the last launch on this thread took
const char* last_kernel();

// build (opx_build.cu)
void compute_layout(const SceneHost& s, opx_scene_layout* lay, size_t* tmp_bytes);
void compute_scene_stats(SceneHost& s);
opx_status build_bvh(SceneHost& s, void* d_scene_ws, void* d_tmp_ws, cudaStream_t stream);

// propagate (opx_propagate.cu)
enum WalkMode { kWalkProduct = 0, kWalkBrute = 1, kWalkBinary = 2 };   // product path / every triangle (debug) / binary tree only (debug)
opx_status configure_device(int* sms = nullptr);      // per-device kernel attributes (dynamic shared memory sizes) and SM count; idempotent, thread-safe
opx_status propagate_common(const opx_scene* scene, WalkMode mode, uint64_t n, const uint64_t* d_n, uint64_t base, const float* o,
                            const float* d, const float* wl, uint64_t seed, uint32_t flags, const opx_hits* out, uint32_t* hitmap,
                            uint64_t* counters, void* stream);
opx_status device_ok();
opx_status launch_propagate(const SceneHost& s, WalkMode mode, uint64_t n, const uint64_t* d_n, uint64_t id_base, const float* o,
                            const float* d, const float* wl, uint64_t seed, uint32_t flags, const opx_hits& out,
                            uint32_t* hitmap, uint64_t* counters, cudaStream_t stream);
// the same launch writing the detected photons only, appended to a list in photon-id order (DetOut above)
opx_status launch_propagate_detected(const SceneHost& s, uint64_t n, const uint64_t* d_n, uint64_t id_base, const float* o,
                                     const float* d, const float* wl, uint64_t seed, uint32_t flags, const opx_detected& list,
                                     uint64_t capacity, uint64_t* d_n_detected, const uint32_t* d_index, void* workspace, uint32_t* hitmap,
                                     uint64_t* counters, cudaStream_t stream);
size_t detected_workspace_bytes(uint64_t n, uint64_t capacity);
// pre-propagation filter (opx_prefilter.cu)
size_t prefilter_workspace_bytes(uint64_t n);
opx_status launch_prefilter(const SceneHost& s, uint64_t n, uint64_t id_base, const float* o, const float* d, const float* wl,
                            uint64_t seed, const uint32_t* factors, uint32_t n_factors, float* oo, float* od, float* owl,
                            uint32_t* oidx, uint64_t capacity, uint64_t* d_n_kept, void* ws, cudaStream_t stream);
opx_status launch_stats(const SceneHost& s, uint64_t n, uint64_t id_base, const float* o, const float* d,
                        const float* wl, uint64_t seed, uint64_t* stats, cudaStream_t stream);
opx_status launch_packet_stats(const SceneHost& s, uint64_t n, uint64_t id_base, const float* o, const float* d,
                               const float* wl, uint64_t seed, const opx_hits& out, uint64_t* stats, cudaStream_t stream);
size_t wide_node_capacity(size_t n_triangles);
void launch_prefilter_scan(uint32_t* counts, uint32_t nb, uint64_t* d_total, cudaStream_t stream);   // exclusive scan in place + total
// Cherenkov emission (opx_emit.cu)
opx_status launch_emit_filtered(const SceneHost& s, const opx_track_steps& st, float n_index, float lambda1, float lambda2, uint64_t n,
                                uint64_t id_base, uint64_t seed, const uint32_t* factors, uint32_t n_factors, float* o, float* d,
                                float* wl, uint32_t* oidx, uint64_t capacity, uint64_t* d_n_kept, void* ws, cudaStream_t stream);
opx_status launch_emit(const opx_track_steps& st, float n_index, float lambda1, float lambda2, uint64_t n, uint64_t id_base,
                       uint64_t seed, float* o, float* d, float* wl, cudaStream_t stream);

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace opx

struct opx_scene : opx::SceneHost {};
