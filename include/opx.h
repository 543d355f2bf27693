/* opx.h -- C ABI of libopx.so: per-photon optical propagation on one B200 (sm_100a).
 *
 * The calls follow the paper's statement of the problem (arXiv:2309.12496; line numbers are
 * /root/reference/PAPER.md):
 *   - geometry  = triangle meshes grouped per material;
 *   - materials = per-material efficiency-vs-wavelength tables: mirror reflectivity, detector
 *                 quantum efficiency, applied in flight per interaction as the
 *                 paper proposes;
 *   - input     = "a vector input of initial positions and momenta", one ray per
 *                 entry, here as origins, unit directions and wavelengths;
 *   - output    = the global hit position of every photon and its 2-D detector
 *                 pixel from the corner point A along two in-plane unit vectors,
 *                 plus the pixel hit-map that replaces the paper's film/bitmap.
 * What each call computes, step by step and operation by operation, is DESIGN.md sections 2 and 3.
 *
 * Conventions
 *   Units: mm, nm.  All floating point data is IEEE binary32.
 *   Ownership: the CALLER owns every device byte (photon arrays, hit records, hit-map, counters,
 *     scene and build workspaces).  The library never allocates or frees device memory.  Host
 *     pointers passed to opx_scene_create are read during that call only.  An opx_scene is host
 *     memory owned by the library until opx_scene_destroy.
 *   Streams: `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls
 *     enqueue work and return without synchronising unless stated; an asynchronous CUDA failure is
 *     reported by the next call as OPX_ERR_CUDA.
 *   Errors: every entry point returns opx_status; nothing throws across the boundary.
 *     opx_last_error() gives a thread-local message for the last non-OK status.
 *   Device: requires compute capability 10.x (B200); anything else => OPX_ERR_UNSUPPORTED_DEVICE.
 *   Threading: a built scene is immutable; concurrent opx_propagate calls on different streams
 *     are allowed.  opx_bvh_build and opx_scene_destroy need the scene to themselves: no other call on
 *     that scene may be running or start until they return.  The host-buffer calls (opx_propagate_host,
 *     opx_propagate_host_detected, opx_tracks_host_detected) share one set of internal streams per scene:
 *     concurrent ones wait for each other, and all of them must be made with the device current on which
 *     the scene was built (OPX_ERR_BAD_STATE otherwise).
 */
#ifndef OPX_H_
#define OPX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct opx_scene opx_scene; /* opaque, host side */

typedef enum {
    OPX_OK = 0,
    OPX_ERR_INVALID_ARG = 1,
    OPX_ERR_BAD_STATE = 2,           /* e.g. propagate before bvh_build */
    OPX_ERR_WORKSPACE_TOO_SMALL = 3,
    OPX_ERR_CUDA = 4,
    OPX_ERR_UNSUPPORTED_DEVICE = 5
} opx_status;

typedef enum { OPX_MAT_ABSORBER = 0, OPX_MAT_MIRROR = 1, OPX_MAT_DETECTOR = 2 } opx_mat_kind;

/* Terminal state of a photon. */
typedef enum {
    OPX_DETECTED = 0,         /* reached a detector pixel and passed the QE draw              */
    OPX_QE_REJECTED = 1,      /* reached a detector pixel, failed the QE draw                 */
    OPX_ABSORBED_SURFACE = 2, /* hit an absorber                                              */
    OPX_ABSORBED_MIRROR = 3,  /* hit a mirror, failed the reflectivity draw                   */
    OPX_DETECTOR_DEAD = 4,    /* hit a detector surface outside its pixel grid                */
    OPX_BOUNCE_LIMIT = 5,     /* reflected max_bounces times                                  */
    OPX_ESCAPED = 6           /* no surface along the segment (also NaN / zero directions)    */
} opx_state;

typedef struct {
    float lambda_min_nm, lambda_max_nm; /* uniform wavelength grid of every table, max > min  */
    uint32_t n_lambda;                  /* points per table, >= 2                             */
    uint32_t max_bounces;               /* reflections before OPX_BOUNCE_LIMIT (16), 1..255   */
    float t_min_mm;                     /* minimum hit distance after a bounce (1e-3), >= 0   */
} opx_scene_params;

/* Form of a material's efficiency table.
 *   LINEAR     n_lambda points on the uniform grid lambda_min..lambda_max, piecewise linear, clamped;
 *   HISTOGRAM  the paper's form ("histograms of 33 nm bin width", "bins of 25 nm"): the
 *              n_lambda values are the contents of n_lambda equal bins tiling [lambda_min, lambda_max]; lower
 *              bin edges inclusive, the end bins extend outwards. */
typedef enum { OPX_TABLE_LINEAR = 0, OPX_TABLE_HISTOGRAM = 1 } opx_table_interp;

typedef struct {
    uint32_t kind;      /* opx_mat_kind                                                        */
    uint32_t interp;    /* opx_table_interp                                                    */
    const float* table; /* HOST, n_lambda values in [0,1]: reflectivity (mirror) or QE         */
                        /* (detector); ignored (may be NULL) for an absorber                   */
} opx_material;

/* Flags of opx_propagate_flags. */
typedef enum {
    OPX_FLAG_NO_EFFICIENCY = 1 /* efficiencies were applied before propagation (opx_prefilter): every mirror
                                  reflects, every detector pixel detects, no random number is drawn */
} opx_flags;

/* Detector pixel grid: a point p maps to a = (p-A).u, b = (p-A).v,
 * iu = floor(a / pitch_u), iv = floor(b / pitch_v); inside iff 0 <= iu < nu and 0 <= iv < nv;
 * pixel id = pixel_base + iv*nu + iu. */
typedef struct {
    float A[3], u[3], v[3]; /* corner point and the two in-plane unit vectors                  */
    float pitch_u, pitch_v; /* > 0                                                             */
    uint32_t nu, nv, pixel_base;
} opx_pixel_frame;

/* One surface = one mesh.  Surface id = index in the `meshes` array; global triangle id = triangles
 * of mesh 0 in order, then mesh 1, ... (used for tie-breaks and for `last triangle` skipping). */
typedef struct {
    const float* vertices;   /* HOST, n_vertices x 3, xyz packed                               */
    uint32_t n_vertices;
    const uint32_t* indices; /* HOST, n_triangles x 3, each < n_vertices                       */
    uint32_t n_triangles;
    uint32_t material;       /* index into `materials`                                         */
    int32_t pixel_frame;     /* index into `frames`; required (>= 0) iff the material is a     */
                             /* detector, ignored otherwise                                    */
    const float* vertex_normals; /* HOST, n_vertices x 3 unit normals (an OBJ file's `vn`), or NULL.  A mirror */
                             /* mesh that carries them reflects about the normal interpolated with the hit's  */
                             /* edge functions instead of the face    */
                             /* normal; components must be finite.  Ignored by detectors and absorbers.       */
} opx_mesh;

/* Per-photon hit records, DEVICE pointers, each of length n (pos, dir: n x 3 packed).
 *   pos     hit point of the last interaction (ESCAPED: origin of the last segment)
 *   dir     direction of arrival (BOUNCE_LIMIT: the reflected direction)
 *   pixel   detector pixel id, -1 unless state is DETECTED or QE_REJECTED
 *   surface surface id of the last hit, -1 for ESCAPED
 *   state   opx_state;  bounces = number of mirror reflections performed */
typedef struct {
    float* pos;
    float* dir;
    int32_t* pixel;
    int32_t* surface;
    uint8_t* state;
    uint8_t* bounces;
} opx_hits;

/* Byte offsets of the arrays opx_bvh_build leaves in the scene workspace (for tests that check
 * the BVH invariants; DESIGN.md section 8 gives the element layouts). */
typedef struct {
    uint64_t nodes;       /* (n_nodes) x 64 B                                                   */
    uint64_t triangles;   /* (n_triangles) x 48 B, leaf order                                   */
    uint64_t normals;     /* (n_triangles) x 16 B, leaf order: n.xyz, surface id bits           */
    uint64_t surfaces;    /* (n_surfaces) x 8 B: material, frame                                */
    uint64_t mat_kinds;   /* (n_materials) x 4 B                                                */
    uint64_t tables;      /* (n_materials) x n_lambda x 4 B                                     */
    uint64_t frames;      /* (n_frames) x 64 B                                                  */
    uint64_t sorted_keys; /* (n_triangles) x 8 B Morton keys in leaf order (kept for checking)  */
    uint64_t parents;     /* (2 n_triangles - 1) x 4 B: parent of internal node i / leaf T-1+i  */
    uint64_t wide_nodes;  /* (wide_node_capacity) x 896 B: 32-wide nodes collapsed from `nodes`  */
    uint64_t wide_node_capacity;
    uint64_t wide_count;  /* uint32: number of 32-wide nodes the build produced; 0 = the wide tree did not fit or is too deep */
    uint64_t vertex_normals; /* (n_triangles) x 36 B: na, nb, nc in GLOBAL triangle-id order; 16 B if no mesh has any */
    uint64_t total_bytes;
} opx_scene_layout;

/* A0.  Validates and flattens the meshes into one global triangle list, computes the face normals
 * and copies tables and frames.  Host only; no CUDA call.
 * Errors: NULL pointers, n_lambda < 2, lambda_max <= lambda_min, max_bounces outside 1..255,
 * negative t_min, material / frame / vertex index out of range, detector mesh without a frame,
 * non-positive pitch, zero-sized pixel grid, table value outside [0,1] or NaN, more than 2^28
 * triangles => OPX_ERR_INVALID_ARG.  n_meshes = 0 (an empty scene) is valid. */
opx_status opx_scene_create(const opx_scene_params* params, const opx_mesh* meshes, uint32_t n_meshes,
                            const opx_material* materials, uint32_t n_materials,
                            const opx_pixel_frame* frames, uint32_t n_frames, opx_scene** out);

/* Sizes of the two device workspaces opx_bvh_build needs: `scene_bytes` must stay alive and
 * untouched for as long as the scene is used; `build_tmp_bytes` may be released once the stream has
 * passed the build. */
opx_status opx_scene_workspace_bytes(const opx_scene* scene, size_t* scene_bytes, size_t* build_tmp_bytes);

/* A1-A4.  GPU LBVH build into the caller's workspaces (both 256-byte aligned device pointers):
 * scene AABB + 63-bit Morton keys of the triangle AABB centres, LSD radix sort, Karras hierarchy,
 * padded bottom-up refit, packing into 64-byte nodes and leaf-ordered triangles, collapse into the 32-wide tree.
 * Uploads the flattened scene first, then enqueues a fixed sequence of kernels on cuda_stream and returns: nothing
 * is read back and the stream is not synchronised (the uploads leave from pageable host memory, so the call returns
 * once the last of them has been staged; the scene's host arrays are not referenced afterwards).  Work that uses the
 * scene must be ordered after the build (same stream, or an event).  May be called again to rebuild.
 * Errors: OPX_ERR_WORKSPACE_TOO_SMALL, OPX_ERR_INVALID_ARG (NULL / misaligned),
 * OPX_ERR_UNSUPPORTED_DEVICE, OPX_ERR_CUDA. */
opx_status opx_bvh_build(opx_scene* scene, void* d_scene_ws, size_t scene_bytes,
                         void* d_tmp_ws, size_t tmp_bytes, void* cuda_stream);

/* A5-A12.  Propagates n photons (DEVICE pointers): origins and dirs n x 3 packed, wavelengths n, in
 * nm.  Directions must be unit length; they are NOT renormalised.  Global photon id = photon_id_base
 * + i keys the random stream (seed, id, bounce), so any chunking gives identical per-id results.
 * Writes the hit records, ADDS detected photons to d_hitmap (n_pixels uint32) and ADDS to
 * d_counters (8 uint64: one per opx_state 0..6, [7] = closest-hit queries); the caller zeroes both.
 * d_hitmap may be NULL only if the scene has no pixels; d_counters may be NULL.  n = 0 is a no-op.
 * Errors: OPX_ERR_BAD_STATE before opx_bvh_build; OPX_ERR_INVALID_ARG for NULL / misaligned
 * (4-byte) pointers; OPX_ERR_CUDA. */
opx_status opx_propagate(const opx_scene* scene, uint64_t n, uint64_t photon_id_base,
                         const float* d_origins, const float* d_dirs, const float* d_wavelengths,
                         uint64_t seed, const opx_hits* out, uint32_t* d_hitmap, uint64_t* d_counters,
                         void* cuda_stream);

/* opx_propagate with `flags` (opx_flags, 0 = opx_propagate) and an optional photon count that lives on the
 * device: if d_n is not NULL the kernels propagate min(n, *d_n) photons (read when the kernels run, so the count
 * written by opx_prefilter on the same stream is used without a host round trip); records beyond it are left
 * untouched.  n then only bounds the launch and the arrays. */
opx_status opx_propagate_flags(const opx_scene* scene, uint64_t n, const uint64_t* d_n, uint64_t photon_id_base,
                               const float* d_origins, const float* d_dirs, const float* d_wavelengths,
                               uint64_t seed, uint32_t flags, const opx_hits* out, uint32_t* d_hitmap,
                               uint64_t* d_counters, void* cuda_stream);

/* Pre-propagation efficiency filter, the paper's own method ("it is advantageous to apply any
 * quantum efficiency and reflectivity effects prior to propagation and discard the associated photons ... For
 * each photon, with its specific wavelength, an accept-reject algorithm was used to model the three
 * efficiencies before propagation").  DESIGN.md 3.9: photon i is kept iff
 *     U(seed, photon_id_base + i, 0; stream 1)  <  e_0(lambda_i) * e_1(lambda_i) * ... (left to right, fp32),
 * e_k = the table of material factors[k] (HOST array of n_factors <= 8 material indices, e.g. detector, mirror 1,
 * mirror 2; a material may repeat; n_factors = 0 keeps everything).  The kept photons are written in input
 * order (stable compaction) to d_out_origins / d_out_dirs (x3) / d_out_wavelengths, their index i to
 * d_out_index (may be NULL), and their number to *d_n_kept (DEVICE uint64, overwritten).  The out arrays hold
 * out_capacity entries each (n is always enough) and must not alias the inputs: survivors beyond out_capacity are
 * not written, but *d_n_kept still receives the TRUE count, so *d_n_kept > out_capacity tells the caller that the
 * list was truncated.  n <= 2^32 - 1.  Trace the survivors with
 * opx_propagate_flags(..., n, d_n_kept, ..., OPX_FLAG_NO_EFFICIENCY, ...).
 * d_workspace: opx_prefilter_workspace_bytes(n) device bytes, 256-byte aligned. */
opx_status opx_prefilter_workspace_bytes(uint64_t n, size_t* bytes);
opx_status opx_prefilter(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                         const float* d_dirs, const float* d_wavelengths, uint64_t seed,
                         const uint32_t* factors, uint32_t n_factors,
                         float* d_out_origins, float* d_out_dirs, float* d_out_wavelengths, uint32_t* d_out_index,
                         uint64_t out_capacity, uint64_t* d_n_kept, void* d_workspace, size_t workspace_bytes,
                         void* cuda_stream);

/* opx_prefilter for callers that cannot allocate device memory.  Some users of this library never get to call
 * cudaMalloc: a plug-in inside an experiment framework (a Geant4 worker, a trigger-farm process) is handed its photon
 * buffers by the framework's memory pool, which has reserved the whole card and forbids allocations of its own; and a
 * worker thread in an event loop that shares the GPU with other threads' streams cannot afford cudaMalloc / cudaFree,
 * which make every stream on the device wait.  Such a caller has input and output arrays but nowhere to put the
 * filter's workspace.  This call needs none: the mask words and per-block counts live in a fixed array compiled into
 * libopx.so (about 2 MiB; every GPU that loads the library's device code holds it until the process exits).
 *   - Arguments, results and errors are those of opx_prefilter without d_workspace / workspace_bytes; the output is the
 *     same bytes opx_prefilter produces.  The caller still owns and passes every input and output array.
 *   - n <= OPX_PREFILTER_NOALLOC_MAX_PHOTONS, otherwise OPX_ERR_INVALID_ARG with a message naming the limit: split the
 *     photons over several calls (photon_id_base keeps the draws identical) or use opx_prefilter.
 *   - The call never allocates or frees device memory, neither directly nor through a library routine: it enqueues the
 *     three kernels of opx_prefilter (for n = 0 one 8-byte memset of *d_n_kept) and returns.
 *   - The first call with n >= 1 on each device looks up where that device keeps the array (one cudaGetSymbolAddress,
 *     which loads the library's device code there if it is not loaded yet) and remembers the answer.  Make that first
 *     call with the device current and before any stream capture begins; a call with n = 0 does not do the look-up.
 *   - All calls on one device share the one array, and it keeps whatever the previous call left in it.  The kernels
 *     overwrite every word they later read, so nothing has to be cleared between calls -- but two calls whose kernels
 *     can run at the same time on one GPU (different streams without an event between them, or two host threads)
 *     overwrite each other's masks and give wrong survivors.  Order such calls on one stream or with events.
 *   - Device ordinals 0..63. */
#define OPX_PREFILTER_NOALLOC_MAX_PHOTONS 16777216ull /* 2^24 photons per call */
opx_status opx_prefilter_noalloc(const opx_scene* scene, uint64_t n, uint64_t photon_id_base, const float* d_origins,
                                 const float* d_dirs, const float* d_wavelengths, uint64_t seed,
                                 const uint32_t* factors, uint32_t n_factors,
                                 float* d_out_origins, float* d_out_dirs, float* d_out_wavelengths, uint32_t* d_out_index,
                                 uint64_t out_capacity, uint64_t* d_n_kept, void* cuda_stream);

/* Track steps for opx_emit_cherenkov: DEVICE pointers.  Step s starts at x[s], runs along the unit vector w[s] for
 * length[s] mm with velocity beta[s]; first (n_steps + 1 entries, non-decreasing, first[0] = 0) is the exclusive
 * prefix sum of the photons emitted per step: global photon g belongs to the step with first[s] <= g < first[s+1].
 * The photon COUNT per step is the caller's (Geant4's, or a Frank-Tamm yield). */
typedef struct {
    const float* x;        /* n_steps x 3 */
    const float* w;        /* n_steps x 3, unit */
    const float* length;   /* n_steps, mm */
    const float* beta;     /* n_steps */
    const uint64_t* first; /* n_steps + 1 */
    uint64_t n_steps;
} opx_track_steps;

/* Cherenkov photons generated on the device from charged-track steps (PAPER.md:71:
 * cos(theta_c) = 1/(n beta); the paper writes Geant4's photons to a file and wants the loop
 * memory-resident).  Photons photon_id_base .. photon_id_base + n - 1 are written to d_origins / d_dirs (n x 3) and
 * d_wavelengths (n) - the arrays opx_propagate and opx_prefilter read - entry g - photon_id_base for photon g:
 * position uniform along its step, polar angle theta_c about the track (along the track if n beta <= 1), azimuth
 * uniform, wavelength with density 1/lambda^2 on [lambda1_nm, lambda2_nm]; operation by operation DESIGN.md 3.12.
 * A photon depends on (seed, g, its step) only, so any split of the id range over calls or GPUs gives the same bits.
 * n_total = first[n_steps] as the HOST knows it: photon_id_base + n > n_total, n_steps = 0 with n > 0, NULL pointers,
 * lambda1 <= 0 or lambda2 <= lambda1, n_index not finite => OPX_ERR_INVALID_ARG.  n = 0 is valid.  Enqueues one
 * kernel on cuda_stream; needs no scene. */
opx_status opx_emit_cherenkov(const opx_track_steps* steps, uint64_t n_total, float n_index, float lambda1_nm,
                              float lambda2_nm, uint64_t n, uint64_t photon_id_base, uint64_t seed, float* d_origins,
                              float* d_dirs, float* d_wavelengths, void* cuda_stream);

/* opx_emit_cherenkov followed by opx_prefilter in one call, without ever writing the photons the filter discards
 * (6 of 7 with the paper's efficiencies): the paper's whole front end - photons from track steps, the three
 * efficiencies applied before propagation - memory-resident.  By definition the
 * result is that of the two calls (DESIGN.md 3.12 then 3.9, nothing new is computed): the survivors among photons
 * photon_id_base .. photon_id_base + n - 1, in id order, in d_out_origins / d_out_dirs / d_out_wavelengths, their
 * offsets g - photon_id_base in d_out_index (may be NULL), their number in *d_n_kept (DEVICE uint64, overwritten).
 * The out arrays hold out_capacity entries each (n covers the worst case, factors with efficiency 1; an upper bound
 * on the kept fraction is enough in practice): survivors beyond out_capacity are not written, and *d_n_kept still
 * receives the TRUE count, so *d_n_kept > out_capacity reports the truncation.  n <= 2^32 - 1.  Arguments and errors as in opx_emit_cherenkov and opx_prefilter;
 * d_workspace: opx_prefilter_workspace_bytes(n) device bytes, 256-byte aligned.  Three launches, no host round trip;
 * trace the survivors with opx_propagate_flags(..., n, d_n_kept, ..., OPX_FLAG_NO_EFFICIENCY, ...). */
opx_status opx_emit_cherenkov_filtered(const opx_scene* scene, const opx_track_steps* steps, uint64_t n_total, float n_index,
                                       float lambda1_nm, float lambda2_nm, uint64_t n, uint64_t photon_id_base, uint64_t seed,
                                       const uint32_t* factors, uint32_t n_factors, float* d_out_origins, float* d_out_dirs,
                                       float* d_out_wavelengths, uint32_t* d_out_index, uint64_t out_capacity,
                                       uint64_t* d_n_kept, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* List of DETECTED photons, DEVICE pointers, each array of `capacity` entries (pos, dir: capacity x 3 packed): what the paper
 * asks the emitter-to-detector loop to produce, "the position of the ray in a list when it interacts with the detector"
 * (PAPER.md:195).  Entry r: global photon id, detector pixel id, hit position, direction of arrival - the fields of the
 * photon's hit record (opx_hits), for photons whose state is OPX_DETECTED only. */
typedef struct {
    uint64_t* id;
    int32_t* pixel;
    float* pos;
    float* dir;
} opx_detected;

/* opx_propagate_flags with a compacted output: instead of one hit record per photon, the photons that end DETECTED are
 * APPENDED to the list `out`, in increasing photon id (stable: the result does not depend on scheduling, two runs give
 * identical bytes).  *d_n_detected (DEVICE uint64) is the list's length: on entry the number of entries already in it
 * (the caller zeroes it once), on exit increased by the number of photons this call detected.  While *d_n_detected <=
 * capacity the list is complete.  Entries that do not fit are dropped but still counted, so *d_n_detected > capacity
 * reports a truncated list; a truncated list holds `capacity` entries in increasing id, not necessarily those with
 * the smallest ids.  Calls that append to the same list must be ordered (same stream, or events): a later call reads
 * the length an earlier one wrote.  Hit-map and counters as in opx_propagate (every photon is counted, whatever its state).  The per-photon
 * results are those of opx_propagate_flags bit for bit: this call only leaves out the 34 B/photon of records
 * nobody asked for.  Three launches and one memset, no host round trip: the propagation kernel stages each tile's
 * detected photons in the workspace in the order the tiles finish, a scan and a gather kernel move them to the list in
 * photon-id order.  d_workspace: opx_propagate_detected_workspace_bytes(n, capacity) device bytes, 256-byte aligned, used
 * while the call's kernels run.  d_index (DEVICE, n entries, may be NULL): when the inputs are the survivors of
 * opx_prefilter / opx_emit_cherenkov_filtered, the index array that call wrote - the list then carries the ORIGINAL
 * photon ids photon_id_base + d_index[i] (increasing, the filters being stable) instead of photon_id_base + i; it
 * changes nothing else.  Needs a scene of two triangles or more (OPX_ERR_BAD_STATE otherwise).  Other arguments
 * and errors as in opx_propagate_flags. */
opx_status opx_propagate_detected_workspace_bytes(uint64_t n, uint64_t capacity, size_t* bytes);
opx_status opx_propagate_detected(const opx_scene* scene, uint64_t n, const uint64_t* d_n, uint64_t photon_id_base,
                                  const float* d_origins, const float* d_dirs, const float* d_wavelengths,
                                  uint64_t seed, uint32_t flags, const uint32_t* d_index, const opx_detected* out,
                                  uint64_t capacity, uint64_t* d_n_detected, void* d_workspace, size_t workspace_bytes,
                                  uint32_t* d_hitmap, uint64_t* d_counters, void* cuda_stream);

/* Size of the device staging workspace opx_propagate_host needs for chunks of `chunk` photons. */
opx_status opx_propagate_host_workspace_bytes(const opx_scene* scene, uint64_t chunk, size_t* bytes);

/* End-to-end form with HOST buffers (pinned memory recommended): origins, dirs, wavelengths and the
 * six record arrays of `out` are host pointers of length n; h_hitmap (n_pixels, +=) and h_counters
 * (8, +=, may be NULL) are host arrays.  Photons are streamed through the caller's device workspace
 * in chunks of at most `chunk` photons (the first and last few are smaller, to shorten the part of the
 * pipeline that cannot overlap), the upload of one chunk, the kernel of the next and the download of a
 * third overlapping on three internal streams forked from and joined into `cuda_stream`.  Synchronises
 * `cuda_stream` before returning.  DESIGN.md 8.5. */
opx_status opx_propagate_host(const opx_scene* scene, uint64_t n, uint64_t photon_id_base,
                              const float* h_origins, const float* h_dirs, const float* h_wavelengths,
                              uint64_t seed, const opx_hits* h_out, uint32_t* h_hitmap,
                              uint64_t* h_counters, void* d_workspace, size_t workspace_bytes,
                              uint64_t chunk, void* cuda_stream);

/* opx_propagate_host with the detected-only output of opx_propagate_detected: photons are uploaded in chunks as in
 * opx_propagate_host, nothing but the list of detected photons (HOST arrays of `capacity` entries in h_out), the hit-map
 * and the counters comes back - 28 B per photon up, 36 B per DETECTED photon down.  *h_n_detected receives the number of
 * detected photons of this call (entries beyond capacity are dropped but counted); the list starts at entry 0.
 * d_workspace: opx_propagate_host_detected_workspace_bytes(scene, chunk, capacity) device bytes, 256-byte aligned.
 * Synchronises `cuda_stream` before returning. */
opx_status opx_propagate_host_detected_workspace_bytes(const opx_scene* scene, uint64_t chunk, uint64_t capacity, size_t* bytes);
opx_status opx_propagate_host_detected(const opx_scene* scene, uint64_t n, uint64_t photon_id_base,
                                       const float* h_origins, const float* h_dirs, const float* h_wavelengths,
                                       uint64_t seed, uint32_t flags, const opx_detected* h_out, uint64_t capacity,
                                       uint64_t* h_n_detected, uint32_t* h_hitmap, uint64_t* h_counters,
                                       void* d_workspace, size_t workspace_bytes, uint64_t chunk, void* cuda_stream);

/* The paper's whole loop, memory-resident (photons are written to a file by Geant4 today, "the rendering
 * loop" should run from memory): track steps in HOST memory in, the list of detected photons in HOST memory out; the photons
 * themselves never exist outside the device.  h_steps holds HOST pointers (opx_track_steps); photons photon_id_base ..
 * photon_id_base + n - 1 of its first[] are generated (opx_emit_cherenkov) and propagated in chunks of at most `chunk` (the
 * first few and the last are shorter; the step table goes up slice by slice and the list comes down chunk by chunk on internal
 * streams while other chunks are traced), the detected ones appended to h_out as in opx_propagate_host_detected.  n_factors = 0: efficiencies drawn in flight
 * (opx_emit_cherenkov then opx_propagate_detected).  n_factors > 0: the paper's own pipeline - the pre-propagation filter
 * on `factors` fused with the emission (opx_emit_cherenkov_filtered), the survivors traced with OPX_FLAG_NO_EFFICIENCY; the
 * list carries the original photon ids either way.  By definition the result is that of those calls.  Moves 40 B per track
 * step up and 36 B per detected photon down.  d_workspace: opx_tracks_host_detected_workspace_bytes(...) device bytes,
 * 256-byte aligned.  chunk <= 2^32 - 1.  Synchronises `cuda_stream` before returning. */
opx_status opx_tracks_host_detected_workspace_bytes(const opx_scene* scene, uint64_t n_steps, uint64_t chunk, uint64_t capacity,
                                                    size_t* bytes);
opx_status opx_tracks_host_detected(const opx_scene* scene, const opx_track_steps* h_steps, uint64_t n_total, float n_index,
                                    float lambda1_nm, float lambda2_nm, uint64_t n, uint64_t photon_id_base, uint64_t seed,
                                    const uint32_t* factors, uint32_t n_factors, const opx_detected* h_out, uint64_t capacity,
                                    uint64_t* h_n_detected, uint32_t* h_hitmap, uint64_t* h_counters, void* d_workspace,
                                    size_t workspace_bytes, uint64_t chunk, void* cuda_stream);

opx_status opx_scene_info(const opx_scene* scene, uint64_t* n_triangles, uint64_t* n_nodes,
                          uint64_t* n_pixels, uint64_t* n_surfaces);
opx_status opx_scene_get_layout(const opx_scene* scene, opx_scene_layout* out);

void opx_scene_destroy(opx_scene* scene);
const char* opx_last_error(void); /* thread-local, never NULL */
const char* opx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* OPX_H_ */
