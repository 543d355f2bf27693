"""Thin Python binding of libopx.so (include/opx.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the CUDA kernels of
csrc/.  There is no CPU fallback: loading fails loudly if the library is missing.
Names follow include/opx.h (opx_scene_create -> Scene(...), opx_bvh_build -> Scene.build(),
opx_propagate -> Scene.propagate(), opx_propagate_host -> Scene.propagate_host()).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "lib", "libopx.so")

STATE_NAMES = ("DETECTED", "QE_REJECTED", "ABSORBED_SURFACE", "ABSORBED_MIRROR", "DETECTOR_DEAD",
               "BOUNCE_LIMIT", "ESCAPED")
OPX_OK, OPX_ERR_INVALID_ARG, OPX_ERR_BAD_STATE, OPX_ERR_WORKSPACE_TOO_SMALL, OPX_ERR_CUDA, \
    OPX_ERR_UNSUPPORTED_DEVICE = range(6)

FLAG_NO_EFFICIENCY = 1                   # opx_flags
PREFILTER_NOALLOC_MAX_PHOTONS = 1 << 24  # OPX_PREFILTER_NOALLOC_MAX_PHOTONS
TABLE_LINEAR, TABLE_HISTOGRAM = 0, 1     # opx_table_interp

# the product boundary (include/opx.h) ...
EXPORTS = ("opx_scene_create", "opx_scene_workspace_bytes", "opx_bvh_build", "opx_propagate",
           "opx_propagate_flags", "opx_prefilter_workspace_bytes", "opx_prefilter", "opx_prefilter_noalloc", "opx_emit_cherenkov",
           "opx_emit_cherenkov_filtered", "opx_propagate_host_workspace_bytes", "opx_propagate_host",
           "opx_propagate_detected_workspace_bytes", "opx_propagate_detected",
           "opx_propagate_host_detected_workspace_bytes", "opx_propagate_host_detected",
           "opx_tracks_host_detected_workspace_bytes", "opx_tracks_host_detected",
           "opx_scene_info", "opx_scene_get_layout", "opx_scene_destroy", "opx_last_error", "opx_version")
# ... and the debugging / measurement exports (include/opx_debug.h) that tests and bench.py use
DEBUG_EXPORTS = ("opx_propagate_brute", "opx_propagate_binary", "opx_profile_begin", "opx_profile_end", "opx_propagate_stats",
                 "opx_propagate_packet_stats", "opx_scene_wide_info", "opx_measure_fp32_peak", "opx_launch_count", "opx_last_kernel")


class OpxError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"opx status {status}: {message}")
        self.status = status


class SceneParams(C.Structure):
    _fields_ = [("lambda_min_nm", C.c_float), ("lambda_max_nm", C.c_float), ("n_lambda", C.c_uint32),
                ("max_bounces", C.c_uint32), ("t_min_mm", C.c_float)]


class Material(C.Structure):
    _fields_ = [("kind", C.c_uint32), ("interp", C.c_uint32), ("table", C.c_void_p)]


class PixelFrame(C.Structure):
    _fields_ = [("A", C.c_float * 3), ("u", C.c_float * 3), ("v", C.c_float * 3),
                ("pitch_u", C.c_float), ("pitch_v", C.c_float),
                ("nu", C.c_uint32), ("nv", C.c_uint32), ("pixel_base", C.c_uint32)]


class Mesh(C.Structure):
    _fields_ = [("vertices", C.c_void_p), ("n_vertices", C.c_uint32), ("indices", C.c_void_p),
                ("n_triangles", C.c_uint32), ("material", C.c_uint32), ("pixel_frame", C.c_int32),
                ("vertex_normals", C.c_void_p)]


class Hits(C.Structure):
    _fields_ = [("pos", C.c_void_p), ("dir", C.c_void_p), ("pixel", C.c_void_p), ("surface", C.c_void_p),
                ("state", C.c_void_p), ("bounces", C.c_void_p)]


class Detected(C.Structure):
    _fields_ = [("id", C.c_void_p), ("pixel", C.c_void_p), ("pos", C.c_void_p), ("dir", C.c_void_p)]


class TrackSteps(C.Structure):
    _fields_ = [("x", C.c_void_p), ("w", C.c_void_p), ("length", C.c_void_p), ("beta", C.c_void_p), ("first", C.c_void_p),
                ("n_steps", C.c_uint64)]


class SceneLayout(C.Structure):
    _fields_ = [(k, C.c_uint64) for k in ("nodes", "triangles", "normals", "surfaces", "mat_kinds", "tables",
                                          "frames", "sorted_keys", "parents", "wide_nodes", "wide_node_capacity", "wide_count",
                                          "vertex_normals", "total_bytes")]


_lib = None


def load_library(path=LIB_PATH):
    """dlopen libopx.so; raises if it has not been built (`python -m paper_2309_12496_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise OpxError(-1, f"{path} not found: build it with `python paper_2309_12496_b200/build.py` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, u64, u32 = C.c_void_p, C.c_uint64, C.c_uint32
    lib.opx_last_error.restype = C.c_char_p
    lib.opx_version.restype = C.c_char_p
    lib.opx_launch_count.restype = u64
    lib.opx_last_kernel.restype = C.c_char_p
    lib.opx_scene_create.argtypes = [vp, vp, u32, vp, u32, vp, u32, vp]
    lib.opx_scene_workspace_bytes.argtypes = [vp, vp, vp]
    lib.opx_bvh_build.argtypes = [vp, vp, C.c_size_t, vp, C.c_size_t, vp]
    for f in (lib.opx_propagate, lib.opx_propagate_brute, lib.opx_propagate_binary):
        f.argtypes = [vp, u64, u64, vp, vp, vp, u64, vp, vp, vp, vp]
    lib.opx_propagate_flags.argtypes = [vp, u64, vp, u64, vp, vp, vp, u64, u32, vp, vp, vp, vp]
    lib.opx_prefilter_workspace_bytes.argtypes = [u64, vp]
    lib.opx_prefilter.argtypes = [vp, u64, u64, vp, vp, vp, u64, vp, u32, vp, vp, vp, vp, u64, vp, vp, C.c_size_t, vp]
    lib.opx_prefilter_noalloc.argtypes = [vp, u64, u64, vp, vp, vp, u64, vp, u32, vp, vp, vp, vp, u64, vp, vp]
    lib.opx_emit_cherenkov.argtypes = [vp, u64, C.c_float, C.c_float, C.c_float, u64, u64, u64, vp, vp, vp, vp]
    lib.opx_emit_cherenkov_filtered.argtypes = [vp, vp, u64, C.c_float, C.c_float, C.c_float, u64, u64, u64, vp, u32,
                                                vp, vp, vp, vp, u64, vp, vp, C.c_size_t, vp]
    lib.opx_propagate_host_workspace_bytes.argtypes = [vp, u64, vp]
    lib.opx_propagate_host.argtypes = [vp, u64, u64, vp, vp, vp, u64, vp, vp, vp, vp, C.c_size_t, u64, vp]
    lib.opx_propagate_detected_workspace_bytes.argtypes = [u64, u64, vp]
    lib.opx_propagate_detected.argtypes = [vp, u64, vp, u64, vp, vp, vp, u64, u32, vp, vp, u64, vp, vp, C.c_size_t, vp, vp, vp]
    lib.opx_tracks_host_detected_workspace_bytes.argtypes = [vp, u64, u64, u64, vp]
    lib.opx_tracks_host_detected.argtypes = [vp, vp, u64, C.c_float, C.c_float, C.c_float, u64, u64, u64, vp, u32, vp, u64, vp, vp, vp,
                                             vp, C.c_size_t, u64, vp]
    lib.opx_propagate_host_detected_workspace_bytes.argtypes = [vp, u64, u64, vp]
    lib.opx_propagate_host_detected.argtypes = [vp, u64, u64, vp, vp, vp, u64, u32, vp, u64, vp, vp, vp, vp, C.c_size_t, u64, vp]
    lib.opx_profile_begin.argtypes = [vp, u32]
    lib.opx_profile_end.argtypes = [vp, vp, vp, vp]
    lib.opx_propagate_stats.argtypes = [vp, u64, u64, vp, vp, vp, u64, vp, vp]
    lib.opx_propagate_packet_stats.argtypes = [vp, u64, u64, vp, vp, vp, u64, vp, vp, vp]
    lib.opx_scene_wide_info.argtypes = [vp, vp, vp]
    lib.opx_measure_fp32_peak.argtypes = [vp, vp, vp]
    lib.opx_scene_info.argtypes = [vp, vp, vp, vp, vp]
    lib.opx_scene_get_layout.argtypes = [vp, vp]
    lib.opx_scene_destroy.argtypes = [vp]
    _lib = lib
    return lib


def _check(status):
    if status != OPX_OK:
        raise OpxError(status, load_library().opx_last_error().decode())


def measure_fp32_peak(device="cuda"):
    """opx_measure_fp32_peak -> TFLOP/s of the FP32 FMA micro-benchmark on the current device."""
    import torch
    scratch = torch.zeros(4, dtype=torch.float32, device=device)
    out = C.c_double()
    _check(load_library().opx_measure_fp32_peak(C.byref(out), scratch.data_ptr(),
                                                C.c_void_p(torch.cuda.current_stream(device).cuda_stream)))
    return out.value


def upload_track_steps(steps, device="cuda"):
    """Host step table (dict x, w, length, beta float32; first uint64 -- e.g. workloads.TrackSource.steps()) -> the
    same dict as CUDA tensors plus n_total = first[-1] as a Python int (first as an int64 view of the uint64 bits)."""
    import torch
    out = {k: torch.from_numpy(np.ascontiguousarray(steps[k], dtype=np.float32)).to(device) for k in ("x", "w", "length", "beta")}
    first = np.ascontiguousarray(steps["first"], dtype=np.uint64)
    out["first"] = torch.from_numpy(first.view(np.int64)).to(device)
    out["n_total"] = int(first[-1]) if len(first) else 0
    return out


def emit_cherenkov(dev_steps, n, photon_id_base=0, seed=0, n_index=1.0014, lambda1=200.0, lambda2=600.0, out=None, stream=None):
    """opx_emit_cherenkov on an uploaded step table -> (origins (n,3), dirs (n,3), wavelengths (n,)) CUDA tensors."""
    import torch
    dev = dev_steps["first"].device
    if out is None:
        out = (torch.empty((n, 3), dtype=torch.float32, device=dev), torch.empty((n, 3), dtype=torch.float32, device=dev),
               torch.empty(n, dtype=torch.float32, device=dev))
    st = TrackSteps(dev_steps["x"].data_ptr(), dev_steps["w"].data_ptr(), dev_steps["length"].data_ptr(),
                    dev_steps["beta"].data_ptr(), dev_steps["first"].data_ptr(), int(dev_steps["length"].shape[0]))
    s = stream if stream is not None else torch.cuda.current_stream(dev)
    _check(load_library().opx_emit_cherenkov(C.byref(st), int(dev_steps["n_total"]), n_index, lambda1, lambda2, int(n),
                                             int(photon_id_base), int(seed), out[0].data_ptr(), out[1].data_ptr(),
                                             out[2].data_ptr(), C.c_void_p(s.cuda_stream)))
    return out


def launch_count():
    return int(load_library().opx_launch_count())


def last_kernel():
    """opx_last_kernel: the propagation-kernel instantiation the last propagate call of this thread launched."""
    return load_library().opx_last_kernel().decode()


def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class Scene:
    """opx_scene handle.  `scene` is any object with the fields of workloads.Scene (meshes,
    materials, frames, lambda_min, lambda_max, n_lambda, max_bounces, t_min)."""

    def __init__(self, scene):
        lib = load_library()
        keep = []
        mats = (Material * max(1, len(scene.materials)))()
        for k, m in enumerate(scene.materials):
            t = np.ascontiguousarray(m["table"], dtype=np.float32)
            keep.append(t)
            mats[k].kind, mats[k].interp, mats[k].table = int(m["kind"]), int(m.get("interp", TABLE_LINEAR)), t.ctypes.data
        frames = (PixelFrame * max(1, len(scene.frames)))()
        for k, f in enumerate(scene.frames):
            frames[k].A[:] = [float(x) for x in f["A"]]
            frames[k].u[:] = [float(x) for x in f["u"]]
            frames[k].v[:] = [float(x) for x in f["v"]]
            frames[k].pitch_u, frames[k].pitch_v = f["pitch_u"], f["pitch_v"]
            frames[k].nu, frames[k].nv, frames[k].pixel_base = f["nu"], f["nv"], f["pixel_base"]
        meshes = (Mesh * max(1, len(scene.meshes)))()
        for k, m in enumerate(scene.meshes):
            v = np.ascontiguousarray(m["vertices"], dtype=np.float32)
            i = np.ascontiguousarray(m["indices"], dtype=np.uint32)
            keep += [v, i]
            meshes[k].vertices, meshes[k].n_vertices = v.ctypes.data, len(v)
            meshes[k].indices, meshes[k].n_triangles = i.ctypes.data, len(i)
            meshes[k].material, meshes[k].pixel_frame = int(m["material"]), int(m["frame"])
            if m.get("vertex_normals") is not None:
                vn = np.ascontiguousarray(m["vertex_normals"], dtype=np.float32)
                if vn.shape != v.shape:
                    raise OpxError(OPX_ERR_INVALID_ARG, "vertex_normals must have the shape of vertices")
                keep.append(vn)
                meshes[k].vertex_normals = vn.ctypes.data
        params = SceneParams(scene.lambda_min, scene.lambda_max, scene.n_lambda, scene.max_bounces, scene.t_min)
        handle = C.c_void_p()
        _check(lib.opx_scene_create(C.byref(params), meshes, len(scene.meshes), mats, len(scene.materials),
                                    frames, len(scene.frames), C.byref(handle)))
        self._h = handle
        nt, nn, npix, ns = C.c_uint64(), C.c_uint64(), C.c_uint64(), C.c_uint64()
        _check(lib.opx_scene_info(self._h, C.byref(nt), C.byref(nn), C.byref(npix), C.byref(ns)))
        self.n_triangles, self.n_nodes, self.n_pixels, self.n_surfaces = nt.value, nn.value, npix.value, ns.value
        self.workspace = None
        self._ws = {}       # cached device workspaces, one per (kind, device, stream): see _workspace()

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.opx_scene_destroy(self._h)
            self._h = None

    # ---------------------------------------------------------------------------------- build
    def workspace_bytes(self):
        a, b = C.c_size_t(), C.c_size_t()
        _check(load_library().opx_scene_workspace_bytes(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def layout(self):
        lay = SceneLayout()
        _check(load_library().opx_scene_get_layout(self._h, C.byref(lay)))
        return {k: getattr(lay, k) for k, _ in SceneLayout._fields_}

    def build(self, device="cuda", stream=None, keep_tmp=False):
        """opx_bvh_build into torch-owned workspaces; returns self."""
        import torch
        scene_b, tmp_b = self.workspace_bytes()
        self.workspace = torch.empty(scene_b + 256, dtype=torch.uint8, device=device)
        tmp = torch.empty(tmp_b + 256, dtype=torch.uint8, device=device)
        st = stream if stream is not None else torch.cuda.current_stream(device)
        _check(load_library().opx_bvh_build(self._h, _aligned(self.workspace), scene_b, _aligned(tmp), tmp_b,
                                            C.c_void_p(st.cuda_stream)))
        st.synchronize()
        if keep_tmp:
            self._tmp = tmp
        return self

    # ------------------------------------------------------------------------------ propagate
    def alloc_records(self, n, device="cuda"):
        import torch
        return dict(pos=torch.empty((n, 3), dtype=torch.float32, device=device),
                    dir=torch.empty((n, 3), dtype=torch.float32, device=device),
                    pixel=torch.empty(n, dtype=torch.int32, device=device),
                    surface=torch.empty(n, dtype=torch.int32, device=device),
                    state=torch.empty(n, dtype=torch.uint8, device=device),
                    bounces=torch.empty(n, dtype=torch.uint8, device=device))

    def alloc_accumulators(self, device="cuda"):
        import torch
        return (torch.zeros(max(1, self.n_pixels), dtype=torch.int32, device=device),
                torch.zeros(8, dtype=torch.int64, device=device))

    def propagate(self, origins, dirs, wavelengths, seed=0, photon_id_base=0, records=None, hitmap=None,
                  counters=None, stream=None, brute=False, flags=0, n_dev=None, binary=False):
        """opx_propagate on device tensors.  hitmap (int32 view of uint32) and counters (int64 view of
        uint64) are accumulated into; pass zeroed tensors or None to have them created.
        flags / n_dev (int64 CUDA tensor of one element: photon count left on the device by prefilter)
        select opx_propagate_flags.  brute / binary select the debug walks of include/opx_debug.h."""
        import torch
        n = int(wavelengths.shape[0])
        for t, shape in ((origins, (n, 3)), (dirs, (n, 3)), (wavelengths, (n,))):
            if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == shape):
                raise OpxError(OPX_ERR_INVALID_ARG, "photon tensors must be contiguous float32 CUDA tensors (n,3),(n,3),(n,)")
        dev = wavelengths.device
        if records is None:
            records = self.alloc_records(n, dev)
        if hitmap is None or counters is None:
            hm, ct = self.alloc_accumulators(dev)
            hitmap = hm if hitmap is None else hitmap
            counters = ct if counters is None else counters
        h = Hits(*(records[k].data_ptr() for k in ("pos", "dir", "pixel", "surface", "state", "bounces")))
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        if flags or n_dev is not None:
            if brute or binary:
                raise OpxError(OPX_ERR_INVALID_ARG, "the debug walks take no flags")
            _check(load_library().opx_propagate_flags(
                self._h, n, None if n_dev is None else n_dev.data_ptr(), int(photon_id_base), origins.data_ptr(),
                dirs.data_ptr(), wavelengths.data_ptr(), int(seed), int(flags), C.byref(h), hitmap.data_ptr(),
                counters.data_ptr(), C.c_void_p(st.cuda_stream)))
        else:
            lib = load_library()
            fn = lib.opx_propagate_brute if brute else (lib.opx_propagate_binary if binary else lib.opx_propagate)
            _check(fn(self._h, n, int(photon_id_base), origins.data_ptr(), dirs.data_ptr(), wavelengths.data_ptr(),
                      int(seed), C.byref(h), hitmap.data_ptr(), counters.data_ptr(), C.c_void_p(st.cuda_stream)))
        out = dict(records)
        out["hitmap"], out["counters"] = hitmap[:self.n_pixels], counters
        return out

    def alloc_detected(self, capacity, device="cuda"):
        """Device arrays of an opx_detected list + its length (int64 view of uint64, zero)."""
        import torch
        return dict(id=torch.empty(capacity, dtype=torch.int64, device=device), pixel=torch.empty(capacity, dtype=torch.int32, device=device),
                    pos=torch.empty((capacity, 3), dtype=torch.float32, device=device),
                    dir=torch.empty((capacity, 3), dtype=torch.float32, device=device),
                    n_detected=torch.zeros(1, dtype=torch.int64, device=device))

    def _workspace(self, kind, nbytes, device, stream):
        """Cached scratch tensor of at least nbytes + 256 bytes for calls of `kind` on `device` and `stream`.  Calls on
        different streams or devices never share one (they could run at the same time); `stream` None is for the
        host-buffer calls, which synchronise before they return.  A buffer that has to grow is handed back to torch's
        allocator only after the work already queued on its stream (record_stream)."""
        import torch
        device = torch.device(device)
        if device.index is None:
            device = torch.device("cuda", torch.cuda.current_device())
        key = (kind, device.index, None if stream is None else int(stream.cuda_stream))
        ws = self._ws.get(key)
        if ws is None or ws.numel() < nbytes + 256:
            if ws is not None and stream is not None:
                ws.record_stream(stream)
            ws = self._ws[key] = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
        return ws

    def propagate_detected(self, origins, dirs, wavelengths, seed=0, photon_id_base=0, capacity=None, out=None, hitmap=None,
                           counters=None, stream=None, flags=0, n_dev=None, index=None):
        """opx_propagate_detected: the DETECTED photons appended to `out` (alloc_detected) in photon-id order; out["n_detected"]
        is the running length on the device.  No per-photon records are written."""
        import torch
        n = int(wavelengths.shape[0])
        dev = wavelengths.device
        if out is None:
            out = self.alloc_detected(n if capacity is None else int(capacity), dev)
        cap = int(out["id"].shape[0])
        if hitmap is None or counters is None:
            hm, ct = self.alloc_accumulators(dev)
            hitmap = hm if hitmap is None else hitmap
            counters = ct if counters is None else counters
        lib = load_library()
        need = C.c_size_t()
        _check(lib.opx_propagate_detected_workspace_bytes(n, cap, C.byref(need)))
        d = Detected(*(out[k].data_ptr() for k in ("id", "pixel", "pos", "dir")))
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        ws = self._workspace("detected", need.value, dev, st)
        _check(lib.opx_propagate_detected(self._h, n, None if n_dev is None else n_dev.data_ptr(), int(photon_id_base),
                                          origins.data_ptr(), dirs.data_ptr(), wavelengths.data_ptr(), int(seed), int(flags),
                                          None if index is None else index.data_ptr(), C.byref(d), cap, out["n_detected"].data_ptr(), _aligned(ws), need.value,
                                          hitmap.data_ptr(), counters.data_ptr(), C.c_void_p(st.cuda_stream)))
        res = dict(out)
        res["hitmap"], res["counters"] = hitmap[:self.n_pixels], counters
        return res

    def propagate_host_detected(self, origins, dirs, wavelengths, seed=0, photon_id_base=0, capacity=None, chunk=1 << 20, out=None,
                                stream=None, device="cuda", flags=0):
        """opx_propagate_host_detected: host photon buffers in, the list of detected photons (host) + hit-map + counters out."""
        import torch
        lib = load_library()
        n = int(wavelengths.shape[0])
        chunk = max(1, min(int(chunk), max(n, 1)))
        if out is None:
            out = alloc_host_detected(max(1, n if capacity is None else int(capacity)), self.n_pixels)
        cap = int(out["id"].shape[0])
        need = C.c_size_t()
        _check(lib.opx_propagate_host_detected_workspace_bytes(self._h, chunk, cap, C.byref(need)))
        ws = self._workspace("host", need.value, torch.device(device), None)
        ptr = (lambda t: t.data_ptr()) if isinstance(wavelengths, torch.Tensor) else (lambda a: a.ctypes.data)
        d = Detected(*(out[k].data_ptr() for k in ("id", "pixel", "pos", "dir")))
        nd = C.c_uint64(0)
        st = stream if stream is not None else torch.cuda.current_stream(device)
        _check(lib.opx_propagate_host_detected(self._h, n, int(photon_id_base), ptr(origins), ptr(dirs), ptr(wavelengths), int(seed),
                                               int(flags), C.byref(d), cap, C.byref(nd), out["hitmap"].data_ptr(),
                                               out["counters"].data_ptr(), _aligned(ws), need.value, chunk,
                                               C.c_void_p(st.cuda_stream)))
        out["n_detected"] = int(nd.value)
        return out

    def tracks_host_detected(self, steps, n, factors=(), photon_id_base=0, seed=0, n_index=1.0014, lambda1=200.0, lambda2=600.0,
                             capacity=None, chunk=1 << 24, out=None, stream=None, device="cuda"):
        """opx_tracks_host_detected: `steps` = dict of HOST numpy arrays (x, w (S,3), length, beta (S,) float32, first (S+1,) uint64)
        in, list of detected photons (host) + hit-map + counters out.  factors: () = efficiencies in flight, else the paper's
        pre-propagation filter on those materials."""
        import torch
        lib = load_library()
        x, w = np.ascontiguousarray(steps["x"], np.float32), np.ascontiguousarray(steps["w"], np.float32)
        ln, be = np.ascontiguousarray(steps["length"], np.float32), np.ascontiguousarray(steps["beta"], np.float32)
        first = np.ascontiguousarray(steps["first"], np.uint64)
        S = len(ln)
        ts = TrackSteps(x.ctypes.data, w.ctypes.data, ln.ctypes.data, be.ctypes.data, first.ctypes.data, S)
        chunk = max(1, min(int(chunk), max(int(n), 1)))
        if out is None:
            out = alloc_host_detected(max(1, int(n) if capacity is None else int(capacity)), self.n_pixels)
        cap = int(out["id"].shape[0])
        need = C.c_size_t()
        _check(lib.opx_tracks_host_detected_workspace_bytes(self._h, S, chunk, cap, C.byref(need)))
        ws = self._workspace("host", need.value, torch.device(device), None)
        fac = (C.c_uint32 * max(1, len(factors)))(*factors)
        d = Detected(*(out[k].data_ptr() for k in ("id", "pixel", "pos", "dir")))
        nd = C.c_uint64(0)
        st = stream if stream is not None else torch.cuda.current_stream(device)
        _check(lib.opx_tracks_host_detected(self._h, C.byref(ts), int(first[-1]), n_index, lambda1, lambda2, int(n), int(photon_id_base),
                                            int(seed), fac, len(factors), C.byref(d), cap, C.byref(nd), out["hitmap"].data_ptr(),
                                            out["counters"].data_ptr(), _aligned(ws), need.value, chunk,
                                            C.c_void_p(st.cuda_stream)))
        out["n_detected"] = int(nd.value)
        return out

    def prefilter(self, origins, dirs, wavelengths, factors, seed=0, photon_id_base=0, out=None, stream=None, capacity=None):
        """opx_prefilter on device tensors -> dict(origins, dirs, wavelengths, index (int32 view of uint32),
        n_kept (int64 CUDA tensor of one element)); the first n_kept entries of the arrays are the survivors in
        input order.  No host synchronisation: pass out["n_kept"] as `n_dev` to propagate().  capacity (default n)
        sizes the output arrays; n_kept > capacity means the list was truncated."""
        import torch
        n = int(wavelengths.shape[0])
        dev = wavelengths.device
        if out is None:
            cap = int(n if capacity is None else capacity)
            out = dict(origins=torch.empty((cap, 3), dtype=torch.float32, device=dev),
                       dirs=torch.empty((cap, 3), dtype=torch.float32, device=dev),
                       wavelengths=torch.empty(cap, dtype=torch.float32, device=dev),
                       index=torch.empty(cap, dtype=torch.int32, device=dev),
                       n_kept=torch.zeros(1, dtype=torch.int64, device=dev))
        need = C.c_size_t()
        _check(load_library().opx_prefilter_workspace_bytes(n, C.byref(need)))
        ws = out.get("workspace")
        if ws is None or ws.numel() < need.value + 256:
            ws = out["workspace"] = torch.empty(need.value + 256, dtype=torch.uint8, device=dev)
        fac = (C.c_uint32 * max(1, len(factors)))(*[int(f) for f in factors])
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        idx = out.get("index")
        _check(load_library().opx_prefilter(
            self._h, n, int(photon_id_base), origins.data_ptr(), dirs.data_ptr(), wavelengths.data_ptr(), int(seed),
            fac, len(factors), out["origins"].data_ptr(), out["dirs"].data_ptr(), out["wavelengths"].data_ptr(),
            None if idx is None else idx.data_ptr(), int(out["wavelengths"].shape[0]), out["n_kept"].data_ptr(), _aligned(ws),
            need.value, C.c_void_p(st.cuda_stream)))
        return out

    def prefilter_noalloc(self, origins, dirs, wavelengths, factors, out, seed=0, photon_id_base=0, stream=None):
        """opx_prefilter_noalloc: prefilter() for a caller that may not allocate device memory (a plug-in living on buffers
        a framework's pool handed it, a worker thread that must not stall the other streams of its GPU with cudaMalloc).
        Nothing is allocated here either: `out` is required and must already hold the caller's tensors origins (cap, 3),
        dirs (cap, 3), wavelengths (cap,) float32, n_kept (1,) int64 and optionally index (cap,) int32; the scratch is
        the library's built-in array, so n <= PREFILTER_NOALLOC_MAX_PHOTONS (OpxError otherwise) and calls that could
        overlap on one GPU must be ordered by the caller.  Same survivors, same order, same bytes as prefilter()."""
        import torch
        n = int(wavelengths.shape[0])
        fac = (C.c_uint32 * max(1, len(factors)))(*[int(f) for f in factors])
        st = stream if stream is not None else torch.cuda.current_stream(wavelengths.device)
        idx = out.get("index")
        _check(load_library().opx_prefilter_noalloc(
            self._h, n, int(photon_id_base), origins.data_ptr(), dirs.data_ptr(), wavelengths.data_ptr(), int(seed),
            fac, len(factors), out["origins"].data_ptr(), out["dirs"].data_ptr(), out["wavelengths"].data_ptr(),
            None if idx is None else idx.data_ptr(), int(out["wavelengths"].shape[0]), out["n_kept"].data_ptr(),
            C.c_void_p(st.cuda_stream)))
        return out

    def emit_cherenkov_filtered(self, dev_steps, n, factors, photon_id_base=0, seed=0, n_index=1.0014, lambda1=200.0,
                                lambda2=600.0, out=None, stream=None, capacity=None):
        """opx_emit_cherenkov_filtered on an uploaded step table -> the dict prefilter() returns (origins, dirs,
        wavelengths, index, n_kept, workspace).  capacity (default n) sizes the output arrays."""
        import torch
        dev = dev_steps["first"].device
        cap = int(n if capacity is None else capacity)
        if out is None:
            out = dict(origins=torch.empty((cap, 3), dtype=torch.float32, device=dev),
                       dirs=torch.empty((cap, 3), dtype=torch.float32, device=dev),
                       wavelengths=torch.empty(cap, dtype=torch.float32, device=dev),
                       index=torch.empty(cap, dtype=torch.int32, device=dev),
                       n_kept=torch.zeros(1, dtype=torch.int64, device=dev))
        need = C.c_size_t()
        _check(load_library().opx_prefilter_workspace_bytes(int(n), C.byref(need)))
        ws = out.get("workspace")
        if ws is None or ws.numel() < need.value + 256:
            ws = out["workspace"] = torch.empty(need.value + 256, dtype=torch.uint8, device=dev)
        st = TrackSteps(dev_steps["x"].data_ptr(), dev_steps["w"].data_ptr(), dev_steps["length"].data_ptr(),
                        dev_steps["beta"].data_ptr(), dev_steps["first"].data_ptr(), int(dev_steps["length"].shape[0]))
        fac = (C.c_uint32 * max(1, len(factors)))(*[int(f) for f in factors])
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        idx = out.get("index")
        _check(load_library().opx_emit_cherenkov_filtered(
            self._h, C.byref(st), int(dev_steps["n_total"]), n_index, lambda1, lambda2, int(n), int(photon_id_base), int(seed),
            fac, len(factors), out["origins"].data_ptr(), out["dirs"].data_ptr(), out["wavelengths"].data_ptr(),
            None if idx is None else idx.data_ptr(), int(out["wavelengths"].shape[0]), out["n_kept"].data_ptr(), _aligned(ws),
            need.value, C.c_void_p(s.cuda_stream)))
        return out

    def profile_begin(self, max_calls):
        """opx_profile_begin: record per-kernel CUDA events for the next max_calls propagate calls."""
        self._prof_max = int(max_calls)
        _check(load_library().opx_profile_begin(self._h, self._prof_max))

    def profile_end(self):
        """opx_profile_end -> (ms_propagate[], ms_bin[]) per recorded call."""
        a = (C.c_float * self._prof_max)()
        b = (C.c_float * self._prof_max)()
        n = C.c_uint32()
        _check(load_library().opx_profile_end(self._h, a, b, C.byref(n)))
        return list(a[:n.value]), list(b[:n.value])

    def propagate_stats(self, origins, dirs, wavelengths, seed=0, photon_id_base=0, stream=None):
        """opx_propagate_stats -> dict(segments, nodes, triangle_tests, interactions)."""
        import torch
        n = int(wavelengths.shape[0])
        stats = torch.zeros(4, dtype=torch.int64, device=wavelengths.device)
        st = stream if stream is not None else torch.cuda.current_stream(wavelengths.device)
        _check(load_library().opx_propagate_stats(self._h, n, int(photon_id_base), origins.data_ptr(), dirs.data_ptr(),
                                                  wavelengths.data_ptr(), int(seed), stats.data_ptr(),
                                                  C.c_void_p(st.cuda_stream)))
        v = stats.cpu().tolist()
        return dict(segments=v[0], nodes=v[1], triangle_tests=v[2], interactions=v[3])

    def propagate_packet_stats(self, origins, dirs, wavelengths, seed=0, photon_id_base=0, records=None, stream=None):
        """opx_propagate_packet_stats -> (records, dict(beam_segments, fallback_segments, wide_visits,
        beam_triangles, stack_overflows)) of the instrumented product kernel."""
        import torch
        n = int(wavelengths.shape[0])
        dev = wavelengths.device
        if records is None:
            records = self.alloc_records(n, dev)
        stats = torch.zeros(64, dtype=torch.int64, device=dev)
        h = Hits(*(records[k].data_ptr() for k in ("pos", "dir", "pixel", "surface", "state", "bounces")))
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        _check(load_library().opx_propagate_packet_stats(self._h, n, int(photon_id_base), origins.data_ptr(), dirs.data_ptr(),
                                                         wavelengths.data_ptr(), int(seed), C.byref(h), stats.data_ptr(),
                                                         C.c_void_p(st.cuda_stream)))
        v = stats.cpu().tolist()
        return records, dict(beam_segments=v[0], fallback_segments=v[1], wide_visits=v[2], beam_triangles=v[3],
                             stack_overflows=v[4], lane_culls=v[5], raw=v)

    def wide_info(self):
        """opx_scene_wide_info -> (wide nodes built, capacity)."""
        a, b = C.c_uint64(), C.c_uint64()
        _check(load_library().opx_scene_wide_info(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def propagate_host(self, origins, dirs, wavelengths, seed=0, photon_id_base=0, chunk=1 << 20, out=None,
                       stream=None, device="cuda"):
        """opx_propagate_host: host (pinned torch or numpy) buffers in, host buffers out."""
        import torch
        lib = load_library()
        n = int(wavelengths.shape[0])
        chunk = max(1, min(int(chunk), max(n, 1)))
        need = C.c_size_t()
        _check(lib.opx_propagate_host_workspace_bytes(self._h, chunk, C.byref(need)))
        ws = self._workspace("host", need.value, torch.device(device), None)
        if out is None:
            out = alloc_host_records(n, self.n_pixels)
        ptr = (lambda t: t.data_ptr()) if isinstance(wavelengths, torch.Tensor) else (lambda a: a.ctypes.data)
        h = Hits(*(out[k].data_ptr() for k in ("pos", "dir", "pixel", "surface", "state", "bounces")))
        st = stream if stream is not None else torch.cuda.current_stream(device)
        _check(lib.opx_propagate_host(self._h, n, int(photon_id_base), ptr(origins), ptr(dirs), ptr(wavelengths),
                                      int(seed), C.byref(h), out["hitmap"].data_ptr(), out["counters"].data_ptr(),
                                      _aligned(ws), need.value, chunk, C.c_void_p(st.cuda_stream)))
        return out


def alloc_host_records(n, n_pixels):
    """Pinned host buffers for opx_propagate_host (hitmap and counters zeroed)."""
    import torch
    pin = torch.cuda.is_available()
    mk = lambda shape, dt: torch.empty(shape, dtype=dt, pin_memory=pin)
    out = dict(pos=mk((n, 3), torch.float32), dir=mk((n, 3), torch.float32), pixel=mk((n,), torch.int32),
               surface=mk((n,), torch.int32), state=mk((n,), torch.uint8), bounces=mk((n,), torch.uint8),
               hitmap=torch.zeros(max(1, n_pixels), dtype=torch.int32, pin_memory=pin),
               counters=torch.zeros(8, dtype=torch.int64, pin_memory=pin))
    return out


def alloc_host_detected(capacity, n_pixels):
    """Pinned host buffers for opx_propagate_host_detected (hitmap and counters zeroed)."""
    import torch
    pin = torch.cuda.is_available()
    mk = lambda shape, dt: torch.empty(shape, dtype=dt, pin_memory=pin)
    return dict(id=mk((capacity,), torch.int64), pixel=mk((capacity,), torch.int32), pos=mk((capacity, 3), torch.float32),
                dir=mk((capacity, 3), torch.float32), hitmap=torch.zeros(max(1, n_pixels), dtype=torch.int32, pin_memory=pin),
                counters=torch.zeros(8, dtype=torch.int64, pin_memory=pin))


def _aligned(t, a=256):
    """256-byte aligned pointer inside a tensor allocated with >= a spare bytes."""
    p = t.data_ptr()
    return C.c_void_p((p + a - 1) // a * a)
