"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT.

ctypes/numpy front end of oracle/opx_oracle.cpp (a plain scalar CPU tracer with brute-force
all-triangle closest hit, written from PAPER.md and DESIGN.md section 3).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs import this
package.  It imports nothing from paper_2309_12496_b200 and shares no code with it.
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

STATE_NAMES = ("DETECTED", "QE_REJECTED", "ABSORBED_SURFACE", "ABSORBED_MIRROR", "DETECTOR_DEAD",
               "BOUNCE_LIMIT", "ESCAPED")
DETECTED, QE_REJECTED, ABSORBED_SURFACE, ABSORBED_MIRROR, DETECTOR_DEAD, BOUNCE_LIMIT, ESCAPED = range(7)


class Frame(C.Structure):
    _fields_ = [("A", C.c_float * 3), ("u", C.c_float * 3), ("v", C.c_float * 3),
                ("pitch_u", C.c_float), ("pitch_v", C.c_float),
                ("nu", C.c_uint32), ("nv", C.c_uint32), ("pixel_base", C.c_uint32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_uniform.restype = C.c_float
        _lib.oracle_uniform.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32]
        _lib.oracle_table_lerp.restype = C.c_double
        _lib.oracle_table_lerp.argtypes = [C.c_int, C.c_void_p, C.c_uint32, C.c_float, C.c_float, C.c_float]
        _lib.oracle_hit_triangle.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        _lib.oracle_pixel_map.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.oracle_table_value.restype = C.c_double
        _lib.oracle_table_value.argtypes = [C.c_int, C.c_void_p, C.c_uint32, C.c_uint32, C.c_float, C.c_float, C.c_float]
        _lib.oracle_uniform_stream.restype = C.c_float
        _lib.oracle_uniform_stream.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32]
        _lib.oracle_prefilter.restype = C.c_uint64
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# ------------------------------------------------------------------------------ unit functions
def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c), _p(k), _p(out))
    return out


def uniform(seed, g, b):
    return float(lib().oracle_uniform(int(seed), int(g), int(b)))


def table_lerp(table, lam, lmin=200.0, lmax=600.0, fp64=False):
    t = _f32(table)
    return float(lib().oracle_table_lerp(int(fp64), _p(t), len(t), lmin, lmax, float(lam)))


NO_EFFICIENCY = 1          # trace flag: efficiencies were applied by prefilter(), surfaces act with probability 1
LINEAR, HISTOGRAM = 0, 1   # table forms


def uniform_stream(seed, g, b, stream):
    return float(lib().oracle_uniform_stream(int(seed), int(g), int(b), int(stream)))


def table_value(table, lam, interp=LINEAR, lmin=200.0, lmax=600.0, fp64=False):
    t = _f32(table)
    return float(lib().oracle_table_value(int(fp64), _p(t), len(t), int(interp), lmin, lmax, float(lam)))


def _mat_interp(scene):
    return np.ascontiguousarray([m.get("interp", LINEAR) for m in scene.materials], dtype=np.uint32)


def _tri_vnormals(scene):
    """(T, 3, 3) vertex normals per triangle in global triangle order, zeros for a mesh without the optional
    "vertex_normals" (V, 3) entry; None when no mesh of the scene has one."""
    if not any(m.get("vertex_normals") is not None for m in scene.meshes):
        return None
    out = []
    for m in scene.meshes:
        idx = m["indices"].astype(np.int64)
        vn = m.get("vertex_normals")
        out.append(np.zeros((len(idx), 3, 3), np.float32) if vn is None else _f32(vn)[idx])
    return np.ascontiguousarray(np.concatenate(out, axis=0))


def shading_normal(o, d, tri, vnormals, fp64=False):
    """Shading normal where the ray meets the triangle -> (n (3,), uvw (3,)) or None on a miss."""
    o, d, v, n9 = _f32(o), _f32(d), _f32(tri).reshape(9), _f32(vnormals).reshape(9)
    out, uvw = np.zeros(3), np.zeros(3)
    if not lib().oracle_shading_normal(int(fp64), _p(o), _p(d), _p(v), _p(n9), _p(out), _p(uvw)):
        return None
    return out, uvw


def emit_cherenkov(steps, n, id_base=0, seed=0, n_index=1.0014, lambda1=200.0, lambda2=600.0):
    """Cherenkov photons id_base .. id_base+n-1 from track steps.  `steps`: dict with x (S,3),
    w (S,3), length (S,), beta (S,) float32 and first (S+1,) uint64.  Returns origins, dirs (n,3), wavelengths (n,)."""
    x, w, ln, be = _f32(steps["x"]).reshape(-1, 3), _f32(steps["w"]).reshape(-1, 3), _f32(steps["length"]), _f32(steps["beta"])
    first = np.ascontiguousarray(steps["first"], dtype=np.uint64)
    assert len(first) == len(ln) + 1 == len(be) + 1 == len(x) + 1 == len(w) + 1
    o, d, lam = np.zeros((n, 3), np.float32), np.zeros((n, 3), np.float32), np.zeros(n, np.float32)
    rc = lib().oracle_emit_cherenkov(C.c_uint64(len(ln)), _p(x), _p(w), _p(ln), _p(be), _p(first), C.c_float(n_index),
                                     C.c_float(lambda1), C.c_float(lambda2), C.c_uint64(n), C.c_uint64(id_base),
                                     C.c_uint64(seed), _p(o), _p(d), _p(lam))
    if rc != 0:
        raise ValueError("oracle_emit_cherenkov: a photon id lies beyond the last step")
    return o, d, lam


def prefilter(scene, wavelengths, factors, seed=0, id_base=0):
    """Pre-propagation efficiency filter: one accept-reject per photon on the product of the
    efficiencies of the materials listed in `factors`.  Returns keep (n,) uint8, index (n_kept,) uint32, prob (n,)."""
    wl = _f32(wavelengths).reshape(-1)
    n = len(wl)
    mat_table = np.ascontiguousarray(np.stack([m["table"] for m in scene.materials]), dtype=np.float32)
    interp = _mat_interp(scene)
    fac = np.ascontiguousarray(factors, dtype=np.uint32)
    keep, index, prob = np.zeros(n, np.uint8), np.zeros(n, np.uint32), np.zeros(n, np.float32)
    kept = lib().oracle_prefilter(_p(mat_table), _p(interp), C.c_uint32(len(interp)), C.c_uint32(mat_table.shape[1]),
                                  C.c_float(scene.lambda_min), C.c_float(scene.lambda_max), _p(fac), C.c_uint32(len(fac)),
                                  C.c_uint64(n), C.c_uint64(id_base), _p(wl), C.c_uint64(seed), _p(keep), _p(index), _p(prob))
    if kept == 2 ** 64 - 1:
        raise ValueError("oracle_prefilter: factor is not a material index")
    return Result(keep=keep, index=index[:kept], prob=prob)


def reflect(d, n, fp64=False):
    d, n, out = _f64(d), _f64(n), np.zeros(3)
    lib().oracle_reflect(int(fp64), _p(d), _p(n), _p(out))
    return out


def face_normal(tri):
    v, out = _f32(tri).reshape(9), np.zeros(3)
    lib().oracle_face_normal(_p(v), _p(out))
    return out


def make_frame(f):
    fr = Frame()
    fr.A[:], fr.u[:], fr.v[:] = list(map(float, f["A"])), list(map(float, f["u"])), list(map(float, f["v"]))
    fr.pitch_u, fr.pitch_v = f["pitch_u"], f["pitch_v"]
    fr.nu, fr.nv, fr.pixel_base = f["nu"], f["nv"], f["pixel_base"]
    return fr


def pixel_map(frame, p, fp64=False):
    fr = make_frame(frame)
    p = _f64(p)
    iu, iv = C.c_int32(), C.c_int32()
    ok = lib().oracle_pixel_map(int(fp64), C.byref(fr), _p(p), C.byref(iu), C.byref(iv))
    return bool(ok), iu.value, iv.value


def hit_triangle(o, d, tri, tmin=0.0, fp64=False):
    o, d, v = _f32(o), _f32(d), _f32(tri).reshape(9)
    t = C.c_double()
    h = lib().oracle_hit_triangle(int(fp64), _p(o), _p(d), _p(v), float(tmin), C.byref(t))
    return (True, t.value) if h else (False, None)


# ------------------------------------------------------------------------------------ tracers
class Result(dict):
    """pos, dir (n,3) float64; pixel, surface, tri (n,) int32; state, bounces (n,) uint8;
    segments (n,) uint32; hitmap (n_pixels,) uint32; counters (8,) uint64."""
    __getattr__ = dict.__getitem__


def trace_mesh(scene, origins, dirs, wavelengths, seed=0, id_base=0, ids=None, fp64=False,
               n_threads=None, flags=0):
    """Brute-force trace of `scene` (a workloads.Scene-like object: meshes, materials, frames,
    lambda_min/max, n_lambda, max_bounces, t_min)."""
    o, d, wl = _f32(origins).reshape(-1, 3), _f32(dirs).reshape(-1, 3), _f32(wavelengths).reshape(-1)
    n = len(wl)
    tri, tri_surface = scene.flat_triangles()
    tri = np.ascontiguousarray(tri.reshape(-1, 9))
    surf_mat = np.ascontiguousarray([m["material"] for m in scene.meshes], dtype=np.uint32)
    surf_frame = np.ascontiguousarray([m["frame"] for m in scene.meshes], dtype=np.int32)
    mat_kind = np.ascontiguousarray([m["kind"] for m in scene.materials], dtype=np.uint32)
    mat_table = np.ascontiguousarray(np.stack([m["table"] for m in scene.materials]), dtype=np.float32)
    frames = (Frame * max(1, len(scene.frames)))(*[make_frame(f) for f in scene.frames])
    return trace_mesh_arrays(tri, tri_surface, surf_mat, surf_frame, mat_kind, mat_table,
                             scene.lambda_min, scene.lambda_max, frames, len(scene.frames),
                             scene.max_bounces, scene.t_min, scene.n_pixels, o, d, wl, seed, id_base,
                             ids, fp64, n_threads, mat_interp=_mat_interp(scene), flags=flags,
                             tri_vnormal=_tri_vnormals(scene))


def trace_mesh_arrays(tri, tri_surface, surf_mat, surf_frame, mat_kind, mat_table, lmin, lmax, frames,
                      n_frames, max_bounces, t_min, n_pixels, o, d, wl, seed=0, id_base=0, ids=None,
                      fp64=False, n_threads=None, mat_interp=None, flags=0, tri_vnormal=None):
    n = len(wl)
    if n_threads is None:
        n_threads = os.cpu_count() or 1
    ids_arr = None if ids is None else np.ascontiguousarray(ids, dtype=np.uint64)
    r = Result(pos=np.zeros((n, 3)), dir=np.zeros((n, 3)), pixel=np.zeros(n, np.int32),
               surface=np.zeros(n, np.int32), tri=np.zeros(n, np.int32), state=np.zeros(n, np.uint8),
               bounces=np.zeros(n, np.uint8), segments=np.zeros(n, np.uint32),
               hitmap=np.zeros(max(1, n_pixels), np.uint32), counters=np.zeros(8, np.uint64))
    interp_arr = None if mat_interp is None else np.ascontiguousarray(mat_interp, dtype=np.uint32)
    vn_arr = None if tri_vnormal is None else np.ascontiguousarray(tri_vnormal, dtype=np.float32).reshape(-1, 9)
    assert vn_arr is None or len(vn_arr) == len(tri_surface)
    rc = lib().oracle_trace_mesh_ex2(
        C.c_int(int(fp64)), _p(interp_arr), C.c_uint32(flags), _p(vn_arr), _p(tri), _p(tri_surface), C.c_uint64(len(tri_surface)),
        _p(surf_mat), _p(surf_frame), C.c_uint32(len(surf_mat)),
        _p(mat_kind), _p(mat_table), C.c_uint32(len(mat_kind)), C.c_uint32(mat_table.shape[1]),
        C.c_float(lmin), C.c_float(lmax), frames, C.c_uint32(n_frames),
        C.c_uint32(max_bounces), C.c_float(t_min),
        C.c_uint64(n), _p(ids_arr), C.c_uint64(id_base), _p(o), _p(d), _p(wl), C.c_uint64(seed),
        _p(r["pos"]), _p(r["dir"]), _p(r["pixel"]), _p(r["surface"]), _p(r["tri"]), _p(r["state"]),
        _p(r["bounces"]), _p(r["segments"]), _p(r["hitmap"]), _p(r["counters"]), C.c_int(n_threads))
    if rc != 0:
        raise ValueError(f"oracle_trace_mesh: invalid scene (code {rc})")
    r["hitmap"] = r["hitmap"][:n_pixels]
    r["n_threads"] = n_threads
    return r


def detected_list(result, id_base=0, ids=None):
    """The list PAPER.md:195 asks for ("writes the position of the ray in a list when it interacts with the detector"): the
    records of the photons whose state is DETECTED, in photon order.  `result` is what trace_mesh returned for photons
    id_base + i (or ids[i]).  Returns Result(id (k,) uint64, pixel (k,) int32, pos, dir (k,3))."""
    idx = np.nonzero(np.asarray(result["state"]) == DETECTED)[0]
    gid = (np.uint64(id_base) + idx.astype(np.uint64)) if ids is None else np.asarray(ids, dtype=np.uint64)[idx]
    return Result(id=gid, pixel=result["pixel"][idx].copy(), pos=result["pos"][idx].copy(), dir=result["dir"][idx].copy(), index=idx)


def trace_analytic_toy(scene, origins, dirs, wavelengths, seed=0, id_base=0, with_box=True,
                       det_half=300.0):
    """Config 0 with the mirror as an exact sphere (fp64).  `scene` is workloads.toy_rich_scene():
    its .info holds the closed-form geometry; tables and frame are taken from it.  det_half = -1
    removes the detector rectangle, with_box=False the enclosure (pin P8 traces the mirror alone)."""
    o, d, wl = _f32(origins).reshape(-1, 3), _f32(dirs).reshape(-1, 3), _f32(wavelengths).reshape(-1)
    n, g = len(wl), scene.info
    refl = next(m["table"] for m in scene.materials if m["kind"] == 1)
    qe = next(m["table"] for m in scene.materials if m["kind"] == 2)
    fr = make_frame(scene.frames[0])
    box = next((m for m in scene.meshes if m["name"] == "enclosure"), None)
    lo = _f64(box["vertices"].min(axis=0)) if (box is not None and with_box) else None
    hi = _f64(box["vertices"].max(axis=0)) if (box is not None and with_box) else None
    r = Result(pos=np.zeros((n, 3)), dir=np.zeros((n, 3)), pixel=np.zeros(n, np.int32),
               surface=np.zeros(n, np.int32), state=np.zeros(n, np.uint8), bounces=np.zeros(n, np.uint8))
    v = lambda k: _f64(g[k])
    keep = [v(k) for k in ("C", "V", "ex", "ey", "a", "D", "du", "dv")]
    lib().oracle_trace_analytic_toy(
        _p(keep[0]), C.c_double(g["R"]), _p(keep[1]), _p(keep[2]), _p(keep[3]), _p(keep[4]),
        C.c_double(g["half"]), _p(keep[5]), _p(keep[6]), _p(keep[7]), C.c_double(det_half), C.c_double(det_half),
        C.byref(fr), _p(lo), _p(hi), _p(_f32(refl)), _p(_f32(qe)), C.c_uint32(scene.n_lambda),
        C.c_float(scene.lambda_min), C.c_float(scene.lambda_max), C.c_uint32(scene.max_bounces),
        C.c_double(scene.t_min), C.c_uint64(n), C.c_uint64(id_base), _p(o), _p(d), _p(wl), C.c_uint64(seed),
        _p(r["pos"]), _p(r["dir"]), _p(r["pixel"]), _p(r["surface"]), _p(r["state"]), _p(r["bounces"]))
    return r
