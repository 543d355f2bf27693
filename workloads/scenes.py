"""Procedural scenes standing in for the paper's GDML -> FreeCAD -> Mefisto -> OBJ
meshes (section 4.1), which are not in the container.

Every scene is a list of triangle meshes grouped per material (PAPER.md:91, 97:
mirrors share one BSDF/material, the detector has its own), per-material
wavelength tables and detector pixel frames given, as in the
paper, by a corner point A and two in-plane unit vectors.
All geometry is computed in float64 and rounded to float32 exactly once.

No ray tracing, table lookup or RNG of the method lives here.
"""
from dataclasses import dataclass, field

import numpy as np

MAT_ABSORBER, MAT_MIRROR, MAT_DETECTOR = 0, 1, 2
PIXEL_PITCH_MM = 2.88           # BASELINE.json configs 0 and 3
N_LAMBDA = 64                   # BASELINE.json config 1: 64-point tables
LAMBDA_MIN_NM, LAMBDA_MAX_NM = 200.0, 600.0


TABLE_LINEAR, TABLE_HISTOGRAM = 0, 1     # opx_table_interp (include/opx.h)


@dataclass
class Scene:
    """Plain container; field names follow include/opx.h."""
    meshes: list = field(default_factory=list)      # dicts: vertices, indices, material, frame, name
    materials: list = field(default_factory=list)   # dicts: kind, table (n_lambda,) float32
    frames: list = field(default_factory=list)      # dicts: A,u,v (3,) f32, pitch_u, pitch_v, nu, nv, pixel_base
    lambda_min: float = LAMBDA_MIN_NM
    lambda_max: float = LAMBDA_MAX_NM
    n_lambda: int = N_LAMBDA
    max_bounces: int = 16
    t_min: float = 1e-3
    info: dict = field(default_factory=dict)        # closed-form constants for the tests

    @property
    def n_triangles(self):
        return int(sum(len(m["indices"]) for m in self.meshes))

    @property
    def n_pixels(self):
        return int(max((f["pixel_base"] + f["nu"] * f["nv"] for f in self.frames), default=0))

    def add_mesh(self, name, vertices, indices, material, frame=-1, vertex_normals=None):
        """vertex_normals: optional (V, 3) unit normals (an OBJ file's `vn` records): a mirror mesh that carries
        them reflects about the interpolated normal."""
        v = np.ascontiguousarray(np.asarray(vertices, dtype=np.float64).astype(np.float32))
        i = np.ascontiguousarray(np.asarray(indices, dtype=np.uint32).reshape(-1, 3))
        vn = None
        if vertex_normals is not None:
            vn = np.ascontiguousarray(np.asarray(vertex_normals, dtype=np.float64).astype(np.float32))
            assert vn.shape == v.shape
        self.meshes.append(dict(name=name, vertices=v, indices=i, material=int(material),
                                frame=int(frame), vertex_normals=vn))
        return len(self.meshes) - 1

    def add_material(self, kind, table, interp=TABLE_LINEAR):
        t = np.ascontiguousarray(np.asarray(table, dtype=np.float64).astype(np.float32))
        assert t.shape == (self.n_lambda,)
        self.materials.append(dict(kind=int(kind), table=t, interp=int(interp)))
        return len(self.materials) - 1

    def add_frame(self, A, u, v, pitch_u, pitch_v, nu, nv, pixel_base):
        f32 = lambda x: np.ascontiguousarray(np.asarray(x, dtype=np.float64).astype(np.float32))
        self.frames.append(dict(A=f32(A), u=f32(u), v=f32(v), pitch_u=float(np.float32(pitch_u)),
                                pitch_v=float(np.float32(pitch_v)), nu=int(nu), nv=int(nv),
                                pixel_base=int(pixel_base)))
        return len(self.frames) - 1

    def flat_triangles(self):
        """(T,3,3) float32 vertices and (T,) int32 surface (= mesh index) in global
        triangle-id order: meshes in order, triangles in order within each mesh."""
        tris = [m["vertices"][m["indices"].astype(np.int64)] for m in self.meshes]
        surf = [np.full(len(m["indices"]), s, dtype=np.int32) for s, m in enumerate(self.meshes)]
        tris.append(np.zeros((0, 3, 3), np.float32))
        surf.append(np.zeros(0, np.int32))
        return (np.ascontiguousarray(np.concatenate(tris, axis=0)),
                np.ascontiguousarray(np.concatenate(surf)))


# ----------------------------------------------------------------------------- tables
def lambda_grid(n_lambda=N_LAMBDA, lo=LAMBDA_MIN_NM, hi=LAMBDA_MAX_NM):
    return lo + (hi - lo) * np.arange(n_lambda, dtype=np.float64) / (n_lambda - 1)


def flat_tables(reflectivity=0.9, qe=0.25):
    """Config 0: flat reflectivity 0.9 and flat QE 0.25 as constant 64-point tables."""
    return (np.full(N_LAMBDA, reflectivity), np.full(N_LAMBDA, qe))


def c2_tables():
    """Config 1: reflectivity ramping 0.85 -> 0.95 and a QE peaking at 0.30 near 400 nm.
    Shapes only: the paper's curves (Fig. 3: QE peak 35 % near 450 nm,
    R between 94 % and 89 %) come from a TDR that is not in the container."""
    lam = lambda_grid()
    refl = 0.85 + 0.10 * np.arange(N_LAMBDA) / (N_LAMBDA - 1)
    qe = 0.30 * np.exp(-0.5 * ((lam - 400.0) / 90.0) ** 2)
    return refl, qe


def paper_histogram_tables():
    """The paper's table form: QE as a histogram of 33 nm bins, reflectivity in bins of
    25 nm, both written on ONE grid of 400 bins of 1 nm over 200-600 nm (every bin edge is a whole nm, so the
    1 nm grid holds both binnings exactly).  Shapes only (QE peaking 35 % near 450 nm, R falling from 94 % to
    89 %): the measured curves of Ref. [14] are not in the container."""
    lam = LAMBDA_MIN_NM + 0.5 + np.arange(400)                       # centres of the 1 nm bins
    centre33 = LAMBDA_MIN_NM + 33.0 * (np.floor((lam - LAMBDA_MIN_NM) / 33.0) + 0.5)
    centre25 = LAMBDA_MIN_NM + 25.0 * (np.floor((lam - LAMBDA_MIN_NM) / 25.0) + 0.5)
    qe = 0.35 * np.exp(-0.5 * ((centre33 - 450.0) / 110.0) ** 2)
    refl = 0.94 - 0.05 * (centre25 - 212.5) / 375.0
    return refl, qe


# ------------------------------------------------------------------------- mesh helpers
def _quad(c, eu, ev, hu, hv):
    """Two triangles for the rectangle c +- hu*eu +- hv*ev: (v00,v10,v11),(v00,v11,v01)."""
    c, eu, ev = (np.asarray(x, dtype=np.float64) for x in (c, eu, ev))
    verts = np.array([c - hu * eu - hv * ev, c + hu * eu - hv * ev,
                      c + hu * eu + hv * ev, c - hu * eu + hv * ev])
    return verts, np.array([[0, 1, 2], [0, 2, 3]], dtype=np.uint32)


def _grid_patch(origin, eu, ev, nu, nv, du, dv, lift=None):
    """(nu+1)x(nv+1) vertices origin + i*du*eu + j*dv*ev (+ lift(x,y)), each cell split into
    (v00,v11,v10) and (v00,v01,v11); vertex index j*(nu+1)+i."""
    i = np.arange(nu + 1, dtype=np.float64) * du
    j = np.arange(nv + 1, dtype=np.float64) * dv
    X, Y = np.meshgrid(i, j, indexing="xy")        # shape (nv+1, nu+1), X varies fastest
    P = (np.asarray(origin, np.float64)[None, None, :] + X[..., None] * np.asarray(eu, np.float64)
         + Y[..., None] * np.asarray(ev, np.float64))
    if lift is not None:
        P = P + lift(X, Y)
    verts = P.reshape(-1, 3)
    ii, jj = np.meshgrid(np.arange(nu), np.arange(nv), indexing="xy")
    v00 = (jj * (nu + 1) + ii).ravel()
    v10, v01, v11 = v00 + 1, v00 + (nu + 1), v00 + (nu + 2)
    tris = np.empty((2 * nu * nv, 3), dtype=np.uint32)
    tris[0::2] = np.stack([v00, v11, v10], axis=1)
    tris[1::2] = np.stack([v00, v01, v11], axis=1)
    return verts, tris


def _box(lo, hi, nx=1, ny=1, nz=1):
    """Closed axis-aligned box, each face an (n x n) grid of cells split in two."""
    lo, hi = np.asarray(lo, np.float64), np.asarray(hi, np.float64)
    ex, ey, ez = np.eye(3)
    d = hi - lo
    faces = [  # origin, eu, ev, nu, nv, du, dv
        (lo, ex, ey, nx, ny, d[0] / nx, d[1] / ny),
        (lo + d[2] * ez, ex, ey, nx, ny, d[0] / nx, d[1] / ny),
        (lo, ex, ez, nx, nz, d[0] / nx, d[2] / nz),
        (lo + d[1] * ey, ex, ez, nx, nz, d[0] / nx, d[2] / nz),
        (lo, ey, ez, ny, nz, d[1] / ny, d[2] / nz),
        (lo + d[0] * ex, ey, ez, ny, nz, d[1] / ny, d[2] / nz),
    ]
    V, T, base = [], [], 0
    for f in faces:
        v, t = _grid_patch(*f)
        V.append(v)
        T.append(t + base)
        base += len(v)
    return np.concatenate(V), np.concatenate(T).astype(np.uint32)


# ---------------------------------------------------------------------------- toy RICH
def toy_rich_scene(tables="c2", cells=100, enclosure=True, smooth=False):
    """BASELINE.json configs 0-2: one spherical mirror cap (R = 2400 mm, square 800 mm
    aperture, vertex at z = 1200 mm, tilted 0.25 rad about +x) tessellated into
    2*cells^2 triangles, a 600x600 mm detector quad perpendicular to the reflected axis at
    R/2 from the mirror vertex with a 208x208 grid of 2.88 mm pixels, and an absorbing
    axis-aligned box around everything ("everything else is absorbing").
    smooth=True gives the mirror mesh vertex normals (the unit vectors from each vertex towards the
    centre of curvature, what an OBJ export of the sphere carries as `vn`): SURVEY.md 8(f) row f3.
    """
    R, tilt, zv, half = 2400.0, 0.25, 1200.0, 400.0
    V = np.array([0.0, 0.0, zv])
    ex = np.array([1.0, 0.0, 0.0])
    ey = np.array([0.0, np.cos(tilt), np.sin(tilt)])
    a = np.array([0.0, np.sin(tilt), -np.cos(tilt)])          # vertex -> centre of curvature
    C = V + R * a
    r = np.array([0.0, np.sin(2 * tilt), -np.cos(2 * tilt)])  # reflected chief ray
    D = V + 0.5 * R * r
    du = np.array([1.0, 0.0, 0.0])
    dv = np.cross(-r, du)

    sc = Scene()
    interp = TABLE_LINEAR
    if tables == "paper_hist":
        sc.n_lambda, interp = 400, TABLE_HISTOGRAM
        refl, qe = paper_histogram_tables()
    else:
        refl, qe = flat_tables() if tables == "flat" else c2_tables()
    m_abs = sc.add_material(MAT_ABSORBER, np.zeros(sc.n_lambda))
    m_mir = sc.add_material(MAT_MIRROR, refl, interp)
    m_det = sc.add_material(MAT_DETECTOR, qe, interp)

    step = 2 * half / cells
    sag = lambda X, Y: (R - np.sqrt(R * R - (X - half) ** 2 - (Y - half) ** 2))[..., None] * a
    mv, mt = _grid_patch(V - half * ex - half * ey, ex, ey, cells, cells, step, step, lift=sag)
    sc.add_mesh("mirror", mv, mt, m_mir, vertex_normals=(C[None, :] - mv) / R if smooth else None)

    npix = int(np.floor(600.0 / PIXEL_PITCH_MM))              # 208
    halfgrid = 0.5 * npix * PIXEL_PITCH_MM                    # 299.52
    fr = sc.add_frame(D - halfgrid * du - halfgrid * dv, du, dv, PIXEL_PITCH_MM, PIXEL_PITCH_MM,
                      npix, npix, 0)
    dvv, dtt = _quad(D, du, dv, 300.0, 300.0)
    sc.add_mesh("detector", dvv, dtt, m_det, frame=fr)

    if enclosure:
        allv = np.concatenate([mv, dvv, np.zeros((1, 3))])
        lo = np.floor(allv.min(axis=0) - 100.0)
        hi = np.ceil(allv.max(axis=0) + 100.0)
        bv, bt = _box(lo, hi)
        sc.add_mesh("enclosure", bv, bt, m_abs)

    sc.info = dict(m_abs=m_abs, m_mir=m_mir, m_det=m_det,
                   R=R, tilt=tilt, V=V, C=C, a=a, ex=ex, ey=ey, half=half, r=r, D=D, du=du, dv=dv,
                   facet_circumradius=step * np.sqrt(2) / 2, pixel_grid=npix)
    return sc


# ------------------------------------------------------------------- LHCb-RICH1-like scene
def _hex_fan(k):
    """Unit pointy-top hexagon (circumradius 1) subdivided into 6*k^2 near-equilateral
    triangles; returns 2-D vertices and triangle indices (shared vertices merged)."""
    pts, index = [], {}

    def vid(p):
        key = (round(p[0] * 1e9), round(p[1] * 1e9))
        if key not in index:
            index[key] = len(pts)
            pts.append(p)
        return index[key]

    tris = []
    corners = [np.array([np.sin(np.pi / 3 * s), np.cos(np.pi / 3 * s)]) for s in range(7)]
    for s in range(6):
        p, q = corners[s], corners[s + 1]
        bary = lambda i, j: (i * p + j * q) / k          # centre is the origin
        for i in range(k):
            for j in range(k - i):
                tris.append((vid(bary(i, j)), vid(bary(i + 1, j)), vid(bary(i, j + 1))))
                if j < k - i - 1:
                    tris.append((vid(bary(i + 1, j)), vid(bary(i + 1, j + 1)), vid(bary(i, j + 1))))
    return np.array(pts), np.array(tris, dtype=np.uint32)


def lhcb_like_scene(enclosure_pitch=11.3, edge=5.0, th1=0.40, d1=900.0, d2=455.0):
    """BASELINE.json config 3: an LHCb-RICH1-like scene of ~1e6 triangles.

    Two mirror-symmetric halves (sigma = +-1 in y).  Per half: two spherical primary-mirror
    quadrants (R = 2710 mm), each tiled by 16 hexagons with 2 mm gaps; 8 flat secondary
    mirror tiles on a 5 mm grid (maximum edge 5 mm); a detector plane of
    25x20 modules of 64x64 mm, each module one surface with its own 8x8 frame of 2.88 mm
    pixels.  Absorbing backing plates 1 mm behind every mirror tile and an absorbing box
    tessellated at `enclosure_pitch` bring the scene to ~1e6 triangles.  Positions are
    this build's choice (the config gives counts and radii only); see DESIGN.md.
    th1 = tilt of each primary half about x, d1 = primary vertex -> flat mirror centre,
    d2 = flat mirror centre -> detector plane; the defaults keep the flat mirrors outside the
    250 + 53 mrad light cone of the tracks, so that ~63 % of C3-style photons reach a detector
    plane after two reflections (checked with the oracle).
    """
    sc = Scene()
    refl, qe = c2_tables()
    m_abs = sc.add_material(MAT_ABSORBER, np.zeros(N_LAMBDA))
    m_mir = sc.add_material(MAT_MIRROR, refl)
    m_det = sc.add_material(MAT_DETECTOR, qe)

    R, V = 2710.0, np.array([0.0, 0.0, 1400.0])
    ex = np.array([1.0, 0.0, 0.0])
    r_hex = 88.0
    k = int(np.ceil(r_hex / edge))
    hp, ht = _hex_fan(k)
    info = dict(R=R, V=V, halves=[])
    allv = [np.zeros((1, 3))]
    module_id = 0
    for sigma in (+1.0, -1.0):
        a = np.array([0.0, sigma * np.sin(th1), -np.cos(th1)])
        ey = np.array([0.0, np.cos(th1), sigma * np.sin(th1)])
        C = V + R * a
        # ---- primary: 2 quadrants x 16 hexagons (pointy-top honeycomb, 4 columns x 4 rows)
        w = np.sqrt(3.0) * r_hex
        for quad in (-1.0, +1.0):
            for row in range(4):
                for col in range(4):
                    cx = (col + 0.5 + 0.5 * (row & 1)) * w + 4.0          # local |x| in (4, ~690)
                    cy = (row * 1.5 + 1.0) * r_hex + 4.0                   # local sigma*y in (4, ~580)
                    xy = hp * (r_hex - 2.0 / np.sqrt(3.0)) + np.array([cx, cy])
                    X, Y = quad * xy[:, 0], sigma * xy[:, 1]
                    s = R - np.sqrt(R * R - X * X - Y * Y)
                    P = V + X[:, None] * ex + Y[:, None] * ey + s[:, None] * a
                    sc.add_mesh("primary", P, ht, m_mir)
                    back = C + (P - C) * ((R + 1.0) / R)
                    sc.add_mesh("primary_backing", back, ht, m_abs)
                    allv.append(back)
        # ---- secondary flat mirror: 4 x 2 tiles of 380 x 350 mm on a 5 mm grid
        r1 = np.array([0.0, sigma * np.sin(2 * th1), -np.cos(2 * th1)])
        r2 = np.array([0.0, sigma * np.cos(th1), np.sin(th1)])
        M = V + d1 * r1
        n = (r1 - r2) / np.linalg.norm(r1 - r2)       # faces the incoming light (n . r1 > 0 side is the back)
        e1 = ex
        e2 = np.cross(n, e1)
        for ti in range(4):
            for tj in range(2):
                org = M + (ti - 2) * 382.0 * e1 + (tj - 1) * 352.0 * e2 + 1.0 * e1 + 1.0 * e2
                fv, ft = _grid_patch(org, e1, e2, 76, 70, 5.0, 5.0)
                sc.add_mesh("secondary", fv, ft, m_mir)
                sc.add_mesh("secondary_backing", fv + 1.0 * n, ft, m_abs)
                allv.append(fv)
        # ---- detector plane: 25 x 20 modules of 64 mm, each its own surface + pixel frame
        D = M + d2 * r2
        du = ex
        dv = np.cross(-r2, du)
        halfgrid = 4 * PIXEL_PITCH_MM
        for mj in range(20):
            for mi in range(25):
                c = D + (mi - 12) * 64.0 * du + (mj - 9.5) * 64.0 * dv
                fr = sc.add_frame(c - halfgrid * du - halfgrid * dv, du, dv, PIXEL_PITCH_MM,
                                  PIXEL_PITCH_MM, 8, 8, 64 * module_id)
                qv, qt = _quad(c, du, dv, 32.0, 32.0)
                sc.add_mesh("module", qv, qt, m_det, frame=fr)
                allv.append(qv)
                module_id += 1
        info["halves"].append(dict(sigma=sigma, a=a, C=C, r1=r1, r2=r2, M=M, n=n, D=D, du=du, dv=dv))
    # ---- absorbing enclosure ("enclosure and support structure")
    allv = np.concatenate(allv)
    lo = np.floor(allv.min(axis=0) - 100.0)
    hi = np.ceil(allv.max(axis=0) + 100.0)
    nx, ny, nz = (int(np.ceil(d / enclosure_pitch)) for d in (hi - lo))
    bv, bt = _box(lo, hi, nx, ny, nz)
    sc.add_mesh("enclosure", bv, bt, m_abs)
    info.update(lo=lo, hi=hi, n_modules=module_id)
    sc.info = info
    return sc
