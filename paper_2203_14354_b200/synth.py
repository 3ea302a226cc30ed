"""Seeded synthetic inputs shared by the CUDA path and the oracle.

This module holds *no* arithmetic of the method (no intersection, no optics, no
RNG of the propagation): it only writes the triangle meshes, the optical tables
and the photon batches of BASELINE.json's configs C0..C4
as plain numpy arrays.  The identical arrays are handed to `oracle/` and to
`libdarwinopt.so`.

Stands in for the paper's CAD-imported DARWIN model (section
2.1; line 191, section 3 "average LCE" workload), which is not available
(PAPER.md line 432).  Units: mm, ns, nm.

Conventions:
  * triangle normal n_g = normalize((v1-v0) x (v2-v0)) points from the
    triangle's INNER material to its OUTER material;
  * every component owns its vertices (no welding); coincident vertices of
    neighbouring components are bit-identical fp32 values;
  * materials: 0 LXe, 1 GXe, 2 solid (never entered), 3 absorbing gas of C0;
  * surfaces : 0 PTFE, 1 photocathode, 2 steel, 3 perfect detector of C0.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

MAT_LXE, MAT_GXE, MAT_SOLID, MAT_C0GAS = 0, 1, 2, 3
SURF_PTFE, SURF_CATHODE, SURF_STEEL, SURF_PERFECT = 0, 1, 2, 3
MAT_QUARTZ, SURF_BLACK, SURF_SIPM = 4, 4, 5        # design variants (design_optics / tpc_design)
LAMBDA_NM = 175.0
INF = float("inf")


@dataclasses.dataclass
class Geometry:
    """Triangle mesh + per-triangle codes, all numpy, C-contiguous."""
    xyz: np.ndarray        # [V,3] float32
    idx: np.ndarray        # [T,3] int32
    mat_inner: np.ndarray  # [T] int32
    mat_outer: np.ndarray  # [T] int32
    surface: np.ndarray    # [T] int32, -1 = none (Fresnel)
    channel: np.ndarray    # [T] int32, -1 = not a sensor
    n_channels: int = 0
    info: dict = dataclasses.field(default_factory=dict)

    @property
    def n_tri(self) -> int:
        return int(self.idx.shape[0])

    @property
    def n_vert(self) -> int:
        return int(self.xyz.shape[0])


@dataclasses.dataclass
class Optics:
    """Wavelength-tabulated materials and surfaces on a uniform lambda grid."""
    n_lambda: int
    lambda0: float
    dlambda: float
    refr_index: np.ndarray   # [M,n_lambda] float32
    abs_len: np.ndarray      # [M,n_lambda] float32 (+inf = off)
    scat_len: np.ndarray     # [M,n_lambda] float32 (+inf = off)
    detect: np.ndarray       # [S,n_lambda] float32
    reflect_diffuse: np.ndarray
    reflect_specular: np.ndarray
    transmit: np.ndarray
    # thin-film surfaces (optional): film_on [S] int32 (1 = the surface is a film), film_n / film_k / film_d [S,n_lambda] float32
    # (index, extinction, thickness in nm); for a film surface `detect` is the probability that a photon absorbed in it is detected
    film_on: np.ndarray | None = None
    film_n: np.ndarray | None = None
    film_k: np.ndarray | None = None
    film_d: np.ndarray | None = None


@dataclasses.dataclass
class Photons:
    """SoA photon batch (52 B per photon)."""
    pos: np.ndarray   # [3,N] float32  (x,y,z rows)
    dir: np.ndarray   # [3,N] float32
    pol: np.ndarray   # [3,N] float32
    wavelength: np.ndarray  # [N] float32
    t0: np.ndarray    # [N] float32
    id_base: int = 0

    @property
    def n(self) -> int:
        return int(self.t0.shape[0])

    def slice(self, a: int, b: int) -> "Photons":
        return Photons(np.ascontiguousarray(self.pos[:, a:b]), np.ascontiguousarray(self.dir[:, a:b]),
                       np.ascontiguousarray(self.pol[:, a:b]), np.ascontiguousarray(self.wavelength[a:b]),
                       np.ascontiguousarray(self.t0[a:b]), self.id_base + a)


# --------------------------------------------------------------------------- optics
def default_optics(ptfe_reflectivity: float = 0.95, qe: float = 0.3, steel_specular: float = 0.5,
                   n_lambda: int = 1, lambda0: float = LAMBDA_NM, dlambda: float = 1.0) -> Optics:
    """Flat tables for BASELINE.json configs (Table 2 of the paper, PAPER.md 150-171,
    where BASELINE.json's config values override the paper's: reading G16)."""
    def tab(vals):
        return np.repeat(np.asarray(vals, dtype=np.float32)[:, None], n_lambda, axis=1).copy()
    #             LXe      GXe     solid  C0 gas
    n = tab([1.69, 1.0, 1.0, 1.0])
    la = tab([50000.0, 5.0e5, INF, 2000.0])
    ls = tab([400.0, 2.0e5, INF, INF])
    #             PTFE  cathode steel  perfect
    det = tab([0.0, qe, 0.0, 1.0])
    rd = tab([ptfe_reflectivity, 0.0, 0.0, 0.0])
    rs = tab([0.0, 0.0, steel_specular, 0.0])
    tr = tab([0.0, 0.0, 0.0, 0.0])
    return Optics(n_lambda, lambda0, dlambda, n, la, ls, det, rd, rs, tr)


# --------------------------------------------------------------------------- meshes
def icosphere(radius: float = 1000.0, subdiv: int = 4) -> tuple[np.ndarray, np.ndarray]:
    """Icosahedron on `radius`, `subdiv` midpoint subdivisions re-projected to the sphere.
    Returns (xyz float32 [V,3], idx int32 [T,3]) with outward normals.  subdiv=4: 2562 / 5120."""
    t = (1.0 + math.sqrt(5.0)) / 2.0
    v = [(-1, t, 0), (1, t, 0), (-1, -t, 0), (1, -t, 0), (0, -1, t), (0, 1, t),
         (0, -1, -t), (0, 1, -t), (t, 0, -1), (t, 0, 1), (-t, 0, -1), (-t, 0, 1)]
    verts = [np.asarray(p, dtype=np.float64) / math.sqrt(1 + t * t) for p in v]
    faces = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4),
             (11, 10, 2), (10, 7, 6), (7, 1, 8), (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8),
             (3, 8, 9), (4, 9, 5), (2, 4, 11), (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    for _ in range(subdiv):
        cache: dict[tuple[int, int], int] = {}

        def mid(a: int, b: int) -> int:
            key = (a, b) if a < b else (b, a)
            if key not in cache:
                m = verts[a] + verts[b]
                verts.append(m / np.linalg.norm(m))
                cache[key] = len(verts) - 1
            return cache[key]
        nf = []
        for a, b, c in faces:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            nf += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        faces = nf
    xyz = (np.asarray(verts) * radius).astype(np.float32)
    idx = np.asarray(faces, dtype=np.int32)
    # make all normals point outward
    p0, p1, p2 = (xyz[idx[:, i]].astype(np.float64) for i in range(3))
    flip = np.einsum("ij,ij->i", np.cross(p1 - p0, p2 - p0), p0 + p1 + p2) < 0
    idx[flip] = idx[flip][:, [0, 2, 1]]
    return np.ascontiguousarray(xyz), np.ascontiguousarray(idx)


class _MeshBuilder:
    def __init__(self):
        self.v, self.t, self.mi, self.mo, self.s, self.c = [], [], [], [], [], []
        self.nv = 0

    def add(self, xyz, idx, mat_inner, mat_outer, surface, channel):
        xyz = np.asarray(xyz, dtype=np.float64).reshape(-1, 3)
        idx = np.asarray(idx, dtype=np.int64).reshape(-1, 3)
        n = idx.shape[0]
        self.v.append(xyz.astype(np.float32))
        self.t.append((idx + self.nv).astype(np.int32))
        self.nv += xyz.shape[0]
        for lst, val in ((self.mi, mat_inner), (self.mo, mat_outer), (self.s, surface), (self.c, channel)):
            lst.append(np.broadcast_to(np.asarray(val, dtype=np.int32), (n,)).copy())

    def build(self, n_channels=0, info=None) -> Geometry:
        cat = np.concatenate
        return Geometry(np.ascontiguousarray(cat(self.v)), np.ascontiguousarray(cat(self.t)),
                        cat(self.mi), cat(self.mo), cat(self.s), cat(self.c), n_channels, info or {})


def _ring(radius: float, n_seg: int) -> np.ndarray:
    a = 2.0 * np.pi * np.arange(n_seg) / n_seg
    return np.stack([radius * np.cos(a), radius * np.sin(a)], axis=1)


def _fan(cx, cy, z, ring_xy, up: bool):
    """Triangle fan: centre + closed ring; normal +z if `up` else -z."""
    n = ring_xy.shape[0]
    xyz = np.concatenate([[[cx, cy, z]], np.column_stack([ring_xy[:, 0] + cx, ring_xy[:, 1] + cy, np.full(n, z)])])
    j = np.arange(n)
    a, b = 1 + j, 1 + (j + 1) % n
    idx = np.stack([np.zeros(n, dtype=np.int64), a, b] if up else [np.zeros(n, dtype=np.int64), b, a], axis=1)
    return xyz, idx


def _wall_band(ring_xy, z0, z1):
    """Extruded polygon band between z0<z1, outward normals, 2 triangles per segment."""
    n = ring_xy.shape[0]
    lo = np.column_stack([ring_xy, np.full(n, z0)])
    hi = np.column_stack([ring_xy, np.full(n, z1)])
    xyz = np.concatenate([lo, hi])
    j = np.arange(n)
    jn = (j + 1) % n
    idx = np.concatenate([np.stack([j, jn, n + jn], axis=1), np.stack([j, n + jn, n + j], axis=1)])
    return xyz, idx


def hex_centres(pitch: float, r_max: float) -> np.ndarray:
    """Hexagonal lattice points (one at the origin) with |c| <= r_max, sorted by (y, x)."""
    m = int(r_max / (pitch * math.sqrt(3) / 2)) + 2
    pts = []
    for j in range(-m, m + 1):
        for i in range(-2 * m, 2 * m + 1):
            x, y = pitch * (i + 0.5 * j), pitch * math.sqrt(3) / 2 * j
            if x * x + y * y <= r_max * r_max + 1e-9:
                pts.append((round(y, 6), round(x, 6), x, y))
    pts.sort()
    return np.asarray([(p[2], p[3]) for p in pts], dtype=np.float64)


def _wire_grid(mb: _MeshBuilder, z: float, R: float, pitch: float, radius: float, seg_len: float,
               mat_outer: int, n_side: int = 8):
    """Parallel wires along y at x = k*pitch, |x| <= R-5; each an n_side prism cut into ~seg_len pieces."""
    kmax = int(math.floor((R - pitch) / pitch + 1e-9))
    ang = (np.arange(n_side) + 0.5) * (2 * np.pi / n_side)
    ox, oz = radius * np.cos(ang), radius * np.sin(ang)
    n_tri = 0
    for k in range(-kmax, kmax + 1):
        x = k * pitch
        Y = math.sqrt(R * R - x * x) + 1.0
        nseg = max(1, int(math.ceil(2 * Y / seg_len)))
        ys = np.linspace(-Y, Y, nseg + 1)
        # vertices: (nseg+1) rings of n_side
        vx = np.tile(x + ox, nseg + 1)
        vz = np.tile(z + oz, nseg + 1)
        vy = np.repeat(ys, n_side)
        xyz = np.column_stack([vx, vy, vz])
        s = np.arange(nseg)[:, None] * n_side
        j = np.arange(n_side)[None, :]
        jn = (j + 1) % n_side
        a, b, c, d = s + j, s + jn, s + n_side + jn, s + n_side + j   # ring s: a,b ; ring s+1: d,c
        # outward normal: around the axis (+y) the angle runs x->z; (b-a) x (d-a) must point outward.
        # tangent (x->z sense) x (+y) = inward, so use (a, d, c), (a, c, b).
        idx = np.concatenate([np.stack([a, d, c], axis=-1).reshape(-1, 3), np.stack([a, c, b], axis=-1).reshape(-1, 3)])
        mb.add(xyz, idx, MAT_SOLID, mat_outer, SURF_STEEL, -1)
        n_tri += idx.shape[0]
    return n_tri, 2 * kmax + 1


def tpc(R: float, z_liq: float, height: float, n_seg: int = 256, pmt_pitch: float = 81.0,
        pmt_diam: float = 76.2, pmt_tris: int = 64, wires: bool = False, wire_pitch: float = 5.0,
        wire_radius: float = 0.108, wire_seg: float = 20.0) -> Geometry:
    """Synthetic dual-phase TPC of BASELINE.json configs 1-4."""
    mb = _MeshBuilder()
    ring = _ring(R, n_seg)
    # wall: 2 bands split at the liquid level
    mb.add(*_wall_band(ring, 0.0, z_liq), MAT_LXE, MAT_SOLID, SURF_PTFE, -1)
    mb.add(*_wall_band(ring, z_liq, height), MAT_GXE, MAT_SOLID, SURF_PTFE, -1)
    # caps (normals out of the xenon)
    mb.add(*_fan(0, 0, 0.0, ring, up=False), MAT_LXE, MAT_SOLID, SURF_PTFE, -1)
    mb.add(*_fan(0, 0, height, ring, up=True), MAT_GXE, MAT_SOLID, SURF_PTFE, -1)
    # liquid surface: inner LXe below, outer GXe above, no surface -> Fresnel
    mb.add(*_fan(0, 0, z_liq, ring, up=True), MAT_LXE, MAT_GXE, -1, -1)
    # PMT photocathode disks floating 1 mm in front of the caps, same medium on both sides
    centres = hex_centres(pmt_pitch, R - (pmt_diam / 2 + 1.0))
    disk = _ring(pmt_diam / 2, pmt_tris)
    n_pmt = centres.shape[0]
    for i, (cx, cy) in enumerate(centres):
        mb.add(*_fan(cx, cy, 1.0, disk, up=True), MAT_LXE, MAT_LXE, SURF_CATHODE, i)
    for i, (cx, cy) in enumerate(centres):
        mb.add(*_fan(cx, cy, height - 1.0, disk, up=False), MAT_GXE, MAT_GXE, SURF_CATHODE, n_pmt + i)
    info = dict(R=R, z_liq=z_liq, height=height, n_pmt_per_array=n_pmt, pmt_centres=centres, grids=[])
    if wires:
        for name, zg, mo in (("cathode", 50.0, MAT_LXE), ("gate", z_liq - 2.5, MAT_LXE), ("anode", z_liq + 2.5, MAT_GXE)):
            nt, nw = _wire_grid(mb, zg, R, wire_pitch, wire_radius, wire_seg, mo)
            info["grids"].append(dict(name=name, z=zg, n_wires=nw, n_tri=nt))
    return mb.build(n_channels=2 * n_pmt, info=info)


def design_optics(ptfe_reflectivity: float = 0.95, qe: float = 0.3, sipm_pde: float = 0.24, quartz_n: float = 1.6) -> Optics:
    """default_optics plus what the design variants need: material 4 = quartz window (index 1.6, absorption
    length 1 m, no scattering), surface 4 = black (absorbs everything), surface 5 = SiPM (detects with the photon detection
    efficiency, absorbs the rest).  Values are stand-ins of the right size; the paper tabulates none of them."""
    o = default_optics(ptfe_reflectivity, qe)
    col = lambda v: np.full((1, o.n_lambda), v, np.float32)   # noqa: E731
    cat = np.concatenate
    return dataclasses.replace(
        o, refr_index=cat([o.refr_index, col(quartz_n)]), abs_len=cat([o.abs_len, col(1000.0)]), scat_len=cat([o.scat_len, col(INF)]),
        detect=cat([o.detect, col(0.0), col(sipm_pde)]), reflect_diffuse=cat([o.reflect_diffuse, col(0.0), col(0.0)]),
        reflect_specular=cat([o.reflect_specular, col(0.0), col(0.0)]), transmit=cat([o.transmit, col(0.0), col(0.0)]))


def _frustum(cx, cy, r0, z0, r1, z1, n: int):
    """Open cone frustum between the circle (r0, z0) and the circle (r1, z1), 2 triangles per segment."""
    a, b = _ring(r0, n), _ring(r1, n)
    xyz = np.concatenate([np.column_stack([a[:, 0] + cx, a[:, 1] + cy, np.full(n, z0)]),
                          np.column_stack([b[:, 0] + cx, b[:, 1] + cy, np.full(n, z1)])])
    j = np.arange(n)
    jn = (j + 1) % n
    idx = np.concatenate([np.stack([j, jn, n + jn], axis=1), np.stack([j, n + jn, n + j], axis=1)])
    return xyz, idx


def tpc_design(R: float, z_liq: float, height: float, n_seg: int = 256, pmt_pitch: float = 81.0, pmt_diam: float = 76.2,
               pmt_tris: int = 32, detailed_pmt: bool = False, side_sensors: bool = False, window: float = 5.0, cone: float = 10.0,
               tile_fill: float = 0.9) -> Geometry:
    """Design variants of the synthetic TPC (the paper's section 5 studies).
    detailed_pmt: every PMT is a quartz window (a closed cylinder `window` thick: front face quartz|xenon without a surface, i.e.
      Fresnel; back face the photocathode, quartz|solid; rim black) standing on the cap on a closed black skirt, with a conical PTFE reflector opening from the
      window's edge towards the xenon over `cone` mm.  Needs height - z_liq > window + cone + 2.
    side_sensors: the liquid part of the wall carries one rectangular sensor per wall segment and row (rows as high as a segment is
      wide), `tile_fill` of the cell in each direction, floating 1 mm in front of the PTFE: n_seg x rows channels after the PMTs'.
    Materials and surfaces of design_optics()."""
    mb = _MeshBuilder()
    ring = _ring(R, n_seg)
    mb.add(*_wall_band(ring, 0.0, z_liq), MAT_LXE, MAT_SOLID, SURF_PTFE, -1)
    mb.add(*_wall_band(ring, z_liq, height), MAT_GXE, MAT_SOLID, SURF_PTFE, -1)
    mb.add(*_fan(0, 0, 0.0, ring, up=False), MAT_LXE, MAT_SOLID, SURF_PTFE, -1)
    mb.add(*_fan(0, 0, height, ring, up=True), MAT_GXE, MAT_SOLID, SURF_PTFE, -1)
    mb.add(*_fan(0, 0, z_liq, ring, up=True), MAT_LXE, MAT_GXE, -1, -1)
    r_pmt = pmt_diam / 2
    r_cell = pmt_pitch / 2 - 0.5
    centres = hex_centres(pmt_pitch, R - (pmt_pitch / 2 + 1.0))
    disk = _ring(r_pmt, pmt_tris)
    n_pmt = centres.shape[0]
    if detailed_pmt and height - z_liq <= window + cone + 2.0:
        raise ValueError("tpc_design: the gas gap is too small for the top PMTs")
    for top in (False, True):
        med = MAT_GXE if top else MAT_LXE
        sgn = -1.0 if top else 1.0
        z_back = height - 1.0 if top else 1.0
        for i, (cx, cy) in enumerate(centres):
            ch = (n_pmt if top else 0) + i
            if not detailed_pmt:
                mb.add(*_fan(cx, cy, z_back, disk, up=not top), med, med, SURF_CATHODE, ch)
                continue
            z_front = z_back + sgn * window
            mb.add(*_fan(cx, cy, z_front, disk, up=not top), MAT_QUARTZ, med, -1, -1)                 # window face: Fresnel
            mb.add(*_fan(cx, cy, z_back, disk, up=top), MAT_QUARTZ, MAT_SOLID, SURF_CATHODE, ch)      # photocathode behind the window
            xyz, idx = _wall_band(disk + [cx, cy], min(z_back, z_front), max(z_back, z_front))
            mb.add(xyz, idx, MAT_QUARTZ, med, SURF_BLACK, -1)                                         # rim
            # skirt from the photocathode to the cap: nothing gets under the window (the space behind it is declared solid)
            z_cap = height if top else 0.0
            mb.add(*_wall_band(disk + [cx, cy], min(z_back, z_cap), max(z_back, z_cap)), MAT_SOLID, med, SURF_BLACK, -1)
            mb.add(*_frustum(cx, cy, r_pmt + 0.05, z_front, r_cell, z_front + sgn * cone, pmt_tris), med, med, SURF_PTFE, -1)
    n_chan = 2 * n_pmt
    info = dict(R=R, z_liq=z_liq, height=height, n_pmt_per_array=n_pmt, pmt_centres=centres, grids=[], detailed_pmt=detailed_pmt,
                n_side=0, z_min=(1.0 + window + cone + 1.0) if detailed_pmt else 2.0, r_margin=3.0 if side_sensors else 1.0)
    if side_sensors:
        dphi = 2 * np.pi / n_seg
        cell = 2 * R * np.sin(dphi / 2)                               # width of a wall segment = height of a row
        z_lo = info["z_min"] if detailed_pmt else 2.0
        rows = int((z_liq - 1.0 - z_lo) // cell)
        r_plane = R * np.cos(dphi / 2) - 1.0                          # 1 mm in front of the flat wall segment
        j = np.arange(n_seg)[None, :]
        k = np.arange(rows)[:, None]
        a0, a1 = (j + 0.5 - tile_fill / 2) * dphi, (j + 0.5 + tile_fill / 2) * dphi
        rr = r_plane / np.cos(tile_fill * dphi / 2)
        z0, z1 = z_lo + (k + 0.5 - tile_fill / 2) * cell, z_lo + (k + 0.5 + tile_fill / 2) * cell
        full = lambda v: np.broadcast_to(v, (rows, n_seg))   # noqa: E731
        corners = [(a0, z0), (a1, z0), (a1, z1), (a0, z1)]
        xyz = np.stack([np.stack([full(rr * np.cos(a)), full(rr * np.sin(a)), full(z)], axis=-1) for a, z in corners], axis=2)   # [rows, n_seg, 4, 3]
        base = 4 * np.arange(rows * n_seg)[:, None]
        idx = np.concatenate([base + [0, 1, 2], base + [0, 2, 3]], axis=1).reshape(-1, 3)
        chan = np.repeat(n_chan + np.arange(rows * n_seg), 2)
        mb.add(xyz.reshape(-1, 3), idx, MAT_LXE, MAT_LXE, SURF_SIPM, chan)
        info["n_side"] = rows * n_seg
        info["side_rows"] = rows
        n_chan += rows * n_seg
    return mb.build(n_channels=n_chan, info=info)


def sphere_detector(radius: float = 1000.0, subdiv: int = 4, material: int = MAT_C0GAS,
                    surface: int = SURF_PERFECT) -> Geometry:
    """C0: every triangle of the icosphere is its own detector channel."""
    xyz, idx = icosphere(radius, subdiv)
    T = idx.shape[0]
    return Geometry(xyz, idx, np.full(T, material, np.int32), np.full(T, MAT_SOLID, np.int32),
                    np.full(T, surface, np.int32), np.arange(T, dtype=np.int32), T, dict(R=radius))


def box(lo, hi, mat_inner: int, mat_outer: int, surface: int, channel: int = -1) -> Geometry:
    """Axis-aligned closed box, outward normals, 12 triangles (used by unit tests)."""
    lo, hi = np.asarray(lo, float), np.asarray(hi, float)
    c = np.array([[lo[0], lo[1], lo[2]], [hi[0], lo[1], lo[2]], [hi[0], hi[1], lo[2]], [lo[0], hi[1], lo[2]],
                  [lo[0], lo[1], hi[2]], [hi[0], lo[1], hi[2]], [hi[0], hi[1], hi[2]], [lo[0], hi[1], hi[2]]])
    q = [(0, 3, 2, 1), (4, 5, 6, 7), (0, 1, 5, 4), (2, 3, 7, 6), (1, 2, 6, 5), (3, 0, 4, 7)]
    idx = []
    for a, b, cc, d in q:
        idx += [(a, b, cc), (a, cc, d)]
    mb = _MeshBuilder()
    mb.add(c, np.asarray(idx), mat_inner, mat_outer, surface, channel)
    return mb.build(n_channels=max(0, channel + 1))


def merge(*geoms: Geometry) -> Geometry:
    mb = _MeshBuilder()
    for g in geoms:
        mb.add(g.xyz, g.idx, g.mat_inner, g.mat_outer, g.surface, g.channel)
    return mb.build(n_channels=max(g.n_channels for g in geoms))


# --------------------------------------------------------------------------- photons
def moved(g: Geometry, kind: str) -> Geometry:
    """The same triangles at new vertex positions, of the kind a design sweep makes (inputs of dw_refit_bvh).
    'affine': the whole detector stretched and shifted (every box changes, long triangles change their number of pieces);
    'component': everything above 60 % of the height lifted by 2 % of it (one part moves, the triangles across the cut stretch);
    'jitter': every vertex displaced by up to 0.2 % of the size (seeded)."""
    xyz = g.xyz.astype(np.float64)
    lo, hi = xyz.min(0), xyz.max(0)
    size = float((hi - lo).max())
    if kind == "affine":
        out = (xyz - lo) * np.array([1.07, 0.94, 1.11]) + lo + np.array([3.0, -2.0, 5.0])
    elif kind == "component":
        out = xyz.copy()
        out[xyz[:, 2] > lo[2] + 0.6 * (hi[2] - lo[2]), 2] += 0.02 * (hi[2] - lo[2])
    elif kind == "jitter":
        out = xyz + np.random.default_rng(5).uniform(-0.002 * size, 0.002 * size, xyz.shape)
    else:
        raise ValueError(f"unknown motion '{kind}'")
    return dataclasses.replace(g, xyz=np.ascontiguousarray(out, dtype=np.float32))


def isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    """[3,n] float64 unit vectors, cos(theta) uniform in [-1,1], phi uniform."""
    ct = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2 * np.pi, n)
    st = np.sqrt(np.maximum(0.0, 1 - ct * ct))
    return np.stack([st * np.cos(ph), st * np.sin(ph), ct])


def transverse_pol(rng: np.random.Generator, k: np.ndarray) -> np.ndarray:
    """normalize(k x r) for an independent isotropic r ("random transverse")."""
    r = isotropic(rng, k.shape[1])
    e = np.cross(k.T, r.T).T
    nrm = np.linalg.norm(e, axis=0)
    bad = nrm < 1e-6
    if bad.any():  # re-draw the (measure-zero) parallel cases deterministically
        r[:, bad] = np.roll(k[:, bad], 1, axis=0) * np.array([[1.0], [-1.0], [0.5]])
        e = np.cross(k.T, r.T).T
        nrm = np.linalg.norm(e, axis=0)
    return e / nrm


def _finish(rng, pos, t0=None, id_base=0) -> Photons:
    n = pos.shape[1]
    k = isotropic(rng, n)
    e = transverse_pol(rng, k)
    k32 = k.astype(np.float32)
    e32 = e.astype(np.float32)
    return Photons(np.ascontiguousarray(pos.astype(np.float32)), np.ascontiguousarray(k32), np.ascontiguousarray(e32),
                   np.full(n, LAMBDA_NM, np.float32),
                   np.zeros(n, np.float32) if t0 is None else np.ascontiguousarray(t0.astype(np.float32)), id_base)


def photons_point(seed: int, n: int, origin=(0.0, 0.0, 0.0), id_base: int = 0) -> Photons:
    rng = np.random.Generator(np.random.PCG64([seed, id_base]))
    pos = np.repeat(np.asarray(origin, float)[:, None], n, axis=1)
    return _finish(rng, pos, None, id_base)


def photons_in_liquid(seed: int, n: int, R: float, z_liq: float, exclude_z=(), id_base: int = 0, z_min: float = 2.0,
                      r_margin: float = 1.0) -> Photons:
    """Uniform in the liquid: r = (R-r_margin) sqrt(u), z in [z_min, z_liq-1]; slabs |z-zg|<0.5 excluded (C3)."""
    rng = np.random.Generator(np.random.PCG64([seed, id_base]))
    r = (R - r_margin) * np.sqrt(rng.uniform(0, 1, n))
    ph = rng.uniform(0, 2 * np.pi, n)
    z = rng.uniform(z_min, z_liq - 1.0, n)
    for _ in range(64):
        bad = np.zeros(n, bool)
        for zg in exclude_z:
            bad |= np.abs(z - zg) < 0.5
        if not bad.any():
            break
        z[bad] = rng.uniform(z_min, z_liq - 1.0, int(bad.sum()))
    pos = np.stack([r * np.cos(ph), r * np.sin(ph), z])
    return _finish(rng, pos, None, id_base)


def photons_s2_spot(seed: int, n: int, centre, radius: float = 1.0, tau_ns: float = 27.0, id_base: int = 0) -> Photons:
    """C4: uniform in a ball of `radius` around `centre`, start times t0 = -tau ln u."""
    rng = np.random.Generator(np.random.PCG64([seed, id_base]))
    d = isotropic(rng, n)
    rr = radius * np.cbrt(rng.uniform(0, 1, n))
    pos = np.asarray(centre, float)[:, None] + d * rr
    t0 = -tau_ns * np.log(1.0 - rng.uniform(0, 1, n))
    return _finish(rng, pos, t0, id_base)


# --------------------------------------------------------------------------- configs
@dataclasses.dataclass
class Config:
    name: str
    geometry: Geometry
    optics: Optics
    n_photons: int
    seed: int
    max_steps: int
    make_photons: callable   # (n, id_base) -> Photons
    notes: str = ""


_GEOM_CACHE: dict = {}


def _tpc_cached(key, **kw) -> Geometry:
    if key not in _GEOM_CACHE:
        _GEOM_CACHE[key] = tpc(**kw)
    return _GEOM_CACHE[key]


def config(i: int, ptfe_reflectivity: float = 0.95) -> Config:
    """BASELINE.json configs[i] (0-indexed), SURVEY.md section 8d table."""
    if i == 0:
        g = sphere_detector(1000.0, 4)
        return Config("C0 absorbing sphere", g, default_optics(), 100_000, 1, 10,
                      lambda n, base=0: photons_point(1, n, (0, 0, 0), base),
                      "expected detected fraction exp(-0.5)")
    if i == 1:
        g = _tpc_cached("c1", R=250.0, z_liq=495.0, height=500.0)
        return Config("C1 small LXe TPC", g, default_optics(ptfe_reflectivity), 1_000_000, 2, 2000,
                      lambda n, base=0: photons_in_liquid(2, n, 250.0, 495.0, (), base))
    if i == 2:
        g = _tpc_cached("c2", R=1300.0, z_liq=2600.0, height=2605.0)
        return Config("C2 DARWIN-scale TPC", g, default_optics(ptfe_reflectivity), 10_000_000, 3, 2000,
                      lambda n, base=0: photons_in_liquid(3, n, 1300.0, 2600.0, (), base))
    if i in (3, 4):
        g = _tpc_cached("c3", R=1300.0, z_liq=2600.0, height=2605.0, wires=True)
        zs = tuple(gr["z"] for gr in g.info["grids"])
        if i == 3:
            return Config("C3 DARWIN-scale TPC + electrodes", g, default_optics(ptfe_reflectivity), 10_000_000, 4, 2000,
                          lambda n, base=0: photons_in_liquid(4, n, 1300.0, 2600.0, zs, base))
        return Config("C4 S2 spot sweep", g, default_optics(ptfe_reflectivity), 100_000_000, 5, 2000,
                      lambda n, base=0: photons_s2_spot(5, n, (400.0, 200.0, 2600.0 + 1.25), 1.0, 27.0, base),
                      "batches of 1e7, photon_id_base = b*1e7; PTFE reflectivity in {0.90,0.95,0.99}")
    raise ValueError(f"no config {i}")


DESIGN_VARIANTS = ("baseline", "detailed_pmt", "side_sensors", "both")


def config_design(variant: str = "both", scale: int = 1) -> Config:
    """Design variants at the size of C1 (scale 1: R = 250 mm) or C2 (scale 2: R = 1300 mm).  The gas gap is
    60 mm so that the detailed top PMTs fit.  'baseline' is the same detector with plain photocathode disks and a bare wall."""
    if variant not in DESIGN_VARIANTS:
        raise ValueError(f"unknown design variant '{variant}'")
    R, z_liq = (250.0, 495.0) if scale == 1 else (1300.0, 2600.0)
    kw = dict(detailed_pmt=variant in ("detailed_pmt", "both"), side_sensors=variant in ("side_sensors", "both"))
    key = ("design", variant, scale)
    if key not in _GEOM_CACHE:
        _GEOM_CACHE[key] = tpc_design(R, z_liq, z_liq + 60.0, **kw)
    g = _GEOM_CACHE[key]
    seed = 40 + DESIGN_VARIANTS.index(variant)
    return Config(f"design variant '{variant}' at C{scale} size", g, design_optics(), 1_000_000 if scale == 1 else 10_000_000, seed, 2000,
                  lambda n, base=0: photons_in_liquid(seed, n, R, z_liq, (), base, z_min=g.info["z_min"], r_margin=g.info["r_margin"]))


# ---------------------------------------------------------------------------------------------------------------------
# Emission sources.  Plain parameter sets: no arithmetic of the method lives here.
FWHM_TO_SIGMA = 1.0 / 2.3548200450309493        # 1 / (2 sqrt(2 ln 2))
SHAPE_POINT, SHAPE_CYLINDER, SHAPE_BALL = 0, 1, 2


def source(shape=SHAPE_CYLINDER, centre=(0.0, 0.0, 0.0), radius=0.0, z0=0.0, z1=0.0, lambda_mean=174.8, lambda_fwhm=10.2,
           t_start=0.0, tau1=3.5, tau3=24.0, f_singlet=0.66) -> dict:
    """PAPER.md line 144 and Table 2 (lines 155-160): Gaussian spectrum 174.8 nm / FWHM 10.2 nm, two-exponential time profile with
    tau_1 = 3.5 ns, tau_3 = 24 ns, singlet fraction 0.66 (nuclear recoils) or 0.22 (electronic recoils)."""
    return dict(shape=int(shape), centre=tuple(float(v) for v in centre), radius=float(radius), z0=float(z0), z1=float(z1),
                lambda_mean=float(lambda_mean), lambda_sigma=float(lambda_fwhm) * FWHM_TO_SIGMA, t_start=float(t_start),
                tau1=float(tau1), tau3=float(tau3), f_singlet=float(f_singlet))


def source_for(i: int, recoil: str = "NR") -> dict:
    """The liquid volume of config i (1..3) as a cylinder source, or the S2 spot of config 4 as a ball source."""
    fs = 0.66 if recoil == "NR" else 0.22
    if i == 1:
        return source(SHAPE_CYLINDER, (0, 0, 0), 249.0, 2.0, 494.0, f_singlet=fs)
    if i in (2, 3):
        return source(SHAPE_CYLINDER, (0, 0, 0), 1299.0, 2.0, 2599.0, f_singlet=fs)
    if i == 4:
        return source(SHAPE_BALL, (400.0, 200.0, 2601.25), 1.0, tau1=27.0, tau3=27.0, f_singlet=1.0)
    raise ValueError(i)


# ---------------------------------------------------------------------------------------------------------------------
# Dispersive tables: five wavelength nodes, so that the linear interpolation of S3 is a live path once photons carry the
# emission spectrum.  SYNTHETIC dispersion (the paper tabulates values at 175 nm only, Table 2): chosen to pass through the
# config values at 175 nm and to vary by amounts of the order of the paper's quoted spreads.
DISPERSIVE_GRID = (165.0, 5.0, 5)        # lambda0, dlambda, nodes: 165, 170, 175, 180, 185 nm


def dispersive_optics(ptfe_reflectivity: float = 0.95, qe: float = 0.3) -> Optics:
    l0, dl, nl = DISPERSIVE_GRID
    lam = l0 + dl * np.arange(nl)
    rows = lambda *r: np.asarray(r, np.float32)
    flat = lambda v: np.full(nl, v, np.float32)
    n = rows(1.69 - 0.008 * (lam - 175.0), flat(1.0), flat(1.0), flat(1.0))                       # LXe 1.77 .. 1.61
    la = rows(50000.0 * (1.0 + 0.02 * (lam - 175.0)), flat(5.0e5), flat(INF), 2000.0 + 40.0 * (lam - 175.0))
    ls = rows(400.0 * (lam / 175.0) ** 4, flat(2.0e5), flat(INF), flat(INF))                      # Rayleigh ~ lambda^4
    det = rows(flat(0.0), qe + 0.005 * (lam - 175.0), flat(0.0), flat(1.0))
    rd = rows(ptfe_reflectivity + 0.002 * (lam - 175.0), flat(0.0), flat(0.0), flat(0.0))
    rs = rows(flat(0.0), flat(0.0), flat(0.5), flat(0.0))
    tr = rows(flat(0.0), flat(0.0), flat(0.0), flat(0.0))
    return Optics(nl, l0, dl, n, la, ls, det, rd, rs, tr)


def config_dispersive(i: int = 1) -> Config:
    """Config i (1 or 2) with the dispersive tables and photons that carry the emission spectrum (174.8 nm, FWHM 10.2 nm,
    drawn by the harness, so that some wavelengths fall outside the table and exercise the clamping)."""
    base = config(i)

    def make(n, id_base=0):
        ph = base.make_photons(n, id_base)
        rng = np.random.Generator(np.random.PCG64([base.seed, id_base, 77]))
        lam = rng.normal(174.8, 10.2 * FWHM_TO_SIGMA, ph.n).astype(np.float32)
        return Photons(ph.pos, ph.dir, ph.pol, lam, ph.t0, ph.id_base)
    return Config(base.name + " (dispersive tables)", base.geometry, dispersive_optics(), base.n_photons, base.seed, base.max_steps, make,
                  "synthetic dispersion on five wavelength nodes")


def with_film(op: Optics, surface: int, nf: float, kf: float, d_nm: float, detect: float | None = None) -> Optics:
    """Copy of `op` in which `surface` is a thin film (index nf + i kf, thickness d_nm, flat in wavelength).
    Table 8 of the paper (PAPER.md 356-357): silicon 0.81 + 1.86 i."""
    S, nl = op.detect.shape
    on = np.zeros(S, np.int32) if op.film_on is None else op.film_on.copy()
    fn = np.ones((S, nl), np.float32) if op.film_n is None else op.film_n.copy()
    fk = np.zeros((S, nl), np.float32) if op.film_k is None else op.film_k.copy()
    fd = np.zeros((S, nl), np.float32) if op.film_d is None else op.film_d.copy()
    on[surface] = 1; fn[surface] = nf; fk[surface] = kf; fd[surface] = d_nm
    det = op.detect.copy()
    if detect is not None:
        det[surface] = detect
    return dataclasses.replace(op, detect=det, film_on=on, film_n=fn, film_k=fk, film_d=fd)
