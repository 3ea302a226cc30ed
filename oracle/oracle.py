"""ctypes front end of oracle/oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It imports nothing from the CUDA path; inputs are plain numpy arrays
(normally those written by paper_2203_14354_b200.synth, which holds no method arithmetic).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "oracle.cpp"
_LIB = _HERE / "liboracle.so"

FATE_NAMES = ("detected", "bulk_absorbed", "surface_absorbed", "escaped", "truncated", "nan_abort")
FATE_DETECTED, FATE_BULK_ABSORBED, FATE_SURFACE_ABSORBED, FATE_ESCAPED, FATE_TRUNCATED, FATE_NAN_ABORT = range(6)
H_RAYLEIGH, H_REFLECT_DIFFUSE, H_REFLECT_SPECULAR, H_SURFACE_TRANSMIT = 0x10, 0x20, 0x40, 0x80
H_FRESNEL_REFLECT, H_FRESNEL_REFRACT, H_TIR = 0x100, 0x200, 0x400
H_FILM = 0x1000


def build(force: bool = False) -> Path:
    """Compile oracle.cpp with g++ (no CUDA, no external libraries)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-ffp-contract=off",
                               str(_SRC), "-o", str(tmp)])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        vp, i32, i64, u32, u64, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64, C.c_double
        L.orc_create.restype = vp
        L.orc_destroy.argtypes = [vp]
        L.orc_hardware_threads.restype = C.c_int
        L.orc_set_materials.argtypes = [vp, C.c_int, C.c_int, f64, f64, vp, vp, vp]
        L.orc_set_surfaces.argtypes = [vp, C.c_int, C.c_int, f64, f64, vp, vp, vp, vp]
        L.orc_set_films.argtypes = [vp, C.c_int, C.c_int, f64, f64, vp, vp, vp, vp]
        L.orc_set_geometry.argtypes = [vp, i64, vp, i64, vp, vp, vp, vp, vp]
        L.orc_build_bvh.argtypes = [vp]
        L.orc_first_hit.argtypes = [vp, i64] + [vp] * 7 + [C.c_int, vp, vp, C.c_int]
        L.orc_propagate.argtypes = ([vp, i64] + [vp] * 11 + [u64, u64, i32, C.c_int] + [vp] * 8 +
                                    [i64, vp, i64, f64, f64, vp, vp, vp, C.c_int])
        L.orc_emit.argtypes = [C.c_int, vp, f64, f64, f64, f64, f64, f64, f64, f64, f64, u64, u64, i64, vp]
        L.orc_film_coefficients.argtypes = [f64] * 7 + [vp]
        L.orc_film.argtypes = [f64] * 6 + [vp, vp, vp, f64, vp]
        L.orc_film.restype = C.c_int
        L.orc_philox4x32_10.argtypes = [vp, vp, vp]
        L.orc_uniforms.argtypes = [u64, u64, u32, u32, vp]
        L.orc_rayleigh.argtypes = [vp, vp, u64, u64, u32]
        L.orc_rayleigh.restype = C.c_int
        L.orc_lambert.argtypes = [vp, vp, vp, u64, u64, u32]
        L.orc_specular.argtypes = [vp, vp, vp]
        L.orc_fresnel.argtypes = [f64, f64, vp, vp, vp, f64, vp]
        L.orc_fresnel.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def hardware_threads() -> int:
    return int(lib().orc_hardware_threads())


class Oracle:
    """One scene (geometry + optical tables) in the double-precision CPU tracker."""

    def __init__(self, geometry=None, optics=None, bvh: bool | None = None):
        self.L = lib()
        self.h = C.c_void_p(self.L.orc_create())
        self.use_bvh = False
        self.n_chan = 0
        if optics is not None:
            self.set_optics(optics)
        if geometry is not None:
            self.set_geometry(geometry)
            if bvh is None:
                bvh = geometry.n_tri > 5000
            if bvh:
                self.build_bvh()

    def __del__(self):
        try:
            self.L.orc_destroy(self.h)
        except Exception:
            pass

    def set_optics(self, o):
        self.L.orc_set_materials(self.h, o.refr_index.shape[0], o.n_lambda, o.lambda0, o.dlambda,
                                 _p(_f32(o.refr_index)), _p(_f32(o.abs_len)), _p(_f32(o.scat_len)))
        self.L.orc_set_surfaces(self.h, o.detect.shape[0], o.n_lambda, o.lambda0, o.dlambda, _p(_f32(o.detect)),
                                _p(_f32(o.reflect_diffuse)), _p(_f32(o.reflect_specular)), _p(_f32(o.transmit)))
        if getattr(o, "film_on", None) is not None:            # thin-film surfaces, on the surfaces' grid
            self.L.orc_set_films(self.h, o.detect.shape[0], o.n_lambda, o.lambda0, o.dlambda, _p(_i32(o.film_on)),
                                 _p(_f32(o.film_n)), _p(_f32(o.film_k)), _p(_f32(o.film_d)))

    def set_geometry(self, g):
        self.n_chan = int(g.n_channels)
        self.L.orc_set_geometry(self.h, g.n_vert, _p(_f32(g.xyz)), g.n_tri, _p(_i32(g.idx)), _p(_i32(g.mat_inner)),
                                _p(_i32(g.mat_outer)), _p(_i32(g.surface)), _p(_i32(g.channel)))
        self.use_bvh = False

    def build_bvh(self) -> int:
        n = self.L.orc_build_bvh(self.h)
        self.use_bvh = True
        return n

    def first_hit(self, origin, direction, exclude=None, use_bvh: bool | None = None, nthreads: int | None = None):
        """origin, direction: [3,n] float32.  Returns (tri int32[n], dist float64[n])."""
        o, d = _f32(origin), _f32(direction)
        n = o.shape[1]
        tri = np.empty(n, np.int32)
        dist = np.empty(n, np.float64)
        ex = None if exclude is None else _i32(exclude)
        ub = self.use_bvh if use_bvh is None else use_bvh
        self.L.orc_first_hit(self.h, n, _p(o[0]), _p(o[1]), _p(o[2]), _p(d[0]), _p(d[1]), _p(d[2]), _p(ex), int(ub),
                             _p(tri), _p(dist), nthreads or hardware_threads())
        return tri, dist

    def propagate(self, ph, seed: int, max_steps: int, n_bins: int = 0, t_min: float = 0.0, dt: float = 1.0,
                  use_bvh: bool | None = None, nthreads: int | None = None, full: bool = True) -> dict:
        """ph: synth.Photons.  Returns dict of per-photon arrays and histograms (numpy)."""
        n = ph.n
        pos, k, e = _f32(ph.pos), _f32(ph.dir), _f32(ph.pol)
        wl, t0 = _f32(ph.wavelength), _f32(ph.t0)
        out = dict(flags=np.zeros(n, np.uint32), channel=np.full(n, -1, np.int32), t=np.zeros(n, np.float64),
                   steps=np.zeros(n, np.uint32), last_tri=np.full(n, -1, np.int32))
        if full:
            out.update(pos=np.zeros((3, n)), dir=np.zeros((3, n)), pol=np.zeros((3, n)))
        out.update(chan_count=np.zeros(self.n_chan, np.uint64), time_hist=np.zeros(n_bins, np.uint64),
                   fate_count=np.zeros(8, np.uint64), total_steps=np.zeros(1, np.uint64))
        ub = self.use_bvh if use_bvh is None else use_bvh
        self.L.orc_propagate(self.h, n, _p(pos[0]), _p(pos[1]), _p(pos[2]), _p(k[0]), _p(k[1]), _p(k[2]),
                             _p(e[0]), _p(e[1]), _p(e[2]), _p(wl), _p(t0), int(ph.id_base), int(seed), int(max_steps),
                             int(ub), _p(out["flags"]), _p(out["channel"]), _p(out["t"]), _p(out["steps"]),
                             _p(out["last_tri"]), _p(out.get("pos")), _p(out.get("dir")), _p(out.get("pol")),
                             self.n_chan, _p(out["chan_count"]), n_bins, float(t_min), float(dt), _p(out["time_hist"]),
                             _p(out["fate_count"]), _p(out["total_steps"]), nthreads or hardware_threads())
        out["fate"] = out["flags"] & 0xF
        return out


# ---- single pieces (for the pins)
def philox4x32_10(ctr, key):
    c = np.asarray(ctr, np.uint32)
    k = np.asarray(key, np.uint32)
    o = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(o))
    return o


def uniforms(seed, photon, step, block):
    o = np.zeros(4)
    lib().orc_uniforms(seed, photon, step, block, _p(o))
    return o


def rayleigh(k, e, seed, pid, step=0):
    k = np.array(k, np.float64)
    e = np.array(e, np.float64)
    it = lib().orc_rayleigh(_p(k), _p(e), seed, pid, step)
    return k, e, it


def lambert(nhat, seed, pid, step=0):
    n = np.array(nhat, np.float64)
    k = np.zeros(3)
    e = np.zeros(3)
    lib().orc_lambert(_p(n), _p(k), _p(e), seed, pid, step)
    return k, e


def specular(nhat, k, e):
    n = np.array(nhat, np.float64)
    k = np.array(k, np.float64)
    e = np.array(e, np.float64)
    lib().orc_specular(_p(n), _p(k), _p(e))
    return k, e


def fresnel(n1, n2, nhat, k, e, u):
    n = np.array(nhat, np.float64)
    k = np.array(k, np.float64)
    e = np.array(e, np.float64)
    R = C.c_double(0.0)
    oc = lib().orc_fresnel(float(n1), float(n2), _p(n), _p(k), _p(e), float(u), C.byref(R))
    return oc, R.value, k, e


def emit(source: dict, seed: int, id_base: int, n: int):
    """Emission: n photons of `source` (keys of paper_2203_14354_b200.synth.source()), fp64.
    Returns a dict of arrays: pos [3,n], dir [3,n], pol [3,n], wavelength [n], t0 [n]."""
    out = np.empty((11, n), np.float64)
    c3 = np.ascontiguousarray(source["centre"], np.float64)
    lib().orc_emit(int(source["shape"]), _p(c3), float(source["radius"]), float(source["z0"]), float(source["z1"]),
                   float(source["lambda_mean"]), float(source["lambda_sigma"]), float(source["t_start"]), float(source["tau1"]),
                   float(source["tau3"]), float(source["f_singlet"]), int(seed), int(id_base), int(n), _p(out))
    return dict(pos=out[0:3], dir=out[3:6], pol=out[6:9], wavelength=out[9], t0=out[10])


def film_coefficients(n1, nf, kf, d_nm, n3, lambda_nm, cos1):
    """Thin-film surface: (Rs, Rp, Ts, Tp) for a film nf + i kf of thickness d between n1 and n3."""
    out = np.zeros(4)
    lib().orc_film_coefficients(float(n1), float(nf), float(kf), float(d_nm), float(n3), float(lambda_nm), float(cos1), _p(out))
    return tuple(out)


def film(n1, nf, kf, d_nm, n3, lambda_nm, nhat, k, e, u):
    """One surface event on a film: returns (outcome 0 reflect / 1 transmit / 2 absorbed, k', e', R, T)."""
    kk, ee, rt = np.array(k, np.float64), np.array(e, np.float64), np.zeros(2)
    oc = lib().orc_film(float(n1), float(nf), float(kf), float(d_nm), float(n3), float(lambda_nm),
                        _p(np.ascontiguousarray(nhat, np.float64)), _p(kk), _p(ee), float(u), _p(rt))
    return oc, kk, ee, rt[0], rt[1]


# ---- ray cast of the mesh: the definition written out, the first-hit query S1 per pixel
def camera_rays(eye, forward, up, fov_y_deg, width, height):
    """PAPER.md line 138 ("Chroma rendering", insert of Fig. 1) names a rendering of the mesh and no camera model; the pinhole camera of
    include/darwinopt.h (dw_camera) is the reading: f = unit(forward), r = unit(f x up), u = r x f, t = tan(fov_y / 2); pixel (i, j),
    i to the right and j downwards, looks along unit(f + x t (width / height) r + y t u) with x = 2 (i + 0.5) / width - 1,
    y = 1 - 2 (j + 0.5) / height.  Returns directions [3, height * width] float64, pixel (i, j) at column j * width + i."""
    f = np.asarray(forward, np.float64)
    f = f / np.linalg.norm(f)
    r = np.cross(f, np.asarray(up, np.float64))
    r = r / np.linalg.norm(r)
    u = np.cross(r, f)
    t = np.tan(np.radians(np.float64(fov_y_deg)) / 2.0)
    i = np.arange(width, dtype=np.float64)[None, :]
    j = np.arange(height, dtype=np.float64)[:, None]
    x = np.broadcast_to(2.0 * (i + 0.5) / width - 1.0, (height, width)).reshape(-1)
    y = np.broadcast_to(1.0 - 2.0 * (j + 0.5) / height, (height, width)).reshape(-1)
    d = f[:, None] + (x * t * (width / height))[None, :] * r[:, None] + (y * t)[None, :] * u[:, None]
    return d / np.linalg.norm(d, axis=0)


def render(oracle, geometry, eye, forward, up, fov_y_deg, width, height, use_bvh=None):
    """Per pixel the nearest triangle along the camera ray (id, distance) and shade = round(255 |n . d|), n the unit normal of that
    triangle; (-1, inf, 0) where nothing is hit.  `oracle` is an Oracle holding `geometry`.  Arrays [height, width]."""
    d = camera_rays(eye, forward, up, fov_y_deg, width, height)
    n = d.shape[1]
    o = np.repeat(np.asarray(eye, np.float32)[:, None], n, axis=1)
    d32 = d.astype(np.float32)            # the query takes single-precision rays (as every first-hit comparison does) ...
    tri, dist = oracle.first_hit(o, d32, exclude=None, use_bvh=use_bvh)
    V = np.asarray(geometry.xyz, np.float64)
    I = np.asarray(geometry.idx)[np.maximum(tri, 0)]
    nrm = np.cross(V[I[:, 1]] - V[I[:, 0]], V[I[:, 2]] - V[I[:, 0]])
    nrm /= np.linalg.norm(nrm, axis=1)[:, None]
    cosang = np.abs(np.einsum("ij,ji->i", nrm, d32.astype(np.float64)))   # ... and shades with the direction it was given
    shade = np.where(tri >= 0, np.floor(255.0 * cosang + 0.5), 0.0).astype(np.uint8)
    return tri.reshape(height, width), dist.reshape(height, width), shade.reshape(height, width)


# ---- design-study reductions: plain counting, which is their definition
def tally(flags, channel, t, last_tri, photons_per_source, channel_group, n_groups, tri_component, n_components,
          n_bins=0, t_min=0.0, dt=1.0):
    """LCE = photons hitting the photosensitive area / photons generated, per source position and per sensor
    array (group); line 211: arrival times of the detected photons (for t90); lines 267-271, Table 6: absorbed photons by the
    component that absorbed them.  Photon i belongs to source i // photons_per_source."""
    flags, channel, last_tri = np.asarray(flags), np.asarray(channel), np.asarray(last_tri)
    n = flags.shape[0]
    ns = -(-n // photons_per_source) if n else 0
    out = dict(detected=np.zeros((ns, n_groups), np.uint64), time_hist=np.zeros((ns, n_bins), np.uint64),
               fate_by_source=np.zeros((ns, 8), np.uint64), absorbed_by_component=np.zeros(n_components, np.uint64))
    fate = flags & 0xF
    for i in range(n):
        s = i // photons_per_source
        out["fate_by_source"][s, fate[i] & 7] += 1
        if fate[i] == FATE_DETECTED:
            c = channel[i]
            if 0 <= c < len(channel_group) and 0 <= channel_group[c] < n_groups:
                out["detected"][s, channel_group[c]] += 1
            if n_bins > 0:
                b = int(np.floor((np.float32(t[i]) - np.float32(t_min)) / np.float32(dt)))
                out["time_hist"][s, min(max(b, 0), n_bins - 1)] += 1
        elif fate[i] == FATE_SURFACE_ABSORBED:
            tr = last_tri[i]
            if 0 <= tr < len(tri_component) and 0 <= tri_component[tr] < n_components:
                out["absorbed_by_component"][tri_component[tr]] += 1
    return out


def t90_from_hist(hist, t_min, dt, q=0.9):
    """Time by which the fraction q of the detected photons has arrived, from an arrival-time histogram:
    linear interpolation inside the bin where the cumulative count crosses q of the total.  NaN if nothing was detected."""
    h = np.asarray(hist, np.float64)
    tot = h.sum()
    if tot <= 0:
        return float("nan")
    cum = np.cumsum(h)
    b = int(np.searchsorted(cum, q * tot, side="left"))
    below = cum[b - 1] if b > 0 else 0.0
    return float(t_min + dt * (b + (q * tot - below) / h[b]))
