"""Thin ctypes binding of libdarwinopt.so (include/darwinopt.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the library's kernels.
There is no fallback: if the library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

from . import build as _build

_LIB_PATH = Path(__file__).resolve().parent / "libdarwinopt.so"

DW_OK, DW_E_ARG, DW_E_STATE, DW_E_CUDA, DW_E_RANGE = 0, -1, -2, -3, -4
FATE_NAMES = ("detected", "bulk_absorbed", "surface_absorbed", "escaped", "truncated", "nan_abort")
FATE_DETECTED, FATE_BULK_ABSORBED, FATE_SURFACE_ABSORBED, FATE_ESCAPED, FATE_TRUNCATED, FATE_NAN_ABORT = range(6)
H_RAYLEIGH, H_REFLECT_DIFFUSE, H_REFLECT_SPECULAR, H_SURFACE_TRANSMIT = 0x10, 0x20, 0x40, 0x80
H_FRESNEL_REFLECT, H_FRESNEL_REFRACT, H_TIR, H_MEDIUM_MISMATCH = 0x100, 0x200, 0x400, 0x800
H_FILM = 0x1000
PROP_UNBOUNDED_QUERY = 1
PROP_LEGACY_SCHEDULER = 2
PROP_NO_EMPTY_SKIP = 4
COUNTER_NAMES = ("node_visits", "tri_tests", "queries_traced", "queries_skipped", "physics_phases", "lanes_physics", "lanes_rayleigh",
                 "lanes_setup", "lanes_fresh", "iters_node", "lanes_node", "iters_leaf", "lanes_leaf", "fetches", "lanes_fetch", "rayleigh_iters",
                 "first_queries", "first_query_visits", "surface_queries", "surface_query_visits", "surface_query_hits",
                 "bulk_queries", "bulk_query_visits", "bulk_query_hits")

EXPORTS = ("dw_create", "dw_destroy", "dw_last_error", "dw_version", "dw_set_materials", "dw_set_surfaces",
           "dw_set_geometry", "dw_build_bvh", "dw_first_hit", "dw_propagate", "dw_propagate_host",
           "dw_debug_philox", "dw_last_launch", "dw_emit", "dw_set_films", "dw_tally", "dw_probe_peaks", "dw_refit_bvh", "dw_render",
           "dw_tally_finish", "dw_emit_sources", "dw_design_study", "dw_propagate_counters", "dw_design_study_static")
STATIC_MAX_SOURCES, STATIC_MAX_PHOTONS = 4096, 262144       # include/darwinopt.h DW_STATIC_MAX_*

vp, i32, i64, u32, u64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64, C.c_float


class BuildParams(C.Structure):
    _fields_ = [("max_leaf_tris", i32), ("ploc_radius", i32), ("grid_res", i32), ("split_div", i32), ("reserved", i32 * 4)]


class BuildStats(C.Structure):
    _fields_ = [("n_tri", i64), ("n_nodes", i64), ("node_bytes", i64), ("tri_bytes", i64), ("max_depth", i32),
                ("n_leaves", i32), ("scene_lo", f32 * 3), ("scene_hi", f32 * 3), ("build_ms", f32),
                ("ploc_rounds", i32), ("binary_depth", i32), ("grid_res", i32), ("grid_free_cells", i32), ("n_refs", i32), ("split_div", i32)]


class RefitStats(C.Structure):
    _fields_ = [("refit_ms", f32), ("n_levels", i32), ("n_loose_tris", i32), ("grid_free_cells", i32), ("scene_lo", f32 * 3),
                ("scene_hi", f32 * 3), ("area_ratio", f32)]


class Camera(C.Structure):
    _fields_ = [("eye", f32 * 3), ("forward", f32 * 3), ("up", f32 * 3), ("fov_y_deg", f32), ("width", i32), ("height", i32)]


class Photons(C.Structure):
    _fields_ = [("n", i64), ("photon_id_base", u64)] + [(k, vp) for k in
                ("px", "py", "pz", "kx", "ky", "kz", "ex", "ey", "ez", "wavelength", "t0")]


class Results(C.Structure):
    _fields_ = [(k, vp) for k in ("flags", "channel", "t", "steps", "last_tri", "x", "y", "z",
                                  "kx", "ky", "kz", "ex", "ey", "ez")]


class Hists(C.Structure):
    _fields_ = [("n_chan", i64), ("chan_count", vp), ("n_bins", i64), ("t_min", f32), ("dt", f32),
                ("time_hist", vp), ("fate_count", vp), ("total_steps", vp)]


class Source(C.Structure):
    _fields_ = [("shape", i32), ("centre", f32 * 3), ("radius", f32), ("z0", f32), ("z1", f32), ("lambda_mean", f32),
                ("lambda_sigma", f32), ("t_start", f32), ("tau1", f32), ("tau3", f32), ("f_singlet", f32), ("reserved", i32 * 3)]


class TallyTables(C.Structure):
    _fields_ = [("channel_group", vp), ("n_chan", i64), ("n_groups", i32), ("tri_component", vp), ("n_tri_map", i64), ("n_components", i32),
                ("detected", vp), ("time_hist", vp), ("n_bins", i64), ("t_min", f32), ("dt", f32), ("fate_by_source", vp),
                ("absorbed_by_component", vp)]


class PropagateParams(C.Structure):
    _fields_ = [("flags", u32), ("block_threads", i32), ("blocks_per_sm", i32), ("th_phys", i32),
                ("th_leaf", i32), ("reserved", i32 * 3)]


_lib = None


def load(build_if_missing: bool = True) -> C.CDLL:
    """dlopen the C-ABI library (building it in-tree with nvcc first if it is not there)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        if not build_if_missing:
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2203_14354_b200.build`")
        _build.build()
    elif _build.needs_build():                      # sources newer than the library: never run a stale build silently
        if not build_if_missing or not _build.have_nvcc():
            raise RuntimeError(f"{_LIB_PATH} is older than its sources: run `python -m paper_2203_14354_b200.build`")
        _build.build()
    L = C.CDLL(str(_LIB_PATH))
    L.dw_create.argtypes = [C.c_int, C.POINTER(vp)]
    L.dw_destroy.argtypes = [vp]
    L.dw_last_error.argtypes = [vp]
    L.dw_last_error.restype = C.c_char_p
    L.dw_version.restype = C.c_int
    L.dw_set_materials.argtypes = [vp, C.c_int, C.c_int, f32, f32, vp, vp, vp]
    L.dw_set_surfaces.argtypes = [vp, C.c_int, C.c_int, f32, f32, vp, vp, vp, vp]
    L.dw_set_films.argtypes = [vp, C.c_int, C.c_int, f32, f32, vp, vp, vp, vp]
    L.dw_set_geometry.argtypes = [vp, i64, vp, i64, vp, vp, vp, vp, vp, C.c_int]
    L.dw_build_bvh.argtypes = [vp, C.POINTER(BuildParams), C.POINTER(BuildStats), vp]
    L.dw_first_hit.argtypes = [vp, i64] + [vp] * 9 + [vp]
    L.dw_propagate.argtypes = [vp, C.POINTER(Photons), u64, i32, C.POINTER(Results), C.POINTER(Hists),
                               C.POINTER(PropagateParams), vp]
    L.dw_propagate_host.argtypes = [vp, C.POINTER(Photons), u64, i32, C.POINTER(Results), C.POINTER(Hists),
                                    C.POINTER(PropagateParams)]
    L.dw_propagate_counters.argtypes = [vp, C.POINTER(Photons), u64, i32, C.POINTER(PropagateParams), vp]
    L.dw_debug_philox.argtypes = [vp, u64, u64, u32, u32, i64, vp, vp, vp]
    L.dw_emit.argtypes = [vp, C.POINTER(Source), u64, C.POINTER(Photons), vp]
    L.dw_probe_peaks.argtypes = [vp, vp]
    L.dw_tally.argtypes = [vp, C.POINTER(Results), i64, i64, C.POINTER(TallyTables), vp]
    L.dw_tally_finish.argtypes = [vp, C.POINTER(TallyTables), i64, f32, vp, vp, vp]
    L.dw_emit_sources.argtypes = [vp, C.POINTER(Source), i64, i64, u64, C.POINTER(Photons), vp]
    L.dw_design_study.argtypes = [vp, C.POINTER(Source), i64, i64, u64, i32, C.POINTER(TallyTables), i64, f32, vp, vp, vp]
    L.dw_design_study_static.argtypes = [vp, C.POINTER(Source), i64, i64, u64, i32, C.POINTER(TallyTables), f32, vp, vp, vp]
    L.dw_last_launch.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.POINTER(i64)]
    for name in EXPORTS:
        if name not in ("dw_last_error",):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


class DwError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libdarwinopt error {code}: {msg}")
        self.code = code


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _hp(a):
    return None if a is None else a.ctypes.data_as(vp)


def _dp(t):
    """device (or pinned host) pointer of a torch tensor"""
    return None if t is None else vp(t.data_ptr())


def _stream_ptr(stream=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return vp(s.cuda_stream)


class Context:
    """One dw_ctx: a geometry + optical tables + BVH on one CUDA device."""

    def __init__(self, device: int = 0):
        self.L = load()
        h = vp()
        rc = self.L.dw_create(device, C.byref(h))
        if rc != DW_OK:
            raise DwError(rc, self.L.dw_last_error(None).decode())
        self.h = h
        self.device = device
        self.n_chan = 0
        self.stats = None

    def close(self):
        if getattr(self, "h", None):
            self.L.dw_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != DW_OK:
            raise DwError(rc, self.L.dw_last_error(self.h).decode())

    # ---- uploads -------------------------------------------------------------------------------------
    def set_materials(self, refr_index, abs_len, scat_len, lambda0=175.0, dlambda=1.0):
        n, la, ls = (_np(a, np.float32) for a in (refr_index, abs_len, scat_len))
        n = n.reshape(n.shape[0], -1)
        self._check(self.L.dw_set_materials(self.h, n.shape[0], n.shape[1], lambda0, dlambda, _hp(n), _hp(la), _hp(ls)))

    def set_surfaces(self, detect, reflect_diffuse, reflect_specular, transmit, lambda0=175.0, dlambda=1.0):
        d, rd, rs, tr = (_np(a, np.float32) for a in (detect, reflect_diffuse, reflect_specular, transmit))
        d = d.reshape(d.shape[0], -1)
        self._check(self.L.dw_set_surfaces(self.h, d.shape[0], d.shape[1], lambda0, dlambda, _hp(d), _hp(rd), _hp(rs), _hp(tr)))

    def set_optics(self, o):
        self.set_materials(o.refr_index, o.abs_len, o.scat_len, o.lambda0, o.dlambda)
        self.set_surfaces(o.detect, o.reflect_diffuse, o.reflect_specular, o.transmit, o.lambda0, o.dlambda)
        if getattr(o, "film_on", None) is not None:
            self.set_films(o.film_on, o.film_n, o.film_k, o.film_d, o.lambda0, o.dlambda)

    def set_films(self, film_on, film_n, film_k, film_d, lambda0, dlambda):
        """Thin-film surfaces: film_on int32 [S]; index, extinction, thickness (nm) float32 [S, n_lambda] on the
        surfaces' grid.  film_on=None removes all films."""
        if film_on is None:
            self._check(self.L.dw_set_films(self.h, 0, 0, 0.0, 1.0, None, None, None, None))
            return
        on, fn, fk, fd = _np(film_on, np.int32), _np(film_n, np.float32), _np(film_k, np.float32), _np(film_d, np.float32)
        self._check(self.L.dw_set_films(self.h, fn.shape[0], fn.shape[1], lambda0, dlambda, _hp(on), _hp(fn), _hp(fk), _hp(fd)))

    def set_geometry(self, g):
        xyz, idx = _np(g.xyz, np.float32), _np(g.idx, np.int32)
        mi, mo, sf, ch = (_np(a, np.int32) for a in (g.mat_inner, g.mat_outer, g.surface, g.channel))
        self._check(self.L.dw_set_geometry(self.h, xyz.shape[0], _hp(xyz), idx.shape[0], _hp(idx), _hp(mi), _hp(mo),
                                           _hp(sf), _hp(ch), 0))
        self.n_chan = int(g.n_channels)

    def set_geometry_device(self, xyz, idx, mat_inner, mat_outer, surface, channel, n_channels):
        """torch CUDA tensors (float32 [V,3], int32 [T,3], int32 [T] x4)."""
        self._check(self.L.dw_set_geometry(self.h, xyz.shape[0], _dp(xyz), idx.shape[0], _dp(idx), _dp(mat_inner),
                                           _dp(mat_outer), _dp(surface), _dp(channel), 1))
        self.n_chan = int(n_channels)

    def build_bvh(self, max_leaf_tris: int = 0, stream=None, ploc_radius: int = 0, grid_res: int = 0, split_div: int = 0) -> dict:
        p = BuildParams(max_leaf_tris=max_leaf_tris, ploc_radius=ploc_radius, grid_res=grid_res, split_div=split_div)
        st = BuildStats()
        self._check(self.L.dw_build_bvh(self.h, C.byref(p), C.byref(st), _stream_ptr(stream)))
        self.stats = {k: (list(getattr(st, k)) if k.startswith("scene") else getattr(st, k)) for k, _ in BuildStats._fields_}
        return self.stats

    def refit(self, xyz, stream=None) -> dict:
        """New vertex positions (numpy [V,3] or a torch CUDA tensor) for the same triangles, under the tree of the last build_bvh
        (SURVEY.md 8(f) f4): results equal those of a fresh build on the moved geometry, bit for bit."""
        st = RefitStats()
        if hasattr(xyz, "is_cuda") and xyz.is_cuda:
            self._check(self.L.dw_refit_bvh(self.h, xyz.shape[0], _dp(xyz), 1, C.byref(st), _stream_ptr(stream)))
        else:
            a = _np(xyz, np.float32)
            self._check(self.L.dw_refit_bvh(self.h, a.shape[0], _hp(a), 0, C.byref(st), _stream_ptr(stream)))
        return {k: (list(getattr(st, k)) if k.startswith("scene") else getattr(st, k)) for k, _ in RefitStats._fields_}

    # ---- emission -------------------------------------------------------------------
    def emit(self, source: dict, seed: int, n: int, id_base: int = 0, device="cuda:0", stream=None) -> "EmittedPhotons":
        """n scintillation photons of `source` (see synth.source) generated on the device; the result goes to propagate()."""
        out = EmittedPhotons(n, id_base, device)
        self._check(self.L.dw_emit(self.h, C.byref(_source(source)), int(seed), C.byref(out.c), _stream_ptr(stream)))
        return out

    def emit_sources(self, sources, photons_per_source: int, seed: int, n: int | None = None, id_base: int = 0, device="cuda:0",
                     stream=None) -> "EmittedPhotons":
        """One launch for many sources (dw_emit_sources): photon i belongs to sources[i // photons_per_source]."""
        n = len(sources) * int(photons_per_source) if n is None else int(n)
        out = EmittedPhotons(n, id_base, device)
        arr = (Source * len(sources))(*[_source(s) for s in sources])
        self._check(self.L.dw_emit_sources(self.h, arr, len(sources), int(photons_per_source), int(seed), C.byref(out.c), _stream_ptr(stream)))
        return out

    # ---- design-study reductions ------------------------------------------------------
    def tally(self, results, n, photons_per_source, acc: "Tally", stream=None):
        """Accumulate the per-photon `results` (DeviceResults with flags, channel, t, last_tri) into the device tables of `acc`."""
        acc.check_sources(n, photons_per_source)
        self._check(self.L.dw_tally(self.h, C.byref(results.c), int(n), int(photons_per_source), C.byref(acc.c), _stream_ptr(stream)))

    def tally_finish(self, acc: "Tally", quantile: float = 0.9, stream=None):
        """LCE per source and group and t90 per source from the tables of `acc`, computed by the library (dw_tally_finish)."""
        self._check(self.L.dw_tally_finish(self.h, C.byref(acc.c), acc.ns, float(quantile), _dp(acc.lce),
                                           _dp(acc.t90) if acc.nb > 0 else None, _stream_ptr(stream)))

    def design_study(self, sources, photons_per_source, seed, max_steps, channel_group, n_groups, tri_component, n_components,
                     n_bins=2000, t_min=0.0, dt=1.0, sources_per_batch=32, device="cuda:0", quantile=0.9):
        """The paper's design-study loop as ONE library call (dw_design_study): emission of
        all sources of a batch in one launch, propagation, reduction to LCE per source and sensor array, arrival-time histograms,
        t90 and the table of absorbed photons by component.  Photon ids are source_index * photons_per_source + i, so a result does
        not depend on sources_per_batch.  Returns a dict of numpy arrays."""
        import torch
        ns = len(sources)
        acc = Tally(ns, channel_group, n_groups, tri_component, n_components, n_bins, t_min, dt, device)
        arr = (Source * ns)(*[_source(s) for s in sources])
        self._check(self.L.dw_design_study(self.h, arr, ns, int(photons_per_source), int(seed), int(max_steps), C.byref(acc.c),
                                           int(sources_per_batch), float(quantile), _dp(acc.lce), _dp(acc.t90) if acc.nb > 0 else None,
                                           _stream_ptr()))
        torch.cuda.synchronize()
        return acc.numpy()

    def design_study_static(self, sources, photons_per_source, seed, max_steps, acc: "Tally", quantile=0.9, stream=None):
        """dw_design_study_static: the same loop with every scratch buffer in the library's fixed device array, so the call allocates
        nothing (include/darwinopt.h).  `acc` holds the caller's tables (zeroed by the caller) and receives lce / t90.  At most
        STATIC_MAX_SOURCES sources of at most STATIC_MAX_PHOTONS photons each (DW_E_RANGE beyond).  Asynchronous on the stream."""
        ns = len(sources)
        if ns > acc.ns:
            raise ValueError(f"{ns} sources, the tables hold {acc.ns}")
        arr = (Source * ns)(*[_source(s) for s in sources])
        self._check(self.L.dw_design_study_static(self.h, arr, ns, int(photons_per_source), int(seed), int(max_steps), C.byref(acc.c),
                                                  float(quantile), _dp(acc.lce), _dp(acc.t90) if acc.nb > 0 else None, _stream_ptr(stream)))

    def probe_peaks(self) -> dict:
        """Measured issue rates and L2 read bandwidth of this device (include/darwinopt.h dw_probe_peaks)."""
        out = (C.c_double * 4)()
        self._check(self.L.dw_probe_peaks(self.h, out))
        return dict(fma_lane_instr_per_s=out[0], alu_lane_instr_per_s=out[1], mix_lane_instr_per_s=out[2], l2_read_bytes_per_s=out[3])

    # ---- queries -------------------------------------------------------------------------------------
    def first_hit(self, origin, direction, exclude=None, stream=None):
        """origin, direction: torch CUDA float32 [3,n] (rows contiguous).  Returns (tri int32[n], dist float32[n])."""
        import torch
        n = origin.shape[1]
        tri = torch.empty(n, dtype=torch.int32, device=origin.device)
        dist = torch.empty(n, dtype=torch.float32, device=origin.device)
        self._check(self.L.dw_first_hit(self.h, n, _dp(origin[0]), _dp(origin[1]), _dp(origin[2]), _dp(direction[0]),
                                        _dp(direction[1]), _dp(direction[2]), _dp(exclude), _dp(tri), _dp(dist),
                                        _stream_ptr(stream)))
        return tri, dist

    def render(self, eye, forward, up, fov_y_deg: float, width: int, height: int, device="cuda:0", stream=None):
        """Ray cast of the mesh (dw_render).  Returns torch CUDA tensors [height, width]: (tri int32, depth float32, shade uint8)."""
        import torch
        cam = Camera(eye=(f32 * 3)(*eye), forward=(f32 * 3)(*forward), up=(f32 * 3)(*up), fov_y_deg=fov_y_deg, width=width, height=height)
        shape = (max(int(height), 0), max(int(width), 0))
        tri = torch.empty(shape, dtype=torch.int32, device=device)
        depth = torch.empty(shape, dtype=torch.float32, device=device)
        shade = torch.empty(shape, dtype=torch.uint8, device=device)
        self._check(self.L.dw_render(self.h, C.byref(cam), _dp(tri), _dp(depth), _dp(shade), _stream_ptr(stream)))
        return tri, depth, shade

    def propagate_counters(self, ph: "DevicePhotons", seed: int, max_steps: int, flags: int = 0, **kw) -> dict:
        """The instrumented instantiation of the propagation kernel, once over `ph` (dw_propagate_counters): raw event counts."""
        pp = PropagateParams(flags=flags, **kw)
        out = (u64 * 24)()
        self._check(self.L.dw_propagate_counters(self.h, C.byref(ph.c), seed, max_steps, C.byref(pp), out))
        return {k: int(out[i]) for i, k in enumerate(COUNTER_NAMES)}

    def propagate(self, ph: "DevicePhotons", seed: int, max_steps: int, out: "DeviceResults | None" = None,
                  hist: "DeviceHists | None" = None, flags: int = 0, block_threads: int = 0, blocks_per_sm: int = 0,
                  th_phys: int = 0, th_leaf: int = 0, stream=None):
        pp = PropagateParams(flags=flags, block_threads=block_threads, blocks_per_sm=blocks_per_sm, th_phys=th_phys,
                             th_leaf=th_leaf)
        self._check(self.L.dw_propagate(self.h, C.byref(ph.c), seed, max_steps, C.byref(out.c) if out else None,
                                        C.byref(hist.c) if hist else None, C.byref(pp), _stream_ptr(stream)))

    def propagate_host(self, ph: "HostPhotons", seed: int, max_steps: int, out=None, hist=None, flags: int = 0):
        pp = PropagateParams(flags=flags)
        self._check(self.L.dw_propagate_host(self.h, C.byref(ph.c), seed, max_steps, C.byref(out.c) if out else None,
                                             C.byref(hist.c) if hist else None, C.byref(pp)))

    def debug_philox(self, seed, base, step, block, n):
        import torch
        raw = torch.empty((n, 4), dtype=torch.int32, device=f"cuda:{self.device}")
        u = torch.empty((n, 4), dtype=torch.float32, device=f"cuda:{self.device}")
        self._check(self.L.dw_debug_philox(self.h, seed, base, step, block, n, _dp(raw), _dp(u), _stream_ptr()))
        return raw.cpu().numpy().view(np.uint32), u.cpu().numpy()

    def last_launch(self) -> dict:
        g, b, s, n = i32(), i32(), i32(), i64()
        self.L.dw_last_launch(self.h, C.byref(g), C.byref(b), C.byref(s), C.byref(n))
        return dict(grid=g.value, block=b.value, smem=s.value, n_launches=n.value)


_IN = ("px", "py", "pz", "kx", "ky", "kz", "ex", "ey", "ez", "wavelength", "t0")
_OUT_DT = dict(flags="int32", channel="int32", t="float32", steps="int32", last_tri="int32", x="float32", y="float32",
               z="float32", kx="float32", ky="float32", kz="float32", ex="float32", ey="float32", ez="float32")


def _source(src: dict) -> Source:
    return Source(shape=int(src["shape"]), centre=(f32 * 3)(*src["centre"]), radius=src["radius"], z0=src["z0"], z1=src["z1"],
                  lambda_mean=src["lambda_mean"], lambda_sigma=src["lambda_sigma"], t_start=src["t_start"], tau1=src["tau1"],
                  tau3=src["tau3"], f_singlet=src["f_singlet"])


class _PhotonsBase:
    def _fill(self, tensors, n, id_base):
        self.t = tensors
        self.n = n
        self.c = Photons(n=n, photon_id_base=id_base, **{k: vp(tensors[k].data_ptr()) for k in _IN})

    @property
    def nbytes(self):
        return 4 * 11 * self.n


class DevicePhotons(_PhotonsBase):
    """SoA photon batch resident on the device (torch tensors own the memory)."""

    def __init__(self, ph, device="cuda:0"):
        import torch
        rows = dict(px=ph.pos[0], py=ph.pos[1], pz=ph.pos[2], kx=ph.dir[0], ky=ph.dir[1], kz=ph.dir[2],
                    ex=ph.pol[0], ey=ph.pol[1], ez=ph.pol[2], wavelength=ph.wavelength, t0=ph.t0)
        self._fill({k: torch.from_numpy(_np(v, np.float32)).to(device) for k, v in rows.items()}, ph.n, ph.id_base)


class EmittedPhotons(_PhotonsBase):
    """Eleven uninitialised device arrays for Context.emit to fill."""

    def __init__(self, n, id_base=0, device="cuda:0"):
        import torch
        self._fill({k: torch.empty(max(n, 1), dtype=torch.float32, device=device) for k in _IN}, n, id_base)

    def numpy(self):
        g = lambda k: self.t[k][: self.n].cpu().numpy()
        return dict(pos=np.stack([g("px"), g("py"), g("pz")]), dir=np.stack([g("kx"), g("ky"), g("kz")]),
                    pol=np.stack([g("ex"), g("ey"), g("ez")]), wavelength=g("wavelength"), t0=g("t0"))


class HostPhotons(_PhotonsBase):
    """SoA photon batch in pinned host memory (for dw_propagate_host)."""

    def __init__(self, ph, pin=True):
        import torch
        rows = dict(px=ph.pos[0], py=ph.pos[1], pz=ph.pos[2], kx=ph.dir[0], ky=ph.dir[1], kz=ph.dir[2],
                    ex=ph.pol[0], ey=ph.pol[1], ez=ph.pol[2], wavelength=ph.wavelength, t0=ph.t0)
        ts = {}
        for k, v in rows.items():
            t = torch.from_numpy(_np(v, np.float32).copy())
            ts[k] = t.pin_memory() if pin else t
        self._fill(ts, ph.n, ph.id_base)


class _ResultsBase:
    def numpy(self):
        out = {}
        for k, t in self.t.items():
            a = t.cpu().numpy()
            out[k] = a.view(np.uint32) if k in ("flags", "steps") else a
        if "flags" in out:
            out["fate"] = out["flags"] & 0xF
        return out

    @property
    def nbytes(self):
        return sum(t.numel() * t.element_size() for t in self.t.values())


class DeviceResults(_ResultsBase):
    def __init__(self, n, fields=("flags", "channel", "t", "steps", "last_tri", "x", "y", "z"), device="cuda:0"):
        import torch
        self.t = {k: torch.empty(n, dtype=getattr(torch, _OUT_DT[k]), device=device) for k in fields}
        self.c = Results(**{k: vp(t.data_ptr()) for k, t in self.t.items()})


class HostResults(_ResultsBase):
    def __init__(self, n, fields=("flags", "channel", "t", "steps", "last_tri", "x", "y", "z"), pin=True):
        import torch
        self.t = {k: torch.empty(n, dtype=getattr(torch, _OUT_DT[k]), pin_memory=pin) for k in fields}
        self.c = Results(**{k: vp(t.data_ptr()) for k, t in self.t.items()})


class _HistsBase:
    def _make(self, n_chan, n_bins, t_min, dt, **kw):
        import torch
        self.chan_count = torch.zeros(max(n_chan, 1), dtype=torch.int64, **kw)
        self.time_hist = torch.zeros(max(n_bins, 1), dtype=torch.int32, **kw)
        self.fate_count = torch.zeros(8, dtype=torch.int64, **kw)
        self.total_steps = torch.zeros(1, dtype=torch.int64, **kw)
        self.n_chan, self.n_bins = n_chan, n_bins
        self.c = Hists(n_chan=n_chan, chan_count=vp(self.chan_count.data_ptr()), n_bins=n_bins, t_min=t_min, dt=dt,
                       time_hist=vp(self.time_hist.data_ptr()) if n_bins > 0 else None,
                       fate_count=vp(self.fate_count.data_ptr()), total_steps=vp(self.total_steps.data_ptr()))

    def zero_(self):
        for t in (self.chan_count, self.time_hist, self.fate_count, self.total_steps):
            t.zero_()

    def numpy(self):
        return dict(chan_count=self.chan_count.cpu().numpy()[: self.n_chan].astype(np.uint64),
                    time_hist=self.time_hist.cpu().numpy()[: self.n_bins].view(np.uint32).astype(np.uint64),
                    fate_count=self.fate_count.cpu().numpy().astype(np.uint64),
                    total_steps=self.total_steps.cpu().numpy().astype(np.uint64))

    @property
    def nbytes(self):
        return 8 * self.n_chan + 4 * self.n_bins + 64 + 8


class DeviceHists(_HistsBase):
    def __init__(self, n_chan, n_bins=0, t_min=0.0, dt=1.0, device="cuda:0"):
        self._make(n_chan, n_bins, t_min, dt, device=device)


class HostHists(_HistsBase):
    def __init__(self, n_chan, n_bins=0, t_min=0.0, dt=1.0):
        self._make(n_chan, n_bins, t_min, dt)


def write_pgm(path, shade) -> None:
    """An 8-bit image [height, width] (numpy or torch) as a binary PGM file: the headless stand-in for a display."""
    a = shade.cpu().numpy() if hasattr(shade, "cpu") else np.asarray(shade)
    a = np.ascontiguousarray(a, dtype=np.uint8)
    with open(path, "wb") as fh:
        fh.write(b"P5\n%d %d\n255\n" % (a.shape[1], a.shape[0]))
        fh.write(a.tobytes())


def make_context(geometry, optics, device: int = 0, max_leaf_tris: int = 0) -> Context:
    """Upload tables + geometry and build the BVH."""
    ctx = Context(device)
    ctx.set_optics(optics)
    ctx.set_geometry(geometry)
    ctx.build_bvh(max_leaf_tris)
    return ctx


class Tally:
    """Device tables of dw_tally for n_sources sources (zeroed here; dw_tally accumulates)."""

    def __init__(self, n_sources, channel_group, n_groups, tri_component, n_components, n_bins=0, t_min=0.0, dt=1.0, device="cuda:0"):
        import torch
        self.ns, self.G, self.K, self.nb, self.t_min, self.dt = int(n_sources), int(n_groups), int(n_components), int(n_bins), float(t_min), float(dt)
        self.channel_group = torch.from_numpy(_np(channel_group, np.int32)).to(device)
        self.tri_component = torch.from_numpy(_np(tri_component, np.int32)).to(device)
        z = lambda shape, dt_: torch.zeros(shape, dtype=dt_, device=device)
        self.detected = z((max(self.ns, 1), self.G), torch.int64)
        self.time_hist = z((max(self.ns, 1), max(self.nb, 1)), torch.int32)
        self.fate_by_source = z((max(self.ns, 1), 8), torch.int64)
        self.absorbed = z((self.K,), torch.int64)
        self.lce = torch.full((max(self.ns, 1), self.G), float("nan"), dtype=torch.float32, device=device)   # written by the library
        self.t90 = torch.full((max(self.ns, 1),), float("nan"), dtype=torch.float32, device=device)
        self.c = self._tables(0)
        self._limit = self.ns

    def _tables(self, s0):
        return TallyTables(channel_group=vp(self.channel_group.data_ptr()), n_chan=self.channel_group.numel(), n_groups=self.G,
                           tri_component=vp(self.tri_component.data_ptr()), n_tri_map=self.tri_component.numel(), n_components=self.K,
                           detected=vp(self.detected[s0:].data_ptr()), time_hist=vp(self.time_hist[s0:].data_ptr()) if self.nb > 0 else None,
                           n_bins=self.nb, t_min=self.t_min, dt=self.dt, fate_by_source=vp(self.fate_by_source[s0:].data_ptr()),
                           absorbed_by_component=vp(self.absorbed.data_ptr()))

    def view(self, s0, s1):
        """The same tables seen from source s0 on (for a batch that holds sources s0 .. s1 - 1)."""
        v = object.__new__(Tally)
        v.__dict__.update(self.__dict__)
        v.c = self._tables(s0)
        v._limit = s1 - s0
        return v

    def check_sources(self, n, pps):
        if -(-int(n) // int(pps)) > self._limit:
            raise ValueError(f"{n} photons at {pps} per source need more than the {self._limit} sources of these tables")

    def numpy(self):
        """The tables, and lce / t90 as dw_tally_finish / dw_design_study wrote them (NaN until one of them has run)."""
        det = self.detected[: self.ns].cpu().numpy().astype(np.uint64)
        return dict(detected=det, time_hist=self.time_hist[: self.ns, : self.nb].cpu().numpy().view(np.uint32).astype(np.uint64),
                    fate_by_source=self.fate_by_source[: self.ns].cpu().numpy().astype(np.uint64),
                    absorbed_by_component=self.absorbed.cpu().numpy().astype(np.uint64),
                    lce=self.lce[: self.ns].cpu().numpy(), t90=self.t90[: self.ns].cpu().numpy() if self.nb > 0 else None)
