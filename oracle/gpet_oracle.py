"""ctypes binding of oracle/gpet_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It never imports the CUDA package's kernels or binding; it takes the plain dataclasses of
paper_2603_07327_b200.workloads (the shared input recipe) and marshals them into the oracle's own C
structs.  The oracle itself is single-threaded; `simulate(..., threads=k)` only runs disjoint
history ranges side by side (results are independent of k because every draw is a pure function of
(seed, history, stream, index)).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gpet_oracle.c")
_SO = os.path.join(_HERE, "libgpet_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off",
                               "-o", _SO, _SRC, "-lm"])
    return _SO


class _Layer(C.Structure):
    _fields_ = [("n", C.c_int32 * 2), ("pitch", C.c_float * 2), ("reflector", C.c_float * 2),
                ("offset", C.c_float * 2), ("depth", C.c_float), ("gap_before", C.c_float),
                ("crystal_material", C.c_int32), ("gap_material", C.c_int32)]


class _Geometry(C.Structure):
    _fields_ = [("n_panels", C.c_int32), ("pose", C.POINTER(C.c_float)), ("n_modules", C.c_int32 * 2),
                ("module_size", C.c_float * 2), ("module_pitch", C.c_float * 2),
                ("n_layers", C.c_int32), ("layers", C.POINTER(_Layer))]


class _Materials(C.Structure):
    _fields_ = [("n_materials", C.c_int32), ("n_energies", C.c_int32), ("e_min", C.c_float), ("e_step", C.c_float),
                ("mu_pe", C.POINTER(C.c_float)), ("mu_c", C.POINTER(C.c_float)), ("mu_r", C.POINTER(C.c_float))]


class _Source(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pos", C.c_float * 3), ("acol_fwhm_deg", C.c_float), ("activity_bq", C.c_double),
                ("pairs_per_slice", C.c_uint64), ("activity", C.POINTER(C.c_float)), ("phantom", C.POINTER(C.c_uint8)),
                ("phantom_majorant", C.c_int32), ("dims", C.c_int32 * 3), ("voxel", C.c_float * 3), ("origin", C.c_float * 3),
                ("beam_dir", C.c_float * 3), ("positron_fwhm_mm", C.c_float), ("half_life_s", C.c_double), ("duration_s", C.c_double),
                ("act_index", C.POINTER(C.c_uint32)), ("act_cdf", C.POINTER(C.c_uint64)), ("n_active", C.c_uint64),
                ("w_total", C.c_uint64)]


class _Hits(C.Structure):
    _fields_ = [("history", C.POINTER(C.c_uint32)), ("ids", C.POINTER(C.c_uint32))] + \
               [(k, C.POINTER(C.c_float)) for k in ("x", "y", "z", "e", "tof")] + \
               [("capacity", C.c_uint64), ("n", C.c_uint64)]


_COUNTER_NAMES = ("pairs", "searches", "entries", "steps", "step_vacuum", "virtuals", "pe", "compton", "kn_trials",
                  "rayleigh", "cutoffs", "exits", "escapes", "hits", "ph_steps", "ph_compton", "ph_absorbed", "ph_cutoff", "region_crossings")


class _Counters(C.Structure):
    _fields_ = [(k, C.c_uint64) for k in _COUNTER_NAMES]


class _Digitizer(C.Structure):
    _fields_ = [("fwhm_frac", C.c_float), ("ref_keV", C.c_float), ("e_lo", C.c_float), ("e_hi", C.c_float),
                ("window_ns", C.c_double), ("level", C.c_int32)]


class _Singles(C.Structure):
    _fields_ = [("history", C.POINTER(C.c_uint32)), ("ids", C.POINTER(C.c_uint32))] + \
               [(k, C.POINTER(C.c_float)) for k in ("x", "y", "z", "e")] + \
               [("t", C.POINTER(C.c_double)), ("capacity", C.c_uint64), ("n", C.c_uint64)]


class _Coinc(C.Structure):
    _fields_ = [(k, C.POINTER(C.c_uint32)) for k in ("ids_a", "ids_b", "history_a", "history_b")] + \
               [(k, C.POINTER(C.c_float)) for k in ("e_a", "e_b", "dt_ns")] + \
               [("t", C.POINTER(C.c_double)), ("capacity", C.c_uint64), ("n", C.c_uint64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_uniform.restype = C.c_double
        _lib.orc_uniform.argtypes = [C.c_uint32]
        _lib.orc_rayleigh_cos.restype = C.c_double
        _lib.orc_rayleigh_cos.argtypes = [C.c_double]
        _lib.orc_decay_time.restype = C.c_double
        _lib.orc_decay_time.argtypes = [C.POINTER(_Source), C.c_uint64, C.c_uint64, C.c_uint64]
        _lib.orc_decay_sites.argtypes = [C.POINTER(_Source), C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(C.c_double)]
        _lib.orc_decay_sites.restype = None
        _lib.orc_annihilation_sites.argtypes = [C.POINTER(_Source), C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(C.c_double)]
        _lib.orc_annihilation_sites.restype = None
        _lib.orc_det_log.restype = C.c_double
        _lib.orc_det_log.argtypes = [C.c_double]
        _lib.orc_det_log1m.restype = C.c_double
        _lib.orc_det_log1m.argtypes = [C.c_double]
        _lib.orc_decay_count.restype = C.c_uint64
        _lib.orc_decay_count.argtypes = [C.c_double, C.c_double, C.c_double]
        _lib.orc_rotate.argtypes = [C.POINTER(C.c_double)] + [C.c_double] * 4
        _lib.orc_rotate.restype = None
        _lib.orc_mu_lookup.argtypes = [C.POINTER(_Materials), C.c_int, C.c_double, C.POINTER(C.c_double)]
        _lib.orc_mu_lookup.restype = None
        _lib.orc_mu_majorant.argtypes = [C.POINTER(_Materials), C.c_uint32, C.c_double]
        _lib.orc_mu_majorant.restype = C.c_double
        _lib.orc_ring_poses.argtypes = [C.c_int, C.c_double, C.c_double, C.POINTER(C.c_float)]
        _lib.orc_ring_poses.restype = None
        _lib.orc_kn_sample.argtypes = [C.c_uint64, C.c_uint64, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        _lib.orc_simulate.argtypes = [C.POINTER(_Geometry), C.POINTER(_Materials), C.POINTER(_Source), C.c_uint64,
                                      C.c_uint64, C.c_uint64, C.POINTER(_Hits), C.POINTER(C.c_uint64),
                                      C.POINTER(C.c_double), C.POINTER(_Counters)]
        _lib.orc_digitize.argtypes = [C.POINTER(_Source), C.c_uint64, C.c_uint64, C.POINTER(_Hits), C.c_uint64,
                                      C.POINTER(_Digitizer), C.POINTER(_Singles), C.POINTER(_Coinc), C.POINTER(C.c_uint64)]
        _lib.orc_locate.argtypes = [C.POINTER(_Geometry), C.c_int64, C.POINTER(C.c_float), C.POINTER(C.c_uint32)]
        _lib.orc_locate_local.argtypes = [C.POINTER(_Geometry), C.c_int, C.c_int64, C.POINTER(C.c_double),
                                          C.POINTER(C.c_uint32), C.POINTER(C.c_int32)]
        _lib.orc_panel_box.argtypes = [C.POINTER(_Geometry), C.POINTER(C.c_double), C.POINTER(C.c_double)]
        _lib.orc_panel_search.argtypes = [C.POINTER(_Geometry), C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int,
                                          C.POINTER(C.c_double)]
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


# ----------------------------------------------------------------------------- marshalling
def ring_poses(n: int, radius_mm: float, first_angle_deg: float = 0.0) -> np.ndarray:
    pose = np.zeros((n, 12), np.float32)
    lib().orc_ring_poses(n, radius_mm, first_angle_deg, _p(pose, C.c_float))
    return pose


class _Keep:
    """Holds a C struct together with the numpy arrays it points into."""
    def __init__(self, struct, *arrays):
        self.struct, self.arrays = struct, arrays


def _geometry(g) -> _Keep:
    pose = (np.ascontiguousarray(g.panel_pose, np.float32) if g.panel_pose is not None
            else ring_poses(g.n_panels, g.ring_inner_radius_mm, g.ring_first_angle_deg))
    layers = (_Layer * len(g.layers))()
    for i, l in enumerate(g.layers):
        layers[i] = _Layer((C.c_int32 * 2)(*l.n_crystals), (C.c_float * 2)(*l.pitch_mm), (C.c_float * 2)(*l.reflector_mm),
                           (C.c_float * 2)(*l.offset_mm), l.depth_mm, l.gap_before_mm, l.crystal_material, l.gap_material)
    s = _Geometry(g.n_panels, _p(pose, C.c_float), (C.c_int32 * 2)(*g.n_modules), (C.c_float * 2)(*g.module_size_mm),
                  (C.c_float * 2)(*g.module_pitch_mm), len(g.layers), layers)
    return _Keep(s, pose, layers)


def _materials(t) -> _Keep:
    arrs = [np.ascontiguousarray(a, np.float32) for a in (t.mu_pe, t.mu_compton, t.mu_rayleigh)]
    s = _Materials(t.n_materials, t.n_energies, t.e_min_keV, t.e_step_keV, *[_p(a, C.c_float) for a in arrs])
    return _Keep(s, *arrs)


def _source(src) -> _Keep:
    act = None if src.activity is None else np.ascontiguousarray(src.activity, np.float32)
    ph = None if src.phantom_material is None else np.ascontiguousarray(src.phantom_material, np.uint8)
    s = _Source(src.kind, (C.c_float * 3)(*src.pos_mm), src.acolinearity_fwhm_deg, src.activity_bq,
                src.pairs_per_time_slice, None if act is None else _p(act, C.c_float),
                None if ph is None else _p(ph, C.c_uint8), src.phantom_majorant_material,
                (C.c_int32 * 3)(*src.dims), (C.c_float * 3)(*src.voxel_mm), (C.c_float * 3)(*src.origin_mm),
                (C.c_float * 3)(*src.beam_dir), src.positron_fwhm_mm, src.half_life_s, src.duration_s)
    if lib().orc_source_prepare(C.byref(s)) != 0:
        raise ValueError("source has no active voxel")
    return _Keep(s, act, ph)


@dataclass
class Hits:
    history: np.ndarray
    ids: np.ndarray
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    e_keV: np.ndarray
    tof_ns: np.ndarray

    def __len__(self):
        return len(self.history)

    @staticmethod
    def empty(n: int) -> "Hits":
        return Hits(np.zeros(n, np.uint32), np.zeros(n, np.uint32), *[np.zeros(n, np.float32) for _ in range(5)])

    def _struct(self) -> _Hits:
        return _Hits(_p(self.history, C.c_uint32), _p(self.ids, C.c_uint32), _p(self.x, C.c_float), _p(self.y, C.c_float),
                     _p(self.z, C.c_float), _p(self.e_keV, C.c_float), _p(self.tof_ns, C.c_float), len(self.history), 0)

    def head(self, n: int) -> "Hits":
        return Hits(*[getattr(self, k)[:n].copy() for k in ("history", "ids", "x", "y", "z", "e_keV", "tof_ns")])

    @staticmethod
    def concat(parts) -> "Hits":
        return Hits(*[np.concatenate([getattr(p, k) for p in parts]) for k in ("history", "ids", "x", "y", "z", "e_keV", "tof_ns")])


@dataclass
class SimResult:
    hits: Hits
    outcome_hash: Optional[np.ndarray]
    e_escape: Optional[np.ndarray]
    counters: dict


def _simulate_range(g, m, s, first, n, seed, want_hash, want_escape, hits_per_pair):
    cap = int(n * hits_per_pair) + 64
    while True:
        hits = Hits.empty(cap)
        hs = hits._struct()
        hh = np.zeros((n, 2), np.uint64) if want_hash else None
        ee = np.zeros((n, 2), np.float64) if want_escape else None
        cnt = _Counters()
        rc = lib().orc_simulate(C.byref(g.struct), C.byref(m.struct), C.byref(s.struct), first, n, seed, C.byref(hs),
                                None if hh is None else _p(hh, C.c_uint64), None if ee is None else _p(ee, C.c_double),
                                C.byref(cnt))
        if rc != 0:
            raise ValueError(f"oracle rejected the geometry (code {rc})")
        if hs.n <= cap:
            return hits.head(int(hs.n)), hh, ee, {k: int(getattr(cnt, k)) for k in _COUNTER_NAMES}
        cap = int(hs.n) + 64


def simulate(geometry, tables, source, n_pairs: int, seed: int, first_history: int = 0, want_hash: bool = False,
             want_escape: bool = False, threads: int = 1, hits_per_pair: float = 2.0) -> SimResult:
    """Histories [first_history, first_history + n_pairs); hits in (history, photon, sequence) order."""
    g, m, s = _geometry(geometry), _materials(tables), _source(source)
    try:
        threads = max(1, min(threads, n_pairs // 1024 or 1))
        bounds = np.linspace(0, n_pairs, threads + 1).astype(np.int64)
        jobs = [(first_history + int(bounds[i]), int(bounds[i + 1] - bounds[i])) for i in range(threads)]
        if threads == 1:
            parts = [_simulate_range(g, m, s, jobs[0][0], jobs[0][1], seed, want_hash, want_escape, hits_per_pair)]
        else:
            with ThreadPoolExecutor(threads) as ex:
                parts = list(ex.map(lambda j: _simulate_range(g, m, s, j[0], j[1], seed, want_hash, want_escape,
                                                              hits_per_pair), jobs))
    finally:
        lib().orc_source_release(C.byref(s.struct))
    counters = {k: sum(p[3][k] for p in parts) for k in _COUNTER_NAMES}
    return SimResult(Hits.concat([p[0] for p in parts]),
                     np.concatenate([p[1] for p in parts]) if want_hash else None,
                     np.concatenate([p[2] for p in parts]) if want_escape else None, counters)


@dataclass
class Singles:
    history: np.ndarray
    ids: np.ndarray
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    e_keV: np.ndarray
    t_s: np.ndarray


@dataclass
class Coincidences:
    ids_a: np.ndarray
    ids_b: np.ndarray
    history_a: np.ndarray
    history_b: np.ndarray
    e_a: np.ndarray
    e_b: np.ndarray
    dt_ns: np.ndarray
    t_s: np.ndarray


def digitize(source, seed: int, n_pairs_total: int, hits: Hits, dig):
    """hits (any order) -> (kept singles, time-sorted; coincidences; number of singles before the window)."""
    s = _source(source)
    try:
        n = len(hits)
        cap = max(n, 1)
        u32 = lambda: np.zeros(cap, np.uint32)
        f32 = lambda: np.zeros(cap, np.float32)
        sg = Singles(u32(), u32(), f32(), f32(), f32(), f32(), np.zeros(cap, np.float64))
        co = Coincidences(u32(), u32(), u32(), u32(), f32(), f32(), f32(), np.zeros(cap, np.float64))
        ss = _Singles(_p(sg.history, C.c_uint32), _p(sg.ids, C.c_uint32), _p(sg.x, C.c_float), _p(sg.y, C.c_float),
                      _p(sg.z, C.c_float), _p(sg.e_keV, C.c_float), _p(sg.t_s, C.c_double), cap, 0)
        cs = _Coinc(_p(co.ids_a, C.c_uint32), _p(co.ids_b, C.c_uint32), _p(co.history_a, C.c_uint32),
                    _p(co.history_b, C.c_uint32), _p(co.e_a, C.c_float), _p(co.e_b, C.c_float), _p(co.dt_ns, C.c_float),
                    _p(co.t_s, C.c_double), cap, 0)
        d = _Digitizer(dig.blur_fwhm_frac, dig.blur_ref_keV, dig.e_lo_keV, dig.e_hi_keV, dig.window_ns, dig.readout_level)
        hs = hits._struct()
        nall = C.c_uint64(0)
        lib().orc_digitize(C.byref(s.struct), seed, n_pairs_total, C.byref(hs), n, C.byref(d), C.byref(ss), C.byref(cs),
                           C.byref(nall))
        ns, nc = int(ss.n), int(cs.n)
        sg = Singles(*[getattr(sg, k)[:ns].copy() for k in ("history", "ids", "x", "y", "z", "e_keV", "t_s")])
        co = Coincidences(*[getattr(co, k)[:nc].copy() for k in ("ids_a", "ids_b", "history_a", "history_b", "e_a", "e_b",
                                                                   "dt_ns", "t_s")])
        return sg, co, int(nall.value)
    finally:
        lib().orc_source_release(C.byref(s.struct))


def decay_time(source, seed: int, history: int, n_pairs_total: int) -> float:
    s = _source(source)
    try:
        return float(lib().orc_decay_time(C.byref(s.struct), seed, history, n_pairs_total))
    finally:
        lib().orc_source_release(C.byref(s.struct))


def decay_sites(source, seed: int, first: int, n: int) -> np.ndarray:
    s = _source(source)
    try:
        out = np.zeros((n, 3), np.float64)
        lib().orc_decay_sites(C.byref(s.struct), seed, first, n, _p(out, C.c_double))
        return out
    finally:
        lib().orc_source_release(C.byref(s.struct))


def annihilation_sites(source, seed: int, first: int, n: int) -> np.ndarray:
    s = _source(source)
    try:
        out = np.zeros((n, 3), np.float64)
        lib().orc_annihilation_sites(C.byref(s.struct), seed, first, n, _p(out, C.c_double))
        return out
    finally:
        lib().orc_source_release(C.byref(s.struct))


def det_log(z: float) -> float:
    return float(lib().orc_det_log(z))


def det_log1m(y: float) -> float:
    return float(lib().orc_det_log1m(y))


def decay_count(activity_bq: float, half_life_s: float, duration_s: float) -> int:
    return int(lib().orc_decay_count(activity_bq, half_life_s, duration_s))


def rotate(d, ct: float, st: float, cp: float, sp: float) -> np.ndarray:
    v = np.asarray(d, np.float64).copy()
    lib().orc_rotate(_p(v, C.c_double), ct, st, cp, sp)
    return v


def mu_lookup(tables, material: int, e_keV: float) -> np.ndarray:
    m = _materials(tables)
    out = np.zeros(3, np.float64)
    lib().orc_mu_lookup(C.byref(m.struct), material, e_keV, _p(out, C.c_double))
    return out


def mu_majorant(tables, mask: int, e_keV: float) -> float:
    m = _materials(tables)
    return float(lib().orc_mu_majorant(C.byref(m.struct), mask, e_keV))


def locate(geometry, xyz: np.ndarray) -> np.ndarray:
    g = _geometry(geometry)
    xyz = np.ascontiguousarray(xyz, np.float32).reshape(-1, 3)
    ids = np.zeros(len(xyz), np.uint32)
    rc = lib().orc_locate(C.byref(g.struct), len(xyz), _p(xyz, C.c_float), _p(ids, C.c_uint32))
    if rc != 0:
        raise ValueError(f"oracle rejected the geometry (code {rc})")
    return ids


def locate_local(geometry, panel: int, abc: np.ndarray):
    g = _geometry(geometry)
    abc = np.ascontiguousarray(abc, np.float64).reshape(-1, 3)
    ids = np.zeros(len(abc), np.uint32)
    mat = np.zeros(len(abc), np.int32)
    rc = lib().orc_locate_local(C.byref(g.struct), panel, len(abc), _p(abc, C.c_double), _p(ids, C.c_uint32), _p(mat, C.c_int32))
    if rc != 0:
        raise ValueError(f"oracle rejected the geometry (code {rc})")
    return ids, mat


def panel_box(geometry):
    g = _geometry(geometry)
    lo, hi = np.zeros(3), np.zeros(3)
    rc = lib().orc_panel_box(C.byref(g.struct), _p(lo, C.c_double), _p(hi, C.c_double))
    if rc != 0:
        raise ValueError(f"oracle rejected the geometry (code {rc})")
    return lo, hi


def panel_search(geometry, x, d, excl: int = -1):
    g = _geometry(geometry)
    x, d = np.asarray(x, np.float64), np.asarray(d, np.float64)
    t = C.c_double(0.0)
    p = lib().orc_panel_search(C.byref(g.struct), _p(x, C.c_double), _p(d, C.c_double), excl, C.byref(t))
    return int(p), float(t.value)


def philox(counter, key) -> np.ndarray:
    c = np.asarray(counter, np.uint32).copy()
    k = np.asarray(key, np.uint32).copy()
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def kn_sample(seed: int, history: int, e_keV: float):
    eps, ct = C.c_double(0), C.c_double(0)
    n = lib().orc_kn_sample(seed, history, e_keV, C.byref(eps), C.byref(ct))
    return float(eps.value), float(ct.value), int(n)


def kn_sample_prepared(u4: np.ndarray, e_keV: float):
    """Test hook (O29): the Klein-Nishina sampler on a prepared list of trials, rows {u_a, u_b, u_c, azimuth}.
    Returns (eps, cos_theta, trials, azimuth uniform of the returned trial)."""
    u = np.ascontiguousarray(u4, np.float64).reshape(-1, 4)
    eps, ct, ua = C.c_double(0), C.c_double(0), C.c_double(0)
    f = lib().orc_kn_sample_prepared
    f.argtypes = [C.POINTER(C.c_double), C.c_int, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    n = f(_p(u, C.c_double), len(u), e_keV, C.byref(eps), C.byref(ct), C.byref(ua))
    return float(eps.value), float(ct.value), int(n), float(ua.value)


def unpack_ids(ids: np.ndarray):
    ids = np.asarray(ids, np.uint32)
    return {"seq": ids & 15, "photon": (ids >> 4) & 1, "crystal": (ids >> 5) & 8191, "layer": (ids >> 18) & 3,
            "module": (ids >> 20) & 63, "panel": ids >> 26}
