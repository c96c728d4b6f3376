"""Thin Python binding of libgpet.so (include/gpet.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch supplies device memory and streams.
There is no fallback: importing works anywhere, but any call raises if libgpet.so has not been built
(`python -m paper_2603_07327_b200.build`) or no CUDA device is present.
Function names are the C ABI's.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgpet.so")
GPET_IDS_NONE = 0xFFFFFFFF
CHUNK_PAIRS = 512                     # GPET_HIT_CHUNK_PAIRS


class GpetError(RuntimeError):
    pass


# ----------------------------------------------------------------------------- C structs (mirror include/gpet.h)
class _LayerDesc(C.Structure):
    _fields_ = [("n_crystals", C.c_int32 * 2), ("pitch_mm", C.c_float * 2), ("reflector_mm", C.c_float * 2),
                ("offset_mm", C.c_float * 2), ("depth_mm", C.c_float), ("gap_before_mm", C.c_float),
                ("crystal_material", C.c_int32), ("gap_material", C.c_int32)]


class _GeometryDesc(C.Structure):
    _fields_ = [("n_panels", C.c_int32), ("panel_pose", C.POINTER(C.c_float)), ("ring_inner_radius_mm", C.c_float),
                ("ring_first_angle_deg", C.c_float), ("n_modules", C.c_int32 * 2), ("module_size_mm", C.c_float * 2),
                ("module_pitch_mm", C.c_float * 2), ("n_layers", C.c_int32), ("layers", C.POINTER(_LayerDesc))]


class _Source(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pos_mm", C.c_float * 3), ("beam_dir", C.c_float * 3),
                ("acolinearity_fwhm_deg", C.c_float), ("activity_bq", C.c_double), ("pairs_per_time_slice", C.c_uint64),
                ("activity_map", C.c_void_p), ("phantom_material", C.c_void_p), ("phantom_majorant_material", C.c_int32),
                ("dims", C.c_int32 * 3), ("voxel_mm", C.c_float * 3), ("origin_mm", C.c_float * 3),
                ("positron_fwhm_mm", C.c_float), ("half_life_s", C.c_double), ("duration_s", C.c_double)]


class _Hits(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("history", "ids", "x", "y", "z", "e_keV", "tof_ns")] + \
               [("capacity", C.c_uint64), ("n_hits", C.c_void_p), ("outcome_hash", C.c_void_p), ("chunk_fill", C.c_void_p)]


class _Digitizer(C.Structure):
    _fields_ = [("blur_fwhm_frac", C.c_float), ("blur_ref_keV", C.c_float), ("e_lo_keV", C.c_float), ("e_hi_keV", C.c_float),
                ("window_ns", C.c_double), ("readout_level", C.c_int32)]


class _Singles(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("history", "ids", "x", "y", "z", "e_keV", "t_s")] + \
               [("capacity", C.c_uint64), ("n_singles", C.c_void_p)]


class _Coinc(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("ids_a", "ids_b", "history_a", "history_b", "e_a", "e_b", "dt_ns", "t_s")] + \
               [("capacity", C.c_uint64), ("n_coinc", C.c_void_p)]


class _HostOutputs(C.Structure):
    _fields_ = [("hits", _Hits), ("singles", _Singles), ("coinc", _Coinc)]


EXPORTS = ("gpet_geometry_create", "gpet_geometry_destroy", "gpet_geometry_panel_pose", "gpet_geometry_open_faces", "gpet_geometry_bore_radius", "gpet_geometry_locate",
           "gpet_materials_load", "gpet_materials_destroy", "gpet_activity_create", "gpet_activity_destroy",
           "gpet_simulate", "gpet_digitize_scratch_bytes", "gpet_digitize", "gpet_digitize_static", "gpet_run_host", "gpet_last_error",
           "gpet_launch_count", "gpet_set_transport_warps", "gpet_pipeline_create", "gpet_pipeline_submit", "gpet_pipeline_collect",
           "gpet_pipeline_destroy", "gpet_shutdown", "gpet_decay_count")

_lib = None


def lib():
    """Loads libgpet.so; fails loudly if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise GpetError(f"{LIB_PATH} is missing: build it with `python -m paper_2603_07327_b200.build` "
                            "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, u64, i32 = C.c_void_p, C.c_uint64, C.c_int32
        L.gpet_geometry_create.argtypes = [C.POINTER(_GeometryDesc), C.POINTER(vp)]
        L.gpet_geometry_destroy.argtypes = [vp]
        L.gpet_geometry_panel_pose.argtypes = [vp, i32, C.POINTER(C.c_float)]
        L.gpet_geometry_open_faces.argtypes = [vp, i32, C.POINTER(C.c_uint32)]
        L.gpet_geometry_bore_radius.argtypes = [vp, C.POINTER(C.c_float)]
        L.gpet_geometry_locate.argtypes = [vp, C.c_int64, vp, vp]
        L.gpet_materials_load.argtypes = [i32, i32, C.c_float, C.c_float, vp, vp, vp, C.POINTER(vp)]
        L.gpet_materials_destroy.argtypes = [vp]
        L.gpet_activity_create.argtypes = [vp, C.POINTER(i32), C.POINTER(vp)]
        L.gpet_activity_destroy.argtypes = [vp]
        L.gpet_simulate.argtypes = [vp, vp, C.POINTER(_Source), u64, u64, u64, C.POINTER(_Hits), vp]
        L.gpet_digitize_scratch_bytes.argtypes = [u64, u64]
        L.gpet_digitize_scratch_bytes.restype = C.c_size_t
        L.gpet_digitize.argtypes = [C.POINTER(_Source), u64, u64, u64, u64, C.POINTER(_Hits), u64, C.POINTER(_Digitizer),
                                    vp, C.c_size_t, C.POINTER(_Singles), C.POINTER(_Coinc), vp]
        L.gpet_digitize_static.argtypes = [C.POINTER(_Source), u64, u64, u64, u64, C.POINTER(_Hits), u64, C.POINTER(_Digitizer),
                                           C.POINTER(_Singles), C.POINTER(_Coinc), vp]
        L.gpet_run_host.argtypes = [vp, vp, C.POINTER(_Source), u64, u64, u64, u64, C.POINTER(_Digitizer), C.c_double,
                                    C.POINTER(_HostOutputs)]
        L.gpet_pipeline_create.argtypes = [vp, vp, C.POINTER(_Source), C.POINTER(_Digitizer), u64, u64, C.c_double, C.c_uint32, i32, C.POINTER(vp)]
        L.gpet_pipeline_submit.argtypes = [vp, u64, u64, u64]
        L.gpet_pipeline_collect.argtypes = [vp, C.POINTER(_HostOutputs)]
        L.gpet_pipeline_destroy.argtypes = [vp]
        L.gpet_decay_count.argtypes = [C.c_double, C.c_double, C.c_double, C.POINTER(u64)]
        L.gpet_last_error.restype = C.c_char_p
        L.gpet_launch_count.restype = u64
        L.gpet_set_transport_warps.argtypes = [i32]
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise GpetError(f"libgpet error {rc}: {lib().gpet_last_error().decode()}")


def gpet_decay_count(activity_bq: float, half_life_s: float, duration_s: float) -> int:
    n = C.c_uint64(0)
    _check(lib().gpet_decay_count(activity_bq, half_life_s, duration_s, C.byref(n)))
    return int(n.value)


def gpet_launch_count() -> int:
    return int(lib().gpet_launch_count())


def gpet_set_transport_warps(warps: int) -> int:
    """Warps per transport CTA (1..20, 0 = default 20); returns the value in force."""
    return int(lib().gpet_set_transport_warps(int(warps)))


# ----------------------------------------------------------------------------- handles
class _Handle:
    _destroy = None

    def __init__(self, ptr):
        self.ptr = ptr

    def __del__(self):
        try:
            if self.ptr and _lib is not None:
                getattr(_lib, self._destroy)(self.ptr)
        except Exception:
            pass
        self.ptr = None


class Geometry(_Handle):
    _destroy = "gpet_geometry_destroy"


class Materials(_Handle):
    _destroy = "gpet_materials_destroy"


class Activity(_Handle):
    _destroy = "gpet_activity_destroy"


def _fp(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def gpet_geometry_create(g) -> Geometry:
    """g: workloads.Geometry.  panel_pose None = repetition mode (ring)."""
    layers = (_LayerDesc * len(g.layers))()
    for i, l in enumerate(g.layers):
        layers[i] = _LayerDesc((C.c_int32 * 2)(*l.n_crystals), (C.c_float * 2)(*l.pitch_mm), (C.c_float * 2)(*l.reflector_mm),
                               (C.c_float * 2)(*l.offset_mm), l.depth_mm, l.gap_before_mm, l.crystal_material, l.gap_material)
    pose = None if g.panel_pose is None else np.ascontiguousarray(g.panel_pose, np.float32)
    d = _GeometryDesc(g.n_panels, None if pose is None else _fp(pose), g.ring_inner_radius_mm, g.ring_first_angle_deg,
                      (C.c_int32 * 2)(*g.n_modules), (C.c_float * 2)(*g.module_size_mm), (C.c_float * 2)(*g.module_pitch_mm),
                      len(g.layers), layers)
    out = C.c_void_p()
    _check(lib().gpet_geometry_create(C.byref(d), C.byref(out)))
    return Geometry(out.value)


def gpet_geometry_panel_pose(geom: Geometry, panel: int) -> np.ndarray:
    pose = np.zeros(12, np.float32)
    _check(lib().gpet_geometry_panel_pose(geom.ptr, panel, _fp(pose)))
    return pose


def gpet_geometry_open_faces(geom: Geometry, panel: int) -> int:
    mask = C.c_uint32(0)
    _check(lib().gpet_geometry_open_faces(geom.ptr, panel, C.byref(mask)))
    return int(mask.value)


def gpet_geometry_bore_radius(geom: Geometry) -> float:
    r = C.c_float(0.0)
    _check(lib().gpet_geometry_bore_radius(geom.ptr, C.byref(r)))
    return float(r.value)


def gpet_geometry_locate(geom: Geometry, xyz: np.ndarray) -> np.ndarray:
    xyz = np.ascontiguousarray(xyz, np.float32).reshape(-1, 3)
    ids = np.zeros(len(xyz), np.uint32)
    _check(lib().gpet_geometry_locate(geom.ptr, len(xyz), xyz.ctypes.data, ids.ctypes.data))
    return ids


def gpet_materials_load(t) -> Materials:
    """t: workloads.Tables."""
    arrs = [np.ascontiguousarray(a, np.float32) for a in (t.mu_pe, t.mu_compton, t.mu_rayleigh)]
    out = C.c_void_p()
    _check(lib().gpet_materials_load(t.n_materials, t.n_energies, t.e_min_keV, t.e_step_keV, arrs[0].ctypes.data,
                                     arrs[1].ctypes.data, arrs[2].ctypes.data, C.byref(out)))
    return Materials(out.value)


def gpet_activity_create(activity: np.ndarray, dims) -> Activity:
    a = np.ascontiguousarray(activity, np.float32)
    out = C.c_void_p()
    _check(lib().gpet_activity_create(a.ctypes.data, (C.c_int32 * 3)(*dims), C.byref(out)))
    return Activity(out.value)


class DeviceSource:
    """workloads.Source marshalled once: holds the activity handle and the phantom map on the device."""

    def __init__(self, src, device="cuda"):
        import torch
        self.src = src
        self.activity = gpet_activity_create(src.activity, src.dims) if src.kind == 1 else None
        self.phantom = None
        if src.kind == 1 and src.phantom_material is not None:
            self.phantom = torch.from_numpy(np.ascontiguousarray(src.phantom_material, np.uint8)).to(device)
        self.struct = _source_struct(src, self.activity.ptr if self.activity else None,
                                     self.phantom.data_ptr() if self.phantom is not None else None)


def _source_struct(src, activity_ptr, phantom_ptr) -> _Source:
    return _Source(src.kind, (C.c_float * 3)(*src.pos_mm), (C.c_float * 3)(*src.beam_dir), src.acolinearity_fwhm_deg,
                   src.activity_bq, src.pairs_per_time_slice, activity_ptr, phantom_ptr, src.phantom_majorant_material,
                   (C.c_int32 * 3)(*src.dims), (C.c_float * 3)(*src.voxel_mm), (C.c_float * 3)(*src.origin_mm),
                   src.positron_fwhm_mm, src.half_life_s, src.duration_s)


# ----------------------------------------------------------------------------- device buffers (torch tensors)
@dataclass
class HitBuffer:
    history: "torch.Tensor"
    ids: "torch.Tensor"
    x: "torch.Tensor"
    y: "torch.Tensor"
    z: "torch.Tensor"
    e_keV: "torch.Tensor"
    tof_ns: "torch.Tensor"
    n_hits: "torch.Tensor"                 # int64[1] device counter
    outcome_hash: Optional["torch.Tensor"] = None
    chunk_fill: Optional["torch.Tensor"] = None   # int32[n_chunks + 1]: chunked layout (include/gpet.h), else dense

    @staticmethod
    def allocate(capacity: int, n_hash: int = 0, device="cuda") -> "HitBuffer":
        """n_hash = number of histories to hash (2 words each: photon A, photon B)."""
        import torch
        i32 = lambda: torch.empty(capacity, dtype=torch.int32, device=device)
        f32 = lambda: torch.empty(capacity, dtype=torch.float32, device=device)
        return HitBuffer(i32(), i32(), f32(), f32(), f32(), f32(), f32(), torch.zeros(1, dtype=torch.int64, device=device),
                         torch.empty(2 * n_hash, dtype=torch.int64, device=device) if n_hash else None)

    @staticmethod
    def allocate_chunked(n_pairs: int, hits_per_pair: float, n_hash: int = 0, device="cuda") -> "HitBuffer":
        """Chunked layout for one batch of n_pairs: a region of ceil(512 * hits_per_pair) entries per 512-pair chunk."""
        import torch
        n_chunks = (n_pairs + CHUNK_PAIRS - 1) // CHUNK_PAIRS
        cap = min(2048, max(1, int(np.ceil(CHUNK_PAIRS * hits_per_pair))))
        hb = HitBuffer.allocate(n_chunks * cap, n_hash, device)
        hb.chunk_fill = torch.zeros(n_chunks + 1, dtype=torch.int32, device=device)
        return hb

    def reset(self):
        """Zeroes the counters (before the next gpet_simulate into this buffer); enqueued on the current stream."""
        self.n_hits.zero_()
        if self.chunk_fill is not None:
            self.chunk_fill.zero_()

    @property
    def capacity(self) -> int:
        return int(self.history.numel())

    def struct(self) -> _Hits:
        return _Hits(self.history.data_ptr(), self.ids.data_ptr(), self.x.data_ptr(), self.y.data_ptr(), self.z.data_ptr(),
                     self.e_keV.data_ptr(), self.tof_ns.data_ptr(), self.capacity, self.n_hits.data_ptr(),
                     self.outcome_hash.data_ptr() if self.outcome_hash is not None else None,
                     self.chunk_fill.data_ptr() if self.chunk_fill is not None else None)

    def dropped(self) -> int:
        """Hits dropped for lack of room: dense layout n_hits - capacity, chunked layout the last chunk_fill word."""
        if self.chunk_fill is not None:
            return int(self.chunk_fill[-1].item())
        return max(0, self.count() - self.capacity)

    def count(self) -> int:
        return int(self.n_hits.item())

    def to_numpy(self):
        """Valid entries as numpy arrays (uint32 / float32), buffer order (chunked layout: chunk by chunk)."""
        if self.chunk_fill is not None:
            fill = self.chunk_fill[:-1].cpu().numpy().astype(np.int64)
            cap = self.capacity // len(fill)
            sel = (np.arange(cap)[None, :] < np.minimum(fill, cap)[:, None]).ravel()
            u = lambda t: t.cpu().numpy().view(np.uint32)[:len(sel)][sel]
            f = lambda t: t.cpu().numpy()[:len(sel)][sel]
            return dict(history=u(self.history), ids=u(self.ids), x=f(self.x), y=f(self.y), z=f(self.z), e_keV=f(self.e_keV),
                        tof_ns=f(self.tof_ns))
        n = min(self.count(), self.capacity)
        u = lambda t: t[:n].cpu().numpy().view(np.uint32)
        f = lambda t: t[:n].cpu().numpy()
        return dict(history=u(self.history), ids=u(self.ids), x=f(self.x), y=f(self.y), z=f(self.z), e_keV=f(self.e_keV),
                    tof_ns=f(self.tof_ns))


@dataclass
class SinglesBuffer:
    history: "torch.Tensor"
    ids: "torch.Tensor"
    x: "torch.Tensor"
    y: "torch.Tensor"
    z: "torch.Tensor"
    e_keV: "torch.Tensor"
    t_s: "torch.Tensor"
    n_singles: "torch.Tensor"

    @staticmethod
    def allocate(capacity: int, device="cuda") -> "SinglesBuffer":
        import torch
        i32 = lambda: torch.empty(capacity, dtype=torch.int32, device=device)
        f32 = lambda: torch.empty(capacity, dtype=torch.float32, device=device)
        return SinglesBuffer(i32(), i32(), f32(), f32(), f32(), f32(), torch.empty(capacity, dtype=torch.float64, device=device),
                             torch.zeros(1, dtype=torch.int64, device=device))

    def struct(self) -> _Singles:
        return _Singles(self.history.data_ptr(), self.ids.data_ptr(), self.x.data_ptr(), self.y.data_ptr(), self.z.data_ptr(),
                        self.e_keV.data_ptr(), self.t_s.data_ptr(), int(self.history.numel()), self.n_singles.data_ptr())

    def to_numpy(self):
        n = min(int(self.n_singles.item()), int(self.history.numel()))
        return dict(history=self.history[:n].cpu().numpy().view(np.uint32), ids=self.ids[:n].cpu().numpy().view(np.uint32),
                    x=self.x[:n].cpu().numpy(), y=self.y[:n].cpu().numpy(), z=self.z[:n].cpu().numpy(),
                    e_keV=self.e_keV[:n].cpu().numpy(), t_s=self.t_s[:n].cpu().numpy())


@dataclass
class CoincBuffer:
    ids_a: "torch.Tensor"
    ids_b: "torch.Tensor"
    history_a: "torch.Tensor"
    history_b: "torch.Tensor"
    e_a: "torch.Tensor"
    e_b: "torch.Tensor"
    dt_ns: "torch.Tensor"
    t_s: "torch.Tensor"
    n_coinc: "torch.Tensor"

    @staticmethod
    def allocate(capacity: int, device="cuda") -> "CoincBuffer":
        import torch
        i32 = lambda: torch.empty(capacity, dtype=torch.int32, device=device)
        f32 = lambda: torch.empty(capacity, dtype=torch.float32, device=device)
        return CoincBuffer(i32(), i32(), i32(), i32(), f32(), f32(), f32(), torch.empty(capacity, dtype=torch.float64, device=device),
                           torch.zeros(1, dtype=torch.int64, device=device))

    @property
    def capacity(self) -> int:
        return int(self.ids_a.numel())

    def struct(self) -> _Coinc:
        return _Coinc(self.ids_a.data_ptr(), self.ids_b.data_ptr(), self.history_a.data_ptr(), self.history_b.data_ptr(),
                      self.e_a.data_ptr(), self.e_b.data_ptr(), self.dt_ns.data_ptr(), self.t_s.data_ptr(),
                      int(self.ids_a.numel()), self.n_coinc.data_ptr())

    def to_numpy(self):
        n = min(int(self.n_coinc.item()), int(self.ids_a.numel()))
        u = lambda t: t[:n].cpu().numpy().view(np.uint32)
        return dict(ids_a=u(self.ids_a), ids_b=u(self.ids_b), history_a=u(self.history_a), history_b=u(self.history_b),
                    e_a=self.e_a[:n].cpu().numpy(), e_b=self.e_b[:n].cpu().numpy(), dt_ns=self.dt_ns[:n].cpu().numpy(),
                    t_s=self.t_s[:n].cpu().numpy())


def _stream_ptr(stream) -> Optional[int]:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream or None


# ----------------------------------------------------------------------------- the two hot calls
def gpet_simulate(geom: Geometry, mats: Materials, source: DeviceSource, first_history: int, n_pairs: int, seed: int,
                  hits: HitBuffer, stream=None) -> None:
    """Enqueues the transport of histories [first_history, first_history + n_pairs) on `stream` (default:
    torch's current stream).  Appends to `hits` (the caller zeroes hits.n_hits)."""
    hs = hits.struct()
    _check(lib().gpet_simulate(geom.ptr, mats.ptr, C.byref(source.struct), first_history, n_pairs, seed, C.byref(hs),
                               _stream_ptr(stream)))


def gpet_digitize_scratch_bytes(n_pairs: int, n_hits: int) -> int:
    return int(lib().gpet_digitize_scratch_bytes(n_pairs, n_hits))


def gpet_digitize(source: DeviceSource, seed: int, n_pairs_total: int, first_history: int, n_pairs: int, hits: HitBuffer,
                  n_hits: int, dig, scratch, singles: Optional[SinglesBuffer], coinc: CoincBuffer, stream=None) -> None:
    """dig: workloads.Digitizer; scratch: uint8 device tensor of >= gpet_digitize_scratch_bytes(n_pairs, n_hits)."""
    d = _Digitizer(dig.blur_fwhm_frac, dig.blur_ref_keV, dig.e_lo_keV, dig.e_hi_keV, dig.window_ns, dig.readout_level)
    hs, cs = hits.struct(), coinc.struct()
    ss = singles.struct() if singles is not None else None
    _check(lib().gpet_digitize(C.byref(source.struct), seed, n_pairs_total, first_history, n_pairs, C.byref(hs), n_hits,
                               C.byref(d), scratch.data_ptr(), int(scratch.numel()), C.byref(ss) if ss is not None else None,
                               C.byref(cs), _stream_ptr(stream)))


GPET_STATIC_SCRATCH_BYTES = 64 << 20


def gpet_digitize_static(source: DeviceSource, seed: int, n_pairs_total: int, first_history: int, n_pairs: int, hits: HitBuffer,
                         n_hits: int, dig, singles: Optional[SinglesBuffer], coinc: CoincBuffer, stream=None) -> None:
    """gpet_digitize without a scratch argument, for callers that cannot allocate device memory (the GPU is already
    committed to the host program's pool, or the call runs once per time slice where a cudaMalloc would stall the device).
    The workspace is a 64 MiB array built into libgpet.so: batches with gpet_digitize_scratch_bytes(n_pairs, n_hits) above
    GPET_STATIC_SCRATCH_BYTES raise GpetError; calls share the array, so keep them ordered on one stream; make the first
    call on a device during set-up.  Same output as gpet_digitize (see include/gpet.h)."""
    d = _Digitizer(dig.blur_fwhm_frac, dig.blur_ref_keV, dig.e_lo_keV, dig.e_hi_keV, dig.window_ns, dig.readout_level)
    hs, cs = hits.struct(), coinc.struct()
    ss = singles.struct() if singles is not None else None
    _check(lib().gpet_digitize_static(C.byref(source.struct), seed, n_pairs_total, first_history, n_pairs, C.byref(hs), n_hits,
                                      C.byref(d), C.byref(ss) if ss is not None else None, C.byref(cs), _stream_ptr(stream)))


GPET_WANT_HITS, GPET_WANT_SINGLES, GPET_WANT_HASH = 1, 2, 4


class HostOutputs:
    """Pinned host arrays for one batch's outputs (mirror of gpet_host_outputs) + the three counters."""

    def __init__(self, cap: int, n_pairs: int = 0, want_hits=False, want_singles=False, want_hash=False):
        import torch
        pin = lambda dt, n=cap: torch.empty(n, dtype=dt, pin_memory=True)
        self.cap = cap
        self.counts = torch.zeros(3, dtype=torch.int64, pin_memory=True)
        self.coinc = [pin(torch.int32) for _ in range(4)] + [pin(torch.float32) for _ in range(3)] + [pin(torch.float64)]
        self.hits = [pin(torch.int32) for _ in range(2)] + [pin(torch.float32) for _ in range(5)] if want_hits else None
        self.singles = ([pin(torch.int32) for _ in range(2)] + [pin(torch.float32) for _ in range(4)] + [pin(torch.float64)]
                        if want_singles else None)
        self.hash = pin(torch.int64, 2 * n_pairs) if want_hash else None
        cnt = self.counts
        out = _HostOutputs()
        if self.hits is not None:
            out.hits = _Hits(*[t.data_ptr() for t in self.hits], cap, cnt[0:].data_ptr(), None)
        else:
            out.hits = _Hits(None, None, None, None, None, None, None, 0, cnt[0:].data_ptr(), None)
        if self.hash is not None:
            out.hits.outcome_hash = self.hash.data_ptr()
        if self.singles is not None:
            out.singles = _Singles(*[t.data_ptr() for t in self.singles], cap, cnt[1:].data_ptr())
        else:
            out.singles = _Singles(None, None, None, None, None, None, None, 0, cnt[1:].data_ptr())
        out.coinc = _Coinc(*[t.data_ptr() for t in self.coinc], cap, cnt[2:].data_ptr())
        self.struct = out

    def want(self) -> int:
        return (GPET_WANT_HITS if self.hits is not None else 0) | (GPET_WANT_SINGLES if self.singles is not None else 0) | \
               (GPET_WANT_HASH if self.hash is not None else 0)

    def result(self):
        c = self.counts
        return dict(n_hits=int(c[0]), n_singles=int(c[1]), n_coinc=int(c[2]))

    def __getitem__(self, k):            # dict-style access used by older callers: host["coinc"], host["hits"], ...
        return getattr(self, k)


class Pipeline(_Handle):
    """gpet_pipeline: a stream of batches with host outputs, two in flight (include/gpet.h)."""
    _destroy = "gpet_pipeline_destroy"

    def __init__(self, geom: Geometry, mats: Materials, src, dig, n_pairs_total: int, max_pairs_per_batch: int,
                 hits_per_pair: float = 2.0, want: int = 0, n_slots: int = 2):
        self.geom, self.mats = geom, mats                              # keep the handles alive
        self.activity = gpet_activity_create(src.activity, src.dims) if src.kind == 1 else None
        self.phantom = None
        if src.kind == 1 and src.phantom_material is not None:
            self.phantom = np.ascontiguousarray(src.phantom_material, np.uint8)
        s = _source_struct(src, self.activity.ptr if self.activity else None, self.phantom.ctypes.data if self.phantom is not None else None)
        d = _Digitizer(dig.blur_fwhm_frac, dig.blur_ref_keV, dig.e_lo_keV, dig.e_hi_keV, dig.window_ns, dig.readout_level)
        out = C.c_void_p()
        _check(lib().gpet_pipeline_create(geom.ptr, mats.ptr, C.byref(s), C.byref(d), n_pairs_total, max_pairs_per_batch,
                                          hits_per_pair, want, n_slots, C.byref(out)))
        super().__init__(out.value)

    def submit(self, first_history: int, n_pairs: int, seed: int) -> None:
        _check(lib().gpet_pipeline_submit(self.ptr, first_history, n_pairs, seed))

    def collect(self, host: HostOutputs) -> dict:
        _check(lib().gpet_pipeline_collect(self.ptr, C.byref(host.struct)))
        return host.result()


def gpet_shutdown() -> None:
    _check(lib().gpet_shutdown())


def gpet_run_host(geom: Geometry, mats: Materials, src, n_pairs_total: int, first_history: int, n_pairs: int, seed: int, dig,
                  hits_per_pair: float = 2.0, want_hits: bool = False, want_singles: bool = False, want_hash: bool = False,
                  host=None):
    """Whole path with HOST outputs (pinned torch tensors, reused when `host` is passed back in).
    src: workloads.Source (its phantom map is a host array here).  Returns (HostOutputs, counts)."""
    cap = int(n_pairs * hits_per_pair) + 1024
    if host is None or host.cap < cap:
        host = HostOutputs(cap, n_pairs, want_hits, want_singles, want_hash)
    activity = gpet_activity_create(src.activity, src.dims) if src.kind == 1 else None
    ph = None
    if src.kind == 1 and src.phantom_material is not None:
        ph = np.ascontiguousarray(src.phantom_material, np.uint8)
    s = _source_struct(src, activity.ptr if activity else None, ph.ctypes.data if ph is not None else None)
    d = _Digitizer(dig.blur_fwhm_frac, dig.blur_ref_keV, dig.e_lo_keV, dig.e_hi_keV, dig.window_ns, dig.readout_level)
    _check(lib().gpet_run_host(geom.ptr, mats.ptr, C.byref(s), n_pairs_total, first_history, n_pairs, seed, C.byref(d),
                               hits_per_pair, C.byref(host.struct)))
    return host, host.result()
