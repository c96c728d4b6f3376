"""Seeded, synthetic inputs shared by the CUDA path and the oracle (and by nothing else).

This module holds the *input recipe* only: scanner descriptors, attenuation tables, the hot-rod
phantom and the per-config run parameters of BASELINE.json's C0..C4.
It contains none of the method's arithmetic (no transport, no sampling, no lattice lookup, no
digitizer): both sides receive these plain arrays / dataclasses and marshal them into their own
structures.  Citations: PAPER.md:33-37 (what a user configures), PAPER.md:47 (pitch = crystal +
gap), PAPER.md:61-67 (sources, windows), BASELINE.json configs[0..4] (numbers).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List, Optional, Sequence, Tuple

import numpy as np

F18_HALF_LIFE_S = 109.77 * 60.0     # 18F (1.6e8 atoms <-> 1.70e-2 MBq)
# physical constants used to build the synthetic tables (BASELINE.json C0)
R_E_CM = 2.8179403262e-13          # classical electron radius [cm]
ME_C2_KEV = 510.99895              # electron rest energy [keV]
N_E_LYSO_CM3 = 2.05e24             # BASELINE C0
N_E_WATER_CM3 = 3.3428e23          # water, 1 g/cm3
E_MIN_KEV, E_STEP_KEV, N_ENERGIES = 10.0, 1.0, 502   # 10..511 keV on a 1 keV grid


# ----------------------------------------------------------------------------- plain data
@dataclass(frozen=True)
class Layer:
    """One crystal layer, front (index 0) to back.  PAPER.md:35-37."""
    n_crystals: Tuple[int, int]            # along local u (tangential), v (axial)
    pitch_mm: Tuple[float, float]          # crystal size + reflector gap
    reflector_mm: Tuple[float, float]      # gap between neighbours, half on each side of a cell
    offset_mm: Tuple[float, float]         # lattice origin relative to the module's low corner
    depth_mm: float
    gap_before_mm: float = 0.0             # inter-layer gap in front of this layer
    crystal_material: int = 0
    gap_material: int = -1                 # -1 = vacuum


@dataclass(frozen=True)
class Geometry:
    """Panel -> module -> layer -> crystal hierarchy.  PAPER.md:33-41 (Fig. 1)."""
    n_panels: int
    layers: Tuple[Layer, ...]
    n_modules: Tuple[int, int] = (1, 1)
    module_size_mm: Tuple[float, float] = (0.0, 0.0)
    module_pitch_mm: Tuple[float, float] = (0.0, 0.0)
    # repetition mode: a ring about z
    ring_inner_radius_mm: float = 0.0
    ring_first_angle_deg: float = 0.0
    # non-repetition mode: explicit poses, n_panels x 12 (front-face centre, u, v, w)
    panel_pose: Optional[np.ndarray] = None


@dataclass(frozen=True)
class Source:
    kind: int = 0                          # 0 point, 1 voxel activity map, 2 pencil beam (test rays)
    pos_mm: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    acolinearity_fwhm_deg: float = 0.0
    activity_bq: float = 1.0e6
    pairs_per_time_slice: int = 0          # 0 = one slice holding all pairs
    activity: Optional[np.ndarray] = None           # float32 [nz, ny, nx] (x fastest)
    phantom_material: Optional[np.ndarray] = None   # uint8   [nz, ny, nx]; 0 vacuum, k>0 -> material k-1
    phantom_majorant_material: int = -1             # material whose mu_tot bounds every phantom voxel
    dims: Tuple[int, int, int] = (0, 0, 0)          # nx, ny, nz
    voxel_mm: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    origin_mm: Tuple[float, float, float] = (0.0, 0.0, 0.0)   # low corner of voxel (0,0,0)
    beam_dir: Tuple[float, float, float] = (1.0, 0.0, 0.0)    # kind 2: direction of photon A (B is opposite)
    positron_fwhm_mm: float = 0.0          # 0 = annihilation at the emission site, as in the paper
    half_life_s: float = 0.0               # > 0: decay law over duration_s, activity_bq = initial activity
    duration_s: float = 0.0


@dataclass(frozen=True)
class Digitizer:
    blur_fwhm_frac: float = 0.15
    blur_ref_keV: float = 511.0
    e_lo_keV: float = 350.0
    e_hi_keV: float = 650.0
    window_ns: float = 4.0
    readout_level: int = 1                 # 0 crystal, 1 module, 2 panel


@dataclass(frozen=True)
class Tables:
    """mu tables, 1/mm, fp32, [n_materials][n_energies]; the same arrays go to both sides."""
    e_min_keV: float
    e_step_keV: float
    mu_pe: np.ndarray
    mu_compton: np.ndarray
    mu_rayleigh: np.ndarray

    @property
    def n_materials(self) -> int:
        return int(self.mu_pe.shape[0])

    @property
    def n_energies(self) -> int:
        return int(self.mu_pe.shape[1])


@dataclass(frozen=True)
class Run:
    """One (geometry, source, seed, n_pairs) case of a config."""
    name: str
    geometry: Geometry
    source: Source
    n_pairs: int
    seed: int
    digitizer: Digitizer = field(default_factory=Digitizer)


# ----------------------------------------------------------------------------- tables
def kn_total_cross_section_cm2(e_keV: np.ndarray) -> np.ndarray:
    """Closed-form total Klein-Nishina cross-section per free electron (fp64)."""
    k = np.asarray(e_keV, dtype=np.float64) / ME_C2_KEV
    l = np.log1p(2.0 * k)
    t1 = (1.0 + k) / k ** 2 * (2.0 * (1.0 + k) / (1.0 + 2.0 * k) - l / k)
    t2 = l / (2.0 * k)
    t3 = (1.0 + 3.0 * k) / (1.0 + 2.0 * k) ** 2
    return 2.0 * math.pi * R_E_CM ** 2 * (t1 + t2 - t3)


def energy_grid() -> np.ndarray:
    return E_MIN_KEV + E_STEP_KEV * np.arange(N_ENERGIES, dtype=np.float64)


def tables(with_water: bool = True) -> Tables:
    """Material 0 = LYSO (BASELINE C0 formulas); material 1 = water (C4).

    Computed in fp64 and rounded to fp32 once; the rounded arrays are *the* input.
    """
    e = energy_grid()
    sig = kn_total_cross_section_cm2(e)                       # cm^2 per electron
    pe = [0.029 * (511.0 / e) ** 3]
    co = [N_E_LYSO_CM3 * sig * 0.1]                           # 1/cm -> 1/mm
    ra = [0.002 * (511.0 / e) ** 2]
    if with_water:
        pe.append(2.0e-6 * (511.0 / e) ** 3)                  # synthetic, same shape as C0's
        co.append(N_E_WATER_CM3 * sig * 0.1)
        ra.append(np.zeros_like(e))                           # C4 lists only KN + photoelectric
    f32 = lambda rows: np.ascontiguousarray(np.stack(rows).astype(np.float32))
    return Tables(E_MIN_KEV, E_STEP_KEV, f32(pe), f32(co), f32(ra))


# ----------------------------------------------------------------------------- geometries
def _lyso_layer(n, pitch, gap, depth, offset=(0.0, 0.0), gap_before=0.0) -> Layer:
    return Layer((n, n) if isinstance(n, int) else tuple(n), (pitch, pitch), (gap, gap),
                 tuple(offset), depth, gap_before, 0, -1)


def geometry_c0() -> Geometry:
    """C0: one flat panel = one module of 8x8 crystals, 1.5 mm pitch (1.4 + 0.1), 10 mm deep,
    front-face centre at (50, 0, 0) facing the origin."""
    pose = np.array([[50.0, 0.0, 0.0,   0.0, 1.0, 0.0,   0.0, 0.0, 1.0,   1.0, 0.0, 0.0]], np.float32)
    return Geometry(1, (_lyso_layer(8, 1.5, 0.1, 10.0),), (1, 1), (12.0, 12.0), (12.0, 12.0),
                    panel_pose=pose)


def _ring(layers: Sequence[Layer]) -> Geometry:
    """12 panels on a 55 mm inner radius, 2 (tangential) x 4 (axial) modules of 16 mm."""
    return Geometry(12, tuple(layers), (2, 4), (16.0, 16.0), (16.0, 16.0),
                    ring_inner_radius_mm=55.0, ring_first_angle_deg=0.0)


def geometry_c1() -> Geometry:
    return _ring([_lyso_layer(16, 1.0, 0.1, 10.0)])


def geometry_c2(gap_mm: float = 0.1) -> Geometry:
    """Aligned split: 5 mm + gap + 5 mm (BASELINE C2; gap 0 is the paper's own split)."""
    return _ring([_lyso_layer(16, 1.0, 0.1, 5.0), _lyso_layer(16, 1.0, 0.1, 5.0, gap_before=gap_mm)])


def geometry_c3() -> Geometry:
    """Offset dual layer: 15x15 x 6 mm front, shifted half a pitch on both axes, 0.1 mm gap,
    16x16 x 4 mm back (BASELINE C3; construction as PAPER.md:47)."""
    return _ring([_lyso_layer(15, 1.0, 0.1, 6.0, offset=(0.5, 0.5)),
                  _lyso_layer(16, 1.0, 0.1, 4.0, gap_before=0.1)])


def _paper_ring(layers: Sequence[Layer]) -> Geometry:
    """The paper's own scanner: 10 panels at R = 85 mm, six axial modules of 51 mm with 7 mm gaps
    (panel 10 x 51 x 341 mm), 1.0 mm pitch = 0.92 mm crystal + 0.08 mm air.  Context only."""
    return Geometry(10, tuple(layers), (1, 6), (51.0, 51.0), (51.0, 58.0), ring_inner_radius_mm=85.0)


def geometry_paper_1cl() -> Geometry:
    """H2RSPET-1CL: one layer of 51 x 51 crystals, 10 mm deep."""
    return _paper_ring([Layer((51, 51), (1.0, 1.0), (0.08, 0.08), (0.0, 0.0), 10.0)])


def geometry_paper_split() -> Geometry:
    """H2RSPET-1CL-split: two radially connected 5 mm crystals (no gap)."""
    return _paper_ring([Layer((51, 51), (1.0, 1.0), (0.08, 0.08), (0.0, 0.0), 5.0),
                        Layer((51, 51), (1.0, 1.0), (0.08, 0.08), (0.0, 0.0), 5.0)])


def geometry_paper_2cl() -> Geometry:
    """H2RSPET-2CL: inner 50 x 50 layer shifted by half a pitch over an outer 51 x 51 layer, 5 mm each."""
    return _paper_ring([Layer((50, 50), (1.0, 1.0), (0.08, 0.08), (0.5, 0.5), 5.0),
                        Layer((51, 51), (1.0, 1.0), (0.08, 0.08), (0.0, 0.0), 5.0)])


# ----------------------------------------------------------------------------- hot-rod phantom (C4)
ROD_DIAMETERS_MM = (0.75, 1.0, 1.25, 1.5, 1.75, 2.0)


def hot_rod_centres(r_max_mm: float = 13.0) -> List[Tuple[float, float, float]]:
    """(x, y, diameter) of every rod.  Layout is this build's (BASELINE C4 gives only diameters and the
    2d spacing): sector s has its bisector at 60*s + 30 deg, a triangular lattice with the apex
    towards the axis at radius 2d, row j at radius 2d + j*sqrt(3)*d with j+1 rods spaced 2d; a row
    is kept while all its rods lie inside r_max."""
    rods = []
    for s, d in enumerate(ROD_DIAMETERS_MM):
        th = math.radians(60.0 * s + 30.0)
        ex, ey = math.cos(th), math.sin(th)          # along the bisector
        px, py = -ey, ex                             # across it
        j = 0
        while True:
            r = 2.0 * d + j * math.sqrt(3.0) * d
            row = [(r * ex + (2.0 * i - j) * d * px, r * ey + (2.0 * i - j) * d * py) for i in range(j + 1)]
            if any(math.hypot(x, y) + 0.5 * d > r_max_mm for x, y in row):
                break
            rods += [(x, y, d) for x, y in row]
            j += 1
    return rods


def hot_rod_phantom(n: int = 128, voxel_mm: float = 0.25):
    """128^3 x 0.25 mm grid centred on the origin; water cylinder d=30 x 20 mm along z (material
    value 2 = material index 1 = water), vacuum elsewhere; activity 1.0 in voxels whose centre is
    inside a rod and |z| < 10 mm.  Returns (activity f32 [nz,ny,nx], material u8 [nz,ny,nx], origin)."""
    origin = -0.5 * n * voxel_mm
    c = origin + (np.arange(n) + 0.5) * voxel_mm
    x, y = np.meshgrid(c, c, indexing="xy")              # [ny, nx]
    in_z = np.abs(c) < 10.0
    water2d = (x * x + y * y) < 15.0 ** 2
    rod2d = np.zeros_like(water2d)
    for rx, ry, d in hot_rod_centres():
        rod2d |= ((x - rx) ** 2 + (y - ry) ** 2) < (0.5 * d) ** 2
    material = np.zeros((n, n, n), np.uint8)
    activity = np.zeros((n, n, n), np.float32)
    material[in_z] = np.where(water2d, 2, 0).astype(np.uint8)
    activity[in_z] = rod2d.astype(np.float32)
    return activity, material, (origin, origin, origin)


# ----------------------------------------------------------------------------- the paper's Derenzo phantom
DERENZO_DIAMETERS_MM = (0.3, 0.4, 0.5, 0.625, 0.75, 1.0)
DERENZO_ROD_COUNTS = (6, 10, 15, 21, 28, 36)           # triangular numbers: 3 .. 8 rows
DERENZO_ACTIVITY_BQ_PER_MM3 = 92.1                     # 9.21e-5 MBq/mm3
DERENZO_BOX_MM = 40.25


def derenzo_rod_centres(apex_radius_mm: float = 2.5) -> List[Tuple[float, float, float]]:
    """(x, y, diameter) of the 116 rods: six triangular sectors forming a hexagon, sector s on the bisector at 60 s + 30
    degrees, rods of one diameter d per sector on a triangular lattice with centre spacing 2 d, apex towards
    the axis.  The paper gives diameters, counts and spacing; the apex radius (2.5 mm) is this build's choice."""
    rods = []
    for s, (d, n) in enumerate(zip(DERENZO_DIAMETERS_MM, DERENZO_ROD_COUNTS)):
        rows = int(round((math.sqrt(8 * n + 1) - 1) / 2))
        assert rows * (rows + 1) // 2 == n
        th = math.radians(60.0 * s + 30.0)
        ex, ey = math.cos(th), math.sin(th)
        px, py = -ey, ex
        for j in range(rows):
            r = apex_radius_mm + j * math.sqrt(3.0) * d
            rods += [(r * ex + (2.0 * i - j) * d * px, r * ey + (2.0 * i - j) * d * py, d) for i in range(j + 1)]
    return rods


def derenzo_phantom(voxel_mm: float = 0.125, z_voxel_mm: float = 0.25):
    """Water box of 40.25 mm on a grid of 0.125 x 0.125 x 0.25 mm voxels (322 x 322 x 161: the transaxial
    pitch resolves the 0.3 mm rods, the axial one is the paper's reconstruction pitch); activity 1.0 in voxels whose centre
    lies in a rod and |z| < 10 mm (2 cm rods).  Returns (activity f32 [nz,ny,nx], material u8, origin, dims, voxel sizes)."""
    n = int(round(DERENZO_BOX_MM / voxel_mm)); nz = int(round(DERENZO_BOX_MM / z_voxel_mm))
    o = -0.5 * DERENZO_BOX_MM
    c = o + (np.arange(n) + 0.5) * voxel_mm
    cz = o + (np.arange(nz) + 0.5) * z_voxel_mm
    x, y = np.meshgrid(c, c, indexing="xy")
    rod2d = np.zeros((n, n), bool)
    for rx, ry, d in derenzo_rod_centres():
        rod2d |= ((x - rx) ** 2 + (y - ry) ** 2) < (0.5 * d) ** 2
    activity = np.zeros((nz, n, n), np.float32)
    activity[np.abs(cz) < 10.0] = rod2d.astype(np.float32)
    material = np.full((nz, n, n), 2, np.uint8)                        # water (material index 1) everywhere in the box
    return activity, material, (o, o, o), (n, n, nz), (voxel_mm, voxel_mm, z_voxel_mm)


def derenzo_activity_bq() -> float:
    """Total activity of the rods: sum n_i pi d_i^2 / 4 x 20 mm x 9.21e-5 MBq/mm3 = 95.26 kBq."""
    vol = sum(n * math.pi * d * d / 4.0 * 20.0 for d, n in zip(DERENZO_DIAMETERS_MM, DERENZO_ROD_COUNTS))
    return vol * DERENZO_ACTIVITY_BQ_PER_MM3


def source_derenzo(duration_s: float = 12.0) -> Source:
    """The Derenzo source of the paper's Table 1 (12 s of 18F decay): voxel activity map inside the water
    box, decay law on [R34], positron range off, 0.5 deg acolinearity as in BASELINE's ring configs."""
    act, mat, org, dims, vox = derenzo_phantom()
    return Source(1, (0.0, 0.0, 0.0), 0.5, derenzo_activity_bq(), 0, act, mat, 1, dims, vox, org,
                  half_life_s=F18_HALF_LIFE_S, duration_s=duration_s)


def source_point(pos=(0.0, 0.0, 0.0), acolinearity_fwhm_deg=0.5, activity_bq=1.0e6) -> Source:
    return Source(0, tuple(float(v) for v in pos), acolinearity_fwhm_deg, activity_bq)


def source_beam(pos, direction, acolinearity_fwhm_deg=0.0, activity_bq=1.0e6) -> Source:
    """Deterministic test ray: photon A along `direction`, photon B opposite (north_star: indexing on
    deterministic test rays)."""
    return Source(2, tuple(float(v) for v in pos), acolinearity_fwhm_deg, activity_bq,
                  beam_dir=tuple(float(v) for v in direction))


def source_hot_rods(pairs_per_time_slice: int = 0) -> Source:
    act, mat, org = hot_rod_phantom()
    return Source(1, (0.0, 0.0, 0.0), 0.5, 1.0e6, pairs_per_time_slice, act, mat, 1,
                  (128, 128, 128), (0.25, 0.25, 0.25), org)


# ----------------------------------------------------------------------------- configs C0..C4
def config_runs(name: str, n_pairs: Optional[int] = None) -> List[Run]:
    """All runs of one BASELINE config.  n_pairs overrides the full size."""
    name = name.upper()
    if name == "C0":
        return [Run("C0", geometry_c0(), source_point(acolinearity_fwhm_deg=0.0), n_pairs or 100_000, 1)]
    if name == "C1":
        return [Run("C1", geometry_c1(), source_point(), n_pairs or 10_000_000, 2)]
    if name == "C2":
        return [Run(f"C2_x{int(x)}", geometry_c2(), source_point((x, 0.0, 0.0)), n_pairs or 10_000_000, 30 + i)
                for i, x in enumerate((0.0, 5.0, 10.0, 25.0, 50.0))]
    if name == "C3":
        runs, i = [], 0
        for z in (0.0, 16.0):
            for x in range(0, 55, 5):
                runs.append(Run(f"C3_x{x}_z{int(z)}", geometry_c3(), source_point((float(x), 0.0, z)),
                                n_pairs or 10_000_000, 400 + i))
                i += 1
        return runs
    if name == "C4":
        n = n_pairs or 1_000_000_000
        return [Run("C4", geometry_c3(), source_hot_rods(pairs_per_time_slice=max(1, n // 16)), n, 5)]
    if name in ("P1", "P2", "P3"):      # the paper's own scanners with a centred point source (context)
        geom = {"P1": geometry_paper_1cl, "P2": geometry_paper_split, "P3": geometry_paper_2cl}[name]()
        dig = Digitizer(0.16, 511.0, 350.0, 700.0, 3.0, 1)
        return [Run(name, geom, source_point(), n_pairs or 10_000_000, 60 + int(name[1]), dig)]
    if name in ("T1", "T2", "T3"):      # the paper's Table 1: Derenzo source, 12 s of decay, on its three scanners
        geom = {"T1": geometry_paper_1cl, "T2": geometry_paper_split, "T3": geometry_paper_2cl}[name]()
        src = source_derenzo()
        lam = math.log(2.0) / src.half_life_s
        n = n_pairs or int(round(src.activity_bq / lam * -math.expm1(-lam * src.duration_s)))
        return [Run(name, geom, src, n, 70 + int(name[1]), Digitizer(0.16, 511.0, 350.0, 700.0, 3.0, 1))]
    raise ValueError(f"unknown config {name!r}")


def with_pairs(run: Run, n_pairs: int) -> Run:
    return replace(run, n_pairs=n_pairs)
