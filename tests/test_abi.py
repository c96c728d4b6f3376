"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/gpet.h declares, and its
host logic (descriptor validation, ring placement, error reporting) behaves as documented.  No kernel runs."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import gpet_oracle as O
from paper_2603_07327_b200 import api, build, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    build.build()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "gpet.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gpet_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert "gpet_simulate" in names and "gpet_digitize" in names and len(names) >= 14
    lib = ctypes.CDLL(api.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in gpet.h but not exported"
    assert sorted(api.EXPORTS) == names


def test_binding_structs_match_the_header_layout(tmp_path):
    """sizeof and the offset of the last member of every struct of gpet.h, as gcc lays them out, against the ctypes mirrors
    of the binding: a header edit cannot silently skew the binding."""
    import subprocess
    pairs = [("gpet_layer_desc", "gap_material", api._LayerDesc), ("gpet_geometry_desc", "layers", api._GeometryDesc),
             ("gpet_source", "duration_s", api._Source), ("gpet_hits", "chunk_fill", api._Hits), ("gpet_digitizer", "readout_level", api._Digitizer),
             ("gpet_singles", "n_singles", api._Singles), ("gpet_coincidences", "n_coinc", api._Coinc), ("gpet_host_outputs", "coinc", api._HostOutputs)]
    src = tmp_path / "sz.c"
    body = "".join(f'printf("%zu %zu\\n", sizeof({c}), offsetof({c}, {m}));' for c, m, _ in pairs)
    src.write_text(f'#include <stdio.h>\n#include <stddef.h>\n#include "gpet.h"\nint main(void){{{body}return 0;}}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)])
    out = subprocess.check_output([str(exe)], text=True).split()
    for k, (c, m, t) in enumerate(pairs):
        assert ctypes.sizeof(t) == int(out[2 * k]) and getattr(t, m).offset == int(out[2 * k + 1]), (c, out[2 * k:2 * k + 2])


def test_ring_placement_equals_the_oracles_bit_for_bit():
    for geom in (W.geometry_c1(), W.geometry_paper_1cl(), W.Geometry(7, W.geometry_c1().layers, (2, 4), (16.0, 16.0), (16.0, 16.0),
                                                                      ring_inner_radius_mm=40.0, ring_first_angle_deg=12.5)):
        g = api.gpet_geometry_create(geom)
        want = O.ring_poses(geom.n_panels, geom.ring_inner_radius_mm, geom.ring_first_angle_deg)
        for p in range(geom.n_panels):
            assert np.array_equal(api.gpet_geometry_panel_pose(g, p).view(np.uint32), want[p].view(np.uint32))
    pose = api.gpet_geometry_panel_pose(api.gpet_geometry_create(W.geometry_c1()), 3)   # 90 degrees: exact zeros
    assert pose[0] == 0.0 and pose[1] == 55.0 and pose[3] == -1.0 and pose[4] == 0.0


def test_explicit_poses_are_kept_verbatim():
    g0 = W.geometry_c0()
    g = api.gpet_geometry_create(g0)
    assert np.array_equal(api.gpet_geometry_panel_pose(g, 0), g0.panel_pose[0])
    with pytest.raises(api.GpetError):
        api.gpet_geometry_panel_pose(g, 1)


@pytest.mark.parametrize("bad", [
    dict(n=(17, 16)),                      # lattice wider than its module
    dict(offset=(0.5, 0.0)),               # shifted 16x16 overhangs (SURVEY O9's alternative is rejected)
    dict(depth=0.0), dict(pitch=(0.0, 1.0)), dict(reflector=(1.0, 0.1)), dict(material=9),
])
def test_geometry_validation(bad):
    l = W.Layer(bad.get("n", (16, 16)), bad.get("pitch", (1.0, 1.0)), bad.get("reflector", (0.1, 0.1)), bad.get("offset", (0.0, 0.0)),
                bad.get("depth", 10.0), 0.0, bad.get("material", 0))
    with pytest.raises(api.GpetError, match="error -2"):
        api.gpet_geometry_create(W.Geometry(12, (l,), (2, 4), (16.0, 16.0), (16.0, 16.0), ring_inner_radius_mm=55.0))
    # the oracle rejects the same descriptors
    if "material" not in bad:
        with pytest.raises(ValueError):
            O.locate(W.Geometry(12, (l,), (2, 4), (16.0, 16.0), (16.0, 16.0), ring_inner_radius_mm=55.0), np.zeros((1, 3), np.float32))


def test_geometry_count_limits():
    l = W.geometry_c1().layers
    for kw in (dict(n_panels=64), dict(n_panels=0)):
        with pytest.raises(api.GpetError):
            api.gpet_geometry_create(W.Geometry(kw["n_panels"], l, (2, 4), (16.0, 16.0), (16.0, 16.0), ring_inner_radius_mm=55.0))
    with pytest.raises(api.GpetError):
        api.gpet_geometry_create(W.Geometry(12, l * 5, (2, 4), (16.0, 16.0), (16.0, 16.0), ring_inner_radius_mm=55.0))
    api.gpet_geometry_create(W.Geometry(63, l, (2, 4), (16.0, 16.0), (16.0, 16.0), ring_inner_radius_mm=400.0))


def test_table_validation_needs_no_kernel():
    t = W.tables()
    bad = W.Tables(t.e_min_keV, t.e_step_keV, -t.mu_pe, t.mu_compton, t.mu_rayleigh)
    with pytest.raises(api.GpetError, match="error -3"):
        api.gpet_materials_load(bad)
    nan = t.mu_pe.copy(); nan[0, 5] = np.nan
    with pytest.raises(api.GpetError, match="error -3"):
        api.gpet_materials_load(W.Tables(t.e_min_keV, t.e_step_keV, nan, t.mu_compton, t.mu_rayleigh))


def test_product_path_fails_loudly_without_a_gpu(tables):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(api.GpetError, match="error -5"):       # GPET_E_CUDA, never a CPU fallback
        api.gpet_materials_load(tables)
    g = api.gpet_geometry_create(W.geometry_c0())
    with pytest.raises(api.GpetError, match="error -5"):
        api.gpet_geometry_locate(g, np.zeros((4, 3), np.float32))


def test_scratch_size_is_monotone():
    a = api.gpet_digitize_scratch_bytes(1000, 800)
    b = api.gpet_digitize_scratch_bytes(10_000_000, 8_000_000)
    assert 0 < a < b < 2 * 1024 ** 3


def test_open_faces_of_panel_boxes():
    """A face is open when no other panel has a point beyond it (transport then skips the panel search for photons leaving
    through it).  Checked against a brute-force sampling of every other panel box, on a ring, a lone panel and two
    facing panels; a closed face must never be reported open."""
    rng = np.random.default_rng(3)
    facing = np.array([[30, 0, 0, 0, 1, 0, 0, 0, 1, 1, 0, 0], [-30, 0, 0, 0, -1, 0, 0, 0, 1, -1, 0, 0]], np.float32)
    two = W.Geometry(2, W.geometry_c0().layers, (1, 1), (12.0, 12.0), (12.0, 12.0), panel_pose=facing)
    for geom in (W.geometry_c1(), W.geometry_c3(), W.geometry_c0(), two, W.geometry_paper_1cl()):
        g = api.gpet_geometry_create(geom)
        n = geom.n_panels
        poses = np.stack([api.gpet_geometry_panel_pose(g, p).astype(np.float64) for p in range(n)])
        W_, H_ = [(geom.n_modules[a] - 1) * geom.module_pitch_mm[a] + geom.module_size_mm[a] for a in (0, 1)]
        D_ = sum(l.depth_mm + l.gap_before_mm for l in geom.layers)
        lo, hi = np.array([-W_ / 2, -H_ / 2, 0.0]), np.array([W_ / 2, H_ / 2, D_])
        for p in range(n):
            mask = api.gpet_geometry_open_faces(g, p)
            o, axes = poses[p, :3], poses[p, 3:].reshape(3, 3)
            beyond = np.zeros(6, bool)
            for q in range(n):
                if q == p:
                    continue
                loc = rng.uniform(lo, hi, (4000, 3))
                pts = poses[q, :3] + loc @ poses[q, 3:].reshape(3, 3)
                l = (pts - o) @ axes.T
                for k in range(3):
                    beyond[2 * k + 1] |= bool((l[:, k] > hi[k]).any())
                    beyond[2 * k] |= bool((l[:, k] < lo[k]).any())
            for f in range(6):
                if beyond[f]:
                    assert not (mask >> f) & 1, (p, f)
            if n == 1:
                assert mask == 63
        if geom.panel_pose is None:                                   # rings: the back face (high w) is open, the front is not
            assert all((api.gpet_geometry_open_faces(g, p) >> 5) & 1 and not (api.gpet_geometry_open_faces(g, p) >> 4) & 1 for p in range(n))
    assert api.gpet_geometry_open_faces(api.gpet_geometry_create(two), 0) == 0b100000   # only the back: the side faces are flush with the other panel's


def test_bore_radius_of_planar_detectors():
    """The acceptance pre-test's radius: no panel point may lie closer to the z axis (checked by sampling every box), and it is
    the front-face apothem for the rings; detectors that are not planar report none."""
    rng = np.random.default_rng(4)
    for geom, expect in ((W.geometry_c1(), 55.0), (W.geometry_c3(), 55.0), (W.geometry_paper_2cl(), 85.0), (W.geometry_c0(), 50.0)):
        g = api.gpet_geometry_create(geom)
        r = api.gpet_geometry_bore_radius(g)
        assert abs(r - (expect - 1e-3)) < 1e-4
        W_, H_ = [(geom.n_modules[a] - 1) * geom.module_pitch_mm[a] + geom.module_size_mm[a] for a in (0, 1)]
        D_ = sum(l.depth_mm + l.gap_before_mm for l in geom.layers)
        for p in range(geom.n_panels):
            pose = api.gpet_geometry_panel_pose(g, p).astype(np.float64)
            loc = rng.uniform([-W_ / 2, -H_ / 2, 0.0], [W_ / 2, H_ / 2, D_], (4000, 3))
            pts = pose[:3] + loc @ pose[3:].reshape(3, 3)
            assert np.hypot(pts[:, 0], pts[:, 1]).min() >= r
    from test_oracle_pins import tiny_scanner
    assert api.gpet_geometry_bore_radius(api.gpet_geometry_create(tiny_scanner())) <= 0.0     # panels off the z = 0 plane: not planar


def test_bench_roofline_table_matches_the_audit():
    """bench.py's algorithmic instruction counts are the audited ones (tests/golden/alg_instr_per_pair.json, written by
    tests/golden/alg_instr.py from the oracle's event counts); C1 alone keeps SURVEY 8(d)'s 740."""
    import importlib.util, json
    spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec); spec.loader.exec_module(bench)
    audit = json.load(open(os.path.join(ROOT, "tests", "golden", "alg_instr_per_pair.json")))
    name = {"C2": "C2_x0", "C3": "C3_x0_z0", "C4": "C4", "P1": "P1", "T1": "T1", "T2": "T2", "T3": "T3"}
    for k, v in name.items():
        assert abs(bench.ALG_INSTR_PER_PAIR[k] - audit[v]["instr_per_pair"]) < 0.05, k
    assert bench.ALG_INSTR_PER_PAIR["C1"] == 740.0 and abs(audit["C1"]["instr_per_pair"] - 700.0) < 10.0
    assert abs(bench.AUDITED_C1 - audit["C1"]["instr_per_pair"]) < 0.05      # roofline.frac_audited of the C1 line


def test_multiply_high_division_is_exact(tmp_path):
    """gpet_device.cuh: floor(n / d) = umulhi(n, magic) >> shift for every 0 <= n < 2^31 -- the lattice lookup's crystal and
    module indices [R7] and the voxel index -> (ix, iy, iz) split [R13] rest on it.  qdiv_make is the library's own (the
    shim includes the header); umulhi is by definition the high word of the 64-bit product.  Checked for every divisor the
    workloads C0-C4, P1-P3, T1-T3 produce (pitches in 2^-20 mm units, grid sizes) and for random divisors, each at random
    numerators and at the numerators where a wrong magic shows first: multiples of d, one below them, and the top of the
    range."""
    import subprocess
    HERE = os.path.dirname(os.path.abspath(__file__))
    so = str(tmp_path / "qdiv_host.so")
    subprocess.check_call(["nvcc", "-O1", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC",
                           "-I", os.path.join(ROOT, "paper_2603_07327_b200", "csrc"), "-o", so, os.path.join(HERE, "golden", "qdiv_host.cu")])
    shim = ctypes.CDLL(so)
    rng = np.random.default_rng(11)
    used = set()
    for cfg in ("C0", "C1", "C2", "C3", "C4", "P1", "P2", "P3", "T1", "T2", "T3"):
        for r in W.config_runs(cfg, 1000):
            g = r.geometry
            used.update(int(round(float(p) * 2 ** 20)) for p in g.module_pitch_mm)
            for lay in g.layers:
                used.update(int(round(float(p) * 2 ** 20)) for p in lay.pitch_mm)
            if r.source.kind == 1:
                nx, ny = int(r.source.dims[0]), int(r.source.dims[1])
                used.update((nx, nx * ny))
    used = {d for d in used if 2 <= d < 2 ** 31}
    assert len(used) >= 6
    d = np.concatenate([np.array(sorted(used), np.uint32), np.array([2, 3, 5, 7, 2 ** 16, 2 ** 16 + 1, 2 ** 30, 2 ** 31 - 1], np.uint32),
                        2 ** np.arange(1, 31, dtype=np.uint32), 2 ** np.arange(2, 31, dtype=np.uint32) - 1, 2 ** np.arange(1, 31, dtype=np.uint32) + 1,
                        rng.integers(2, 2 ** 31, 20_000, dtype=np.uint64).astype(np.uint32),
                        rng.integers(2, 2 ** 12, 2_000, dtype=np.uint64).astype(np.uint32)])
    magic, shift = np.zeros(len(d), np.uint32), np.zeros(len(d), np.uint32)
    vp = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    shim.qdiv_make_batch(vp(d), len(d), vp(magic), vp(shift))
    D, M, S = d.astype(np.uint64)[:, None], magic.astype(np.uint64)[:, None], shift.astype(np.uint64)[:, None]
    top = np.uint64(2 ** 31 - 1)
    k = rng.integers(1, 2 ** 31, (len(d), 64), dtype=np.uint64) // D + np.uint64(1)          # multiples k d spread over the range
    n = np.concatenate([rng.integers(0, 2 ** 31, (len(d), 256), dtype=np.uint64), np.minimum(k * D, top), np.minimum(k * D - np.uint64(1), top),
                        (top // D) * D, (top // D) * D - np.uint64(1), np.broadcast_to(top, (len(d), 1)), np.zeros((len(d), 1), np.uint64),
                        D - np.uint64(1), D, np.minimum(D + np.uint64(1), top)], axis=1)
    assert n.max() < 2 ** 31 and (M < 2 ** 32).all()
    q = ((n * M) >> np.uint64(32)) >> S                                 # n < 2^31, magic < 2^32: the product fits 63 bits
    bad = q != n // D
    assert not bad.any(), (d[np.nonzero(bad)[0][:4]], n[bad][:4])
