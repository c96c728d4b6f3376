"""Pins of the oracle (oracle/gpet_oracle.c) to things other than itself: published Philox vectors and
cuRAND's own round function, closed forms, invariants, library routines and brute force on tiny inputs
(BASELINE.json north_star).  CPU only."""
import ctypes
import math
import os
import subprocess

import numpy as np
import pytest
from scipy import integrate, stats

from oracle import gpet_oracle as O
from paper_2603_07327_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
C_MM_NS = 299.792458
Q = 2.0 ** 20


# ----------------------------------------------------------------------------- helpers
def const_tables(pe, c, r, n_mat=1):
    f = lambda v: np.full((n_mat, W.N_ENERGIES), v, np.float32)
    return W.Tables(W.E_MIN_KEV, W.E_STEP_KEV, f(pe), f(c), f(r))


def slab(depth=10.0, lateral=12.0, n=1, gap=0.0, dist=50.0, layers=None):
    """One panel = one module facing the origin from +x: u = +y, v = +z, w = +x."""
    pose = np.array([[dist, 0, 0, 0, 1, 0, 0, 0, 1, 1, 0, 0]], np.float32)
    if layers is None:
        layers = (W.Layer((n, n), (lateral / n,) * 2, (gap, gap), (0.0, 0.0), depth),)
    return W.Geometry(1, tuple(layers), (1, 1), (lateral, lateral), (lateral, lateral), panel_pose=pose)


def beam(direction=(1, 0, 0), pos=(0, 0, 0), acol=0.0):
    return W.source_beam(pos, direction, acol)


# ----------------------------------------------------------------------------- P1 Philox
def test_philox_published_vectors():
    for line in open(os.path.join(HERE, "golden", "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        assert list(O.philox(w[0:4], w[4:6])) == w[6:10]


def test_philox_equals_curand_header(tmp_path):
    so = str(tmp_path / "philox_curand_host.so")
    subprocess.check_call(["g++", "-O1", "-shared", "-fPIC", "-I/usr/local/cuda/include", "-o", so,
                           os.path.join(HERE, "golden", "philox_curand_host.cpp")])
    ref = ctypes.CDLL(so)
    rng = np.random.default_rng(7)
    for _ in range(2000):
        c = rng.integers(0, 2 ** 32, 4, dtype=np.uint64).astype(np.uint32)
        k = rng.integers(0, 2 ** 32, 2, dtype=np.uint64).astype(np.uint32)
        out = np.zeros(4, np.uint32)
        ref.curand_philox_host(c.ctypes.data_as(ctypes.c_void_p), k.ctypes.data_as(ctypes.c_void_p),
                               out.ctypes.data_as(ctypes.c_void_p))
        assert np.array_equal(O.philox(c, k), out)


def test_uniform_is_open_interval_and_fp32_exact():
    lib = O.lib()
    for x in (0, 511, 512, 2 ** 31, 2 ** 31 + 512, 0xFFFFFDFF, 2 ** 32 - 1):
        u = lib.orc_uniform(x)
        assert 0.0 < u < 1.0 and float(np.float32(u)) == u
    assert lib.orc_uniform(0) == 2.0 ** -24 and lib.orc_uniform(2 ** 32 - 1) == 1.0 - 2.0 ** -24


# ----------------------------------------------------------------------------- tables
def test_mu_lookup_equals_library_interpolation(tables):
    e_grid = W.energy_grid()
    rng = np.random.default_rng(3)
    for e in list(rng.uniform(10.0, 511.0, 300)) + [10.0, 10.5, 510.999, 511.0, 100.0]:
        for m in range(tables.n_materials):
            got = O.mu_lookup(tables, m, float(e))
            want = [np.interp(e, e_grid, t[m].astype(np.float64)) for t in (tables.mu_pe, tables.mu_compton, tables.mu_rayleigh)]
            assert np.allclose(got, want, rtol=1e-12, atol=0)
        tot = [sum(np.interp(e, e_grid, t[m].astype(np.float64)) for t in (tables.mu_pe, tables.mu_compton, tables.mu_rayleigh))
               for m in range(tables.n_materials)]
        assert math.isclose(O.mu_majorant(tables, 0b11, float(e)), max(tot), rel_tol=1e-9)
        assert math.isclose(O.mu_majorant(tables, 0b10, float(e)), tot[1], rel_tol=1e-9)


def test_table_compton_is_the_integral_of_the_klein_nishina_pdf(tables):
    """Ties the mu_C input table (closed-form sigma_KN) to the differential cross-section that the
    sampler's pdf is checked against below."""
    for e in (60.0, 170.0, 511.0):
        k = e / W.ME_C2_KEV
        dsdo = lambda c: 0.5 * W.R_E_CM ** 2 * (1 / (1 + k * (1 - c))) ** 2 * (1 / (1 + k * (1 - c)) + (1 + k * (1 - c)) - (1 - c * c))
        sig = 2 * math.pi * integrate.quad(dsdo, -1, 1, epsabs=0, epsrel=1e-12)[0]
        assert math.isclose(sig, float(W.kn_total_cross_section_cm2(e)), rel_tol=1e-10)
        i = int(round(e - 10))
        assert math.isclose(tables.mu_compton[0, i], W.N_E_LYSO_CM3 * sig * 0.1, rel_tol=1e-6)
    assert math.isclose(tables.mu_compton[0, -1], 0.05874, rel_tol=2e-4)      # SURVEY O11's printed value


# ----------------------------------------------------------------------------- P2 Woodcock / free path
def test_slab_transmission_and_depth_distribution():
    mu, L, n = 0.05, 10.0, 400_000
    res = O.simulate(slab(L), const_tables(mu, 0, 0), beam(), n, seed=11, want_escape=True, threads=4)
    unscattered = np.mean(res.e_escape[:, 0] == 511.0)
    p = math.exp(-mu * L)
    assert abs(unscattered - p) < 4 * math.sqrt(p * (1 - p) / n)
    assert np.all(res.e_escape[:, 1] == 511.0)                        # photon B flies away from the slab
    depth = res.hits.x.astype(np.float64) - 50.0
    assert len(depth) == n - int(round(unscattered * n))
    cdf = lambda d: (1 - np.exp(-mu * d)) / (1 - math.exp(-mu * L))
    assert stats.kstest(depth, cdf).pvalue > 1e-3
    assert np.all(res.hits.e_keV == 511.0)


def test_lattice_line_through_crystal_and_through_reflector(tables):
    g = W.geometry_c0()                                              # crystal 4 spans y in [0.05, 1.45)
    t = W.Tables(tables.e_min_keV, tables.e_step_keV, tables.mu_pe[:1], tables.mu_compton[:1], np.zeros_like(tables.mu_rayleigh[:1]))
    n = 300_000
    res = O.simulate(g, t, beam(pos=(0, 0.75, 0.75)), n, seed=12, want_escape=True, threads=4)
    mu_tot = float(t.mu_pe[0, -1]) + float(t.mu_compton[0, -1])
    p = math.exp(-mu_tot * 10.0)
    # unscattered = left with the full energy (no Rayleigh in these tables)
    assert abs(np.mean(res.e_escape[:, 0] == 511.0) - p) < 4 * math.sqrt(p * (1 - p) / n)
    res = O.simulate(g, t, beam(pos=(0, 0.01, 0.75)), 50_000, seed=13, want_escape=True)      # inside the reflector gap
    assert len(res.hits) == 0 and np.all(res.e_escape == 511.0)
    c = res.counters
    assert c["steps"] > c["exits"] and c["step_vacuum"] == c["steps"] - c["exits"]          # only virtual steps in vacuum


# ----------------------------------------------------------------------------- P3 interaction mix
def test_first_interaction_fractions_at_511(tables):
    needle = slab(depth=30.0, lateral=0.02)                          # scattered photons leave sideways at once
    lyso = W.Tables(tables.e_min_keV, tables.e_step_keV, tables.mu_pe[:1], tables.mu_compton[:1], tables.mu_rayleigh[:1])
    n = 400_000
    c = O.simulate(needle, lyso, beam(), n, seed=14, threads=4).counters
    tot = c["pe"] + c["compton"] + c["rayleigh"]
    mu = np.array([lyso.mu_pe[0, -1], lyso.mu_compton[0, -1], lyso.mu_rayleigh[0, -1]], np.float64)
    want = mu / mu.sum()
    assert np.allclose(want, [0.3232, 0.6545, 0.0223], atol=2e-4)    # SURVEY P3's printed fractions
    for got, w in zip((c["pe"], c["compton"], c["rayleigh"]), want):
        assert abs(got / tot - w) < 4 * math.sqrt(w * (1 - w) / tot) + 1e-3
    p_int = 1 - math.exp(-mu.sum() * 30.0)
    assert abs(tot / n - p_int) < 0.004


def test_interaction_mix_with_energy_independent_tables():
    t = const_tables(0.03, 0.05, 0.01)
    c = O.simulate(slab(10.0, 40.0, n=4, gap=0.0), t, beam(), 300_000, seed=15, threads=4).counters
    tot = c["pe"] + c["compton"] + c["rayleigh"]
    for got, w in zip((c["pe"], c["compton"], c["rayleigh"]), (1 / 3, 5 / 9, 1 / 9)):
        assert abs(got / tot - w) < 4 * math.sqrt(w * (1 - w) / tot)
    assert c["virtuals"] == 0                                        # one material everywhere: no virtual collisions in it


# ----------------------------------------------------------------------------- P4 Klein-Nishina
@pytest.mark.parametrize("e_keV", [511.0, 170.0, 60.0])
def test_klein_nishina_angles(e_keV):
    n = 120_000
    smp = np.array([O.kn_sample(99, h, e_keV) for h in range(n)])
    eps, ct, trials = smp[:, 0], smp[:, 1], smp[:, 2]
    k = e_keV / W.ME_C2_KEV
    assert np.allclose(eps, 1 / (1 + k * (1 - ct)), rtol=1e-12)      # Compton kinematics
    pdf = lambda c: (1 / (1 + k * (1 - c))) ** 2 * (1 / (1 + k * (1 - c)) + (1 + k * (1 - c)) - (1 - c * c))
    edges = np.linspace(-1, 1, 41)
    mass = np.array([integrate.quad(pdf, a, b)[0] for a, b in zip(edges[:-1], edges[1:])])
    obs = np.histogram(ct, edges)[0]
    assert stats.chisquare(obs, mass / mass.sum() * n).pvalue > 1e-3
    mean_eps = integrate.quad(lambda c: pdf(c) / (1 + k * (1 - c)), -1, 1)[0] / mass.sum()
    assert abs(eps.mean() - mean_eps) < 4 * eps.std() / math.sqrt(n)
    if e_keV == 511.0:
        assert abs(mean_eps - 0.6555) < 5e-4                          # SURVEY P4's printed value
    assert 1.2 < trials.mean() < 1.6                                  # acceptance 0.67..0.74


def test_klein_nishina_trial_cap():
    """SURVEY 8(c) O29 / [R20]: after 64 rejected trials the 64th is taken as it stands.  Honest draws never get there
    (acceptance >= 0.67 per trial: p < 1e-30), so the sampler runs on a prepared list: u_c just below 1 rejects every
    trial (g < 1 away from forward scattering), each trial carries its own u_b and azimuth.  The result must be the
    64th trial's -- not the first, not the initial eps = 1, not a 65th -- with Compton kinematics intact; a list that
    accepts at trial 3 stops there; and the honest sampler never comes near the cap."""
    e_keV = 511.0
    k = e_keV / W.ME_C2_KEV
    e0 = 1.0 / (1.0 + 2.0 * k)
    rows = np.zeros((80, 4))
    rows[:, 0] = 0.999                                                # u_a: always the second branch, eps^2 uniform in [e0^2, 1]
    rows[:, 1] = np.linspace(0.2, 0.8, 80)                            # u_b: a different eps per trial
    rows[:, 2] = 1.0 - 2.0 ** -30                                     # u_c: reject
    rows[:, 3] = (np.arange(80) + 0.5) / 80.0                         # azimuth: names the trial that was returned
    eps, ct, trials, ua = O.kn_sample_prepared(rows, e_keV)
    assert trials == 64 and ua == rows[63, 3]
    want = math.sqrt(e0 * e0 + (1.0 - e0 * e0) * rows[63, 1])        # that branch's inverse cdf at the 64th u_b
    assert abs(eps - want) < 1e-15 and e0 <= eps <= 1.0
    assert abs(eps - 1.0 / (1.0 + k * (1.0 - ct))) < 1e-14 and -1.0 <= ct <= 1.0
    rows[2, 2] = 0.0                                                  # trial 3 accepts
    eps3, ct3, trials3, ua3 = O.kn_sample_prepared(rows, e_keV)
    assert trials3 == 3 and ua3 == rows[2, 3] and abs(eps3 - math.sqrt(e0 * e0 + (1.0 - e0 * e0) * rows[2, 1])) < 1e-15
    rows[:, 0] = 0.0                                                  # first branch: eps = exp(-a1 u_b), same cap
    rows[2, 2] = 1.0 - 2.0 ** -30
    eps, ct, trials, ua = O.kn_sample_prepared(rows, e_keV)
    assert trials == 64 and abs(eps - e0 ** rows[63, 1]) < 1e-15 and abs(eps - 1.0 / (1.0 + k * (1.0 - ct))) < 1e-14
    assert max(O.kn_sample(5, h, e_keV)[2] for h in range(50_000)) < 40


# ----------------------------------------------------------------------------- P5 Rayleigh, rotation, acolinearity
def test_rayleigh_inverts_the_thomson_cdf():
    lib = O.lib()
    for u in np.linspace(1e-6, 1 - 1e-6, 501):
        c = lib.orc_rayleigh_cos(u)
        assert -1 <= c <= 1 and abs(0.375 * (c + c ** 3 / 3) + 0.5 - u) < 1e-12


def test_rotation_is_a_rigid_rotation_about_d():
    rng = np.random.default_rng(5)
    for _ in range(200):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        th, p1, p2 = rng.uniform(0, math.pi), rng.uniform(0, 2 * math.pi), rng.uniform(0, 2 * math.pi)
        a = O.rotate(d, math.cos(th), math.sin(th), math.cos(p1), math.sin(p1))
        b = O.rotate(d, math.cos(th), math.sin(th), math.cos(p2), math.sin(p2))
        assert abs(np.linalg.norm(a) - 1) < 1e-14 and abs(a @ d - math.cos(th)) < 1e-13
        pa, pb = a - (a @ d) * d, b - (b @ d) * d
        assert abs(pa @ pb - math.sin(th) ** 2 * math.cos(p1 - p2)) < 1e-13      # azimuth is a true angle about d
    assert np.allclose(O.rotate([0, 0, -1.0], 0.0, 1.0, 1.0, 0.0) @ np.array([0, 0, -1.0]), 0.0)   # pole is regular


def test_acolinearity_projects_to_a_gaussian_of_the_stated_fwhm():
    n, dist = 200_000, 1000.0
    pose = np.array([[-dist, 0, 0, 0, 1, 0, 0, 0, 1, -1, 0, 0]], np.float32)       # faces photon B (-x)
    g = W.Geometry(1, (W.Layer((1, 1), (400.0, 400.0), (0, 0), (0, 0), 1.0),), (1, 1), (400.0, 400.0), (400.0, 400.0), panel_pose=pose)
    res = O.simulate(g, const_tables(1000.0, 0, 0), beam(acol=0.5), n, seed=16, threads=4)
    h = res.hits
    assert len(h) == n and np.all((h.ids >> 4) & 1 == 1)
    sigma = math.radians(0.5) / 2.354820045 * dist
    for lateral in (h.y.astype(np.float64), h.z.astype(np.float64)):
        assert abs(lateral.std() / sigma - 1) < 0.01 and abs(lateral.mean()) < 4 * sigma / math.sqrt(n)
        assert stats.kstest(lateral / sigma, "norm").pvalue > 1e-3


# ----------------------------------------------------------------------------- P6 solid angle
def test_point_source_acceptance_equals_the_analytic_solid_angle(tables):
    n = 2_000_000
    r = W.config_runs("C0")[0]
    c = O.simulate(r.geometry, tables, r.source, n, r.seed, threads=8).counters
    a = b = 6.0; d = 50.0
    omega = 4 * math.asin(a * b / math.sqrt((a * a + d * d) * (b * b + d * d)))
    p = 2 * omega / (4 * math.pi)
    assert abs(p - 0.0090375) < 1e-7                                  # SURVEY P6's printed value
    assert abs(c["entries"] / n - p) < 4 * math.sqrt(p / n)
    assert c["searches"] == 2 * n + c["exits"] and c["escapes"] == 2 * n - c["pe"] - c["cutoffs"]


# ----------------------------------------------------------------------------- P7 split layer is exact
def test_zero_gap_split_is_bit_identical_to_the_single_layer(tables):
    n = 60_000
    a = O.simulate(W.geometry_c1(), tables, W.source_point(), n, seed=2, threads=8)
    b = O.simulate(W.geometry_c2(gap_mm=0.0), tables, W.source_point(), n, seed=2, threads=8)
    assert len(a.hits) == len(b.hits) > 30_000
    for k in ("history", "x", "y", "z", "e_keV", "tof_ns"):
        assert np.array_equal(getattr(a.hits, k), getattr(b.hits, k))
    layer_mask = np.uint32(3 << 18)
    assert np.array_equal(a.hits.ids & ~layer_mask, b.hits.ids & ~layer_mask)
    pose = O.ring_poses(12, 55.0)
    p = b.hits.ids >> 26
    xyz = np.stack([b.hits.x, b.hits.y, b.hits.z], 1).astype(np.float64)
    depth = np.einsum("ij,ij->i", xyz - pose[p, 0:3], pose[p, 9:12].astype(np.float64))
    clear = np.abs(depth - 5.0) > 1e-4
    assert np.array_equal(((b.hits.ids >> 18) & 3)[clear], (depth[clear] >= 5.0).astype(np.uint32))
    assert 0.3 < np.mean((b.hits.ids >> 18) & 3) < 0.5               # both layers are populated


# ----------------------------------------------------------------------------- P8 energy conservation
def test_energy_is_conserved_per_photon(tables):
    n = 100_000
    res = O.simulate(W.geometry_c3(), tables, W.source_point((25.0, 0, 8.0)), n, seed=17, want_escape=True, threads=8)
    dep = np.zeros((n, 2))
    np.add.at(dep, (res.hits.history, (res.hits.ids >> 4) & 1), res.hits.e_keV.astype(np.float64))
    assert np.max(np.abs(dep + res.e_escape - 511.0)) < 1e-3
    assert 0.5 < len(res.hits) / n < 2.0


def test_long_histories_saturate_the_sequence_counter_and_still_conserve_energy():
    """SURVEY 8(c) O31 / [R9], PAPER.md:43 ("transported step by step until it either exited the panel or fell below the
    cutoff energy"): a thick Compton-only slab, where a photon scatters dozens of times.  Almost half the photons make
    16 or more deposits; the 4-bit sequence number counts 0..14 and then stays at 15 (it must not wrap), the hits of a
    photon come out in path order (time of flight never decreases: that is what orders the saturated ones), every
    deposit is one Compton event of the counters, and deposits + what leaves = 511 keV for every photon.  A semi-infinite
    homogeneous slab has no length scale but 1/mu, so the discrete outcome cannot depend on mu: ten times the attenuation
    gives the same hits at a tenth of the depth."""
    n = 5000
    res = O.simulate(slab(800.0, 1600.0), const_tables(0, 0.05, 0), beam(), n, seed=31, want_escape=True, threads=8)
    h = res.hits
    photon = (h.ids >> 4) & 1
    assert np.all(photon == 0)                                        # photon B flies away from the slab
    cnt = np.bincount(h.history, minlength=n)
    assert np.mean(cnt >= 16) > 0.3 and cnt.max() > 40                # the regime: long histories are common
    start = np.cumsum(cnt) - cnt
    rank = np.arange(len(h)) - np.repeat(start, cnt)                  # position of a hit in its photon's track, as emitted
    assert np.all(np.diff(h.history.astype(np.int64)) >= 0)
    assert np.array_equal(h.ids & 15, np.minimum(rank, 15))           # 0, 1, ..., 14, 15, 15, 15, ...
    same = np.diff(h.history.astype(np.int64)) == 0
    assert np.all(np.diff(h.tof_ns.astype(np.float64))[same] >= 0)
    c = res.counters
    assert len(h) == c["compton"] == c["hits"] and c["cutoffs"] + c["exits"] == n
    dep = np.zeros(n); np.add.at(dep, h.history, h.e_keV.astype(np.float64))
    assert np.max(np.abs(dep + res.e_escape[:, 0] - 511.0)) < 2e-3 and np.all(res.e_escape[:, 1] == 511.0)
    r10 = O.simulate(slab(800.0, 1600.0), const_tables(0, 0.5, 0), beam(), n, seed=31, want_escape=True, threads=8)
    assert np.array_equal(r10.hits.ids, h.ids) and np.array_equal(r10.hits.history, h.history)
    assert np.allclose((r10.hits.x.astype(np.float64) - 50.0) * 10.0, h.x.astype(np.float64) - 50.0, rtol=1e-4, atol=1e-3)
    assert np.allclose(r10.hits.e_keV, h.e_keV, rtol=0, atol=1e-4)


# ----------------------------------------------------------------------------- P9 indexing by brute force
def tiny_scanner():
    th = math.radians(37.0)
    poses = np.array([[20, 0, 0, 0, 1, 0, 0, 0, 1, 1, 0, 0],
                      [-20, 3, 1, 0, -1, 0, 0, 0, 1, -1, 0, 0],
                      [25 * math.cos(th), 25 * math.sin(th), -2, -math.sin(th), math.cos(th), 0, 0, 0, 1, math.cos(th), math.sin(th), 0]],
                     np.float32)
    layers = (W.Layer((3, 2), (1.25, 1.5), (0.25, 0.125), (0.125, 0.25), 2.0),
              W.Layer((2, 2), (1.5, 1.25), (0.0, 0.25), (0.5, 0.0), 3.0, gap_before_mm=0.5))
    return W.Geometry(3, layers, (2, 2), (4.0, 3.5), (4.5, 4.0), panel_pose=poses)


def brute_force_boxes(g):
    """Every crystal as an explicit box in panel-local Q units from the low corner (nested loops)."""
    q = lambda v: int(round(float(np.float32(v)) * Q))
    boxes = []
    for mx in range(g.n_modules[0]):
        for my in range(g.n_modules[1]):
            c0 = 0
            for li, l in enumerate(g.layers):
                c0 += q(l.gap_before_mm)
                for ix in range(l.n_crystals[0]):
                    for iy in range(l.n_crystals[1]):
                        lo, hi = [], []
                        for a, (m, i) in enumerate(((mx, ix), (my, iy))):
                            base = m * q(g.module_pitch_mm[a]) + q(l.offset_mm[a]) + i * q(l.pitch_mm[a])
                            gp = q(l.reflector_mm[a])
                            lo.append(base + gp // 2); hi.append(base + q(l.pitch_mm[a]) - (gp - gp // 2))
                        boxes.append((lo[0], hi[0], lo[1], hi[1], c0, c0 + q(l.depth_mm),
                                      (mx + g.n_modules[0] * my) << 20 | li << 18 | (ix + l.n_crystals[0] * iy) << 5))
                c0 += q(l.depth_mm)
    W_q = (g.n_modules[0] - 1) * q(g.module_pitch_mm[0]) + q(g.module_size_mm[0])
    H_q = (g.n_modules[1] - 1) * q(g.module_pitch_mm[1]) + q(g.module_size_mm[1])
    return boxes, W_q, H_q, c0


def brute_locate(g, boxes, W_q, H_q, D_q, xyz):
    out = np.full(len(xyz), 0xFFFFFFFF, np.uint32)
    pose = g.panel_pose.astype(np.float64)
    for i, x in enumerate(xyz.astype(np.float64)):
        for p in range(g.n_panels):
            r = x - pose[p, 0:3]
            a, b, c = (r[0] * pose[p, 3] + r[1] * pose[p, 4] + r[2] * pose[p, 5], r[0] * pose[p, 6] + r[1] * pose[p, 7] + r[2] * pose[p, 8],
                       r[0] * pose[p, 9] + r[1] * pose[p, 10] + r[2] * pose[p, 11])
            qa, qb, qc = math.floor(a * Q) + (W_q >> 1), math.floor(b * Q) + (H_q >> 1), math.floor(c * Q)
            if not (0 <= qa < W_q and 0 <= qb < H_q and 0 <= qc < D_q):
                continue
            for (a0, a1, b0, b1, c0, c1, code) in boxes:
                if a0 <= qa < a1 and b0 <= qb < b1 and c0 <= qc < c1:
                    out[i] = (p << 26) | code
                    break
            break                                                     # lowest panel containing the point decides
    return out


def test_indexing_against_brute_force_enumeration():
    g = tiny_scanner()
    boxes, W_q, H_q, D_q = brute_force_boxes(g)
    assert len(boxes) == 4 * (6 + 4) and (W_q, H_q, D_q) == (int(8.5 * Q), int(7.5 * Q), int(5.5 * Q))
    rng = np.random.default_rng(8)
    pts = []
    for p in range(3):                                               # random points in and around every panel
        loc = rng.uniform([-4.6, -4.1, -0.3], [4.6, 4.1, 5.8], (1500, 3))
        pose = g.panel_pose[p].astype(np.float64)
        pts.append(pose[0:3] + loc[:, :1] * pose[3:6] + loc[:, 1:2] * pose[6:9] + loc[:, 2:3] * pose[9:12])
    # points exactly on faces (dyadic coordinates, axis-aligned panel 0): half-open intervals decide
    grid = np.arange(-4.25, 4.26, 0.125)
    ga, gb, gc = np.meshgrid(grid, grid[2:-2], np.arange(0.0, 5.51, 0.25), indexing="ij")
    pts.append(np.stack([20.0 + gc.ravel(), ga.ravel(), gb.ravel()], 1))
    xyz = np.concatenate(pts).astype(np.float32)
    got = O.locate(g, xyz)
    want = brute_locate(g, boxes, W_q, H_q, D_q, xyz)
    assert np.array_equal(got, want)
    inside = got != 0xFFFFFFFF
    assert 0.2 < inside.mean() < 0.8
    u = O.unpack_ids(got[inside])
    assert set(u["panel"]) == {0, 1, 2} and set(u["module"]) == {0, 1, 2, 3} and set(u["layer"]) == {0, 1}
    assert set(u["crystal"][u["layer"] == 0]) == set(range(6)) and set(u["crystal"][u["layer"] == 1]) == set(range(4))


def test_half_open_faces_in_the_local_frame():
    g = W.geometry_c0()                                              # 12 x 12 x 10, pitch 1.5, gap 0.1 -> 0.05 each side
    h = 2.0 ** -20
    pts = np.array([[-6 + 0.05 - h, 0.7, 1], [-6 + 0.05, 0.7, 1], [-6 + 1.45 - h, 0.7, 1], [-6 + 1.45, 0.7, 1],
                    [0.7, 0.7, 0.0], [0.7, 0.7, -h], [0.7, 0.7, 10 - h], [0.7, 0.7, 10.0], [5.95 - h, 5.95 - h, 5], [5.95, 5.0, 5]])
    # quantised edges: 0.05 mm -> 52429 Q (rounded up), 1.45 = pitch - (gap - gap//2)
    ids, mat = O.locate_local(g, 0, pts)
    qgap = int(round(float(np.float32(0.1)) * Q)); lo = (qgap // 2) / Q; hi = 1.5 - (qgap - qgap // 2) / Q
    pts2 = np.array([[-6 + lo - h, 0.7, 1], [-6 + lo, 0.7, 1], [-6 + hi - h, 0.7, 1], [-6 + hi, 0.7, 1]])
    ids2, mat2 = O.locate_local(g, 0, pts2)
    assert list(mat2) == [-1, 0, 0, -1] and list(ids2 >> 5 & 8191) [1:3] == [4 * 8, 4 * 8]
    assert list(mat[4:8]) == [0, -1, 0, -1]
    assert ids[8] >> 5 & 8191 == 63 and mat[9] == -1


# ----------------------------------------------------------------------------- panel search by marching
def test_panel_search_against_marching(tables):
    g = W.geometry_c3()
    pose = O.ring_poses(12, 55.0).astype(np.float64)
    lo, hi = O.panel_box(g)
    assert np.allclose(lo, [-16, -32, 0]) and np.allclose(hi, [16, 32, 10.1], atol=1e-6)
    rng = np.random.default_rng(9)
    n_hit = 0
    for _ in range(150):
        x = rng.uniform(-30, 30, 3) * [1, 1, 0.5]
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        p, t = O.panel_search(g, x, d)
        ts = np.arange(0.0, 140.0, 0.01)
        pts = x + ts[:, None] * d
        first = (-1, np.inf)
        for q in range(12):
            r = pts - pose[q, 0:3]
            loc = np.stack([r @ pose[q, 3:6], r @ pose[q, 6:9], r @ pose[q, 9:12]], 1)
            ins = np.all((loc >= lo) & (loc < hi), 1)
            if ins.any() and ts[ins.argmax()] < first[1] - 1e-9:
                first = (q, ts[ins.argmax()])
        if first[0] < 0:
            # a march in 0.01 mm steps can miss a corner clip shorter than the step, never a long chord
            assert p < 0 or t > 0
            continue
        n_hit += 1
        assert p >= 0 and abs(t - first[1]) <= 0.0101 + 1e-9
        if p != first[0]:                                            # only legitimate in the overlap wedge
            assert abs(t - first[1]) <= 0.0101
    assert n_hit > 60
    assert O.panel_search(g, [0, 0, 0], [1, 0, 0], excl=0)[0] == -1  # excluded panel is skipped
    assert O.panel_search(g, [0, 0, 0], [1, 0, 0])[0] == 0 and abs(O.panel_search(g, [0, 0, 0], [1, 0, 0])[1] - 55.0) < 1e-5


# ----------------------------------------------------------------------------- P10 / P11 paper's own checks
def test_centred_source_symmetry(tables):
    n = 200_000
    h = O.simulate(W.geometry_c1(), tables, W.source_point(), n, seed=2, threads=8).hits
    counts = np.bincount(h.ids >> 26, minlength=12)
    assert stats.chisquare(counts).pvalue > 1e-3                      # equal counts in all panels
    up, down = int(np.sum(h.z > 0)), int(np.sum(h.z < 0))            # PAPER.md:87 symmetric axial profile
    assert abs(up - down) < 4 * math.sqrt(up + down)


def test_dual_layer_signature(tables):
    n = 200_000
    pose = O.ring_poses(12, 55.0).astype(np.float64)

    def local(h):
        p = h.ids >> 26
        r = np.stack([h.x, h.y, h.z], 1).astype(np.float64) - pose[p, 0:3]
        return np.stack([np.einsum("ij,ij->i", r, pose[p, 3 * k + 3:3 * k + 6]) for k in range(3)], 1)

    h1 = O.simulate(W.geometry_c1(), tables, W.source_point(), n, seed=2, threads=8).hits
    h3 = O.simulate(W.geometry_c3(), tables, W.source_point(), n, seed=2, threads=8).hits
    l1, l3 = local(h1), local(h3)
    front = np.sum((h3.ids >> 18) & 3 == 0) / np.sum(l1[:, 2] < 6.0)
    assert 0.86 < front < 0.92                                        # (15/16)^2 = 0.879 of the crystal area
    back = np.sum((h3.ids >> 18) & 3 == 1) / np.sum(l1[:, 2] >= 6.0)
    assert 0.93 < back < 1.07                                         # deeper region matches
    # lateral shift of the front layer = the offset: cell phase measured from the module corner
    f = (h3.ids >> 18) & 3 == 0
    for axis, half in ((0, 16.0), (1, 32.0)):
        phase0 = np.mod(l3[f, axis] + half - 0.5, 1.0)
        phase1 = np.mod(l3[~f, axis] + half, 1.0)
        for ph in (phase0, phase1):
            assert ph.min() >= 0.05 - 1e-4 and ph.max() <= 0.95 + 1e-4
    assert (h3.ids[f] >> 5 & 8191).max() == 15 * 15 - 1 and (h3.ids[~f] >> 5 & 8191).max() == 16 * 16 - 1


# ----------------------------------------------------------------------------- P12 time of flight
def test_first_hit_time_of_flight():
    g = W.geometry_c1()
    src = W.source_point((10.0, -5.0, 3.0), acolinearity_fwhm_deg=0.5)
    h = O.simulate(g, const_tables(0.09, 0, 0), src, 50_000, seed=18, threads=4).hits     # PE only: every hit is a first interaction
    dist = np.sqrt((h.x.astype(np.float64) - 10) ** 2 + (h.y.astype(np.float64) + 5) ** 2 + (h.z.astype(np.float64) - 3) ** 2)
    assert len(h) > 20_000 and np.max(np.abs(h.tof_ns - dist / C_MM_NS)) < 2e-6
    assert np.all(h.ids & 15 == 0)


# ----------------------------------------------------------------------------- P13 adder + coincidences by brute force
def brute_digitize(hits, t0, dig):
    """O(N^2)-style restatement of SURVEY O24-O27 with the blur switched off (sigma = 0)."""
    sh = {0: 5, 1: 20, 2: 26}[dig.readout_level]
    groups = {}
    for i in range(len(hits)):
        groups.setdefault((int(hits.history[i]), int(hits.ids[i]) >> sh), []).append(i)
    singles = []
    for (hist, unit), idx in groups.items():
        e = sum(float(hits.e_keV[i]) for i in idx)
        best = min(idx, key=lambda i: (-float(hits.e_keV[i]), int(hits.ids[i]) & 31))
        if dig.e_lo_keV <= e < dig.e_hi_keV:
            singles.append((t0[hist] + min(float(hits.tof_ns[i]) for i in idx) * 1e-9, hist, unit, int(hits.ids[best]), e))
    singles.sort(key=lambda s: s[:3])
    coinc, used = [], [False] * len(singles)
    for i, s in enumerate(singles):
        if used[i]:
            continue
        members = [j for j in range(i, len(singles)) if not used[j] and singles[j][0] - s[0] < dig.window_ns * 1e-9]
        for j in members:
            used[j] = True
        if len(members) == 2 and (singles[members[0]][3] >> 26) != (singles[members[1]][3] >> 26):
            coinc.append((singles[members[0]][3], singles[members[1]][3], singles[members[0]][1], singles[members[1]][1]))
    return singles, coinc


@pytest.mark.parametrize("level", [0, 1, 2])
def test_adder_and_coincidences_against_brute_force(tables, level):
    n = 6000
    src = W.source_point((5.0, 0, 0), activity_bq=2.0e8)             # very hot: plenty of randoms and multiples
    hits = O.simulate(W.geometry_c3(), tables, src, n, seed=19).hits
    dig = W.Digitizer(blur_fwhm_frac=0.0, e_lo_keV=200.0, e_hi_keV=600.0, window_ns=4.0, readout_level=level)
    sg, co, n_all = O.digitize(src, 19, n, hits, dig)
    t0 = {h: O.decay_time(src, 19, h, n) for h in set(int(x) for x in hits.history)}
    singles, coinc = brute_digitize(hits, t0, dig)
    assert len(sg.history) == len(singles) > 1000
    assert [int(x) for x in sg.history] == [s[1] for s in singles] and [int(x) for x in sg.ids] == [s[3] for s in singles]
    assert np.allclose(sg.t_s, [s[0] for s in singles], rtol=0, atol=1e-15) and np.allclose(sg.e_keV, [s[4] for s in singles], atol=1e-3)
    assert len(co.ids_a) == len(coinc) > 50
    assert [(int(a), int(b), int(c), int(d)) for a, b, c, d in zip(co.ids_a, co.ids_b, co.history_a, co.history_b)] == coinc
    assert np.sum(co.history_a != co.history_b) > 10                 # randoms exist at this activity
    assert np.all(co.dt_ns >= 0) and np.all(co.dt_ns < 4.0)
    # hit order must not matter
    perm = np.random.default_rng(1).permutation(len(hits))
    shuffled = O.Hits(*[getattr(hits, k)[perm] for k in ("history", "ids", "x", "y", "z", "e_keV", "tof_ns")])
    sg2, co2, _ = O.digitize(src, 19, n, shuffled, dig)
    assert np.array_equal(sg2.ids, sg.ids) and np.array_equal(co2.ids_a, co.ids_a) and np.array_equal(sg2.t_s, sg.t_s)


def test_low_activity_has_only_true_coincidences(tables):
    n = 100_000
    src = W.source_point(activity_bq=10.0)
    hits = O.simulate(W.geometry_c1(), tables, src, n, seed=20, threads=8).hits
    sg, co, n_all = O.digitize(src, 20, n, hits, W.Digitizer())
    assert len(co.ids_a) > 2000 and np.all(co.history_a == co.history_b)
    assert 0.45 < n_all / n < 0.65 and 0.25 < len(sg.history) / n < 0.42   # 0.54 singles, 0.33 kept per pair
    assert np.all(np.diff(sg.t_s) >= 0)


# ----------------------------------------------------------------------------- P14 blur
def test_energy_blur_width_and_window():
    n = 200_000
    src = beam()
    hits = O.simulate(slab(10.0), const_tables(5.0, 0, 0), src, n, seed=21, threads=4).hits
    assert len(hits) == n and np.all(hits.e_keV == 511.0)
    dig = W.Digitizer(blur_fwhm_frac=0.15, blur_ref_keV=511.0, e_lo_keV=0.0, e_hi_keV=2000.0, window_ns=4.0)
    sg, _, _ = O.digitize(src, 21, n, hits, dig)
    sigma = 0.15 * 511.0 / 2.354820045                               # FWHM 76.65 keV at the photopeak
    assert abs(sg.e_keV.std() / sigma - 1) < 0.01 and abs(sg.e_keV.mean() - 511.0) < 4 * sigma / math.sqrt(n)
    assert stats.kstest((sg.e_keV.astype(np.float64) - 511.0) / sigma, "norm").pvalue > 1e-3
    dig = W.Digitizer(blur_fwhm_frac=0.15, blur_ref_keV=511.0, e_lo_keV=350.0, e_hi_keV=650.0)
    sg2, _, _ = O.digitize(src, 21, n, hits, dig)
    keep = (sg.e_keV >= 350.0) & (sg.e_keV < 650.0)
    assert len(sg2.e_keV) == int(keep.sum()) and sg2.e_keV.min() >= 350.0 and sg2.e_keV.max() < 650.0
    # sigma ~ sqrt(E): a 127.75 keV deposit (E/4) has half the sigma of the photopeak
    quarter = O.Hits(hits.history, hits.ids, hits.x, hits.y, hits.z, np.full(n, 127.75, np.float32), hits.tof_ns)
    sg3, _, _ = O.digitize(src, 21, n, quarter, W.Digitizer(0.15, 511.0, 0.0, 2000.0))
    assert abs(sg3.e_keV.std() / (sigma / 2) - 1) < 0.01


# ----------------------------------------------------------------------------- P15 voxel source, decay times
def test_voxel_source_is_uniform_over_active_voxels():
    src = W.source_hot_rods()
    n = 2_000_000
    xyz = O.decay_sites(src, 5, 0, n)
    v = np.floor((xyz + 16.0) / 0.25).astype(np.int64)
    flat = (v[:, 2] * 128 + v[:, 1]) * 128 + v[:, 0]
    active = np.flatnonzero(src.activity.ravel() > 0)
    assert len(active) == 130_720
    assert np.all(np.isin(flat, active))
    counts = np.bincount(np.searchsorted(active, flat), minlength=len(active))
    assert stats.chisquare(counts).pvalue > 1e-3
    frac = (xyz + 16.0) / 0.25 - v
    assert np.all(np.abs(frac.mean(0) - 0.5) < 4 / math.sqrt(12 * n)) and frac.min() > 0 and frac.max() < 1


def test_decay_times_fill_their_time_slice():
    src = W.Source(activity_bq=1.0e6, pairs_per_time_slice=1000)
    t = np.array([O.decay_time(src, 3, h, 4000) for h in range(4000)])
    assert np.all(np.floor(t / 1e-3).astype(int) == np.arange(4000) // 1000)
    assert stats.kstest(np.mod(t, 1e-3) / 1e-3, "uniform").pvalue > 1e-3
    assert len(np.unique(t)) == 4000
    t1 = np.array([O.decay_time(W.Source(activity_bq=2.0e6), 3, h, 4000) for h in range(100)])
    assert np.all(t1 < 4000 / 2.0e6)


def test_phantom_attenuation(tables):
    """C4's water cylinder (d = 30 mm, 20 mm long): photons born at the centre leave it unscattered with
    probability <exp(-mu_water * chord)> over isotropic directions (vacuum voxels are virtual
    collisions that consume no draw).  The detector material is made transparent so that
    'left with 511 keV' means 'no interaction in the phantom' (water has no Rayleigh here)."""
    act, mat, org = W.hot_rod_phantom()
    one = np.zeros_like(act); one[64, 64, 64] = 1.0
    src = W.Source(1, (0, 0, 0), 0.0, 1e6, 0, one, mat, 1, (128, 128, 128), (0.25,) * 3, org)
    n = 200_000
    zero = np.zeros((1, W.N_ENERGIES), np.float32)
    wt = W.Tables(10.0, 1.0, np.concatenate([zero, tables.mu_pe[1:2]]), np.concatenate([zero, tables.mu_compton[1:2]]),
                  np.concatenate([zero, zero]))
    res = O.simulate(W.geometry_c1(), wt, src, n, seed=5, want_escape=True, threads=8)
    c = res.counters
    mu_w = float(wt.mu_pe[1, -1]) + float(wt.mu_compton[1, -1])
    cz = np.linspace(-1, 1, 400_001); sz = np.sqrt(1 - cz ** 2)
    chord = np.minimum(15.0 / np.maximum(sz, 1e-12), 10.0 / np.maximum(np.abs(cz), 1e-12))
    p_free = float(np.exp(-mu_w * chord).mean())
    got = float(np.mean(res.e_escape == 511.0))
    assert abs(got - p_free) < 4 * math.sqrt(p_free * (1 - p_free) / (2 * n)) + 5e-4
    assert 0.85 < p_free < 0.88 and len(res.hits) == 0
    assert c["ph_absorbed"] < 0.01 * c["ph_compton"] and c["ph_steps"] > 2 * n
    assert abs(math.fsum(res.e_escape.ravel()) / (2 * n) - 511.0) < 25.0   # scattered photons keep most of their energy


def test_leaving_the_phantom_keeps_the_line_of_flight(tables):
    """a gamma escaping from the phantom is taken to its panel along its line of flight.  With an
    all-vacuum phantom the acceptance of C0's panel must therefore still be the analytic solid angle
    2*Omega/4pi = 0.0090375, and first hits must keep tof = |x - source| / c.  A Woodcock step
    (mean free path of the water majorant: ~104 mm) that carried the photon past the panel on leaving the grid
    would lose most entries [R17]."""
    act, mat, org = W.hot_rod_phantom()
    one = np.zeros_like(act); one[64, 64, 64] = 1.0
    src = W.Source(1, (0, 0, 0), 0.0, 1e6, 0, one, np.zeros_like(mat), 1, (128, 128, 128), (0.25,) * 3, org)
    n = 2_000_000
    res = O.simulate(W.geometry_c0(), tables, src, n, seed=8, threads=8)
    c = res.counters
    expect = 0.0090375 * n
    assert abs(c["entries"] - expect) < 4 * math.sqrt(expect) + 0.004 * expect      # voxel is 0.125 mm off-centre
    assert c["ph_steps"] >= 2 * n and c["ph_compton"] == 0
    first = (res.hits.ids & 15) == 0
    site = O.decay_sites(src, 8, 0, n)[res.hits.history[first]]
    xyz = np.stack([res.hits.x, res.hits.y, res.hits.z], 1)[first]
    direct = np.linalg.norm(xyz - site, axis=1) / 299.792458
    unscattered = np.abs(res.hits.tof_ns[first] - direct) < 1e-4
    assert unscattered.mean() > 0.9                                  # the rest scattered in the crystal first


def test_randoms_rate_follows_the_singles_rate(tables):
    """random coincidences (members from different histories) occur at ~ tau * S^2 for the rate S of
    singles without a kept partner, reduced by the same-panel veto (11/12 on a uniformly lit 12-panel ring).  Order-of-magnitude invariant of the window rule [R27] and of the decay-time model [R16]."""
    n, A, tau = 200_000, 1.0e7, 4.0e-9
    src = W.source_point(activity_bq=A)
    hits = O.simulate(W.geometry_c1(), tables, src, n, seed=23, threads=8).hits
    sg, co, _ = O.digitize(src, 23, n, hits, W.Digitizer())
    T = n / A
    # a window holding a true pair plus a stranger has three members and is dropped, so randoms form among the singles
    # whose partner was not kept: histories with exactly one kept single
    per_history = np.bincount(sg.history.astype(np.int64), minlength=n)
    lonely = int(np.sum(per_history == 1))
    expect = lonely * (lonely / T) * tau * (11.0 / 12.0)
    randoms = int(np.sum(co.history_a != co.history_b))
    assert expect > 250 and 0.8 * expect < randoms < 1.2 * expect, (randoms, expect)
    # and it scales with the activity: a tenth of the activity gives about a tenth of the randoms per single
    src2 = W.source_point(activity_bq=A / 10)
    sg2, co2, _ = O.digitize(src2, 23, n, hits, W.Digitizer())
    r2 = int(np.sum(co2.history_a != co2.history_b))
    assert len(sg2.ids) == len(sg.ids) and 0.05 * randoms < r2 < 0.2 * randoms


# ----------------------------------------------------------------------------- branches no config reaches
def test_constant_fraction_blur():
    """[R25] blur_ref_keV = 0 selects sigma = (R / 2.3548) * E: the relative width is the same at every energy, and the
    blurred energies are Gaussian (KS) at two energies."""
    n = 200_000
    src = beam()
    hits = O.simulate(slab(10.0), const_tables(5.0, 0, 0), src, n, seed=22, threads=4).hits
    assert len(hits) == n
    for e in (511.0, 127.75):
        h = O.Hits(hits.history, hits.ids, hits.x, hits.y, hits.z, np.full(n, e, np.float32), hits.tof_ns)
        sg, _, _ = O.digitize(src, 22, n, h, W.Digitizer(0.15, 0.0, 0.0, 5000.0))
        sigma = 0.15 / 2.354820045 * e
        assert abs(sg.e_keV.std() / sigma - 1) < 0.01, (e, sg.e_keV.std(), sigma)
        assert stats.kstest((sg.e_keV.astype(np.float64) - e) / sigma, "norm").pvalue > 1e-3
    # and it differs from the photopeak-referenced model away from the reference energy (sqrt(E) law: twice as wide at E/4)
    sg_ref, _, _ = O.digitize(src, 22, n, h, W.Digitizer(0.15, 511.0, 0.0, 5000.0))
    assert abs(sg_ref.e_keV.std() / sg.e_keV.std() - 2.0) < 0.03


def test_weighted_activity_map_is_sampled_in_proportion():
    """[R13] decay sites follow the activity: a three-valued map on a small grid, chi-square of the voxel counts
    against the activities themselves (the integer weights rint(a / a_max * 2^20) and the `first cumulative weight
    above the target` search sit in between), plus the uniform position inside the voxel."""
    rng = np.random.default_rng(3)
    dims = (6, 5, 4)                                                   # nx, ny, nz
    act = rng.choice(np.array([0.0, 0.05, 0.3, 1.0], np.float32), size=(dims[2], dims[1], dims[0]), p=[0.4, 0.2, 0.2, 0.2])
    src = W.Source(1, (0, 0, 0), 0.0, 1e6, 0, act, None, -1, dims, (0.5, 0.25, 1.0), (-1.5, -0.625, -2.0))
    n = 1_000_000
    xyz = O.decay_sites(src, 8, 0, n)
    v = np.floor((xyz - np.array(src.origin_mm)) / np.array(src.voxel_mm)).astype(np.int64)
    assert v.min() >= 0 and np.all(v.max(0) < np.array(dims))
    flat = (v[:, 2] * dims[1] + v[:, 1]) * dims[0] + v[:, 0]          # x fastest
    counts = np.bincount(flat, minlength=act.size).astype(np.float64)
    a = act.ravel().astype(np.float64)
    assert np.all(counts[a == 0] == 0)                                 # nothing is born where there is no activity
    live = a > 0
    assert live.sum() > 40 and len(np.unique(a[live])) == 3
    assert stats.chisquare(counts[live], n * a[live] / a[live].sum()).pvalue > 1e-3
    # ratio of the two extreme populations: 0.05 / 1.0 (a dropped weight scaling or an off-by-one in the search shows here)
    r = counts[a == np.float32(0.05)].sum() / counts[a == 1.0].sum() / ((a == np.float32(0.05)).sum() / (a == 1.0).sum())
    assert abs(r / 0.05 - 1) < 0.03
    frac = (xyz - np.array(src.origin_mm)) / np.array(src.voxel_mm) - v
    assert np.all(np.abs(frac.mean(0) - 0.5) < 4 / math.sqrt(12 * n))


def fnv_events(events):
    """[R23] FNV-1a over (type, payload) pairs, vectorised over histories -- restated here to label photons by their
    event sequence.  events: list of (type, payload) with payload an int or a uint64 array."""
    P = np.uint64(0x100000001B3)
    h = np.uint64(0xCBF29CE484222325)
    with np.errstate(over="ignore"):
        for t, p in events:
            h = (h ^ np.uint64(t)) * P
            h = (h ^ np.asarray(p, np.uint64)) * P
    return h


def closed_cube(half=40.0):
    """Six panels closing a cube about the origin, one gapless crystal each: every photon is caught, at its entry point
    when the material is a strong pure absorber."""
    faces = [((1, 0, 0), (0, 1, 0), (0, 0, 1)), ((-1, 0, 0), (0, -1, 0), (0, 0, 1)), ((0, 1, 0), (-1, 0, 0), (0, 0, 1)),
             ((0, -1, 0), (1, 0, 0), (0, 0, 1)), ((0, 0, 1), (1, 0, 0), (0, 1, 0)), ((0, 0, -1), (1, 0, 0), (0, -1, 0))]
    poses = np.array([np.concatenate([half * np.array(w, float), u, v, w]) for w, u, v in faces], np.float32)
    side = 2 * half                                                    # the six boxes touch along the cube's edges without overlapping
    lay = (W.Layer((1, 1), (side, side), (0.0, 0.0), (0.0, 0.0), 10.0),)
    return W.Geometry(6, lay, (1, 1), (side, side), (side, side), panel_pose=poses)


def phantom_rayleigh_setup(mu_r=0.1):
    """A 0.4 mm cube of a thin, purely Rayleigh-scattering medium (material 1) around a point-like activity at the origin,
    inside the closed cube of strong photo-absorbers (material 0): photon B of a pair whose photon A scattered exactly
    once shows the original axis, photon A's entry point the deflected direction.  The medium is thin (2 % of the
    photons scatter) so that `exactly once` selects deflection angles almost without bias (a backscattered photon has a
    longer way out: the bias of <cos> is ~ mu * 0.05 mm)."""
    dims = (4, 4, 4)
    act = np.zeros((4, 4, 4), np.float32); act[1:3, 1:3, 1:3] = 1.0
    mat = np.full((4, 4, 4), 2, np.uint8)                              # value 2 = material index 1
    src = W.Source(1, (0, 0, 0), 0.0, 1e6, 0, act, mat, 1, dims, (0.1, 0.1, 0.1), (-0.2, -0.2, -0.2))
    f = lambda a, b: np.stack([np.full(W.N_ENERGIES, a, np.float32), np.full(W.N_ENERGIES, b, np.float32)])
    # absorber: photoelectric only, 0.2 mm mean depth (a stronger one would put 5e-5 of the first collisions within fp32
    # rounding of the entry face, where the CUDA path and the oracle may disagree on `inside`); medium: Rayleigh only
    t = W.Tables(W.E_MIN_KEV, W.E_STEP_KEV, f(5.0, 0.0), f(0.0, 0.0), f(0.0, mu_r))
    return closed_cube(), t, src


def single_rayleigh_deflections(hits, hashes, n):
    """cos(theta) and azimuth of the deflection of photons A that scattered exactly once in the phantom while their
    partner B left it unscattered -- selected by the event hash [R23] rebuilt from the hit's own panel and ids."""
    ids = hits["ids"]; hist = hits["history"].astype(np.int64)
    photon = (ids >> 4) & 1
    pos = np.stack([hits["x"], hits["y"], hits["z"]], 1).astype(np.float64)
    first = (ids & 15) == 0
    ia = np.full(n, -1); ib = np.full(n, -1)
    ia[hist[first & (photon == 0)]] = np.flatnonzero(first & (photon == 0))
    ib[hist[first & (photon == 1)]] = np.flatnonzero(first & (photon == 1))
    both = np.flatnonzero((ia >= 0) & (ib >= 0))
    a, b = ia[both], ib[both]
    strip = lambda i: (ids[i] & ~np.uint32(31)).astype(np.uint64)
    want_a = fnv_events([(11, 0), (14, 0), (1, (ids[a] >> 26).astype(np.uint64)), (4, strip(a))])   # PH_RAYLEIGH, PH_LEAVE, ENTER, PE
    want_b = fnv_events([(14, 0), (1, (ids[b] >> 26).astype(np.uint64)), (4, strip(b))])            # PH_LEAVE, ENTER, PE
    sel = (hashes[both, 0] == want_a) & (hashes[both, 1] == want_b)
    a, b = a[sel], b[sel]
    axis = -pos[b] / np.linalg.norm(pos[b], axis=1, keepdims=True)     # B flies along -d: A started along +d
    out = pos[a] / np.linalg.norm(pos[a], axis=1, keepdims=True)
    e1 = np.cross(axis, [0.3, -0.5, 0.8]); e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
    e2 = np.cross(axis, e1)
    return np.sum(axis * out, 1), np.arctan2(np.sum(out * e2, 1), np.sum(out * e1, 1))


def check_thomson(c, phi):
    assert len(c) > 25_000
    # the scattering point lies within 0.35 mm of the origin, 40 mm from the faces: angles are good to ~0.01 rad
    assert abs(c.mean()) < 0.012 and abs((c ** 2).mean() - 0.4) < 0.01, (c.mean(), (c ** 2).mean())
    cdf = lambda x: 0.375 * (x + x ** 3 / 3.0) + 0.5
    assert stats.kstest(c, cdf).pvalue > 1e-4
    assert stats.kstest(phi, stats.uniform(-math.pi, 2 * math.pi).cdf).pvalue > 1e-3


def test_phantom_rayleigh_follows_the_thomson_distribution():
    """[R17, R20] the phantom's Rayleigh branch (no config's water has mu_R > 0): single deflections follow
    3/8 (1 + cos^2): <cos> = 0, <cos^2> = 2/5, the closed-form cdf (KS), and a uniform azimuth about the flight axis."""
    g, t, src = phantom_rayleigh_setup()
    n = 2_000_000
    res = O.simulate(g, t, src, n, seed=12, want_hash=True, threads=8)
    assert res.counters["ph_compton"] == 0 and res.counters["ph_absorbed"] == 0 and res.counters["rayleigh"] == 0
    check_thomson(*single_rayleigh_deflections(PU_hits(res.hits), res.outcome_hash, n))


def PU_hits(hits):
    return {k: getattr(hits, k) for k in ("history", "ids", "x", "y", "z", "e_keV", "tof_ns")}


def square_ring(width=24.0):
    """Four panels at 0, 90, 180, 270 degrees on a 10 mm apothem (poses exactly representable), wider than the square's
    side (20 mm) so that neighbours overlap at the corners -- the situation of C1..C4's wedge with exact
    arithmetic: a ray along a diagonal reaches two front faces at bit-identical distances."""
    lay = (W.Layer((1, 1), (width, width), (0.0, 0.0), (0.0, 0.0), 5.0),)
    return W.Geometry(4, lay, (1, 1), (width, width), (width, width), ring_inner_radius_mm=10.0)


def test_panel_search_tie_goes_to_the_lowest_index():
    """[R6] equal entry distances -> the lowest panel index.  Diagonal rays of the square ring tie exactly (dx == dy in
    binary), so the rule -- not rounding -- decides; a `<=` in place of `<`, or a descending loop, fails here."""
    g = square_ring()
    s = 1.0 / math.sqrt(2.0)
    for d, want, other in (((s, s, 0), 0, 1), ((s, -s, 0), 0, 3), ((-s, s, 0), 1, 2), ((-s, -s, 0), 2, 3)):
        p, t = O.panel_search(g, [0.0, 0.0, 0.0], list(d))
        assert p == want and abs(t - 10.0 / s) < 1e-12, (d, p, t)
        p2, t2 = O.panel_search(g, [0.0, 0.0, 0.0], list(d), excl=want)    # without it the tie partner is found, same distance
        assert p2 == other and t2 == t
    # two coincident panels (explicit poses): every ray ties
    pose = np.array([[20, 0, 0, 0, 1, 0, 0, 0, 1, 1, 0, 0]] * 2, np.float32)
    twin = W.Geometry(2, square_ring().layers, (1, 1), (24.0, 24.0), (24.0, 24.0), panel_pose=pose)
    rng = np.random.default_rng(4)
    for _ in range(50):
        d = np.array([1.0, rng.uniform(-0.4, 0.4), rng.uniform(-0.4, 0.4)]); d /= np.linalg.norm(d)
        assert O.panel_search(twin, [0.0, 0.0, 0.0], d)[0] == 0 and O.panel_search(twin, [0.0, 0.0, 0.0], d, excl=0)[0] == 1


def test_ring_handedness_against_hand_written_numbers():
    """[R5] u x v = w for every ring panel, and the tangential axis runs counter-clockwise: on C1's ring a point displaced
    along +y from the centre of panel 0 (at +x) lies in a HIGHER crystal column, on panel 3 (at +y) a point displaced
    along -x does.  Expected ids are written out by hand from [R7] / [R9], not taken from the oracle."""
    pose = O.ring_poses(12, 55.0).astype(np.float64)
    for p in range(12):
        u, v, w = pose[p, 3:6], pose[p, 6:9], pose[p, 9:12]
        assert np.allclose(np.cross(u, v), w, atol=1e-7) and np.allclose(pose[p, 0:3], 55.0 * w, atol=1e-5)
        assert abs(math.atan2(w[1], w[0]) - math.radians(30.0 * p if p <= 6 else 30.0 * p - 360.0)) < 1e-6
    g = W.geometry_c1()                                                # 2 x 4 modules of 16 x 16, pitch 1 mm, panel 32 x 64 x 10
    pack = lambda panel, mx, my, ix, iy: (panel << 26) | ((mx + 2 * my) << 20) | ((ix + 16 * iy) << 5)
    pts = np.array([[56.0, 3.5, 0.5],      # panel 0: a = +3.5 -> 19.5 from the low edge: module column 1, crystal column 3; b = 0.5 -> 32.5: module row 2, crystal row 0
                    [56.0, -3.5, 0.5],     # panel 0: a = -3.5 -> 12.5: module column 0, crystal column 12
                    [56.0, 0.5, -20.5],    # panel 0: b = -20.5 -> 11.5: module row 0, crystal row 11; a = 0.5 -> 16.5: module column 1, crystal column 0
                    [-3.5, 56.0, 0.5],     # panel 3 (at +y, u = -x): a = +3.5 -> module column 1, crystal column 3
                    [3.5, 56.0, 0.5],      # panel 3: a = -3.5 -> module column 0, crystal column 12
                    [-56.0, -3.5, 0.5]],   # panel 6 (at -x, u = -y): a = +3.5 -> module column 1, crystal column 3
                   np.float32)
    want = [pack(0, 1, 2, 3, 0), pack(0, 0, 2, 12, 0), pack(0, 1, 0, 0, 11), pack(3, 1, 2, 3, 0), pack(3, 0, 2, 12, 0), pack(6, 1, 2, 3, 0)]
    assert list(O.locate(g, pts)) == want


# ----------------------------------------------------------------------------- decay law, positron range
def test_f18_source_of_the_paper():
    """1.6e8 atoms of 18F are `about 1.70e-2 MBq`; over the 120 s acquisition N0 (1 - exp(-lambda T)) of them
    decay.  [R34] the expected count is what a run simulates (n_pairs_total)."""
    lam = math.log(2.0) / W.F18_HALF_LIFE_S
    a0 = 1.6e8 * lam
    assert abs(a0 / 1.70e4 - 1.0) < 0.015                              # the paper rounds: 1.684e-2 MBq
    n = O.decay_count(a0, W.F18_HALF_LIFE_S, 120.0)
    assert n == round(1.6e8 * (1.0 - math.exp(-lam * 120.0))) == 2_007_947
    assert O.decay_count(1.0e6, 0.0, 10.0) == 10_000_000              # constant activity: A T
    assert abs(O.decay_count(a0, W.F18_HALF_LIFE_S, 1e9) / 1.6e8 - 1.0) < 1e-9    # every atom decays in the end


def test_deterministic_log_equals_the_library_logarithm():
    """[R34] the logarithm restated with +, -, *, / only (so that both sides get bit-identical decay times)."""
    rng = np.random.default_rng(17)
    z = np.concatenate([rng.uniform(0.0, 1.0, 20000), 1.0 - 10.0 ** rng.uniform(-15, -1, 5000), 10.0 ** rng.uniform(-12, 0, 5000), [1.0, 0.5, 0.25]])
    z = z[(z > 0) & (z <= 1.0)]
    got = np.array([O.det_log(float(v)) for v in z])
    want = np.log(z)
    assert np.all(np.abs(got - want) <= 4e-16 * np.maximum(np.abs(want), 1.0))
    y = np.concatenate([10.0 ** rng.uniform(-18, 0, 20000), rng.uniform(0.0, 1.0, 5000), [0.0, 0.25, 0.2499999]])
    y = y[y < 1.0]
    got = np.array([O.det_log1m(float(v)) for v in y])
    want = np.log1p(-y)
    assert np.all(np.abs(got[y > 0] / want[y > 0] - 1.0) < 1e-15) and O.det_log1m(0.0) == 0.0


def test_decay_times_follow_the_truncated_decay_law():
    """[R34] half-life 100 s observed for 250 s: decay times have the cdf (1 - exp(-lambda t)) / (1 - exp(-lambda T)) (KS),
    every time slice covers its own stretch of the time axis, and a half-life far longer than the acquisition gives back
    the constant-activity times of [R16]."""
    lam, T, n = math.log(2.0) / 100.0, 250.0, 20_000
    src = W.Source(activity_bq=1.0, half_life_s=100.0, duration_s=T)
    t = np.array([O.decay_time(src, 9, h, n) for h in range(n)])
    cdf = lambda x: (1.0 - np.exp(-lam * x)) / (1.0 - math.exp(-lam * T))
    assert t.min() > 0 and t.max() < T and stats.kstest(t, cdf).pvalue > 1e-3
    assert abs(np.mean(t < 100.0) - 0.5 / (1.0 - 0.5 ** 2.5)) < 0.01   # half of ALL atoms decay in the first half-life
    src4 = W.Source(activity_bq=1.0, half_life_s=100.0, duration_s=T, pairs_per_time_slice=n // 4)
    t4 = np.array([O.decay_time(src4, 9, h, n) for h in range(n)])
    edges = -np.log(1.0 - np.arange(5) / 4.0 * (1.0 - math.exp(-lam * T))) / lam
    for k in range(4):
        s = t4[k * n // 4:(k + 1) * n // 4]
        assert edges[k] <= s.min() and s.max() <= edges[k + 1]
    assert stats.kstest(t4, cdf).pvalue > 1e-3
    slow = W.Source(activity_bq=50.0, half_life_s=1e12, duration_s=n / 50.0)
    ref = W.Source(activity_bq=50.0)
    for h in (0, 17, n - 1):
        assert abs(O.decay_time(slow, 9, h, n) / O.decay_time(ref, 9, h, n) - 1.0) < 1e-8


def test_decay_times_of_a_cut_short_last_slice_stay_inside_the_acquisition():
    """[R34]: with explicit time slices of B pairs and N not a multiple of B, the last slice holds only N mod B
    histories and covers only the quantile range [kB/N, 1) -- stretching it to a full slice put q above 1, decay times past
    the end of the run (11.8 % of the last slice in the advisor's case) and, for long acquisitions, 1 - qP below 0.  The
    quantile of slice k is q = (kB + u len_k) / N with len_k = min(B, N - kB): every t0 < T, the last slice fills exactly
    the stretch between its edge and T, the other slices are where they were, and the whole run still follows the
    truncated decay law (KS)."""
    lam_of = lambda hl: math.log(2.0) / hl
    # the advisor's case: A0 = 5e7 Bq, half-life 0.02 s, T = 0.05 s, B = 100 000
    hl, T, B = 0.02, 0.05, 100_000
    n = O.decay_count(5.0e7, hl, T)
    assert n % B not in (0, B - 1) and n // B >= 5
    src = W.Source(activity_bq=5.0e7, half_life_s=hl, duration_s=T, pairs_per_time_slice=B)
    k_last = n // B
    last = np.array([O.decay_time(src, 9, h, n) for h in range(k_last * B, n)])
    P = 1.0 - math.exp(-lam_of(hl) * T)
    edge = -math.log(1.0 - (k_last * B / n) * P) / lam_of(hl)
    assert edge <= last.min() and last.max() < T
    assert last.min() < edge + 0.01 * (T - edge) and last.max() > T - 0.01 * (T - edge)      # ... and fills [edge, T)
    prev = np.array([O.decay_time(src, 9, h, n) for h in range((k_last - 1) * B, k_last * B, 37)])
    edge0 = -math.log(1.0 - ((k_last - 1) * B / n) * P) / lam_of(hl)
    assert edge0 <= prev.min() and prev.max() <= edge                                          # full slices unchanged
    # ten half-lives, where the stretched slice used to reach 1 - qP < 0
    hl, T, B, n = 1.0, 10.0, 3_000, 20_000
    src = W.Source(activity_bq=1.0, half_life_s=hl, duration_s=T, pairs_per_time_slice=B)
    t = np.array([O.decay_time(src, 9, h, n) for h in range(n)])
    cdf = lambda x: (1.0 - np.exp(-lam_of(hl) * x)) / (1.0 - math.exp(-lam_of(hl) * T))
    assert np.all(np.isfinite(t)) and t.min() > 0 and t.max() < T
    assert stats.kstest(t, cdf).pvalue > 1e-3
    assert np.all(np.diff([t[k * B:(k + 1) * B].max() for k in range(7)]) > 0)


def test_positron_range_is_an_isotropic_gaussian():
    """[R35] off (the paper's setting): the annihilation point IS the emission site.  On: the displacement is
    Gaussian on every axis with the stated FWHM (PAPER.md:145 quotes 0.102 mm for 18F), uncorrelated between axes."""
    n = 200_000
    off = W.source_point((1.0, -2.0, 3.0))
    assert np.array_equal(O.annihilation_sites(off, 4, 0, 100), O.decay_sites(off, 4, 0, 100))
    on = W.Source(0, (1.0, -2.0, 3.0), 0.5, 1e6, positron_fwhm_mm=0.102)
    d = O.annihilation_sites(on, 4, 0, n) - np.array([1.0, -2.0, 3.0])
    sigma = 0.102 / 2.354820045
    for k in range(3):
        assert stats.kstest(d[:, k] / sigma, "norm").pvalue > 1e-3
    c = np.cov(d.T) / sigma ** 2
    assert np.all(np.abs(c - np.eye(3)) < 0.02)
    # the voxel source is displaced from its sampled site, not from the grid origin
    rods = W.source_hot_rods()
    from dataclasses import replace
    a, b = O.decay_sites(rods, 5, 0, 1000), O.annihilation_sites(replace(rods, positron_fwhm_mm=0.102), 5, 0, 1000)
    assert 0.02 < np.abs(a - b).max() < 0.5 and abs(np.std(a - b) / sigma - 1.0) < 0.1


# ----------------------------------------------------------------------------- majorant regions, 3-4 layers
def two_material_tables(mu0, mu1):
    """Energy-independent photoelectric-only tables for two materials (first interactions = hits)."""
    f = lambda a, b: np.stack([np.full(W.N_ENERGIES, a, np.float32), np.full(W.N_ENERGIES, b, np.float32)])
    z = f(0.0, 0.0)
    return W.Tables(W.E_MIN_KEV, W.E_STEP_KEV, f(mu0, mu1), z, z)


def test_majorant_regions_cross_layer_faces_analytically():
    """[R19] a stack of a light layer (mu 0.02/mm, 4 mm) over a dense one (mu 0.2/mm, 6 mm), homogeneous (no reflector
    gaps), pencil beam along the depth axis: each layer is its own majorant region, so there is NOT ONE virtual
    collision, the unscattered fraction is exp(-mu1 L1 - mu2 L2) and the first-interaction depth follows the
    piecewise-exponential law (KS).  The same stack under one whole-panel majorant would need virtual collisions in
    the light layer -- the regions remove them without changing the physics."""
    mu1, mu2, L1, L2, n = 0.02, 0.2, 4.0, 6.0, 400_000
    layers = (W.Layer((1, 1), (12.0, 12.0), (0.0, 0.0), (0.0, 0.0), L1, 0.0, crystal_material=1),
              W.Layer((1, 1), (12.0, 12.0), (0.0, 0.0), (0.0, 0.0), L2, 0.0, crystal_material=0))
    res = O.simulate(slab(layers=layers), two_material_tables(mu2, mu1), beam(), n, seed=31, want_escape=True, threads=4)
    c = res.counters
    assert c["virtuals"] == 0 and c["step_vacuum"] == 0 and c["region_crossings"] > 0.8 * n
    p = math.exp(-mu1 * L1 - mu2 * L2)
    assert abs(np.mean(res.e_escape[:, 0] == 511.0) - p) < 4 * math.sqrt(p * (1 - p) / n)
    depth = res.hits.x.astype(np.float64) - 50.0
    def cdf(d):
        d = np.asarray(d, np.float64)
        a = 1.0 - np.exp(-mu1 * np.minimum(d, L1))
        b = math.exp(-mu1 * L1) * (1.0 - np.exp(-mu2 * np.maximum(d - L1, 0.0)))
        return (a + b) / (1.0 - p)
    assert stats.kstest(depth, cdf).pvalue > 1e-3
    layer = (res.hits.ids >> 18) & 3
    assert np.all(layer[depth < L1 - 1e-6] == 0) and np.all(layer[depth > L1 + 1e-6] == 1)
    # a photon entering from the BACK crosses the regions the other way
    back = O.simulate(slab(layers=layers), two_material_tables(mu2, mu1), beam(direction=(-1, 0, 0), pos=(70, 0, 0)), n, seed=32, want_escape=True, threads=4)
    assert abs(np.mean(back.e_escape[:, 0] == 511.0) - p) < 4 * math.sqrt(p * (1 - p) / n) and back.counters["virtuals"] == 0
    assert abs(np.mean(((back.hits.ids >> 18) & 3) == 1) - (1 - math.exp(-mu2 * L2)) / (1 - p)) < 0.005
    # same materials in consecutive layers: ONE region, exactly the single-layer run (no region events in the hash)
    same = (W.Layer((1, 1), (12.0, 12.0), (0.0, 0.0), (0.0, 0.0), L1), W.Layer((1, 1), (12.0, 12.0), (0.0, 0.0), (0.0, 0.0), L2))
    a = O.simulate(slab(layers=same), const_tables(0.05, 0, 0), beam(), 20_000, seed=33, want_hash=True)
    b = O.simulate(slab(L1 + L2), const_tables(0.05, 0, 0), beam(), 20_000, seed=33, want_hash=True)
    assert a.counters["region_crossings"] == 0 and np.array_equal(a.hits.x, b.hits.x) and len(a.hits) == len(b.hits) > 7000


def four_layer_scanner():
    """Four stacked layers with their own lattices, offsets, gaps and materials (PAPER.md:35 `the number of layers`,
    PAPER.md:141 three- and four-layer stacks): three majorant regions (materials 0 | 1, 1 | 0)."""
    base = tiny_scanner()
    layers = (W.Layer((3, 2), (1.25, 1.5), (0.25, 0.125), (0.125, 0.25), 1.0, 0.0, 0, -1),
              W.Layer((2, 2), (1.5, 1.25), (0.0, 0.25), (0.5, 0.0), 1.5, 0.25, 1, -1),
              W.Layer((4, 3), (1.0, 1.0), (0.125, 0.125), (0.0, 0.25), 1.25, 0.0, 1, -1),
              W.Layer((2, 1), (2.0, 3.5), (0.5, 0.5), (0.0, 0.0), 2.0, 0.125, 0, 1))
    return W.Geometry(3, layers, (2, 2), (4.0, 3.5), (4.5, 4.0), panel_pose=base.panel_pose)


def test_four_layer_indexing_against_brute_force_enumeration():
    g = four_layer_scanner()
    boxes, W_q, H_q, D_q = brute_force_boxes(g)
    assert len(boxes) == 4 * (6 + 4 + 12 + 2) and D_q == int(6.125 * Q)
    rng = np.random.default_rng(18)
    pts = []
    for p in range(3):
        loc = rng.uniform([-4.6, -4.1, -0.3], [4.6, 4.1, 6.4], (2500, 3))
        pose = g.panel_pose[p].astype(np.float64)
        pts.append(pose[0:3] + loc[:, :1] * pose[3:6] + loc[:, 1:2] * pose[6:9] + loc[:, 2:3] * pose[9:12])
    grid = np.arange(-4.25, 4.26, 0.125)
    ga, gb, gc = np.meshgrid(grid, grid[2:-2], np.arange(0.0, 6.13, 0.125), indexing="ij")
    pts.append(np.stack([20.0 + gc.ravel(), ga.ravel(), gb.ravel()], 1))
    xyz = np.concatenate(pts).astype(np.float32)
    got = O.locate(g, xyz)
    assert np.array_equal(got, brute_locate(g, boxes, W_q, H_q, D_q, xyz))
    u = O.unpack_ids(got[got != 0xFFFFFFFF])
    assert set(u["layer"]) == {0, 1, 2, 3} and set(u["crystal"][u["layer"] == 2]) == set(range(12))


def test_three_and_four_layer_stacks_transport(tables):
    """Energy conservation and region bookkeeping on a 3-layer and the 4-layer mixed-material scanner."""
    for g in (four_layer_scanner(), W.Geometry(3, four_layer_scanner().layers[:3], (2, 2), (4.0, 3.5), (4.5, 4.0), panel_pose=tiny_scanner().panel_pose)):
        res = O.simulate(g, tables, W.source_point((0.0, 0.0, 0.0)), 400_000, seed=35, want_escape=True, threads=4)
        assert res.counters["region_crossings"] > 10_000 and len(res.hits) > 1000
        dep = np.zeros((400_000, 2)); np.add.at(dep, (res.hits.history.astype(np.int64), ((res.hits.ids >> 4) & 1).astype(np.int64)), res.hits.e_keV.astype(np.float64))
        # deposits in the water-like layers' crystals are hits too; only interactions in a non-crystal material leave no hit
        assert np.all(dep + res.e_escape <= 511.0 + 1e-3)
        assert set(np.unique((res.hits.ids >> 18) & 3)) == set(range(len(g.layers)))
