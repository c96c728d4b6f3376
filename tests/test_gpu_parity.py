"""Parity of the CUDA path (through the C ABI) against the oracle.  All tests need a B200: `-m gpu`.

Bars (BASELINE.json north_star): indexing on deterministic rays bit-exact; >= 99.99 % of histories with an
identical outcome hash; for those, |dx| <= 1e-3 mm and |dE| <= 1e-3 keV; per-crystal histograms chi-square
p > 0.01; digitizer output equal on equal input."""
import numpy as np
import pytest

from oracle import gpet_oracle as O
from paper_2603_07327_b200 import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if torch.cuda.is_available():
    import parity_util as PU
    from paper_2603_07327_b200 import api

MIN_MATCH = 0.9999          # north_star
POS_TOL, E_TOL = 1e-3, 1e-3  # mm, keV (north_star)
TOF_TOL = 1e-4              # ns  (= 0.03 mm of path; fp32 path sums differ by ~1e-5 mm)


def run_both(run, tables, n=None, first=0):
    n = n or run.n_pairs
    g, gh, cnt = PU.gpu_simulate(run, tables, n_pairs=n, first_history=first)
    o = O.simulate(run.geometry, tables, run.source, n, run.seed, first_history=first, want_hash=True, threads=16)
    return g, gh, cnt, o


# ----------------------------------------------------------------------------- transport
def test_c0_every_hit(tables):
    """configs[0] in full: 1e5 pairs, seed 1, all hits (crystal id, xyz fp32, E keV) compared."""
    r = W.config_runs("C0")[0]
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] == 1.0 and cnt == len(o.hits) == res["n_hits_compared"] > 400
    assert np.array_equal(g["ids"], o.hits.ids) and np.array_equal(g["history"], o.hits.history)


RING_CASES = [("C1", 0), ("C2", 0), ("C2", 4), ("C3", 0), ("C3", 10), ("C3", 21)]


@pytest.mark.parametrize("cfg,idx", RING_CASES)
def test_ring_parity(tables, cfg, idx):
    """300k pairs span ~1200 blocks of the transport grid and a ragged tail (300k is no multiple of 256)."""
    r = W.config_runs(cfg, 300_001)[idx]
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH, res
    assert abs(cnt - len(o.hits)) <= 60
    assert PU.chi2_crystal_histograms(g["ids"], o.hits.ids) > 0.01
    layers = (g["ids"] >> 18) & 3
    assert layers.max() == len(r.geometry.layers) - 1                 # per-layer ids recorded


def test_c4_phantom_parity(tables):
    r = W.config_runs("C4", 150_000)[0]
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and res["n_hits_compared"] > 20_000, res
    assert o.counters["ph_compton"] > 10_000                         # the phantom really scatters


def test_offset_history_ranges_and_append(tables):
    """first_history offsets the counter-based streams; two appended calls equal one call."""
    r = W.config_runs("C3", 40_000)[5]
    g, gh, cnt, o = run_both(r, tables, n=40_000, first=123_456_789)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, first_history=123_456_789)
    assert res["frac"] >= MIN_MATCH
    geom, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    hb = api.HitBuffer.allocate(200_000)
    api.gpet_simulate(geom, m, s, 123_456_789, 15_000, r.seed, hb)
    api.gpet_simulate(geom, m, s, 123_456_789 + 15_000, 25_000, r.seed, hb)       # appends
    torch.cuda.synchronize()
    two = PU.canonical(hb.to_numpy())
    assert all(np.array_equal(two[k], g[k]) for k in PU.HIT_KEYS)


def test_overflow_is_counted_and_rerun_is_identical(tables):
    r = W.config_runs("C1", 50_000)[0]
    geom, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    small = api.HitBuffer.allocate(1000)
    api.gpet_simulate(geom, m, s, 0, 50_000, r.seed, small)
    torch.cuda.synchronize()
    n = small.count()
    assert n > 30_000 > small.capacity                                # dropped but counted
    runs = []
    for _ in range(2):
        hb = api.HitBuffer.allocate(n)
        api.gpet_simulate(geom, m, s, 0, 50_000, r.seed, hb)
        torch.cuda.synchronize()
        assert hb.count() == n
        runs.append(PU.canonical(hb.to_numpy()))
    assert all(np.array_equal(runs[0][k], runs[1][k]) for k in PU.HIT_KEYS)   # deterministic up to buffer order


def test_degenerate_inputs(tables):
    r = W.config_runs("C1", 1)[0]
    geom, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    hb = api.HitBuffer.allocate(64, n_hash=1)
    api.gpet_simulate(geom, m, s, 0, 0, r.seed, hb)                   # empty batch: no-op
    torch.cuda.synchronize()
    assert hb.count() == 0
    for first in (0, 7, 2 ** 33 + 5):                                 # single histories, also beyond 32 bits
        hb.n_hits.zero_()
        api.gpet_simulate(geom, m, s, first, 1, r.seed, hb)
        torch.cuda.synchronize()
        o = O.simulate(r.geometry, tables, r.source, 1, r.seed, first_history=first, want_hash=True)
        assert hb.count() == len(o.hits) and np.array_equal(hb.outcome_hash.cpu().numpy().view(np.uint64), o.outcome_hash[0])
    # source inside a panel box [R30]
    inside = W.Run("inside", W.geometry_c1(), W.source_point((58.0, 1.0, 2.0)), 20_000, 77)
    g, gh, cnt, o = run_both(inside, tables)
    assert PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash)["frac"] >= MIN_MATCH and cnt > 15_000


# ----------------------------------------------------------------------------- indexing
def test_locate_is_bit_exact(tables):
    from test_oracle_pins import tiny_scanner
    rng = np.random.default_rng(21)
    for geom, span in ((tiny_scanner(), 32.0), (W.geometry_c3(), 70.0), (W.geometry_c0(), 62.0)):
        xyz = rng.uniform(-span, span, (200_000, 3)).astype(np.float32)
        g = api.gpet_geometry_create(geom)
        got = api.gpet_geometry_locate(g, xyz)
        want = O.locate(geom, xyz)
        assert np.array_equal(got, want)
        assert (got != api.GPET_IDS_NONE).sum() > 50
    # dyadic points on crystal / module / layer faces of the axis-aligned C0 panel
    grid = np.arange(-6.5, 6.51, 0.0625, dtype=np.float32)
    a, b, c = np.meshgrid(grid, grid[::4], np.arange(-0.25, 10.5, 0.25, dtype=np.float32), indexing="ij")
    xyz = np.stack([50.0 + c.ravel(), a.ravel(), b.ravel()], 1).astype(np.float32)
    g = api.gpet_geometry_create(W.geometry_c0())
    assert np.array_equal(api.gpet_geometry_locate(g, xyz), O.locate(W.geometry_c0(), xyz))


def test_deterministic_rays_index_bit_exact(tables):
    """north_star: crystal/layer/panel indexing on deterministic test rays is bit-exact.  Pencil beams from
    several points, along and across the lattice, through reflector lines, module gaps and the layer offset."""
    rays = [((0, 0, 0), (1, 0, 0)), ((0, 0.3, 0.4), (1, 0.05, 0.02)), ((5, 1, -3), (0.3, 0.9, 0.1)), ((0, 0, 0), (0.5, 0.866, 0.3)),
            ((10, -4, 20), (-0.7, -0.7, -0.1)), ((0, 0, 0.5), (0, 1, 0)), ((0, 0, 0), (1, 0, 1e-3)), ((30, 30, 0), (1, 0.9, 0)),
            ((0, 0, 31.95), (1, 0.2, 0)), ((2, 3, 4), (-1, 0.01, 0.3))]
    total = 0
    for pos, d in rays:
        r = W.Run("ray", W.geometry_c3(), W.source_beam(pos, d, acolinearity_fwhm_deg=0.0), 4000, 91)
        g, gh, cnt, o = run_both(r, tables)
        assert np.array_equal(gh, o.outcome_hash)                     # every lattice decision of every history
        assert np.array_equal(g["ids"], o.hits.ids)
        total += cnt
    assert total > 20_000


# ----------------------------------------------------------------------------- digitizer
@pytest.mark.parametrize("level,ref_keV", [(0, 511.0), (1, 511.0), (2, 511.0), (1, 0.0)])
def test_digitizer_equals_oracle_on_oracle_hits(tables, level, ref_keV):
    """Same hits in (oracle-made, shuffled) -> singles and coincidences must be identical records, at the three readout
    levels and with the constant-fraction blur (blur_ref_keV = 0 [R25])."""
    n = 300_001
    src = W.source_point((10.0, 0.0, 4.0), activity_bq=5.0e7)         # hot enough for randoms and multiples
    o = O.simulate(W.geometry_c3(), tables, src, n, 404, first_history=1000, threads=8)
    dig = W.Digitizer(0.15, ref_keV, 350.0, 650.0, 4.0, level)
    osg, oco, _ = O.digitize(src, 404, 10 * n, o.hits, dig)
    perm = np.random.default_rng(2).permutation(len(o.hits))
    hb = PU.upload_hits(PU.oracle_hits_dict(o.hits), perm)
    s = api.DeviceSource(src)
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(n, len(o.hits)), dtype=torch.uint8, device="cuda")
    sg, co = api.SinglesBuffer.allocate(len(o.hits)), api.CoincBuffer.allocate(len(o.hits))
    api.gpet_digitize(s, 404, 10 * n, 1000, n, hb, len(o.hits), dig, scratch, sg, co)
    torch.cuda.synchronize()
    gs, gc = sg.to_numpy(), co.to_numpy()
    # Same hits in: every record of the join on (history, unit) is compared -- ids, xyz and the fp64 time bit for bit,
    # |dE| <= 1e-3 keV (the blur runs in fp32 on the device: a single within ~1e-4 keV of a window edge may be kept by
    # one side only, hence a symmetric difference of at most 2 singles, each of which can make or break one pair).
    shift = (5, 20, 26)[level]
    n_cmp = PU.compare_singles(gs, osg, shift, exact=True, max_symdiff=2)
    assert n_cmp >= len(osg.ids) - 2 and n_cmp > 50_000
    n_cmp = PU.compare_coincidences(gc, oco, exact=True, max_symdiff=4)
    assert n_cmp >= len(oco.ids_a) - 4
    assert len(oco.ids_a) > 5000 and np.sum(oco.history_a != oco.history_b) > 50
    assert np.all(np.diff(gs["t_s"]) >= 0)


@pytest.mark.parametrize("slice_pairs,first,n,chunked", [(0, 0, 200_000, False), (50_000, 100_000, 150_000, False), (50_000, 120_000, 150_000, False),
                                                        (50_000, 100_000, 150_016, True), (1_000, 120_500, 150_000, True), (100, 0, 20_000, True)])
def test_digitizer_time_sort_paths(tables, slice_pairs, first, n, chunked):
    """The time sort has two forms: coarse buckets sorted in shared memory when the batch's decay times are uniform over its
    time range (one slice, or whole slices [R16]) and fine counted buckets otherwise (a batch that starts or ends inside
    a slice).  Both must give the oracle's singles and coincidences, record for record, on either hit layout, including
    slices shorter than a chunk of the chunked layout."""
    from dataclasses import replace
    src = replace(W.source_point((10.0, 0.0, 4.0), activity_bq=5.0e7), pairs_per_time_slice=slice_pairs)
    n_total = 400_000
    o = O.simulate(W.geometry_c3(), tables, src, n, 406, first_history=first, threads=8)
    dig = W.Digitizer(0.15, 511.0, 350.0, 650.0, 4.0, 0)
    osg, oco, _ = O.digitize(src, 406, n_total, o.hits, dig)
    oh = PU.oracle_hits_dict(o.hits)
    s = api.DeviceSource(src)
    if chunked:                                                       # oracle hits laid out by 512-pair chunk, as gpet_simulate would
        hb = api.HitBuffer.allocate_chunked(n, 3.0)
        nc = (n + 511) // 512
        cap_c = hb.capacity // nc
        chunk = (oh["history"].astype(np.int64) - first) // 512
        order = np.argsort(chunk, kind="stable"); fill = np.bincount(chunk, minlength=nc)
        assert fill.max() <= cap_c
        pos = chunk[order] * cap_c + (np.arange(len(order)) - np.repeat(np.cumsum(fill) - fill, fill))
        for name, arr in (("history", hb.history), ("ids", hb.ids), ("x", hb.x), ("y", hb.y), ("z", hb.z), ("e_keV", hb.e_keV), ("tof_ns", hb.tof_ns)):
            v = np.ascontiguousarray(oh[name][order])
            arr[torch.from_numpy(pos).cuda()] = torch.from_numpy(v.view(np.int32) if v.dtype == np.uint32 else v).cuda()
        hb.chunk_fill[:nc] = torch.from_numpy(fill.astype(np.int32)).cuda()
        hb.n_hits.fill_(len(order))
        cap = hb.capacity
    else:
        hb = PU.upload_hits(oh, np.random.default_rng(5).permutation(len(o.hits))); cap = len(o.hits)
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(n, cap), dtype=torch.uint8, device="cuda")
    sg, co = api.SinglesBuffer.allocate(cap), api.CoincBuffer.allocate(cap)
    api.gpet_digitize(s, 406, n_total, first, n, hb, cap, dig, scratch, sg, co)
    torch.cuda.synchronize()
    gs = sg.to_numpy()
    assert PU.compare_singles(gs, osg, 5, exact=True, max_symdiff=2) >= len(osg.ids) - 2 > 3000
    assert PU.compare_coincidences(co.to_numpy(), oco, exact=True, max_symdiff=4) >= len(oco.ids_a) - 4 > 200
    assert np.all(np.diff(gs["t_s"]) >= 0)


def test_full_time_bucket_region_is_reported_not_silent(tables):
    """VERDICT r2 weak #5 / ADVICE r2: the coarse time buckets hold 832 records each and assume decay times spread evenly
    over the batch's time range.  Here the hits of ONE slice are presented as a batch of a hundred whole slices: every kept
    single falls into the first 1 % of the range, the regions there fill, and the call must say so (both counters
    UINT64_MAX, gpet.h) instead of returning a short list with rc 0.  The same hits in a batch that ends inside a slice
    take the counting path and give exactly the records of the slice digitized on its own."""
    from dataclasses import replace
    B = 20_000
    src = replace(W.source_point((10.0, 0.0, 4.0), activity_bq=5.0e7), pairs_per_time_slice=B)
    g, m, s = api.gpet_geometry_create(W.geometry_c3()), api.gpet_materials_load(tables), api.DeviceSource(src)
    hb = api.HitBuffer.allocate(3 * B)
    api.gpet_simulate(g, m, s, 0, B, 77, hb)
    torch.cuda.synchronize()
    nh = hb.count()
    assert B // 2 < nh <= hb.capacity
    dig, n_total = W.Digitizer(0.15, 511.0, 350.0, 650.0, 4.0, 0), 400 * B

    def digitize(n_pairs):
        scratch = torch.empty(api.gpet_digitize_scratch_bytes(n_pairs, nh), dtype=torch.uint8, device="cuda")
        sg, co = api.SinglesBuffer.allocate(nh), api.CoincBuffer.allocate(nh)
        api.gpet_digitize(s, 77, n_total, 0, n_pairs, hb, nh, dig, scratch, sg, co)
        torch.cuda.synchronize()
        return sg, co

    sg, co = digitize(100 * B)                                         # whole slices -> coarse regions -> they fill
    assert int(sg.n_singles.item()) == -1 and int(co.n_coinc.item()) == -1      # UINT64_MAX through an int64 tensor
    sg1, co1 = digitize(B)                                             # the slice on its own: uniform, coarse path, complete
    sg2, co2 = digitize(100 * B - 7)                                   # ends inside a slice -> counting path, no limit
    a, b = sg1.to_numpy(), sg2.to_numpy()
    assert len(a["ids"]) > B // 5 and all(np.array_equal(a[k], b[k]) for k in a)
    a, b = co1.to_numpy(), co2.to_numpy()
    assert len(a["ids_a"]) > B // 100 and all(np.array_equal(a[k], b[k]) for k in a)


def test_digitizer_empty_and_tiny(tables):
    src = W.source_point()
    s = api.DeviceSource(src)
    hb = api.HitBuffer.allocate(16)
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(100, 0), dtype=torch.uint8, device="cuda")
    sg, co = api.SinglesBuffer.allocate(16), api.CoincBuffer.allocate(16)
    api.gpet_digitize(s, 1, 100, 0, 100, hb, 0, W.Digitizer(), scratch, sg, co)
    torch.cuda.synchronize()
    assert int(sg.n_singles.item()) == 0 and int(co.n_coinc.item()) == 0


def test_end_to_end_coincidences(tables):
    """GPU hits -> GPU digitizer against oracle hits -> oracle digitizer (C1 shape)."""
    r = W.config_runs("C1", 400_000)[0]
    geom, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    hb = api.HitBuffer.allocate(600_000)
    api.gpet_simulate(geom, m, s, 0, r.n_pairs, r.seed, hb)
    torch.cuda.synchronize()
    nh = hb.count()
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(r.n_pairs, nh), dtype=torch.uint8, device="cuda")
    co = api.CoincBuffer.allocate(nh)
    api.gpet_digitize(s, r.seed, r.n_pairs, 0, r.n_pairs, hb, nh, r.digitizer, scratch, None, co)    # coincidences only
    torch.cuda.synchronize()
    gc = co.to_numpy()
    o = O.simulate(r.geometry, tables, r.source, r.n_pairs, r.seed, threads=8)
    _, oco, _ = O.digitize(r.source, r.seed, r.n_pairs, o.hits, r.digitizer)
    key = lambda c: set(zip(np.asarray(c["history_a"]).tolist(), np.asarray(c["history_b"]).tolist(), (np.asarray(c["ids_a"]) >> 5).tolist(),
                            (np.asarray(c["ids_b"]) >> 5).tolist()))
    kg, ko = key(gc), key(dict(history_a=oco.history_a, history_b=oco.history_b, ids_a=oco.ids_a, ids_b=oco.ids_b))
    assert len(ko) > 20_000 and len(kg ^ ko) <= 1e-3 * len(ko)
    assert 0.05 < len(ko) / r.n_pairs < 0.065                         # ~0.057 coincidences per pair


def test_run_host_matches_device_path(tables):
    r = W.config_runs("C3", 100_000)[3]
    geom, m = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables)
    host, counts = api.gpet_run_host(geom, m, r.source, r.n_pairs, 0, r.n_pairs, r.seed, r.digitizer, want_hits=True, want_singles=True)
    s = api.DeviceSource(r.source)
    hb = api.HitBuffer.allocate(300_000)
    api.gpet_simulate(geom, m, s, 0, r.n_pairs, r.seed, hb)
    torch.cuda.synchronize()
    nh = hb.count()
    assert counts["n_hits"] == nh
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(r.n_pairs, nh), dtype=torch.uint8, device="cuda")
    sg, co = api.SinglesBuffer.allocate(nh), api.CoincBuffer.allocate(nh)
    api.gpet_digitize(s, r.seed, r.n_pairs, 0, r.n_pairs, hb, nh, r.digitizer, scratch, sg, co)
    torch.cuda.synchronize()
    gs, gc = sg.to_numpy(), co.to_numpy()
    assert counts["n_singles"] == len(gs["ids"]) and counts["n_coinc"] == len(gc["ids_a"]) > 4000
    nc = counts["n_coinc"]
    assert np.array_equal(host["coinc"][0][:nc].numpy().view(np.uint32), gc["ids_a"])
    assert np.array_equal(host["coinc"][7][:nc].numpy(), gc["t_s"])
    assert np.array_equal(host["singles"][6][:counts["n_singles"]].numpy(), gs["t_s"])
    hh = {k: host["hits"][i][:nh].numpy() for i, k in enumerate(PU.HIT_KEYS)}
    hh["history"], hh["ids"] = hh["history"].view(np.uint32), hh["ids"].view(np.uint32)
    a, b = PU.canonical(hh), PU.canonical(hb.to_numpy())
    assert all(np.array_equal(a[k], b[k]) for k in PU.HIT_KEYS)


# ----------------------------------------------------------------------------- full size, bench launch configuration
def gpu_product_run(run, tables, hits_per_pair, n=None, reps=2):
    """The PRODUCT build (no outcome hashes, 128 slots per warp, chunked hit layout -- what bench.py times): transport +
    digitizer of one batch.  Returns (hits, singles, coincidences) as numpy dicts and the device time of the two calls."""
    n = n or run.n_pairs
    geom, m, s = api.gpet_geometry_create(run.geometry), api.gpet_materials_load(tables), api.DeviceSource(run.source)
    hb = api.HitBuffer.allocate_chunked(n, hits_per_pair)
    cap = hb.capacity
    sg, co = api.SinglesBuffer.allocate(cap), api.CoincBuffer.allocate(cap // 4)
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(n, cap), dtype=torch.uint8, device="cuda")
    st = torch.cuda.current_stream()
    best = float("inf")
    for rep in range(reps):                                           # best of the passes after the first
        hb.reset()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(st)
        api.gpet_simulate(geom, m, s, 0, n, run.seed, hb, st)
        api.gpet_digitize(s, run.seed, n, 0, n, hb, cap, run.digitizer, scratch, sg, co, st)
        b.record(st)
        torch.cuda.synchronize()
        if rep:
            best = min(best, a.elapsed_time(b))
    assert hb.dropped() == 0, "hit buffer overflow in test"
    assert int(co.n_coinc.item()) <= co.capacity
    return hb.to_numpy(), sg.to_numpy(), co.to_numpy(), best


def whole_run_against_oracle(run, tables, hits_per_pair, min_coinc=100_000, reps=2):
    """One config position at its FULL size through the product build, next to the oracle's whole run: hits of every
    history, then singles and coincidences (each side digitizes its own hits).  Budgets: north_star's 1e-4 of the
    histories may differ in their discrete outcome (fp32 vs fp64 decisions); the records of those histories may differ or
    be missing on one side, so the joins allow 1e-4 of each list (+ 2 for window-edge flips of the blur)."""
    n = run.n_pairs
    g, gs, gc, ms = gpu_product_run(run, tables, hits_per_pair, reps=reps)
    o = O.simulate(run.geometry, tables, run.source, n, run.seed, threads=16)
    res = PU.compare_hits_unhashed(g, PU.oracle_hits_dict(o.hits), n, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and res["n_hits_compared"] >= (1.0 - 5e-4) * len(o.hits), res
    assert PU.chi2_crystal_histograms(g["ids"], o.hits.ids) > 0.01
    osg, oco, _ = O.digitize(run.source, run.seed, n, o.hits, run.digitizer)
    bs, bc = int(1e-4 * len(osg.ids)) + 2, int(1e-4 * len(oco.ids_a)) + 2
    ns = PU.compare_singles(gs, osg, 20, exact=False, max_symdiff=bs, max_bad=bs)
    nc = PU.compare_coincidences(gc, oco, exact=False, max_symdiff=bc, max_bad=bc)
    assert ns >= len(osg.ids) - bs and nc >= len(oco.ids_a) - bc and nc > min_coinc
    assert np.all(np.diff(gs["t_s"]) >= 0) and np.all(np.diff(gc["t_s"]) >= 0)
    res.update(n_hits=len(g["ids"]), n_singles_compared=ns, n_coinc_compared=nc, ms=ms, pairs_per_s=n / (ms * 1e-3))
    return g, o, res


def test_c1_full_size_hash_build_whole_run(tables):
    """configs[1] at its full 1e7 pairs through the parity (hash) build: the outcome hash of EVERY history next to the
    oracle's, every hit of the agreeing histories within tolerance, + properties that hold at any size."""
    r = W.config_runs("C1")[0]
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and res["n_hits_compared"] > 7_600_000, res
    assert 0.76 < cnt / r.n_pairs < 0.79                              # 0.77 hits per pair
    counts = np.bincount(g["ids"] >> 26, minlength=12)
    from scipy import stats
    assert stats.chisquare(counts).pvalue > 1e-4                      # centred source: every panel equally hit
    up, down = int((g["z"] > 0).sum()), int((g["z"] < 0).sum())
    assert abs(up - down) < 5 * np.sqrt(up + down)                    # axial symmetry


def test_c1_full_size_product_build_whole_run(tables):
    """configs[1] at 1e7 pairs in the launch configuration bench.py times (product build, chunked hits, scratch and
    buffers sized the same way): all hits, singles and coincidences next to the oracle's whole run."""
    r = W.config_runs("C1")[0]
    g, o, res = whole_run_against_oracle(r, tables, 1.2)
    print("C1 whole run:", res)
    assert 0.32 < res["n_singles_compared"] / r.n_pairs < 0.35 and 0.055 < res["n_coinc_compared"] / r.n_pairs < 0.060


SWEEP = [("C2", i) for i in range(5)] + [("C3", i) for i in range(22)]
SWEEP_RATE = {}


@pytest.mark.parametrize("cfg,idx", SWEEP)
def test_c2_c3_every_position_at_full_size(tables, cfg, idx):
    """BASELINE.json configs[2] (5 radial offsets) and configs[3] (11 radial x 2 axial offsets): EVERY position at its
    full 1e7 pairs through the product build -- hits, singles and coincidences against the oracle's whole run,
    per-layer ids present, per-crystal chi-square."""
    r = W.config_runs(cfg)[idx]
    g, o, res = whole_run_against_oracle(r, tables, 2.0)
    SWEEP_RATE[(cfg, idx)] = res["pairs_per_s"]
    print(f"{r.name}: {res}")
    assert ((g["ids"] >> 18) & 3).max() == 1 and ((o.hits.ids >> 18) & 3).max() == 1   # both layers recorded
    assert 0.65 < res["n_hits"] / r.n_pairs < 1.50


def test_sweep_rates_are_reported(tables):
    """pairs/s of every sweep position (transport + digitizer, product build).  Off-centre positions produce up to 1.9 x
    the hits of the centred one, so they are not expected to run at the centred rate; the 10 % bar of north_star is for
    the three layer configurations at the same position (test_layer_configurations_run_within_ten_percent)."""
    if not SWEEP_RATE:
        pytest.skip("sweep did not run in this session")
    for k in sorted(SWEEP_RATE):
        print(k, f"{SWEEP_RATE[k]:.3e} pairs/s")
    assert min(SWEEP_RATE.values()) > 1e9


def test_c4_full_run_in_time_slices(tables):
    """configs[4] in full: 1e9 pairs in 16 time slices of 6.25e7, transported through the phantom and the detector and
    digitized to coincidence list-mode, every slice in the launch configuration bench.py times.  One slice is also run
    with outcome hashes and singles output, and the oracle recomputes blocks of its histories (hits, hashes and the
    singles of those histories, which depend on no other history: no pile-up [R24])."""
    r = W.config_runs("C4")[0]
    B = r.source.pairs_per_time_slice
    assert r.n_pairs == 10 ** 9 and B * 16 == r.n_pairs
    geom, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    hb = api.HitBuffer.allocate_chunked(B, 1.2)                       # the layout bench.py times
    cap = hb.capacity
    co = api.CoincBuffer.allocate(cap // 8)
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(B, cap), dtype=torch.uint8, device="cuda")
    n_hits = n_coinc = 0
    t_last = -1.0
    for k in range(16):
        hb.reset()
        api.gpet_simulate(geom, m, s, k * B, B, r.seed, hb)
        api.gpet_digitize(s, r.seed, r.n_pairs, k * B, B, hb, cap, r.digitizer, scratch, None, co)
        torch.cuda.synchronize()
        nh, nc = hb.count(), int(co.n_coinc.item())
        assert hb.dropped() == 0 and nc <= co.capacity
        n_hits += nh; n_coinc += nc
        t = co.t_s[:nc]
        assert float(t[0]) > t_last and bool((t[1:] >= t[:-1]).all())  # list-mode is time-ordered across slices
        assert k * B / 1e6 <= float(t[0]) and float(t[-1]) < (k + 1) * B / 1e6 + 1e-6   # slice k covers its own time interval [R16]
        t_last = float(t[-1])
    assert 0.73 < n_hits / r.n_pairs < 0.76 and 0.036 < n_coinc / r.n_pairs < 0.040
    # one slice again with hashes and singles; oracle on sampled blocks
    k = 11
    del hb, co, scratch
    cap = int(0.9 * B)                                                # dense layout for the slice read back to the host
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(B, cap), dtype=torch.uint8, device="cuda")
    hb = api.HitBuffer.allocate(cap, n_hash=B)
    sg, co = api.SinglesBuffer.allocate(cap), api.CoincBuffer.allocate(cap // 8)
    api.gpet_simulate(geom, m, s, k * B, B, r.seed, hb)
    api.gpet_digitize(s, r.seed, r.n_pairs, k * B, B, hb, cap, r.digitizer, scratch, sg, co)
    torch.cuda.synchronize()
    gh = hb.outcome_hash.cpu().numpy().view(np.uint64).reshape(-1, 2)
    g, gs = hb.to_numpy(), sg.to_numpy()
    rng = np.random.default_rng(6)
    same = tot = n_singles_cmp = 0
    for st in np.concatenate([[0, B - 2048], rng.integers(0, B - 2048, 10)]):
        first = k * B + int(st)
        o = O.simulate(r.geometry, tables, r.source, 2048, r.seed, first_history=first, want_hash=True, threads=4)
        ok = np.all(gh[st:st + 2048] == o.outcome_hash, axis=1)
        same += int(ok.sum()); tot += 2048
        sel = (g["history"] >= first) & (g["history"] < first + 2048)
        part = PU.canonical({kk: v[sel] for kk, v in g.items()})
        PU.compare_hits(part, PU.oracle_hits_dict(o.hits), gh[st:st + 2048], o.outcome_hash, first_history=first,
                        pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
        if ok.all():                                                  # same hits in -> the same singles out
            osg, _, _ = O.digitize(r.source, r.seed, r.n_pairs, o.hits, r.digitizer)
            ss = (gs["history"] >= first) & (gs["history"] < first + 2048)
            # joined on (history, module): always compared; a blurred energy within 1e-4 keV of a window edge may flip one
            n_cmp = PU.compare_singles({kk: v[ss] for kk, v in gs.items()}, osg, 20, exact=False, max_symdiff=1)
            assert n_cmp >= len(osg.ids) - 1
            n_singles_cmp += n_cmp
    assert same / tot >= MIN_MATCH and n_singles_cmp > 3000


# ----------------------------------------------------------------------------- north_star: layers cost nothing
def test_layer_configurations_run_within_ten_percent(tables):
    """north_star / PAPER.md:121 (Table 1: the layer extension adds no measurable time): the single-layer (C1), aligned
    split (C2) and offset dual-layer (C3) rings, centred source, 1e7 pairs, transport + digitizer, must run within 10 %
    of each other in pairs/s."""
    times = {}
    for cfg in ("C1", "C2", "C3"):
        r = W.config_runs(cfg)[0]
        n = r.n_pairs
        geom, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
        cap = int(1.2 * n)
        hb, co = api.HitBuffer.allocate(cap), api.CoincBuffer.allocate(cap // 4)
        scratch = torch.empty(api.gpet_digitize_scratch_bytes(n, cap), dtype=torch.uint8, device="cuda")
        st = torch.cuda.current_stream()
        best = float("inf")
        for rep in range(5):
            hb.n_hits.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st)
            api.gpet_simulate(geom, m, s, 0, n, r.seed, hb, st)
            api.gpet_digitize(s, r.seed, n, 0, n, hb, cap, r.digitizer, scratch, None, co, st)
            b.record(st)
            torch.cuda.synchronize()
            if rep >= 2:
                best = min(best, a.elapsed_time(b))
        assert hb.count() <= cap
        times[cfg] = best
        del hb, co, scratch
    assert max(times.values()) / min(times.values()) < 1.10, times


# ----------------------------------------------------------------------------- sensitivity profiles
def test_sensitivity_profiles_against_the_oracle(tables):
    """S(r, E) over radial offsets and the paper's four energy windows (PAPER.md:63, 16 % blur, 3 ns): the CUDA path's
    coincidence counts equal the oracle's on the same seeded histories (a blurred energy within ~1e-4 keV of a window
    edge, or one of the ~1e-5 mismatching histories, may move a count by one or two), 1CL vs 2CL differ by a few percent
     with the single layer ahead (the offset front layer has less crystal), and the formula is symmetric."""
    from paper_2603_07327_b200 import sensitivity as S
    positions = [(0.0, 0.0, 0.0), (25.0, 0.0, 0.0), (50.0, 0.0, 0.0), (0.0, 0.0, 16.0)]
    n = 200_000
    got = {}
    for name, geom in (("1CL", W.geometry_c1()), ("2CL", W.geometry_c3())):
        got[name] = S.sensitivity(geom, tables, positions, n_pairs=n, seed=70)
        for k, pos in enumerate(positions):
            src = W.source_point(pos, activity_bq=1.7e4)
            o = O.simulate(geom, tables, src, n, 70 + k, threads=8)
            for j, (lo, hi) in enumerate(S.PAPER_WINDOWS_KEV):
                dig = W.Digitizer(0.16, 511.0, lo, hi, 3.0, 1)
                _, oco, _ = O.digitize(src, 70 + k, n, o.hits, dig)
                assert abs(round(got[name][k, j] * n) - len(oco.ids_a)) <= 3, (name, pos, lo, len(oco.ids_a))
    assert np.all(np.diff(got["1CL"], axis=1) < 0)                     # narrower window, fewer coincidences
    d = S.delta_sym_percent(got["1CL"], got["2CL"])
    assert np.all(d > 0.0) and np.all(d < 20.0), d
    assert np.allclose(S.delta_sym_percent(got["2CL"], got["1CL"]), -d)


def test_two_stream_pipeline_gives_the_same_results(tables):
    """gpet_simulate of batch k+1 on one stream beside gpet_digitize of batch k on another (transport CTA of 16 warps, the
    way bench.py's pipeline runs) must give, per batch, exactly the hits-derived coincidences of the serial run."""
    r = W.config_runs("C3", 1_000_000)[3]
    n = r.n_pairs
    geom, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    cap = 2 * n
    def alloc():
        return (api.HitBuffer.allocate(cap), api.CoincBuffer.allocate(cap // 4),
                torch.empty(api.gpet_digitize_scratch_bytes(n, cap), dtype=torch.uint8, device="cuda"))
    ref = []
    hb, co, sc = alloc()
    for k in range(4):                                                # serial reference, default CTA
        hb.n_hits.zero_()
        api.gpet_simulate(geom, m, s, k * n, n, r.seed, hb)
        api.gpet_digitize(s, r.seed, 4 * n, k * n, n, hb, cap, r.digitizer, sc, None, co)
        torch.cuda.synchronize()
        ref.append(co.to_numpy())
    try:
        assert api.gpet_set_transport_warps(16) == 16
        bufs = [alloc(), alloc()]
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        sim_done = [torch.cuda.Event() for _ in range(2)]; dig_done = [torch.cuda.Event() for _ in range(2)]
        got = []
        for k in range(4):
            i = k & 1
            hbi, coi, sci = bufs[i]
            if k >= 2:
                sb.synchronize(); got.append(coi.to_numpy())          # batch k-2 is complete: read it before its buffers are reused
                sa.wait_event(dig_done[i])
            with torch.cuda.stream(sa):
                hbi.n_hits.zero_()
                api.gpet_simulate(geom, m, s, k * n, n, r.seed, hbi, sa)
            sim_done[i].record(sa)
            sb.wait_event(sim_done[i])
            api.gpet_digitize(s, r.seed, 4 * n, k * n, n, hbi, cap, r.digitizer, sci, None, coi, sb)
            dig_done[i].record(sb)
        torch.cuda.synchronize()
        got += [bufs[0][1].to_numpy(), bufs[1][1].to_numpy()]
    finally:
        assert api.gpet_set_transport_warps(0) == 20                  # back to the default CTA
    for a, b in zip(ref, got):
        assert len(a["ids_a"]) > 40_000 and all(np.array_equal(a[k], b[k]) for k in a)


def tilted_box_scanner():
    """Six panels on the faces of a cube around the origin, the whole detector tilted: no panel axis is a coordinate
    axis, so the generic panel search (bounding spheres + 3-D slab tests) and the generic kernel variant run."""
    faces = [((1, 0, 0), (0, 1, 0), (0, 0, 1)), ((-1, 0, 0), (0, -1, 0), (0, 0, 1)), ((0, 1, 0), (-1, 0, 0), (0, 0, 1)),
             ((0, -1, 0), (1, 0, 0), (0, 0, 1)), ((0, 0, 1), (1, 0, 0), (0, 1, 0)), ((0, 0, -1), (1, 0, 0), (0, -1, 0))]
    a, b = np.radians(23.0), np.radians(-11.0)
    rz = np.array([[np.cos(a), -np.sin(a), 0], [np.sin(a), np.cos(a), 0], [0, 0, 1]])
    rx = np.array([[1, 0, 0], [0, np.cos(b), -np.sin(b)], [0, np.sin(b), np.cos(b)]])
    rot = rz @ rx
    poses = []
    for w, u, v in faces:
        w, u, v = (rot @ np.array(t, float) for t in (w, u, v))
        assert np.allclose(np.cross(u, v), w)
        poses.append(np.concatenate([40.0 * w, u, v, w]))
    return W.Geometry(6, W.geometry_c3().layers, (2, 2), (16.0, 16.0), (16.0, 16.0), panel_pose=np.array(poses, np.float32))


@pytest.mark.parametrize("pos", [(0.0, 0.0, 0.0), (12.0, -7.0, 20.0)])
def test_generic_panel_search_parity(tables, pos):
    geom = tilted_box_scanner()
    r = W.Run("tilted", geom, W.source_point(pos), 300_001, 55)
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and cnt > 50_000, res
    assert len(np.unique(g["ids"] >> 26)) == 6 and o.counters["exits"] > 10_000
    # the product build (no hashes) of the same generic variant writes the same hits
    gm, m, s = api.gpet_geometry_create(geom), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    hb = api.HitBuffer.allocate(3 * r.n_pairs)
    api.gpet_simulate(gm, m, s, 0, r.n_pairs, r.seed, hb)
    torch.cuda.synchronize()
    plain = PU.canonical(hb.to_numpy())
    assert all(np.array_equal(plain[k], g[k]) for k in PU.HIT_KEYS)


def test_mixed_materials_virtual_collisions_and_voxel_source_without_phantom(tables):
    """Paths the five configs never reach: a front layer of a lighter material (its own majorant region [R19]), a reflector
    made of matter under the crystal's majorant (virtual collisions (interactions that deposit outside any crystal record
    no hit [R20]), and an activity-map source with no phantom (generic kernel variant)."""
    front = W.Layer((15, 15), (1.0, 1.0), (0.1, 0.1), (0.5, 0.5), 6.0, 0.0, crystal_material=1, gap_material=1)
    back = W.Layer((16, 16), (1.0, 1.0), (0.1, 0.1), (0.0, 0.0), 4.0, 0.1, crystal_material=0, gap_material=1)
    geom = W.Geometry(12, (front, back), (2, 4), (16.0, 16.0), (16.0, 16.0), ring_inner_radius_mm=55.0)
    rods = W.source_hot_rods()
    src = W.Source(1, (0, 0, 0), 0.5, 1e6, 0, rods.activity, None, -1, rods.dims, rods.voxel_mm, rods.origin_mm)
    r = W.Run("mixed", geom, src, 300_001, 77)
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and cnt > 100_000, res
    c = o.counters
    # two majorant regions [R19]: the water-like front layer is homogeneous (no virtual collisions there), the back layer's
    # water-like reflector sits under the LYSO majorant (virtual collisions remain)
    assert c["virtuals"] > 10_000 and c["region_crossings"] > 50_000 and c["ph_steps"] == 0
    layers = (g["ids"] >> 18) & 3
    assert (layers == 0).sum() > 1000 and (layers == 1).sum() > 50_000


# ----------------------------------------------------------------------------- the paper's own scanners
def test_paper_scanners_parity_and_the_split_layer_identity(tables):
    """H2RSPET-1CL / -1CL-split / -2CL (10 panels, R = 85 mm, six 51 x 51 modules): parity with the oracle, and
    the paper's own validation (Fig. 3 left) in its strongest form: with radially connected 5 mm crystals the
    split scanner's hits are bit-identical to the single-layer scanner's except for the layer id (layer = depth >= 5 mm)."""
    out = {}
    for cfg in ("P1", "P2", "P3"):
        r = W.config_runs(cfg, 300_001)[0]
        r2 = W.Run(r.name, r.geometry, r.source, r.n_pairs, 61, r.digitizer)      # one seed for all three
        g, gh, cnt, o = run_both(r2, tables)
        # 341 mm panels: the grazing-entry tail of the position error is longer than on BASELINE's 64 mm rings;
        # histories with a hit beyond 1e-3 mm count against the 99.99 % like any other disagreement
        res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
        assert res["frac"] >= MIN_MATCH and cnt > 350_000, (cfg, res)
        out[cfg] = g
    a, b = out["P1"], out["P2"]
    assert len(a["ids"]) == len(b["ids"])
    strip = ~np.uint32(3 << 18)
    assert np.array_equal(a["ids"] & strip, b["ids"] & strip) and all(np.array_equal(a[k], b[k]) for k in ("history", "x", "y", "z", "e_keV", "tof_ns"))
    assert np.all((a["ids"] >> 18) & 3 == 0) and ((b["ids"] >> 18) & 3).max() == 1
    ratio = len(out["P3"]["ids"]) / len(a["ids"])
    assert 0.96 < ratio < 0.99                                        # paper Table 1: 2 620 170 / 2 671 908 = 0.981


# ----------------------------------------------------------------------------- chunked hit layout (the one bench.py times)
@pytest.mark.parametrize("cfg,idx,n", [("C1", 0, 300_001), ("C3", 10, 200_000), ("C4", 0, 100_000)])
def test_chunked_hit_layout_equals_the_dense_one(tables, cfg, idx, n):
    """gpet_hits.chunk_fill: hits grouped per 512-pair chunk, digitized by a shared-memory sort per chunk.  Same hits as
    the dense layout (as a set) and identical singles and coincidences, record for record; a region that is too small
    drops hits and says so."""
    r = W.config_runs(cfg, n)[idx]
    first = 5_000_000
    geom, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    dense = api.HitBuffer.allocate(3 * n)
    chunk = api.HitBuffer.allocate_chunked(n, 3.0)
    api.gpet_simulate(geom, m, s, first, n, r.seed, dense)
    api.gpet_simulate(geom, m, s, first, n, r.seed, chunk)
    torch.cuda.synchronize()
    assert chunk.count() == dense.count() and chunk.dropped() == 0
    a, b = PU.canonical(dense.to_numpy()), PU.canonical(chunk.to_numpy())
    assert all(np.array_equal(a[k], b[k]) for k in PU.HIT_KEYS)
    fill = chunk.chunk_fill[:-1].cpu().numpy()
    assert len(fill) == (n + 511) // 512 and int(fill.sum()) == dense.count()
    out = []
    for hb in (dense, chunk):
        cap = hb.capacity
        scratch = torch.empty(api.gpet_digitize_scratch_bytes(n, cap), dtype=torch.uint8, device="cuda")
        sg, co = api.SinglesBuffer.allocate(cap), api.CoincBuffer.allocate(cap)
        api.gpet_digitize(s, r.seed, 20_000_000, first, n, hb, cap, r.digitizer, scratch, sg, co)
        torch.cuda.synchronize()
        out.append((sg.to_numpy(), co.to_numpy()))
    (s0, c0), (s1, c1) = out
    assert len(s0["ids"]) > 0.2 * n * (0.3 if cfg == "C4" else 1) and all(np.array_equal(s0[k], s1[k]) for k in s0)
    assert len(c0["ids_a"]) > 100 and all(np.array_equal(c0[k], c1[k]) for k in c0)
    # regions too small: hits are dropped, counted, and the total is still reported
    tight = api.HitBuffer.allocate_chunked(n, 0.25)
    api.gpet_simulate(geom, m, s, first, n, r.seed, tight)
    torch.cuda.synchronize()
    assert tight.count() == dense.count() and tight.dropped() > 0
    assert tight.dropped() == dense.count() - int(np.minimum(tight.chunk_fill[:-1].cpu().numpy(), 128).sum())


# ----------------------------------------------------------------------------- branches no config reaches
def test_weighted_activity_map_parity(tables):
    """[R13] decay sites from a map with unequal activities (integer weights, `first cumulative weight above the target`
    search): outcome hashes and hits against the oracle on C1's ring, and voxel populations in proportion."""
    rng = np.random.default_rng(3)
    dims = (24, 20, 16)
    act = rng.choice(np.array([0.0, 0.05, 0.3, 1.0], np.float32), size=(dims[2], dims[1], dims[0]), p=[0.4, 0.2, 0.2, 0.2])
    src = W.Source(1, (0, 0, 0), 0.5, 1e6, 0, act, None, -1, dims, (0.5, 0.25, 1.0), (-6.0, -2.5, -8.0))
    r = W.Run("weighted", W.geometry_c1(), src, 300_001, 88)
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and cnt > 200_000, res


def test_phantom_rayleigh_parity_and_thomson_distribution(tables):
    """[R17, R20] Rayleigh scattering inside the phantom (no config's water has mu_R > 0): hash parity with the oracle in
    a thick medium (several deflections per photon), and in a thin one the single deflections of the CUDA path's own
    photons follow the Thomson distribution (the same check that pins the oracle)."""
    from test_oracle_pins import phantom_rayleigh_setup, single_rayleigh_deflections, check_thomson
    geom, t, src = phantom_rayleigh_setup(mu_r=4.0)
    r = W.Run("ph_rayleigh", geom, src, 300_001, 12)
    g, gh, cnt, o = run_both(r, t)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and cnt > 0.99 * 2 * r.n_pairs, res   # every photon is caught, bar the open channels along the cube's edges
    geom, t, src = phantom_rayleigh_setup()
    r = W.Run("ph_rayleigh_thin", geom, src, 2_000_000, 12)
    g, gh, cnt = PU.gpu_simulate(r, t)
    check_thomson(*single_rayleigh_deflections(g, gh, r.n_pairs))


def test_panel_search_tie_goes_to_the_lowest_index(tables):
    """[R6] diagonal rays of a square ring reach two overlapping front faces at bit-identical distances: the CUDA path
    must enter the lower-index panel, as the oracle does (pinned on the CPU by exact arithmetic)."""
    from test_oracle_pins import square_ring, const_tables
    geom, t = square_ring(), const_tables(5.0, 0.0, 0.0)
    s2 = float(np.float32(1.0 / np.sqrt(2.0)))
    for d, want_a, want_b in (((s2, s2, 0), 0, 2), ((s2, -s2, 0), 0, 1), ((-s2, s2, 0), 1, 0), ((-s2, -s2, 0), 2, 0)):
        r = W.Run("tie", geom, W.source_beam((0.0, 0.0, 0.0), d), 2000, 5)
        g, gh, cnt, o = run_both(r, t)
        assert np.array_equal(gh, o.outcome_hash) and np.array_equal(g["ids"], o.hits.ids) and cnt == 2 * r.n_pairs
        pa = g["ids"][(g["ids"] >> 4) & 1 == 0] >> 26
        pb = g["ids"][(g["ids"] >> 4) & 1 == 1] >> 26
        assert np.all(pa == want_a) and np.all(pb == want_b), (d, np.unique(pa), np.unique(pb))


def test_ring_handedness_against_hand_written_numbers(tables):
    """[R5] the same hand-written (point -> ids) table that pins the oracle's ring placement, through gpet_geometry_locate."""
    g = api.gpet_geometry_create(W.geometry_c1())
    pack = lambda panel, mx, my, ix, iy: (panel << 26) | ((mx + 2 * my) << 20) | ((ix + 16 * iy) << 5)
    pts = np.array([[56.0, 3.5, 0.5], [56.0, -3.5, 0.5], [56.0, 0.5, -20.5], [-3.5, 56.0, 0.5], [3.5, 56.0, 0.5], [-56.0, -3.5, 0.5]], np.float32)
    want = [pack(0, 1, 2, 3, 0), pack(0, 0, 2, 12, 0), pack(0, 1, 0, 0, 11), pack(3, 1, 2, 3, 0), pack(3, 0, 2, 12, 0), pack(6, 1, 2, 3, 0)]
    assert list(api.gpet_geometry_locate(g, pts)) == want


# ----------------------------------------------------------------------------- decay law, positron range
def test_decay_law_times_are_bit_identical(tables):
    """[R34] a decaying source (half-life 20 ms watched for 50 ms: 2.5 half-lives, both branches of the restated logarithm):
    the digitizer's fp64 decay times equal the oracle's bit for bit, in one slice and in time slices, and so do the
    coincidences built on them; the expected count comes from gpet_decay_count.  The last two cases end with the run: its
    last slice is cut short (N mod B != 0) and must stay inside [0, T] -- once on the fine time buckets (fast
    decay) and once on the coarse ones (half-life 2 s: the rate changes by < 10 % over the batch)."""
    from dataclasses import replace
    a0, T = 5.0e7, 0.05
    n_fast = api.gpet_decay_count(a0, 0.02, T)
    assert n_fast == O.decay_count(a0, 0.02, T) and 1_180_000 < n_fast < 1_195_000
    assert api.gpet_decay_count(1.6e8 * np.log(2.0) / W.F18_HALF_LIFE_S, W.F18_HALF_LIFE_S, 120.0) == 2_007_947
    for th, slice_pairs, first, n in ((0.02, 0, 0, 300_000), (0.02, 100_000, 800_000, 300_000), (0.02, 100_000, 900_000, None),
                                      (2.0, 100_000, 2_300_000, None)):
        n_total = api.gpet_decay_count(a0, th, T)
        assert n_total == O.decay_count(a0, th, T)
        to_the_end = n is None
        if to_the_end:
            n = n_total - first
            assert 150_000 < n < 300_000 and 1000 < n_total % slice_pairs < slice_pairs - 1000      # the run ends inside a slice
        src = replace(W.source_point((10.0, 0.0, 4.0), activity_bq=a0), half_life_s=th, duration_s=T, pairs_per_time_slice=slice_pairs)
        o = O.simulate(W.geometry_c3(), tables, src, n, 405, first_history=first, threads=8)
        dig = W.Digitizer(0.15, 511.0, 350.0, 650.0, 4.0, 1)
        osg, oco, _ = O.digitize(src, 405, n_total, o.hits, dig)
        hb = PU.upload_hits(PU.oracle_hits_dict(o.hits), np.random.default_rng(3).permutation(len(o.hits)))
        s = api.DeviceSource(src)
        scratch = torch.empty(api.gpet_digitize_scratch_bytes(n, len(o.hits)), dtype=torch.uint8, device="cuda")
        sg, co = api.SinglesBuffer.allocate(len(o.hits)), api.CoincBuffer.allocate(len(o.hits))
        api.gpet_digitize(s, 405, n_total, first, n, hb, len(o.hits), dig, scratch, sg, co)
        torch.cuda.synchronize()
        gs = sg.to_numpy()
        assert PU.compare_singles(gs, osg, 20, exact=True, max_symdiff=2) >= len(osg.ids) - 2 > n // 6
        assert PU.compare_coincidences(co.to_numpy(), oco, exact=True, max_symdiff=4) >= len(oco.ids_a) - 4 > n // 100
        assert np.all(np.diff(gs["t_s"]) >= 0)
        if to_the_end:                                                 # decay time <= T, plus a few ns of flight
            assert T - 2e-4 < gs["t_s"].max() < T + 1e-8 and osg.t_s.max() < T + 1e-8
            in_last = gs["history"].astype(np.int64) >= (n_total // slice_pairs) * slice_pairs
            assert in_last.sum() > 1000 and gs["t_s"][in_last].min() > gs["t_s"][~in_last].max() - 1e-8
        else:
            assert gs["t_s"].max() < T
        if first and th < 1.0:                                         # histories 800k.. of 1.19M: late in the decay curve
            assert gs["t_s"].min() > 0.02


def test_long_histories_with_a_saturated_sequence_counter(tables):
    """SURVEY 8(c) O31 / [R9]: a thick Compton-only slab (the oracle pin's regime: almost half the photons
    make 16 or more deposits, up to ~70).  The kernel's 4-bit sequence counter must stay at 15, as the oracle's does, and
    every hit of those long tracks must match: outcome hashes, ids, positions, energies, times -- saturated hits paired in
    time-of-flight order (R9).  That order is unique only while two saturated deposits of a photon are further
    apart than the fp32 error of the path sum: the few histories with two such deposits within 2e-6 ns (0.6 um of path) are
    checked for count and hash only.  Both the hashed comparison and the key join of the product-build helper run."""
    pose = np.array([[50.0, 0, 0, 0, 1, 0, 0, 0, 1, 1, 0, 0]], np.float32)
    # 40 mean free paths deep, +-40 wide: as good as semi-infinite (the oracle pin shows the outcome has no other length scale)
    geom = W.Geometry(1, (W.Layer((1, 1), (160.0, 160.0), (0.0, 0.0), (0.0, 0.0), 80.0),), (1, 1), (160.0, 160.0), (160.0, 160.0), panel_pose=pose)
    f = lambda v: np.full((1, W.N_ENERGIES), v, np.float32)
    t = W.Tables(W.E_MIN_KEV, W.E_STEP_KEV, f(0.0), f(0.5), f(0.0))
    n = 40_000
    r = W.Run("long", geom, W.source_beam((0, 0, 0), (1, 0, 0), 0.0), n, 31)
    g, gh, cnt = PU.gpu_simulate(r, t, hits_per_pair=40.0)
    o = O.simulate(geom, t, r.source, n, r.seed, want_hash=True, threads=16)
    oh = PU.oracle_hits_dict(o.hits)
    per_photon = np.bincount(oh["history"], minlength=n)
    assert np.mean(per_photon >= 16) > 0.3 and per_photon.max() > 40 and np.sum((oh["ids"] & 15) == 15) > 100_000
    same = np.all(np.asarray(gh).reshape(-1, 2) == np.asarray(o.outcome_hash).reshape(-1, 2), axis=1)
    assert same.mean() >= 0.999                                       # long tracks: ~20x the decisions of a C1 history
    assert np.array_equal(np.bincount(g["history"], minlength=n)[same], per_photon[same])     # deposits per photon
    ambiguous = np.zeros(n, bool)
    for h in (g, oh):                                                 # both are in canonical order
        sat = (h["ids"] & 15) == 15
        close = sat[1:] & sat[:-1] & (h["history"][1:] == h["history"][:-1]) & (np.abs(np.diff(h["tof_ns"].astype(np.float64))) < 2e-6)
        ambiguous[h["history"][1:][close]] = True
    assert ambiguous.mean() < 0.02
    keep = lambda h: {k: v[~ambiguous[h["history"]]] for k, v in h.items()}
    g2, o2 = keep(g), keep(oh)
    res = PU.compare_hits(g2, o2, gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= 0.999 and res["n_hits_compared"] > 0.97 * len(oh["ids"]), res
    un = PU.compare_hits_unhashed(g2, o2, n, min_match=0.999, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert un["n_hits_compared"] > 0.97 * len(oh["ids"])


@pytest.mark.parametrize("kind", ["point", "rods_in_phantom"])
def test_positron_range_parity(tables, kind):
    """[R35] positron range switched on (0.5 mm FWHM, five times 18F's: PAPER.md:145): every pair starts at its own
    annihilation point -- outcome hashes and hits against the oracle for a point source on C3's ring and for the hot-rod
    source inside its water phantom."""
    from dataclasses import replace
    if kind == "point":
        r = W.Run("positron", W.geometry_c3(), replace(W.source_point((10.0, 0.0, 4.0)), positron_fwhm_mm=0.5), 300_001, 66)
    else:
        c4 = W.config_runs("C4", 150_000)[0]
        r = replace(c4, source=replace(c4.source, positron_fwhm_mm=0.5))
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and res["n_hits_compared"] > 50_000, res
    # the first hits of photon A no longer lie on lines through ONE point: their time of flight differs from |x - source| / c
    if kind == "point":
        first = (g["ids"] & 31) == 0
        d = np.sqrt((g["x"][first] - 10.0) ** 2 + g["y"][first] ** 2 + (g["z"][first] - 4.0) ** 2) / 299.792458 - g["tof_ns"][first]
        mad = 1.4826 * np.median(np.abs(d - np.median(d))) * 299.792458     # robust: 2 % of the photons are Rayleigh-deflected on the way
        assert 0.1 < mad < 0.4                                         # ~ sigma of the displacement along the line of flight (0.21 mm)


# ----------------------------------------------------------------------------- majorant regions, 3-4 layers
def mixed_ring(n_layers):
    """12-panel ring with a stack of up to four layers of their own lattices and materials (PAPER.md:35 `the number of
    layers`; PAPER.md:141 three- and four-layer stacks): LYSO | water-like crystals in a water-like matrix | LYSO | coarse
    LYSO in a water-like matrix -> up to four majorant regions [R19]."""
    layers = (W.Layer((15, 15), (1.0, 1.0), (0.1, 0.1), (0.5, 0.5), 3.0, 0.0, 0, -1),
              W.Layer((16, 16), (1.0, 1.0), (0.1, 0.1), (0.0, 0.0), 2.0, 0.1, 1, 1),
              W.Layer((16, 16), (1.0, 1.0), (0.1, 0.1), (0.0, 0.0), 2.5, 0.0, 0, -1),
              W.Layer((8, 8), (2.0, 2.0), (0.2, 0.2), (0.0, 0.0), 2.4, 0.1, 0, 1))
    return W.Geometry(12, layers[:n_layers], (2, 4), (16.0, 16.0), (16.0, 16.0), ring_inner_radius_mm=55.0)


@pytest.mark.parametrize("n_layers", [3, 4])
def test_three_and_four_layer_stacks_with_majorant_regions(tables, n_layers):
    """Per-region majorants with analytic region crossing on 3- and 4-layer mixed-material rings: outcome hashes (which
    include every region crossing) and hits against the oracle; every layer records hits."""
    r = W.Run(f"mixed{n_layers}", mixed_ring(n_layers), W.source_point((10.0, 0.0, 4.0)), 300_001, 90 + n_layers)
    g, gh, cnt, o = run_both(r, tables)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and cnt > 100_000, res
    assert o.counters["region_crossings"] > 100_000
    assert set(np.unique((g["ids"] >> 18) & 3)) == set(range(n_layers))
    # the product build (no hashes) writes the same hits
    gm, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    hb = api.HitBuffer.allocate(3 * r.n_pairs)
    api.gpet_simulate(gm, m, s, 0, r.n_pairs, r.seed, hb)
    torch.cuda.synchronize()
    plain = PU.canonical(hb.to_numpy())
    assert all(np.array_equal(plain[k], g[k]) for k in PU.HIT_KEYS)


def test_two_region_slab_transmits_like_the_closed_form(tables):
    """The pin of the oracle's regions (a light layer over a dense one, pencil beam along the depth): the CUDA path gives
    the same outcome for every history, so exp(-mu1 L1 - mu2 L2) and zero virtual collisions carry over."""
    from test_oracle_pins import slab, beam, two_material_tables
    layers = (W.Layer((1, 1), (12.0, 12.0), (0.0, 0.0), (0.0, 0.0), 4.0, 0.0, crystal_material=1),
              W.Layer((1, 1), (12.0, 12.0), (0.0, 0.0), (0.0, 0.0), 6.0, 0.0, crystal_material=0))
    for src in (beam(), beam(direction=(-1, 0, 0), pos=(70, 0, 0)), beam(direction=(1, 0.2, 0.1), pos=(0, -8, -4))):
        r = W.Run("slab2", slab(layers=layers), src, 200_000, 31)
        g, gh, cnt, o = run_both(r, two_material_tables(0.2, 0.02))
        assert np.array_equal(gh, o.outcome_hash) and np.array_equal(g["ids"], o.hits.ids) and cnt > 100_000
        assert o.counters["virtuals"] == 0 and o.counters["region_crossings"] > 50_000


def many_material_tables(n):
    """LYSO, water and n - 2 scaled copies of water (denser and denser `tissues`): inputs for the staging tests."""
    t = W.tables()
    scale = [1.0, 1.0] + [1.0 + 0.4 * k for k in range(1, n - 1)]
    pick = [0, 1] + [1] * (n - 2)
    f = lambda a: np.ascontiguousarray(np.stack([a[p] * np.float32(s) for p, s in zip(pick, scale)]).astype(np.float32))
    return W.Tables(t.e_min_keV, t.e_step_keV, f(t.mu_pe), f(t.mu_compton), f(t.mu_rayleigh))


@pytest.mark.parametrize("n_mat", [3, 6])
def test_many_materials_fit_in_shared_memory(n_mat):
    """The mu tables are staged in shared memory next to the photon pools (8 KB per material at 502 energies): with three
    materials everything still fits, with six (a phantom stages every loaded material) the transport CTA gives up warps
    until it does -- same results either way (the launch used to fail with a bare CUDA error)."""
    from dataclasses import replace
    t = many_material_tables(n_mat)
    # detector stack using three materials
    layers = list(mixed_ring(4).layers)
    layers[2] = replace(layers[2], crystal_material=2)
    geom = replace(mixed_ring(4), layers=tuple(layers))
    r = W.Run("mats_det", geom, W.source_point((10.0, 0.0, 4.0)), 100_000, 97)
    g, gh, cnt, o = run_both(r, t)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and cnt > 30_000, res
    # phantom holding every loaded material but LYSO (concentric shells), on C3's ring
    c4 = W.config_runs("C4", 100_000)[0]
    ph = c4.source.phantom_material.copy()
    zz, yy, xx = np.meshgrid(*[np.arange(128)] * 3, indexing="ij")
    rr = np.sqrt((xx - 63.5) ** 2 + (yy - 63.5) ** 2) * 0.25
    for k in range(2, n_mat):
        ph[(ph > 0) & (rr < 15.0 * (n_mat - k) / (n_mat - 1))] = k + 1
    src = replace(c4.source, phantom_material=ph, phantom_majorant_material=n_mat - 1)
    r = replace(c4, source=src)
    g, gh, cnt, o = run_both(r, t)
    res = PU.compare_hits(g, PU.oracle_hits_dict(o.hits), gh, o.outcome_hash, pos_tol=POS_TOL, e_tol=E_TOL, tof_tol=TOF_TOL)
    assert res["frac"] >= MIN_MATCH and cnt > 30_000 and o.counters["ph_compton"] > 10_000, res
    assert len(np.unique(ph)) == n_mat


def test_bad_inputs_are_rejected_with_a_message(tables):
    """skewed poses, zero totals and phantom voxels pointing at materials that are not loaded."""
    geom = W.geometry_c0()
    pose = geom.panel_pose.copy(); pose[0, 3:6] = (0.0, 0.9, 0.1)        # u no longer a unit vector orthogonal to w
    from dataclasses import replace
    with pytest.raises(api.GpetError, match="orthonormal"):
        api.gpet_geometry_create(replace(geom, panel_pose=pose))
    r = W.config_runs("C1", 1000)[0]
    g, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    hb = api.HitBuffer.allocate(4096)
    api.gpet_simulate(g, m, s, 0, 1000, r.seed, hb)
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(1000, 4096), dtype=torch.uint8, device="cuda")
    with pytest.raises(api.GpetError, match="n_pairs_total"):
        api.gpet_digitize(s, r.seed, 0, 0, 1000, hb, 4096, r.digitizer, scratch, None, api.CoincBuffer.allocate(1024))
    c4 = W.config_runs("C4", 1000)[0]
    bad = c4.source.phantom_material.copy(); bad[64, 64, 64] = 9
    with pytest.raises(api.GpetError, match="material"):
        api.Pipeline(api.gpet_geometry_create(c4.geometry), m, replace(c4.source, phantom_material=bad), c4.digitizer, 1000, 1000)
    pipe = api.Pipeline(g, m, r.source, r.digitizer, 4000, 1000, 3.0, 0, 1)      # a batch may not leave the run
    with pytest.raises(api.GpetError, match="leave the run"):
        pipe.submit(3500, 1000, r.seed)


def test_small_transport_ctas_give_the_same_hits(tables):
    """gpet_set_transport_warps documents 1..20; 1..3 used to be refused as 'tables too large'.  The hits of a
    run are a pure function of (seed, history) [R1], so any CTA size must give the same records."""
    r = W.config_runs("C3", 60_000)[3]
    g, m, s = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables), api.DeviceSource(r.source)
    got = []
    try:
        for w in (0, 1, 3, 7):
            assert api.gpet_set_transport_warps(w) == (w or 20)
            hb = api.HitBuffer.allocate(200_000)
            api.gpet_simulate(g, m, s, 0, r.n_pairs, r.seed, hb)
            torch.cuda.synchronize()
            got.append(PU.canonical(hb.to_numpy()))
    finally:
        assert api.gpet_set_transport_warps(0) == 20
    assert len(got[0]["ids"]) > 30_000
    for h in got[1:]:
        assert all(np.array_equal(got[0][k], h[k]) for k in PU.HIT_KEYS)


# ----------------------------------------------------------------------------- the paper's Table 1 workload
TABLE1 = {}


@pytest.mark.parametrize("cfg", ["T1", "T2", "T3"])
def test_table1_derenzo_runs_against_the_oracle(tables, cfg):
    """the Derenzo source (116 rods of 0.3-1.0 mm in a 40.25 mm water box, 9.21e-5 MBq/mm3, 12 s of 18F
    decay = 1 142 344 decays) on H2RSPET-1CL / -1CL-split / -2CL, whole run through the product build with the decay law
    on [R34]: hits, singles and coincidences against the oracle."""
    r = W.config_runs(cfg)[0]
    assert r.n_pairs == 1_142_344 == api.gpet_decay_count(r.source.activity_bq, r.source.half_life_s, r.source.duration_s)
    g, o, res = whole_run_against_oracle(r, tables, 3.0, min_coinc=50_000, reps=8)   # a 12 s acquisition is a 0.6 ms run: best of 7
    TABLE1[cfg] = dict(hits=res["n_hits"], coinc=res["n_coinc_compared"], ms=res["ms"], g=g)
    print(f"{cfg}: hits/decay {res['n_hits'] / r.n_pairs:.3f} (paper 2.34), coincidences/hit {res['n_coinc_compared'] / res['n_hits']:.4f} "
          f"(paper 0.1415), {res['ms']:.3f} ms per 12 s acquisition (paper: 41 s on a TITAN Xp, I/O included)")
    assert gsafe(res["n_hits"] / r.n_pairs, 1.2, 1.7)


def gsafe(v, lo, hi):
    return lo < v < hi


def test_table1_layer_configurations_cost_the_same(tables):
    """PAPER.md:121 (Table 1): `no measurable increase in simulation time` from 1CL to split to 2CL, here on the Derenzo
    workload with ONE seed for the three scanners (a 12 s acquisition is a 0.6 ms run: different seeds alone move it by a
    few percent); and the split scanner records the single-layer scanner's hits."""
    from dataclasses import replace
    ms, hits = [], []
    for cfg in ("T1", "T2", "T3"):
        r = replace(W.config_runs(cfg)[0], seed=70)
        g, _, _, t = gpu_product_run(r, tables, 3.0, reps=8)
        ms.append(t); hits.append(PU.canonical(g))
    assert max(ms) / min(ms) < 1.10, ms
    strip = ~np.uint32(3 << 18)
    assert np.array_equal(hits[0]["ids"] & strip, hits[1]["ids"] & strip) and np.array_equal(hits[0]["x"], hits[1]["x"])
    assert 0.96 < len(hits[2]["ids"]) / len(hits[0]["ids"]) < 1.0        # paper: 2 620 170 / 2 671 908 = 0.981
