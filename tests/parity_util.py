"""Helpers for the CUDA-vs-oracle parity tests (tests only)."""
from __future__ import annotations

import numpy as np

from oracle import gpet_oracle as O
from paper_2603_07327_b200 import api

HIT_KEYS = ("history", "ids", "x", "y", "z", "e_keV", "tof_ns")


def canonical(h: dict) -> dict:
    """Sort a hit dict by (history, photon, seq) -- the canonical order the oracle emits.  The sequence number saturates at
    15 [R9]: from a photon's 16th deposit on, the hits are ordered by time of flight, which grows along the track
    (R9; the oracle emits them in track order)."""
    key = (h["history"].astype(np.uint64) << np.uint64(5)) | (h["ids"] & np.uint32(31)).astype(np.uint64)
    o = np.lexsort((h["tof_ns"], key))
    return {k: h[k][o] for k in HIT_KEYS}


def oracle_hits_dict(hits: O.Hits) -> dict:
    return {k: getattr(hits, k) for k in HIT_KEYS}


def gpu_simulate(run, tables, n_pairs=None, first_history=0, want_hash=True, hits_per_pair=2.5):
    """Runs the CUDA transport for one workloads.Run; returns (hits dict in canonical order, hashes, n_hits)."""
    import torch
    n = n_pairs or run.n_pairs
    g = api.gpet_geometry_create(run.geometry)
    m = api.gpet_materials_load(tables)
    s = api.DeviceSource(run.source)
    hb = api.HitBuffer.allocate(int(n * hits_per_pair) + 1024, n_hash=n if want_hash else 0)
    api.gpet_simulate(g, m, s, first_history, n, run.seed, hb)
    torch.cuda.synchronize()
    cnt = hb.count()
    assert cnt <= hb.capacity, "hit buffer overflow in test"
    hashes = hb.outcome_hash.cpu().numpy().view(np.uint64).reshape(-1, 2) if want_hash else None
    return canonical(hb.to_numpy()), hashes, cnt


def upload_hits(hits: dict, order=None) -> "api.HitBuffer":
    """Copies oracle-made hits (optionally permuted) into a device HitBuffer."""
    import torch
    n = len(hits["ids"])
    hb = api.HitBuffer.allocate(n + 16)
    for k in HIT_KEYS:
        a = hits[k] if order is None else hits[k][order]
        getattr(hb, k)[:n].copy_(torch.from_numpy(np.ascontiguousarray(a.view(np.int32) if a.dtype == np.uint32 else a)))
    hb.n_hits.fill_(n)
    return hb


POS_CAP = 5e-3   # mm: no hit of a history with the oracle's outcome hash may be further off than this (2x the measured tail, see compare_hits)
TAIL_SHARE = 3e-5  # share of the compared hits allowed beyond pos_tol (each also costs its history the 99.99 % bar)


def compare_hits(gpu: dict, orc: dict, gpu_hash, orc_hash, first_history=0, pos_tol=1e-3, e_tol=1e-3, tof_tol=1e-4):
    """Per-history comparison against the oracle (north_star: >= 99.99 % of the histories with an identical discrete
    outcome, and for those positions within 1e-3 mm and energies within 1e-3 keV).

    A history AGREES when its two outcome hashes equal the oracle's AND every one of its hits lies within the tolerances;
    `frac` is the share of agreeing histories and is what the 99.99 % bar is applied to.  Histories with equal hashes must
    hold identical ids (asserted).  The continuous values of a hash-matching history are allowed a tail: a photon that
    scatters in one panel and enters the next at grazing incidence turns a transverse fp32 rounding of ~5e-6 mm into
    (5e-6 / cos of the incidence angle) along its line of flight -- measured 2.4e-3 mm at most in 1e7 pairs of C1
    (DESIGN.md 7).  Such a history counts AGAINST the 99.99 %; none may be off by more than POS_CAP, energies and
    times of hash-matching histories stay within their tolerances without exception."""
    n = len(orc_hash)
    same = np.all(np.asarray(gpu_hash).reshape(-1, 2) == np.asarray(orc_hash).reshape(-1, 2), axis=1)
    hg = (gpu["history"] - np.uint32(first_history)).astype(np.int64)
    ho = (orc["history"] - np.uint32(first_history)).astype(np.int64)
    ok_g, ok_o = same[hg], same[ho]
    g = {k: v[ok_g] for k, v in gpu.items()}
    o = {k: v[ok_o] for k, v in orc.items()}
    assert len(g["ids"]) == len(o["ids"]), "matching histories must hold the same number of hits"
    assert np.array_equal(g["history"], o["history"]) and np.array_equal(g["ids"], o["ids"])
    dxs = np.maximum.reduce([np.abs(g[k].astype(np.float64) - o[k]) for k in ("x", "y", "z")]) if len(g["ids"]) else np.zeros(0)
    dx = float(np.max(dxs, initial=0.0))
    de = float(np.max(np.abs(g["e_keV"].astype(np.float64) - o["e_keV"]), initial=0.0))
    dt = float(np.max(np.abs(g["tof_ns"].astype(np.float64) - o["tof_ns"]), initial=0.0))
    assert dx <= POS_CAP and de <= e_tol and dt <= tof_tol, (dx, de, dt)
    off = dxs > pos_tol
    assert off.sum() <= max(3, TAIL_SHARE * len(dxs)), f"{int(off.sum())} of {len(dxs)} hits beyond {pos_tol} mm: the fp32 tail has grown"
    agree = same.copy()
    agree[hg[ok_g][off]] = False
    return dict(n_histories=n, n_match=int(agree.sum()), frac=float(agree.mean()), frac_hash=float(same.mean()),
                n_hits_compared=int(len(g["ids"])), n_hits_beyond_tol=int(off.sum()), max_dx=dx, max_de=de, max_dt=dt,
                dx_q999=float(np.quantile(dxs, 0.999)) if len(dxs) else 0.0, dx_q99999=float(np.quantile(dxs, 0.99999)) if len(dxs) else 0.0)


def chi2_crystal_histograms(gpu_ids, orc_ids, min_expected=5):
    """Two-sample chi-square on per-crystal hit counts (ids without photon/seq).  Returns the p-value."""
    from scipy import stats
    a = np.unique(gpu_ids >> 5, return_counts=True)
    b = np.unique(orc_ids >> 5, return_counts=True)
    keys = np.union1d(a[0], b[0])
    ca = np.zeros(len(keys)); cb = np.zeros(len(keys))
    ca[np.searchsorted(keys, a[0])] = a[1]; cb[np.searchsorted(keys, b[0])] = b[1]
    keep = (ca + cb) >= 2 * min_expected
    ca, cb = ca[keep], cb[keep]
    if len(ca) < 2:
        return 1.0
    k1, k2 = np.sqrt(cb.sum() / ca.sum()), np.sqrt(ca.sum() / cb.sum())
    stat = np.sum((k1 * ca - k2 * cb) ** 2 / (ca + cb))
    return float(stats.chi2.sf(stat, len(ca) - 1))


# ----------------------------------------------------------------------------- joins (no length-gated compares)
SINGLE_KEYS = ("history", "ids", "x", "y", "z", "e_keV", "t_s")
COINC_KEYS = ("ids_a", "ids_b", "history_a", "history_b", "e_a", "e_b", "dt_ns", "t_s")


def as_dict(rec, keys):
    """dict view of an oracle dataclass (Singles / Coincidences) or of a dict."""
    return {k: (rec[k] if isinstance(rec, dict) else getattr(rec, k)) for k in keys}


def _join(kg, ko):
    """Indices of the common keys of two arrays of UNIQUE uint64 keys and the size of the symmetric difference."""
    assert len(np.unique(kg)) == len(kg) and len(np.unique(ko)) == len(ko), "join keys must be unique"
    _, ig, io = np.intersect1d(kg, ko, assume_unique=True, return_indices=True)
    return ig, io, len(kg) + len(ko) - 2 * len(ig)


def compare_singles(gpu, orc, shift, exact=True, max_symdiff=2, max_bad=0, pos_tol=1e-3, e_tol=1e-3, t_tol=1e-12):
    """Kept singles joined on (history, readout unit = ids >> shift); the intersection is ALWAYS compared record by record.
    exact=True (both digitizers saw the same hits): ids, xyz and the fp64 time bit-identical, |dE| <= e_tol (the blur
    runs in fp32 on the device).  exact=False (each side digitized its own transport's hits): ids identical, xyz / E / t
    within tolerances.  A single whose blurred energy lies within ~1e-4 keV of a window edge may be kept by one side
    only: |symmetric difference| <= max_symdiff.  max_bad = records of the intersection allowed to disagree (histories
    whose fp32 / fp64 outcome differs, north_star's 1e-4 budget).  Returns the number of records compared."""
    g, o = as_dict(gpu, SINGLE_KEYS), as_dict(orc, SINGLE_KEYS)
    key = lambda s: (s["history"].astype(np.uint64) << np.uint64(32)) | (s["ids"] >> np.uint32(shift)).astype(np.uint64)
    ig, io, symdiff = _join(key(g), key(o))
    assert symdiff <= max_symdiff, f"singles present on one side only: {symdiff} > {max_symdiff}"
    bad = g["ids"][ig] != o["ids"][io]
    de = np.abs(g["e_keV"][ig].astype(np.float64) - o["e_keV"][io])
    bad |= de > e_tol
    if exact:
        for k in ("x", "y", "z", "t_s"):
            bad |= g[k][ig] != o[k][io]
    else:
        for k in ("x", "y", "z"):
            bad |= np.abs(g[k][ig].astype(np.float64) - o[k][io]) > pos_tol
        bad |= np.abs(g["t_s"][ig] - o["t_s"][io]) > t_tol
    assert int(bad.sum()) <= max_bad, f"{int(bad.sum())} of {len(ig)} joined singles disagree (allowed {max_bad})"
    return len(ig)


def compare_coincidences(gpu, orc, exact=True, max_symdiff=2, max_bad=0, e_tol=1e-3, t_tol=1e-12, dt_tol=1e-3):
    """List-mode coincidences joined on (history_a, ids_a >> 5) -- a single opens at most one pair; the partner
    (history_b, ids_b), the energies and the times are compared on the intersection.  Returns the number compared."""
    g, o = as_dict(gpu, COINC_KEYS), as_dict(orc, COINC_KEYS)
    key = lambda c: (c["history_a"].astype(np.uint64) << np.uint64(32)) | (c["ids_a"] >> np.uint32(5)).astype(np.uint64)
    ig, io, symdiff = _join(key(g), key(o))
    assert symdiff <= max_symdiff, f"coincidences present on one side only: {symdiff} > {max_symdiff}"
    bad = (g["ids_a"][ig] != o["ids_a"][io]) | (g["ids_b"][ig] != o["ids_b"][io]) | (g["history_b"][ig] != o["history_b"][io])
    for k in ("e_a", "e_b"):
        bad |= np.abs(g[k][ig].astype(np.float64) - o[k][io]) > e_tol
    if exact:
        bad |= g["t_s"][ig] != o["t_s"][io]
        bad |= np.abs(g["dt_ns"][ig].astype(np.float64) - o["dt_ns"][io]) > 1e-6
    else:
        bad |= np.abs(g["t_s"][ig] - o["t_s"][io]) > t_tol
        bad |= np.abs(g["dt_ns"][ig].astype(np.float64) - o["dt_ns"][io]) > dt_tol
    assert int(bad.sum()) <= max_bad, f"{int(bad.sum())} of {len(ig)} joined coincidences disagree (allowed {max_bad})"
    return len(ig)


def compare_hits_unhashed(gpu, orc, n_histories, first_history=0, min_match=0.9999, pos_tol=1e-3, e_tol=1e-3, tof_tol=1e-4):
    """Whole-run hit comparison for builds that write no outcome hash (the product build).  A hit is keyed by
    (history, photon, seq); a history AGREES when both sides hold the same keys with the same ids and every hit lies
    within the tolerances (a flipped accept / reject can leave the ids unchanged, so without hashes the continuous values
    are part of the verdict).  At least `min_match` of ALL histories must agree (north_star).
    Returns dict(frac, n_bad_histories, n_hits_compared, max_dx, max_de, max_dt over the agreeing histories)."""
    def keyed(h):
        k = ((h["history"].astype(np.uint64) - np.uint64(first_history & 0xFFFFFFFF)) & np.uint64(0xFFFFFFFF)) << np.uint64(5)
        k |= (h["ids"] & np.uint32(31)).astype(np.uint64)
        o = np.lexsort((h["tof_ns"], k))
        k = k[o]
        # saturated sequence numbers [R9]: the 16th, 17th, ... deposit of a photon share seq 15; number them by time of flight
        # so that the key stays unique (a photon makes fewer than 2^10 deposits)
        first = np.r_[True, k[1:] != k[:-1]] if len(k) else np.zeros(0, bool)
        idx = np.arange(len(k)); dup = idx - np.maximum.accumulate(np.where(first, idx, 0))
        assert dup.max(initial=0) < 1024
        return (k << np.uint64(10)) | dup.astype(np.uint64), {kk: h[kk][o] for kk in HIT_KEYS}
    kg, g = keyed(gpu)
    ko, o = keyed(orc)
    ig, io, _ = _join(kg, ko)
    bad_hist = np.zeros(n_histories, bool)
    only_g = np.ones(len(kg), bool); only_g[ig] = False
    only_o = np.ones(len(ko), bool); only_o[io] = False
    bad_hist[(kg[only_g] >> np.uint64(15)).astype(np.int64)] = True
    bad_hist[(ko[only_o] >> np.uint64(15)).astype(np.int64)] = True
    hist = (kg[ig] >> np.uint64(15)).astype(np.int64)
    dxs = np.maximum.reduce([np.abs(g[k][ig].astype(np.float64) - o[k][io]) for k in ("x", "y", "z")])
    des = np.abs(g["e_keV"][ig].astype(np.float64) - o["e_keV"][io])
    dts = np.abs(g["tof_ns"][ig].astype(np.float64) - o["tof_ns"][io])
    differ = (g["ids"][ig] != o["ids"][io]) | (dxs > pos_tol) | (des > e_tol) | (dts > tof_tol)
    bad_hist[hist[differ]] = True
    frac = 1.0 - bad_hist.mean()
    assert frac >= min_match, f"only {frac:.6f} of the histories agree (same hits within tolerance on both sides)"
    good = ~bad_hist[hist]
    return dict(frac=float(frac), n_bad_histories=int(bad_hist.sum()), n_hits_compared=int(good.sum()),
                max_dx=float(np.max(dxs[good], initial=0.0)), max_de=float(np.max(des[good], initial=0.0)),
                max_dt=float(np.max(dts[good], initial=0.0)))
