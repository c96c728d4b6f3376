"""Helpers for the CUDA-vs-oracle parity tests (tests only)."""
from __future__ import annotations

import numpy as np

from oracle import gpet_oracle as O
from paper_2603_07327_b200 import api

HIT_KEYS = ("history", "ids", "x", "y", "z", "e_keV", "tof_ns")


def canonical(h: dict) -> dict:
    """Sort a hit dict by (history, photon, seq) -- the canonical order the oracle emits."""
    key = (h["history"].astype(np.uint64) << np.uint64(5)) | (h["ids"] & np.uint32(31)).astype(np.uint64)
    o = np.argsort(key, kind="stable")
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


def compare_hits(gpu: dict, orc: dict, gpu_hash, orc_hash, first_history=0, pos_tol=1e-3, e_tol=1e-3, tof_tol=1e-4):
    """Per-history comparison.  Returns dict(n_histories, n_match, frac, max_dx, max_de, max_dt).
    Histories whose outcome hash agrees must have identical ids and agree within the tolerances."""
    n = len(orc_hash)
    same = np.all(np.asarray(gpu_hash).reshape(-1, 2) == np.asarray(orc_hash).reshape(-1, 2), axis=1)
    ok_g = same[(gpu["history"] - np.uint32(first_history)).astype(np.int64)]
    ok_o = same[(orc["history"] - np.uint32(first_history)).astype(np.int64)]
    g = {k: v[ok_g] for k, v in gpu.items()}
    o = {k: v[ok_o] for k, v in orc.items()}
    assert len(g["ids"]) == len(o["ids"]), "matching histories must hold the same number of hits"
    assert np.array_equal(g["history"], o["history"]) and np.array_equal(g["ids"], o["ids"])
    dx = max(float(np.max(np.abs(g[k].astype(np.float64) - o[k]), initial=0.0)) for k in ("x", "y", "z"))
    de = float(np.max(np.abs(g["e_keV"].astype(np.float64) - o["e_keV"]), initial=0.0))
    dt = float(np.max(np.abs(g["tof_ns"].astype(np.float64) - o["tof_ns"]), initial=0.0))
    assert dx <= pos_tol and de <= e_tol and dt <= tof_tol, (dx, de, dt)
    return dict(n_histories=n, n_match=int(same.sum()), frac=float(same.mean()), n_hits_compared=int(len(g["ids"])),
                max_dx=dx, max_de=de, max_dt=dt)


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
