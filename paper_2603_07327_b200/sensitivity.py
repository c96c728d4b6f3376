"""Sensitivity profiles S(r, E) and the symmetric difference of PAPER.md:63.

S(r, E) = coincidences accepted with energy window E per simulated annihilation pair, for a point source at r.
Pure orchestration over the C ABI: one gpet_simulate per source position, one gpet_digitize per energy window on the
same hits (the digitizer does not modify the hit buffer).  No arithmetic of the method lives here.
"""
from __future__ import annotations

from dataclasses import replace
from typing import Iterable, Sequence, Tuple

import numpy as np

from . import api, workloads as W

PAPER_WINDOWS_KEV = ((150.0, 700.0), (250.0, 700.0), (350.0, 700.0), (450.0, 700.0))
PAPER_DIGITIZER = W.Digitizer(blur_fwhm_frac=0.16, blur_ref_keV=511.0, e_lo_keV=350.0, e_hi_keV=700.0, window_ns=3.0)


def sensitivity(geometry: W.Geometry, tables: W.Tables, positions: Iterable[Sequence[float]],
                windows: Sequence[Tuple[float, float]] = PAPER_WINDOWS_KEV, n_pairs: int = 1_000_000, seed: int = 1,
                digitizer: W.Digitizer = PAPER_DIGITIZER, activity_bq: float = 1.7e4, hits_per_pair: float = 2.5) -> np.ndarray:
    """Returns S[position, window] (coincidences per pair).  activity_bq defaults to the paper's 1.70e-2 MBq."""
    import torch
    geom, mats = api.gpet_geometry_create(geometry), api.gpet_materials_load(tables)
    cap = int(n_pairs * hits_per_pair) + 1024
    hits, coinc = api.HitBuffer.allocate(cap), api.CoincBuffer.allocate(cap // 2)
    scratch = torch.empty(api.gpet_digitize_scratch_bytes(n_pairs, cap), dtype=torch.uint8, device="cuda")
    out = []
    for k, pos in enumerate(positions):
        source = W.source_point(pos, activity_bq=activity_bq)
        src = api.DeviceSource(source)
        hits.n_hits.zero_()
        api.gpet_simulate(geom, mats, src, 0, n_pairs, seed + k, hits)
        row = []
        for lo, hi in windows:
            dig = replace(digitizer, e_lo_keV=lo, e_hi_keV=hi)
            api.gpet_digitize(src, seed + k, n_pairs, 0, n_pairs, hits, cap, dig, scratch, None, coinc)
            row.append(int(coinc.n_coinc.item()) / n_pairs)
        if hits.count() > cap:
            raise api.GpetError("hit buffer overflow in sensitivity(); raise hits_per_pair")
        out.append(row)
    return np.asarray(out)


def delta_sym_percent(s_1cl: np.ndarray, s_2cl: np.ndarray) -> np.ndarray:
    """200 (S_1CL - S_2CL) / (S_1CL + S_2CL)."""
    s_1cl, s_2cl = np.asarray(s_1cl, np.float64), np.asarray(s_2cl, np.float64)
    return 200.0 * (s_1cl - s_2cl) / (s_1cl + s_2cl)
