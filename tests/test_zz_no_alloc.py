"""gpet_digitize_static: the digitizer for callers that cannot allocate device memory.

Some users of libgpet own every byte of the GPU already (a host program whose memory pool took the whole device at
start-up, so a cudaMalloc for our scratch fails) or digitize one time slice after another in a loop where cudaMalloc and
cudaFree are unwelcome because they can stall all streams of the device.  For them include/gpet.h offers
gpet_digitize_static, which works on a 64 MiB array compiled into the library instead of caller scratch.  It must give
exactly what gpet_digitize gives, call after call, although every call finds the previous call's leftovers in that array.

This file is named to be collected last: under `pytest -x` a failure here must not hide the parity tests."""
import ctypes as C

import numpy as np
import pytest

from paper_2603_07327_b200 import api
from paper_2603_07327_b200 import workloads as W

SINGLES_KEYS = ("history", "ids", "x", "y", "z", "e_keV", "t_s")
COINC_KEYS = ("ids_a", "ids_b", "history_a", "history_b", "e_a", "e_b", "dt_ns", "t_s")


def test_oversize_batch_is_refused_before_any_gpu_work():
    """Beyond GPET_STATIC_SCRATCH_BYTES the call says so (GPET_E_OVERFLOW, both sizes in the text) -- on the host, so this
    runs without a GPU: a caller that cannot allocate learns at once that the batch must be cut into smaller slices."""
    torch = pytest.importorskip("torch")
    n_pairs, cap = 2_000_000, 3_000_000
    assert api.gpet_digitize_scratch_bytes(n_pairs, cap) > api.GPET_STATIC_SCRATCH_BYTES
    assert api.gpet_digitize_scratch_bytes(300_000, 450_000) <= api.GPET_STATIC_SCRATCH_BYTES      # the size gpet.h quotes fits
    hb = api.HitBuffer.allocate(cap, device="cpu")                     # never touched: the size test comes first
    co = api.CoincBuffer.allocate(16, device="cpu")
    src = api._source_struct(W.source_point(), None, None)
    dig = W.Digitizer()
    d = api._Digitizer(dig.blur_fwhm_frac, dig.blur_ref_keV, dig.e_lo_keV, dig.e_hi_keV, dig.window_ns, dig.readout_level)
    hs, cs = hb.struct(), co.struct()
    rc = api.lib().gpet_digitize_static(C.byref(src), 1, n_pairs, 0, n_pairs, C.byref(hs), cap, C.byref(d), None, C.byref(cs), None)
    msg = api.lib().gpet_last_error().decode()
    assert rc == -4, msg
    assert "gpet_digitize_static" in msg and str(api.GPET_STATIC_SCRATCH_BYTES) in msg and "2000000 pairs" in msg


@pytest.mark.gpu
def test_static_scratch_digitizer_equals_the_caller_scratch_one_twice_in_a_row():
    """Two calls in a row on the built-in array, each against gpet_digitize with fresh caller scratch on the same hits.
    The second batch differs from the first in every respect that moves data around in the workspace (fewer pairs, another
    seed, the chunked hit layout, short time slices that start mid-slice -> the fine-bucket time sort), so anything the
    first call left behind and the second failed to clear would show.  The kernels and the inputs are the same on both
    sides and the digitizer's output does not depend on hit order, so the bar is the one the other digitizer tests use
    for equal input: identical records, bit for bit."""
    torch = pytest.importorskip("torch")
    from dataclasses import replace
    tables = W.tables()
    r = W.config_runs("C1", 250_000)[0]
    geom, m = api.gpet_geometry_create(r.geometry), api.gpet_materials_load(tables)
    batches = [dict(n=250_000, first=0, seed=r.seed, slice_pairs=0, chunked=False),
               dict(n=70_016, first=120_500, seed=r.seed + 7, slice_pairs=1_000, chunked=True)]
    for call, b in enumerate(batches):
        src = replace(r.source, activity_bq=5.0e7, pairs_per_time_slice=b["slice_pairs"])     # hot: randoms and multiples too
        s = api.DeviceSource(src)
        n, n_total = b["n"], 400_000
        hb = api.HitBuffer.allocate_chunked(n, 1.5) if b["chunked"] else api.HitBuffer.allocate(int(1.5 * n))
        api.gpet_simulate(geom, m, s, b["first"], n, b["seed"], hb)
        torch.cuda.synchronize()
        assert hb.dropped() == 0 and hb.count() > 0.5 * n
        cap = hb.capacity
        assert api.gpet_digitize_scratch_bytes(n, cap) <= api.GPET_STATIC_SCRATCH_BYTES
        # existing path: caller scratch (filled with ones, so neither side may count on zeros)
        scratch = torch.full((api.gpet_digitize_scratch_bytes(n, cap),), 0xA5, dtype=torch.uint8, device="cuda")
        sg0, co0 = api.SinglesBuffer.allocate(cap), api.CoincBuffer.allocate(cap)
        api.gpet_digitize(s, b["seed"], n_total, b["first"], n, hb, cap, r.digitizer, scratch, sg0, co0)
        # new path: no scratch argument
        sg1, co1 = api.SinglesBuffer.allocate(cap), api.CoincBuffer.allocate(cap)
        api.gpet_digitize_static(s, b["seed"], n_total, b["first"], n, hb, cap, r.digitizer, sg1, co1)
        torch.cuda.synchronize()
        s0, s1, c0, c1 = sg0.to_numpy(), sg1.to_numpy(), co0.to_numpy(), co1.to_numpy()
        assert len(s0["ids"]) == len(s1["ids"]) > 0.2 * n, f"call {call}: singles {len(s0['ids'])} vs {len(s1['ids'])}"
        assert len(c0["ids_a"]) == len(c1["ids_a"]) > 0.02 * n, f"call {call}: coincidences {len(c0['ids_a'])} vs {len(c1['ids_a'])}"
        for k in SINGLES_KEYS:
            assert np.array_equal(s0[k], s1[k]), f"call {call}: singles.{k} differs"
        for k in COINC_KEYS:
            assert np.array_equal(c0[k], c1[k]), f"call {call}: coincidences.{k} differs"
        assert np.all(np.diff(s1["t_s"]) >= 0)
    with pytest.raises(api.GpetError, match="error -4"):               # and the limit holds on the GPU box too
        api.gpet_digitize_static(s, 1, 10_000_000, 0, 2_000_000, api.HitBuffer.allocate(3_000_000), 3_000_000, r.digitizer,
                                 None, api.CoincBuffer.allocate(16))
