"""tpc_tracker_protect_static - the protection flags for callers that cannot allocate device memory.

Some users of the library sit inside a reconstruction framework that took all of the GPU's memory for its own arena when
it started, so a cudaMalloc from their code simply fails; others run in a frame-after-frame loop
where the device-wide stall of cudaMalloc / cudaFree is not acceptable.  For them `tpc_tracker_protect_static` keeps its
one scratch byte per cluster in an array compiled into libtpc_tracker.so (at most PROTECT_STATIC_MAX_CLUSTERS clusters
per frame) instead of in workspace or freshly allocated memory.

The array is shared by every call in the process and is never cleared behind the caller's back, so what these tests
look at is exactly what could go wrong with that: the flags must equal those of the ordinary `tpc_tracker_protect`
(bit for bit - the flags are bytes, the tolerance of every flag comparison in this suite is "identical"), also on the
SECOND call, when the array still holds the marks of the first one; and a frame that does not fit must be refused
without anything being written.

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure, and a problem in
this optional entry point must not hide the parity tests.  It uses nothing left behind by other tests (its own trackers,
its own frames) and passes alone in a fresh process as well as at the end of the whole suite.
"""
import numpy as np
import pytest
import torch

from tests.parity_util import run_gpu
from tpc_synth import default_params, generate_config

pytestmark = pytest.mark.gpu


def _flags(trk, out, road, static):
    """keep[n] (host copy) from the ordinary call or from the no-allocation call; the output buffer is pre-filled with a
    value neither call writes, so an entry that was skipped shows up."""
    keep = torch.full((max(1, out.n_in),), 7, dtype=torch.uint8, device=trk.device)
    if static:
        trk.protect_static(out, road[0], road[1], keep)
    else:
        trk.protect(out, road[0], road[1], keep=keep)
    torch.cuda.synchronize()
    return keep.cpu().numpy()[: out.n_in]


def test_static_scratch_flags_equal_the_ordinary_call_twice_in_a_row():
    import paper_2009_07515_b200 as tpc
    tf = generate_config("cfg3", n_collisions=3)            # ~0.5 M clusters, pile-up and noise: many tiles, ragged tail
    assert tf.n <= tpc.PROTECT_STATIC_MAX_CLUSTERS
    P, trk, out = run_gpu(tf)
    assert out.numpy()["status"] == 0 and out.numpy()["n_tracks"] > 0
    wide, narrow = (3.0, 3.0), (0.25, 0.25)
    want_wide = _flags(trk, out, wide, static=False)
    want_narrow = _flags(trk, out, narrow, static=False)
    assert want_wide.sum() > want_narrow.sum() > 0            # the two roads really give different flags
    # first call: wide road, leaves many marks in the shared array
    got_wide = _flags(trk, out, wide, static=True)
    assert np.array_equal(got_wide, want_wide)
    # second call straight after it: narrow road; any mark surviving from the first call would show up as an extra 1
    got_narrow = _flags(trk, out, narrow, static=True)
    assert np.array_equal(got_narrow, want_narrow)
    # a different, smaller frame on another handle right after: the array is per device, not per handle
    tf2 = generate_config("cfg1")
    P2, trk2, out2 = run_gpu(tf2)
    assert np.array_equal(_flags(trk2, out2, (2.0, 2.0), static=True), _flags(trk2, out2, (2.0, 2.0), static=False))
    # and the first handle again (its frame is still the last one it tracked)
    assert np.array_equal(_flags(trk, out, wide, static=True), want_wide)
    trk.destroy(); trk2.destroy()


def test_static_scratch_call_takes_no_device_memory():
    """Free device memory as the driver reports it is the same before and after a call (the set-up of the first call on
    the device is done beforehand; the output buffer exists already)."""
    tf = generate_config("cfg2", n_tracks=800)
    P, trk, out = run_gpu(tf)
    keep = torch.empty(tf.n, dtype=torch.uint8, device=trk.device)
    trk.protect_static(out, 1.0, 1.0, keep)                 # set-up call
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        trk.protect_static(out, 1.0, 1.0, keep)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    trk.destroy()


def test_frame_beyond_the_static_array_is_refused_and_nothing_is_written():
    import paper_2009_07515_b200 as tpc
    n = tpc.PROTECT_STATIC_MAX_CLUSTERS + 1
    rng = np.random.default_rng(2009_07515)
    tf0 = generate_config("cfg1")
    P = default_params(tf0)
    rx = np.asarray(P["row_x"], np.float32)

    class Frame:                                            # seeded uniform noise clusters, one more than the array holds
        pass
    tf = Frame()
    tf.n = n
    tf.sector = rng.integers(0, P["n_sectors"], n).astype(np.uint8)
    tf.row = rng.integers(0, P["n_rows"], n).astype(np.uint8)
    tf.y = ((rng.random(n) * 2 - 1) * rx[tf.row] * np.float32(P["tan_half_sector"])).astype(np.float32)
    tf.z = (rng.random(n) * 250.0).astype(np.float32)
    P, trk, out = run_gpu(tf, params=P)
    assert out.numpy()["status"] == 0
    keep = torch.full((n,), 7, dtype=torch.uint8, device=trk.device)
    with pytest.raises(RuntimeError, match="built-in scratch"):
        trk.protect_static(out, 1.0, 1.0, keep)
    torch.cuda.synchronize()
    assert bool((keep == 7).all().item())                   # refused before anything was enqueued
    # the ordinary call serves the same frame
    ref = trk.protect(out, 1.0, 1.0, keep=keep)
    torch.cuda.synchronize()
    assert int(ref.max().item()) <= 1
    trk.destroy()
