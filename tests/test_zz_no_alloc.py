"""pvf_histogram_noalloc (include/pvf.h): interval sort + FC + ordered segmented sum for a small batch with the kernels'
scratch in a file-scope static __device__ array -- the entry point for callers that cannot allocate.

Checked against the EXISTING path (pvf_run + pvf_debug_copy_histogram) on calls in a row that share the static array, and
against the oracle.  Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import pvf_oracle as O
from pvf_inputs import make_events, make_weights
import paper_2602_19959_b200 as pkg
from paper_2602_19959_b200 import PVFinder

H_TOL = 2e-5            # histogram tolerance of tests/test_gpu_parity.py: relative to max(|H|, 1)
SORT_FLAGS = pkg.FLAG_TRACK_DROPPED | pkg.FLAG_NONFINITE | pkg.FLAG_BAD_OFFSETS


@pytest.fixture(scope="module", autouse=True)
def _built():
    import __graft_entry__ as entry
    entry.build()
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)


def _existing_path(pvf, ev):
    """H and flags of the batch through pvf_run (pool scratch) + the debug accessor."""
    feat, off = torch.from_numpy(ev.feat).cuda(), torch.from_numpy(ev.event_offsets).cuda()
    E = ev.n_events
    probs = torch.empty(E, 4000, device="cuda")
    pk = pvf.alloc_peaks(E)
    H = torch.empty(E, 40, 8, 100, device="cuda")
    s = torch.cuda.Stream()
    pvf.run(feat, off, E, probs, pk, stream=s)
    pvf.debug_copy_histogram(H, E, stream=s)
    s.synchronize()
    return H, pk["flags"].cpu().numpy().astype(np.uint32) & SORT_FLAGS


def _rel(a, b):
    a, b = a.astype(np.float64), b.astype(np.float64)
    return float((np.abs(a - b) / np.maximum(np.abs(b), 1.0)).max())


@pytest.mark.parametrize("prec,margin", [("simt", 0.0), ("tf32", 0.0), ("bf16", 0.5)])
def test_noalloc_histogram_matches_existing_path_on_calls_in_a_row(prec, margin):
    w = make_weights("peaky", 5)
    big = make_events("run3", 60, 4242)                       # ~11 000 tracks: most of the static scratch
    small = make_events("pileup", 7, 4243)                    # then a smaller batch over the stale contents
    assert big.n_tracks <= pkg.NOALLOC_MAX_TRACKS and big.n_events <= pkg.NOALLOC_MAX_EVENTS
    f = small.feat.copy()
    f[0, 3], f[0, 4] = np.nan, 777.0                          # flags must come through as well
    small = type(small)(f, small.event_offsets, small.pv_z)
    kw = dict(precision="fp32" if prec == "simt" else prec, split_mask=1 if prec == "tf32" else 0,
              boundary_margin_mm=margin)
    if prec == "simt":
        kw["cta_pair"] = False
    pvf = PVFinder(w, max_events=64, max_tracks=max(big.n_tracks, small.n_tracks), **kw)
    s = torch.cuda.Stream()
    outs = []
    for ev in (big, small, big):                              # calls in a row, all through the same static array
        feat, off = torch.from_numpy(ev.feat).cuda(), torch.from_numpy(ev.event_offsets).cuda()
        H = torch.full((ev.n_events, 40, 8, 100), -7.0, device="cuda")
        fl = torch.full((ev.n_events,), -1, dtype=torch.int32, device="cuda")
        pvf.histogram_noalloc(feat, off, ev.n_events, H, fl, stream=s)
        s.synchronize()
        outs.append((H, fl.cpu().numpy().astype(np.uint32)))
    for ev, (H, fl) in zip((big, small, big), outs):
        H_ref, fl_ref = _existing_path(pvf, ev)
        assert _rel(H.cpu().numpy(), H_ref.cpu().numpy()) <= H_TOL
        assert torch.equal(H == 0, H_ref == 0)                # empty intervals are exactly zero in both
        if prec == "simt":
            assert torch.equal(H, H_ref)                      # same kernels, same order: bit for bit
        assert np.array_equal(fl, fl_ref)
        Ho, flo = O.histogram(ev.feat, ev.event_offsets, w.fc_w, w.fc_b, margin)
        assert _rel(H.cpu().numpy(), Ho) <= H_TOL
        assert np.array_equal(fl & (pkg.FLAG_TRACK_DROPPED | pkg.FLAG_NONFINITE), np.asarray(flo, np.uint32))
    assert torch.equal(outs[0][0], outs[2][0])                # the same batch again: identical, stale scratch or not
    assert outs[1][1][0] & pkg.FLAG_NONFINITE and outs[1][1][0] & pkg.FLAG_TRACK_DROPPED
    # flags are optional
    feat, off = torch.from_numpy(small.feat).cuda(), torch.from_numpy(small.event_offsets).cuda()
    H = torch.empty(small.n_events, 40, 8, 100, device="cuda")
    pvf.histogram_noalloc(feat, off, small.n_events, H, None, stream=s)
    s.synchronize()
    assert torch.equal(H, outs[1][0])
    pvf.destroy()


def test_noalloc_allocates_nothing_and_rejects_oversized_batches():
    w = make_weights("rand", 2)
    ev = make_events("run3", 64, 99)
    pvf = PVFinder(w, max_events=4096, max_tracks=1 << 20, precision="tf32", split_mask=1)
    feat, off = torch.from_numpy(ev.feat).cuda(), torch.from_numpy(ev.event_offsets).cuda()
    H = torch.empty(65, 40, 8, 100, device="cuda")
    s = torch.cuda.Stream()
    for _ in range(2):                                        # set-up (address of the static array) happens in the first
        pvf.histogram_noalloc(feat, off, 64, H, None, stream=s)
    s.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for _ in range(20):
        pvf.histogram_noalloc(feat, off, 64, H, None, stream=s)
    s.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before        # device memory in use did not move
    # beyond the static scratch: a clear error, nothing enqueued, whatever the handle's own capacity
    big = make_events("run3", 65, 100)
    fb, ob = torch.from_numpy(big.feat).cuda(), torch.from_numpy(big.event_offsets).cuda()
    with pytest.raises(pkg.PVFError) as ei:
        pvf.histogram_noalloc(fb, ob, 65, H, None, stream=s)
    assert ei.value.status == pkg.PVF_ERR_CAPACITY and "static scratch" in str(ei.value)
    many = make_events("pileup", 64, 101)                     # 64 events but > 16384 tracks
    assert many.n_tracks > pkg.NOALLOC_MAX_TRACKS
    fm, om = torch.from_numpy(many.feat).cuda(), torch.from_numpy(many.event_offsets).cuda()
    with pytest.raises(pkg.PVFError) as ei:
        pvf.histogram_noalloc(fm, om, 64, H, None, stream=s)
    assert ei.value.status == pkg.PVF_ERR_CAPACITY
    pvf.histogram_noalloc(fm, om, 0, H, None, stream=s)       # zero events: a no-op
    pvf.destroy()
