"""Seeded input generators: shapes, statistics of the configs, determinism, sharding."""
import numpy as np
import pytest

from pvf_inputs import make_events, make_weights, shard_events, select_events


def test_config0_event():
    ev = make_events("single", 1, 1000)
    assert ev.n_events == 1 and ev.n_tracks == 40 and ev.feat.shape == (9, 40) and ev.feat.dtype == np.float32
    assert len(ev.pv_z[0]) == 1 and -200 <= ev.pv_z[0][0] < 200
    assert np.max(np.abs(ev.feat[0] - ev.pv_z[0][0])) < 0.6
    assert np.all(ev.feat[3:] > 0)


def test_run3_statistics_and_determinism():
    a = make_events("run3", 2000, 1001)
    b = make_events("run3", 2000, 1001)
    assert np.array_equal(a.feat, b.feat) and np.array_equal(a.event_offsets, b.event_offsets)
    npv = np.array([len(z) for z in a.pv_z])
    assert npv.min() >= 1 and abs(npv.mean() - 5.6) < 0.15          # PAPER.md:11 "5.6 ... per bunch crossing"
    assert abs(a.n_tracks / 2000 - 5.62 * 30 * 1.1) < 6
    assert a.event_offsets[0] == 0 and np.all(np.diff(a.event_offsets) >= 0)
    c = make_events("pileup", 500, 1003)
    assert abs(np.mean([len(z) for z in c.pv_z]) - 10.0) < 0.4
    assert np.std(np.concatenate(c.pv_z)) < 35


def test_select_and_shard():
    a = make_events("run3", 10, 5)
    s = select_events(a, [3, 7])
    assert s.n_events == 2
    assert np.array_equal(s.feat[:, :s.event_offsets[1]], a.feat[:, a.event_offsets[3]:a.event_offsets[4]])
    for n, ws in [(16000, 8), (10, 3), (2, 4), (0, 2)]:
        parts = [shard_events(n, ws, r) for r in range(ws)]
        assert parts[0][0] == 0 and parts[-1][1] == n
        assert all(parts[i][1] == parts[i + 1][0] for i in range(ws - 1))
        sizes = [hi - lo for lo, hi in parts]
        assert max(sizes) - min(sizes) <= 1


@pytest.mark.parametrize("kind", ["rand", "peaky"])
@pytest.mark.parametrize("ch", [64, 32, 16])
def test_weight_shapes(kind, ch):
    w = make_weights(kind, 1, ch)
    assert [a.shape for a in w.fc_w] == [(25, 9)] + [(25, 25)] * 4 + [(800, 25)]
    assert [a.shape for a in w.conv_w] == [(ch, 8, 25), (ch, ch, 15), (ch, ch, 5), (ch, 2 * ch, 15), (ch, 2 * ch, 25), (1, ch, 1)]
    assert all(a.dtype == np.float32 for a in w.fc_w + w.fc_b + w.conv_w + w.conv_b)
    if kind == "rand":  # PyTorch default bound 1/sqrt(fan_in)
        assert np.max(np.abs(w.conv_w[4])) <= 1 / np.sqrt(2 * ch * 25) + 1e-9
        assert np.max(np.abs(w.fc_w[5])) <= 1 / 5.0 + 1e-9
