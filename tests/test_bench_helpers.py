"""Host-side bookkeeping of bench.py (no GPU): byte / FLOP accounting inputs and the roofline denominators."""
import numpy as np

import bench
from pvf_inputs import make_events


def test_nonempty_interval_count_matches_a_direct_count():
    ev = make_events("run3", 50, 7)
    n = bench.nonempty_intervals(ev)
    seen = set()
    for e in range(ev.n_events):
        for t in range(ev.event_offsets[e], ev.event_offsets[e + 1]):
            u = np.float32(np.float32(ev.feat[0, t] + np.float32(200.0)) * np.float32(0.1))
            i = int(np.floor(u))
            if 0 <= i < 40:
                seen.add((e, i))
    assert n == len(seen)
    assert 0.3 < n / (50 * 40) < 0.5          # ~15.7 of 40 intervals hold a track in the run3 model


def test_tensor_peak_selection():
    peaks = {"hbm_gbs": 6459.3, "bf16_tflops": 1668.8, "bf16_tflops_sustained": 1393.8}
    p, note = bench.tensor_peak(peaks, "measured", "bf16", None, sustained=True)
    assert p == 1393.8 and "MEASURED_PEAKS" in note
    p, note = bench.tensor_peak(peaks, "measured", "fp16", None, sustained=False)
    assert p == 1668.8
    p, note = bench.tensor_peak(peaks, "measured", "tf32", None, sustained=True)
    assert abs(p - 1393.8 * 1.1 / 2.25) < 1e-9 and "derived" in note          # no measurement: the derived figure, labelled
    p, note = bench.tensor_peak(peaks, "measured", "tf32", {"burst": 700.0, "sustained": 612.0}, sustained=True)
    assert p == 612.0 and "measured in this run" in note
    p, _ = bench.tensor_peak(peaks, "measured", "fp32", {"burst": 700.0, "sustained": 612.0}, sustained=False)
    assert p == 700.0                                                          # FP32 on the tensor cores: against the TF32 peak


def test_whole_job_rate_and_flop_table():
    assert bench.whole_job_rate(8, 16000, 20, 1000.0) == 8 * 16000 * 20
    # MACs per interval x 2 x 40 intervals
    for ch, macs in ((64, 31_494_400), (32, 8_195_200), (16, 2_209_600)):
        assert abs(bench.UNET_FLOP_PER_EVENT[ch] - 2 * 40 * macs) / (2 * 40 * macs) < 1e-3


def test_unet_mac_count_from_the_topology():
    """31 494 400 MAC per interval at C = 64: e1 8->C k25 L100, e2 C->C k15 L50, b C->C k5 L25,
    d2 2C->C k15 L50, d1 2C->C k25 L100, head C->1 L100."""
    def macs(C):
        return 100 * C * 8 * 25 + 50 * C * C * 15 + 25 * C * C * 5 + 50 * C * 2 * C * 15 + 100 * C * 2 * C * 25 + 100 * C
    assert macs(64) == 31_494_400 and macs(32) == 8_195_200 and macs(16) == 2_209_600


def test_zero_conv_weights_are_a_diagnostic_of_peaky():
    """bench.py --weights zero-conv: `peaky` FC weights, all conv weights and biases zero (power-cap diagnostic)."""
    import numpy as np
    import bench
    from pvf_inputs import make_weights
    w, ref = bench.bench_weights("zero-conv", 32), make_weights("peaky", 1, 32)
    assert all(np.array_equal(a, b) for a, b in zip(w.fc_w, ref.fc_w)) and all(np.array_equal(a, b) for a, b in zip(w.fc_b, ref.fc_b))
    assert all(a.shape == b.shape and not a.any() for a, b in zip(w.conv_w, ref.conv_w))
    assert all(a.shape == b.shape and not a.any() for a, b in zip(w.conv_b, ref.conv_b))
    assert bench.bench_weights("rand", 16).kind == "rand"
