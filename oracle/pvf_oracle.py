"""CPU oracle for PVFinder's per-event inference hot path.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this module.  It shares no code with the CUDA path
(``paper_2602_19959_b200/``) and never imports it; the product never imports this file.

What it is: the model *step by step* as PAPER.md section 2 (lines 27-31) and BASELINE.json config 0
define it, written with numpy in float64 (discrete decisions -- interval assignment and the peak
finder -- are defined in float32 so that they cannot flip between implementations).  Every
function cites the passage it follows; readings of silent/garbled passages are listed in DESIGN.md
("Readings") and tagged [READING] here.

Pins (tests/test_oracle_pins.py, all ``-m "not gpu"``): geometry closed forms, conv1d vs
a naive triple loop and vs torch float64 ``F.conv1d``, delta-kernel and shift identities, FC /
softplus / sigmoid / pool / upsample vs torch float64 routines and closed forms, histogram
permutation invariance + additivity, bias-only output for empty intervals, whole model vs a torch
float64 composition, peak-finder hand cases.
Parity unpinned: the *physics* numbers (>97 % efficiency, 0.03 FP/event) -- they need
the trained weights and LHCb simulation, which do not exist here.
"""
from __future__ import annotations

import numpy as np

# ----------------------------------------------------------------------------------------------
# O1 geometry -- PAPER.md:27 "divides the 400 mm interaction region into 40 intervals of 100 bins
# each"; BASELINE.json config 0: z-region [-200, 200) mm, bins of 0.1 mm.
# ----------------------------------------------------------------------------------------------
Z_MIN_MM = -200.0
N_INTERVALS = 40
N_BINS = 100
BIN_WIDTH_MM = 0.1
N_GLOBAL_BINS = N_INTERVALS * N_BINS  # 4000
FC_CHANNELS = 8                       # PAPER.md:29 "800-bin histogram (8 channels each with 100-bin)"
LEAKY_SLOPE = 0.01                    # BASELINE.json config 0
PEAK_THRESHOLD = np.float32(0.01)     # BASELINE.json config 0 "prob > 0.01"
PEAK_HALFWIDTH = 3                    # "+-3 bins"
MAX_PEAKS = 32                        # "at most 32 peaks per event"

FLAG_PEAK_OVERFLOW = 1
FLAG_TRACK_DROPPED = 2
FLAG_NONFINITE = 4


def bin_centre_mm(g):
    """Centre of global bin g = 100*i + l:  z_c(g) = -200 + (g + 0.5) * 0.1."""
    return Z_MIN_MM + (np.asarray(g, np.float64) + 0.5) * BIN_WIDTH_MM


# ----------------------------------------------------------------------------------------------
# O2 interval assignment + relative z, in float32 with separately rounded operations.
# BASELINE.json config 0: "FC input uses z relative to the track's interval lower edge, scaled to
# [0,1]"; "Each track adds to the interval holding its z_poca".   [READING] the exact float32
# sequence u = (z + 200f) * 0.1f, i = floor(u), zrel = u - i, and the drop rule.
# (A 0.1 mm bin * 100 bins = 10 mm interval, so z/10 mm is the interval coordinate.)
# ----------------------------------------------------------------------------------------------
def assign_intervals(z_poca):
    """Returns (interval int32 [T] (-1 = dropped), zrel float32 [T], nonfinite bool [T])."""
    z = np.asarray(z_poca, np.float32)
    finite = np.isfinite(z)
    zs = np.where(finite, z, np.float32(0.0)).astype(np.float32)
    u = (zs + np.float32(200.0)).astype(np.float32)
    u = (u * np.float32(0.1)).astype(np.float32)
    fl = np.floor(u).astype(np.float32)
    zrel = (u - fl).astype(np.float32)          # exact in float32
    ok = finite & (fl >= np.float32(0.0)) & (fl < np.float32(N_INTERVALS))   # decided on the float: |z| may be 1e30
    interval = np.where(ok, fl, np.float32(-1.0)).astype(np.int32)
    return interval, zrel, ~finite


# ----------------------------------------------------------------------------------------------
# O3 FC stage -- PAPER.md:29 "six FC layers"; BASELINE.json config 0: 9->25->25->25->25->25->800,
# LeakyReLU(0.01) hidden, softplus output.
# ----------------------------------------------------------------------------------------------
def leaky_relu(v, slope=LEAKY_SLOPE):
    return np.where(v >= 0.0, v, slope * v)


def softplus(v):
    """softplus(v) = log(1 + exp(v)), written overflow-free as max(v,0) + log1p(exp(-|v|))
    ([READING] beta = 1, no threshold)."""
    v = np.asarray(v, np.float64)
    return np.maximum(v, 0.0) + np.log1p(np.exp(-np.abs(v)))


def sigmoid(v):
    v = np.asarray(v, np.float64)
    return 1.0 / (1.0 + np.exp(-v))


def fc_forward(x, fc_w, fc_b):
    """x float64 [T, 9] -> contributions float64 [T, 800]; output index o = c*100 + l ([C, L]).

    [READING] feature order x = [zrel, x_poca, y_poca, e0..e5] (PAPER.md:27 says only "nine features").
    """
    h = np.asarray(x, np.float64)
    for k in range(5):
        h = leaky_relu(h @ np.asarray(fc_w[k], np.float64).T + np.asarray(fc_b[k], np.float64))
    return softplus(h @ np.asarray(fc_w[5], np.float64).T + np.asarray(fc_b[5], np.float64))


# ----------------------------------------------------------------------------------------------
# O4 histogram -- PAPER.md:29 "combining each track's contribution into a 800-bin histogram";
# PAPER.md:49 (garbled "B=40, C=64, L=800") read as B = 40 intervals, C = 8, L = 100  [READING].
# ----------------------------------------------------------------------------------------------
def boundary_neighbours(interval, zrel, margin_mm):
    """NEXT-1 -- PAPER.md:49 "tracks on boundaries of intervals are part of two intervals".
    [READING] (the paper gives no margin): a kept track whose z lies within ``margin_mm`` of its
    interval's lower (upper) edge ALSO contributes to the previous (next) interval, there with
    z_rel' = z_rel + 1 (z_rel - 1), i.e. still measured from that interval's lower edge; intervals -1 and
    40 do not exist.  Decisions and z_rel' in float32:  m = margin_mm * 0.1f;  lower side iff
    z_rel < m;  upper side iff z_rel >= 1f - m  (margin < 5 mm, so never both).
    Returns (neighbour int32 [T]: -1 none else the extra interval, zrel2 float32 [T])."""
    f32 = np.float32
    m = f32(f32(margin_mm) * f32(0.1))
    interval = np.asarray(interval, np.int32)
    zrel = np.asarray(zrel, np.float32)
    nb = np.full(interval.shape, -1, np.int32)
    z2 = np.zeros(interval.shape, np.float32)
    if not (m > 0):
        return nb, z2
    assert m < f32(0.5)
    lower = (interval > 0) & (zrel < m)
    upper = (interval >= 0) & (interval < N_INTERVALS - 1) & (zrel >= f32(f32(1.0) - m)) & ~lower
    nb[lower] = interval[lower] - 1
    z2[lower] = (zrel[lower] + f32(1.0)).astype(np.float32)
    nb[upper] = interval[upper] + 1
    z2[upper] = (zrel[upper] - f32(1.0)).astype(np.float32)
    return nb, z2


def histogram(feat, event_offsets, fc_w, fc_b, boundary_margin_mm=0.0):
    """feat float32 [9, T] SoA, event_offsets int [E+1] -> (H float64 [E,40,8,100], flags uint32 [E]).

    H[e,i,c,l] = sum over in-range tracks t of event e with interval(t) = i, in ascending track
    index, of fc(x_t)[c*100 + l]; empty intervals are exactly 0.  With boundary_margin_mm > 0 (NEXT-1)
    boundary tracks add a second contribution to the neighbouring interval (boundary_neighbours).
    """
    feat = np.asarray(feat, np.float32)
    off = np.asarray(event_offsets, np.int64)
    E = off.shape[0] - 1
    interval, zrel, nonfinite = assign_intervals(feat[0])
    nb, zrel2 = boundary_neighbours(interval, zrel, boundary_margin_mm)
    x = feat.astype(np.float64).T.copy()           # [T, 9]
    x[:, 0] = zrel.astype(np.float64)
    H = np.zeros((E, N_INTERVALS, FC_CHANNELS, N_BINS), np.float64)
    flags = np.zeros(E, np.uint32)
    for e in range(E):
        lo, hi = int(off[e]), int(off[e + 1])
        if hi == lo:
            continue
        iv = interval[lo:hi]
        if np.any(iv < 0):
            flags[e] |= FLAG_TRACK_DROPPED
        if np.any(nonfinite[lo:hi]):
            flags[e] |= FLAG_NONFINITE
        keep = np.nonzero(iv >= 0)[0]
        if keep.size == 0:
            continue
        contrib = fc_forward(x[lo:hi][keep], fc_w, fc_b)       # [n, 800]
        for n, t in enumerate(keep):                            # ascending original index
            H[e, iv[t]] += contrib[n].reshape(FC_CHANNELS, N_BINS)
        extra = np.nonzero(nb[lo:hi] >= 0)[0]                   # NEXT-1: second contribution of boundary tracks
        if extra.size:
            x2 = x[lo:hi][extra].copy()
            x2[:, 0] = zrel2[lo:hi][extra].astype(np.float64)
            contrib2 = fc_forward(x2, fc_w, fc_b)
            for n, t in enumerate(extra):
                H[e, nb[lo + t]] += contrib2[n].reshape(FC_CHANNELS, N_BINS)
    return H, flags


# ----------------------------------------------------------------------------------------------
# O5 UNet -- PAPER.md:29 "5-layer UNet architecture (64 channels deployed)"; topology and kernel
# sizes from BASELINE.json config 0.
# ----------------------------------------------------------------------------------------------
def conv1d_same(x, W, b, operand_round=None):
    """Cross-correlation with zero "same" padding p = (k-1)/2 (k odd):
        y[n,co,l] = b[co] + sum_ci sum_j W[co,ci,j] * x[n,ci,l+j-p],   x = 0 outside [0,L).
    x [N,Cin,L], W [Cout,Cin,K], b [Cout] -> [N,Cout,L], float64.  One library matmul per tap j.
    ``operand_round`` (tolerance studies only, never parity): callable applied to both operands.
    """
    x = np.asarray(x, np.float64)
    W = np.asarray(W, np.float64)
    N, Cin, L = x.shape
    Cout, Cin2, K = W.shape
    assert Cin == Cin2 and K % 2 == 1
    if operand_round is not None:
        x = operand_round(x)
        W = operand_round(W)
    p = (K - 1) // 2
    xp = np.zeros((N, Cin, L + 2 * p), np.float64)
    xp[:, :, p:p + L] = x
    y = np.empty((N, Cout, L), np.float64)
    y[:] = np.asarray(b, np.float64)[None, :, None]
    for j in range(K):
        y += np.einsum("oc,ncl->nol", W[:, :, j], xp[:, :, j:j + L], optimize=True)
    return y


def maxpool2(x):
    """y[l] = max(x[2l], x[2l+1]); lengths 100 -> 50 -> 25 leave no remainder."""
    assert x.shape[-1] % 2 == 0
    return np.maximum(x[..., 0::2], x[..., 1::2])


def upsample2_nearest(x):
    """y[l] = x[l // 2]."""
    return np.repeat(x, 2, axis=-1)


def unet_logits(H, conv_w, conv_b, operand_round=None):
    """H float64 [N,8,100] (N independent intervals, zero padded at interval edges: PAPER.md:49
    B = 40 batch items) -> logits float64 [N,100].
    [READING] concat order [upsampled, skip]; skips are the pre-pool activations; LeakyReLU(0.01)
    after each of the five k>1 convs; the 1x1 head has no activation before the sigmoid.
    ``operand_round``: None, or dict layer name -> callable (tolerance studies only).
    """
    rnd = (lambda name: None) if operand_round is None else (lambda name: operand_round.get(name))
    e1 = leaky_relu(conv1d_same(H, conv_w[0], conv_b[0], rnd("e1")))
    e2 = leaky_relu(conv1d_same(maxpool2(e1), conv_w[1], conv_b[1], rnd("e2")))
    bt = leaky_relu(conv1d_same(maxpool2(e2), conv_w[2], conv_b[2], rnd("b")))
    d2 = leaky_relu(conv1d_same(np.concatenate([upsample2_nearest(bt), e2], axis=1),
                                conv_w[3], conv_b[3], rnd("d2")))
    d1 = leaky_relu(conv1d_same(np.concatenate([upsample2_nearest(d2), e1], axis=1),
                                conv_w[4], conv_b[4], rnd("d1")))
    logit = conv1d_same(d1, conv_w[5], conv_b[5], rnd("head"))
    return logit[:, 0, :]


def unet_probs(H, conv_w, conv_b, operand_round=None):
    """O6: P[e, 100*i + l] = float32(sigmoid(logit)).  H [E,40,8,100] -> float32 [E,4000]."""
    E = H.shape[0]
    Hn = np.asarray(H, np.float64).reshape(E * N_INTERVALS, FC_CHANNELS, N_BINS)
    p = sigmoid(unet_logits(Hn, conv_w, conv_b, operand_round))
    return p.reshape(E, N_GLOBAL_BINS).astype(np.float32)


# ----------------------------------------------------------------------------------------------
# O7 peak finder in float32 -- PAPER.md:31 "local maximum detection with learned thresholds";
# BASELINE.json config 0: local max over the 4000 concatenated bins with prob > 0.01, weighted
# centroid over +-3 bins, at most 32 peaks.   [READING] strict-left / non-strict-right maximum,
# first 32 in ascending bin, the exact float32 operation sequence below (no FMA).
# ----------------------------------------------------------------------------------------------
def find_peaks_event(P):
    """P float32 [4000] -> (z float32 [32], prob float32 [32], bin int32 [32], count, n_found)."""
    P = np.asarray(P, np.float32)
    G = P.shape[0]
    f32 = np.float32
    ninf = f32(-np.inf)
    left = np.concatenate([[ninf], P[:-1]]).astype(np.float32)
    right = np.concatenate([P[1:], [ninf]]).astype(np.float32)
    with np.errstate(invalid="ignore"):
        is_peak = (P > PEAK_THRESHOLD) & (P > left) & (P >= right)   # NaN compares false: never a peak
    cand = np.nonzero(is_peak)[0]
    z = np.zeros(MAX_PEAKS, np.float32)
    pr = np.zeros(MAX_PEAKS, np.float32)
    bn = np.full(MAX_PEAKS, -1, np.int32)
    count = min(cand.size, MAX_PEAKS)
    for n in range(count):
        g = int(cand[n])
        lo = max(g - PEAK_HALFWIDTH, 0)
        hi = min(g + PEAK_HALFWIDTH, G - 1)
        s0 = f32(0.0)
        s1 = f32(0.0)
        for j in range(lo, hi + 1):
            s0 = f32(s0 + P[j])
            prod = f32(P[j] * f32(j - g))
            s1 = f32(s1 + prod)
        with np.errstate(invalid="ignore", divide="ignore"):
            delta = f32(s1 / s0)
        t = f32(f32(f32(g) + f32(0.5)) + delta)
        zz = f32(t * f32(0.1))
        zz = f32(zz + f32(-200.0))
        z[n], pr[n], bn[n] = zz, P[g], g
    return z, pr, bn, count, int(cand.size)


def find_peaks(P):
    """P float32 [E,4000] -> dict(z [E,32], prob [E,32], bin [E,32], count [E], flags [E])."""
    P = np.asarray(P, np.float32)
    E = P.shape[0]
    out = dict(z=np.zeros((E, MAX_PEAKS), np.float32), prob=np.zeros((E, MAX_PEAKS), np.float32),
               bin=np.full((E, MAX_PEAKS), -1, np.int32), count=np.zeros(E, np.int32),
               flags=np.zeros(E, np.uint32))
    for e in range(E):
        z, pr, bn, c, n = find_peaks_event(P[e])
        out["z"][e], out["prob"][e], out["bin"][e], out["count"][e] = z, pr, bn, c
        if n > MAX_PEAKS:
            out["flags"][e] |= FLAG_PEAK_OVERFLOW
    return out


# ----------------------------------------------------------------------------------------------
# whole path (call stack of PAPER.md:27-31): tracks -> FC -> histogram -> UNet -> sigmoid -> peaks
# ----------------------------------------------------------------------------------------------
def run(feat, event_offsets, weights, chunk_events=16, want_hist=False, operand_round=None,
        boundary_margin_mm=0.0):
    """Returns dict(probs float32 [E,4000], peaks dict, flags uint32 [E][, hist float64 [E,40,8,100]]).
    Events are processed in chunks only to bound memory; each event's result depends on its own
    tracks alone."""
    feat = np.asarray(feat, np.float32)
    off = np.asarray(event_offsets, np.int64)
    E = off.shape[0] - 1
    probs = np.zeros((E, N_GLOBAL_BINS), np.float32)
    flags = np.zeros(E, np.uint32)
    hist = np.zeros((E, N_INTERVALS, FC_CHANNELS, N_BINS), np.float64) if want_hist else None
    for lo in range(0, E, chunk_events):
        hi = min(lo + chunk_events, E)
        sub_off = off[lo:hi + 1] - off[lo]
        H, fl = histogram(feat[:, off[lo]:off[hi]], sub_off, weights.fc_w, weights.fc_b, boundary_margin_mm)
        probs[lo:hi] = unet_probs(H, weights.conv_w, weights.conv_b, operand_round)
        flags[lo:hi] = fl
        if want_hist:
            hist[lo:hi] = H
    peaks = find_peaks(probs)
    flags |= peaks["flags"]
    out = dict(probs=probs, peaks=peaks, flags=flags)
    if want_hist:
        out["hist"] = hist
    return out


# ----------------------------------------------------------------------------------------------
# O8 peak agreement bookkeeping (criterion of BASELINE.json north_star: positions within 1 bin on
# >= 99.9 % of oracle peaks).  Pure comparison logic, used by tests and bench reports.
# ----------------------------------------------------------------------------------------------
def match_peaks(bins_ref, bins_test, tol=1):
    """Greedy one-to-one match in ascending bin.  Returns (#ref matched, #ref, #test unmatched)."""
    ref = [int(b) for b in bins_ref if b >= 0]
    tst = [int(b) for b in bins_test if b >= 0]
    used = [False] * len(tst)
    matched = 0
    k0 = 0
    for g in ref:
        while k0 < len(tst) and tst[k0] < g - tol:
            k0 += 1
        k = k0
        while k < len(tst) and tst[k] <= g + tol:
            if not used[k]:
                used[k] = True
                matched += 1
                break
            k += 1
    return matched, len(ref), used.count(False)


def tau_stable_peaks(P, bins, tau):
    """Oracle peaks that ANY implementation within max|dP| <= tau must reproduce within +-1 bin
    (DESIGN.md "tau-stable peaks"): P[g] > 0.01 + tau and P[g] - max(P[g-2], P[g+2]) > 2 tau."""
    P = np.asarray(P, np.float64)
    G = P.shape[0]
    keep = []
    for g in bins:
        g = int(g)
        if g < 0:
            continue
        l2 = P[g - 2] if g - 2 >= 0 else -np.inf
        r2 = P[g + 2] if g + 2 < G else -np.inf
        if P[g] > float(PEAK_THRESHOLD) + tau and P[g] - max(l2, r2) > 2.0 * tau:
            keep.append(g)
    return keep
