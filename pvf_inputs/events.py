"""Seeded synthetic LHCb-Run-3-shaped events (stand-in for the paper's simulated events).

The paper's workload is "5.6 primary vertices per bunch crossing on average"
 with nine features per VELO track.  Its simulated
samples are not available; BASELINE.json configs 0-4 define the synthetic stand-ins
generated here.  Nothing of the method is computed in this file.

Track features, Structure-of-Arrays, float32, millimetres:
    feat[0] = z_poca, feat[1] = x_poca, feat[2] = y_poca, feat[3..8] = e0..e5
``event_offsets`` is int32 [n_events+1], ascending, offsets[0] = 0.
"""
from __future__ import annotations

from dataclasses import dataclass
import numpy as np

Z_MIN_MM = -200.0
Z_MAX_MM = 200.0

# name -> (mean PVs, PV z sigma [mm], fixed PV count / tracks or None, fake fraction)
CONFIG_EVENT_MODELS = {
    # BASELINE.json config 0: 1 PV at z~N(0,50) clipped to the region, exactly 40 tracks, no fakes
    "single": dict(mean_pv=None, z_sigma=50.0, fixed_tracks=40, fake_frac=0.0),
    # config 1/2/4: PVs ~ Poisson(5.6) min 1; tracks/PV ~ Poisson(30); +10 % fakes uniform in z
    "run3": dict(mean_pv=5.6, z_sigma=50.0, fixed_tracks=None, fake_frac=0.1),
    # config 3: PVs ~ Poisson(10), z ~ N(0,30), tracks/PV ~ Poisson(30); fakes as run3 (DESIGN.md reading)
    "pileup": dict(mean_pv=10.0, z_sigma=30.0, fixed_tracks=None, fake_frac=0.1),
}


@dataclass
class EventBatch:
    feat: np.ndarray           # float32 [9, n_tracks]  (SoA: row k is feature k)
    event_offsets: np.ndarray  # int32 [n_events + 1]
    pv_z: list                 # per event: float64 array of generated PV z (truth, for reports only)

    @property
    def n_events(self) -> int:
        return int(self.event_offsets.shape[0] - 1)

    @property
    def n_tracks(self) -> int:
        return int(self.event_offsets[-1])


def make_events(model: str, n_events: int, seed: int) -> EventBatch:
    """Draw ``n_events`` events of the named model with numpy ``default_rng(seed)``."""
    m = CONFIG_EVENT_MODELS[model]
    rng = np.random.default_rng(seed)
    E = int(n_events)
    if E == 0:
        return EventBatch(np.zeros((9, 0), np.float32), np.zeros(1, np.int32), [])

    if m["fixed_tracks"] is not None:
        n_pv = np.ones(E, np.int64)
    else:
        n_pv = np.maximum(rng.poisson(m["mean_pv"], size=E), 1).astype(np.int64)
    n_pv_tot = int(n_pv.sum())
    pv_event = np.repeat(np.arange(E), n_pv)
    pv_z = rng.normal(0.0, m["z_sigma"], size=n_pv_tot)
    # "clipped to the region": keep PVs inside [-200, 200)
    pv_z = np.clip(pv_z, Z_MIN_MM, np.nextafter(Z_MAX_MM, 0.0))
    if m["fixed_tracks"] is not None:
        trk_per_pv = np.full(n_pv_tot, m["fixed_tracks"], np.int64)
    else:
        trk_per_pv = rng.poisson(30.0, size=n_pv_tot).astype(np.int64)

    n_real_ev = np.bincount(pv_event, weights=trk_per_pv, minlength=E).astype(np.int64)
    n_fake_ev = np.rint(m["fake_frac"] * n_real_ev).astype(np.int64)
    n_real = int(n_real_ev.sum())
    n_fake = int(n_fake_ev.sum())

    z_real = np.repeat(pv_z, trk_per_pv) + rng.normal(0.0, 0.1, size=n_real)
    ev_real = np.repeat(pv_event, trk_per_pv)
    z_fake = rng.uniform(Z_MIN_MM, Z_MAX_MM, size=n_fake)
    ev_fake = np.repeat(np.arange(E), n_fake_ev)

    z = np.concatenate([z_real, z_fake])
    ev = np.concatenate([ev_real, ev_fake])
    T = z.shape[0]
    x = rng.normal(0.0, 0.05, size=T)
    y = rng.normal(0.0, 0.05, size=T)
    ell = rng.lognormal(mean=-2.0, sigma=0.5, size=(6, T))

    # shuffle within each event: sort by (event, random key)
    key = rng.random(T)
    order = np.lexsort((key, ev))
    feat = np.empty((9, T), np.float32)
    feat[0] = z[order]
    feat[1] = x[order]
    feat[2] = y[order]
    feat[3:9] = ell[:, order]

    counts = np.bincount(ev, minlength=E)
    offsets = np.zeros(E + 1, np.int64)
    np.cumsum(counts, out=offsets[1:])
    assert offsets[-1] < 2**31
    pv_off = np.zeros(E + 1, np.int64)
    np.cumsum(n_pv, out=pv_off[1:])
    pv_list = [pv_z[pv_off[e]:pv_off[e + 1]].copy() for e in range(E)]
    return EventBatch(np.ascontiguousarray(feat), offsets.astype(np.int32), pv_list)


def select_events(batch: EventBatch, idx) -> EventBatch:
    """Sub-batch holding the events ``idx`` (in that order); used for oracle samples."""
    idx = np.asarray(idx, np.int64)
    off = batch.event_offsets.astype(np.int64)
    counts = off[idx + 1] - off[idx]
    new_off = np.zeros(idx.shape[0] + 1, np.int64)
    np.cumsum(counts, out=new_off[1:])
    cols = np.concatenate([np.arange(off[i], off[i + 1]) for i in idx]) if idx.size else np.zeros(0, np.int64)
    feat = np.ascontiguousarray(batch.feat[:, cols])
    return EventBatch(feat, new_off.astype(np.int32), [batch.pv_z[i] for i in idx])


def shard_events(n_events: int, world_size: int, rank: int) -> tuple[int, int]:
    """Contiguous event range [lo, hi) owned by ``rank`` (events are independent: PAPER.md:27, 37).

    Pure bookkeeping for the "replicas only" multi-GPU mode: no collective.
    """
    base, rem = divmod(int(n_events), int(world_size))
    lo = rank * base + min(rank, rem)
    hi = lo + base + (1 if rank < rem else 0)
    return lo, hi
